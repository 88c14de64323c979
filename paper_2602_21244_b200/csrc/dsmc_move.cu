// The minimal DSMC loop around the collision step: free flight + Maxwell walls for the
// 1-D Couette layout (Q30), the gather of a per-particle array into sorted order, and the
// per-cell sampling sums behind the macroscopic fields.  Written from the paper / Q30, independent of
// oracle/.  All three are streaming kernels: coalesced loads, FP32 arithmetic (the sampling sums in FP64), grid =
// a multiple of the SM count.
//
//   k_move_couette   8 B read + 8 B written per particle (x, vx -> x, cell), four particles per thread through
//                    16-byte accesses; vy, vz are touched only by the particles a wall re-emits.  Random numbers: Philox stream 5, counter (particle, bounce, step, 5).
//   k_gather_f32     dst[s] = src[perm[s]]
//   k_sample_cells   one warp per cell, FP64 sums, no atomics
#include <algorithm>

#include "dsmc_device.cuh"
#include "dsmc_internal.h"

namespace dsmc {

struct MoveParams {
  float L, dt, u_wall, rt_wall, srt_wall, accommodation, cells_per_len;
  int32_t n_cells;
  uint32_t seed_lo, seed_hi, step;
};

// one particle: free flight for dt with wall hits; returns the new position, updates v, reports re-emission
__device__ __forceinline__ float move_one(int64_t p, float xx, float &v, float &ny, float &nz, bool &emitted, int &nb,
                                          const MoveParams &P) {
  float t_left = P.dt;
  nb = 0;
  emitted = false;
  for (;;) {
    const float xn = fmaf(v, t_left, xx);
    if (xn >= 0.f && xn <= P.L) return xn;
    if (nb == DSMC_MAX_BOUNCES) return xn < 0.f ? 0.f : P.L;  // give up: park the particle on the wall ahead
    const bool upper = xn > P.L;
    const float wall = upper ? P.L : 0.f;
    t_left -= (wall - xx) / v;
    xx = wall;
    const uint4 r = philox4x32_10((uint32_t)p, (uint32_t)nb, P.step, 5u, P.seed_lo, P.seed_hi);
    if (u01(r.x) < P.accommodation) {  // diffuse re-emission from the wall Maxwellian (flux-weighted normal)
      const float vn = sqrtf(-2.0f * P.rt_wall * logf(u01(r.y)));
      const float rad = P.srt_wall * sqrtf(-2.0f * logf(u01(r.z)));
      float sn, cs;
      sincospif(2.0f * u01(r.w), &sn, &cs);
      v = upper ? -vn : vn;
      ny = fmaf(rad, cs, upper ? P.u_wall : -P.u_wall);
      nz = rad * sn;
      emitted = true;
    } else {
      v = -v;
    }
    ++nb;
  }
}

__device__ __forceinline__ int cell_of(float xx, const MoveParams &P) {
  return max(0, min(P.n_cells - 1, (int)floorf(xx * P.cells_per_len)));
}

// VEC: four consecutive particles per thread through 16-byte loads / stores of x, vx and cell (arrays 16-byte
// aligned); the scalar form serves unaligned arrays and the last n % 4 particles
template <bool VEC>
__global__ void __launch_bounds__(256) k_move_couette(int64_t first, int64_t n, float *__restrict__ x,
                                                     float *__restrict__ vx, float *__restrict__ vy,
                                                     float *__restrict__ vz, int32_t *__restrict__ cell,
                                                     int32_t *__restrict__ bounces, MoveParams P) {
  const int64_t units = VEC ? (n - first) / 4 : n - first;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < units; i += (int64_t)gridDim.x * blockDim.x) {
    if (VEC) {
      const int64_t p0 = first + 4 * i;
      float4 X = *reinterpret_cast<const float4 *>(x + p0);
      float4 V = *reinterpret_cast<const float4 *>(vx + p0);
      float *xs = reinterpret_cast<float *>(&X), *vs = reinterpret_cast<float *>(&V);
      int4 C;
      int *cc = reinterpret_cast<int *>(&C);
      bool any = false;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        float ny = 0.f, nz = 0.f;
        bool emitted;
        int nb;
        xs[u] = move_one(p0 + u, xs[u], vs[u], ny, nz, emitted, nb, P);
        cc[u] = cell_of(xs[u], P);
        any |= nb > 0;
        if (emitted) {
          vy[p0 + u] = ny;
          vz[p0 + u] = nz;
        }
        if (bounces) bounces[p0 + u] = nb;
      }
      *reinterpret_cast<float4 *>(x + p0) = X;
      *reinterpret_cast<int4 *>(cell + p0) = C;
      if (any) *reinterpret_cast<float4 *>(vx + p0) = V;
    } else {
      const int64_t p = first + i;
      float v = vx[p], ny = 0.f, nz = 0.f;
      bool emitted;
      int nb;
      const float xx = move_one(p, x[p], v, ny, nz, emitted, nb, P);
      x[p] = xx;
      cell[p] = cell_of(xx, P);
      if (nb) vx[p] = v;
      if (emitted) {
        vy[p] = ny;
        vz[p] = nz;
      }
      if (bounces) bounces[p] = nb;
    }
  }
}

__global__ void __launch_bounds__(256) k_gather_f32(int64_t n, const int32_t *__restrict__ perm,
                                                   const float *__restrict__ src, float *__restrict__ dst) {
  for (int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; s < n; s += (int64_t)gridDim.x * blockDim.x)
    dst[s] = __ldg(src + __ldg(perm + s));
}

__global__ void __launch_bounds__(256) k_sample_cells(int32_t K, const int32_t *__restrict__ cs,
                                                     const float *__restrict__ vx, const float *__restrict__ vy,
                                                     const float *__restrict__ vz, double *__restrict__ acc) {
  const int lane = threadIdx.x & 31;
  const int wpb = blockDim.x >> 5;
  const int64_t stride = (int64_t)gridDim.x * wpb;
  int64_t k = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5);
  if (k >= K) return;
  int a = __ldg(cs + k), b = __ldg(cs + k + 1);
  for (; k < K; k += stride) {
    // offsets of this warp's next cell: fetched now, used after the sums of this one
    const int64_t kn = k + stride;
    int an = 0, bn = 0;
    if (kn < K) {
      an = __ldg(cs + kn);
      bn = __ldg(cs + kn + 1);
    }
    double s[7] = {0, 0, 0, 0, 0, 0, 0};
    // eight rows of 32 particles per trip: 24 loads in flight per lane (the kernel is latency-bound otherwise)
    for (int p0 = a + lane; p0 < b; p0 += 256) {
      float X[8], Y[8], Z[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int p = p0 + 32 * u;
        const bool in = p < b;
        X[u] = in ? __ldg(vx + p) : 0.f;
        Y[u] = in ? __ldg(vy + p) : 0.f;
        Z[u] = in ? __ldg(vz + p) : 0.f;
      }
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const double x = X[u], y = Y[u], z = Z[u];
        s[0] += x; s[1] += y; s[2] += z;
        s[3] += x * x; s[4] += y * y; s[5] += z * z;
        s[6] += x * y;
      }
    }
#pragma unroll
    for (int u = 0; u < 7; ++u) s[u] = warp_sum(s[u]);
    // one warp owns a cell for the whole launch, so the read-modify-write needs no atomicity; lanes 0..7 each add
    // one of the eight numbers
    double mine = (double)(b - a);
#pragma unroll
    for (int u = 0; u < 7; ++u) mine = lane == u + 1 ? s[u] : mine;
    if (lane < 8) acc[8 * k + lane] += mine;
    a = an;
    b = bn;
  }
}

// f1: NTC candidate counts with carried remainder (Q31).  FP64, one thread per cell; the products are
// rounded one by one (no FMA contraction) so that the floor is taken of the same number on every machine.
__global__ void __launch_bounds__(256) k_ntc_counts(int32_t K, const int32_t *__restrict__ cs,
                                                   const float *__restrict__ cap, double coef,
                                                   double *__restrict__ remainder, int32_t *__restrict__ counts) {
  for (int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; k < K; k += (int64_t)gridDim.x * blockDim.x) {
    const int N = __ldg(cs + k + 1) - __ldg(cs + k);
    if (N < 2) {
      counts[k] = 0;
      continue;
    }
    double m = __dmul_rn(0.5, (double)N * (double)(N - 1));
    m = __dmul_rn(m, coef);
    m = __dmul_rn(m, (double)__ldg(cap + k));
    m = __dadd_rn(m, remainder[k]);
    const double f = floor(m);
    counts[k] = (int32_t)f;
    remainder[k] = __dsub_rn(m, f);
  }
}

// grid of a grid-stride kernel: every resident slot of the device, once (a second, partial wave costs a tail)
template <class Kern>
static int resident_grid(dsmc_ctx *c, Kern kern, int threads, int64_t blocks_of_work) {
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
  return (int)std::max<int64_t>(1, std::min<int64_t>(blocks_of_work, (int64_t)c->num_sms * per_sm));
}

int launch_ntc_counts(dsmc_ctx *c, int32_t K, const int32_t *cs, const float *cap, double coef, double *remainder,
                      int32_t *counts) {
  const int grid = (int)std::min<int64_t>(((int64_t)K + 255) / 256, (int64_t)c->num_sms * 8);
  k_ntc_counts<<<grid, 256, 0, c->stream>>>(K, cs, cap, coef, remainder, counts);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_move_couette(dsmc_ctx *c, int64_t n, float *x, float *vx, float *vy, float *vz, int32_t *cell,
                        int32_t *bounces, const dsmc_couette_params *g, uint64_t seed, uint32_t step) {
  MoveParams P;
  P.L = g->L;
  P.dt = g->dt;
  P.u_wall = g->u_wall;
  P.rt_wall = g->rt_wall;
  P.srt_wall = sqrtf(g->rt_wall);
  P.accommodation = g->accommodation;
  P.cells_per_len = (float)((double)g->n_cells / (double)g->L);
  P.n_cells = g->n_cells;
  P.seed_lo = (uint32_t)(seed & 0xFFFFFFFFu);
  P.seed_hi = (uint32_t)(seed >> 32);
  P.step = step;
  const bool aligned = ((reinterpret_cast<uintptr_t>(x) | reinterpret_cast<uintptr_t>(vx) |
                         reinterpret_cast<uintptr_t>(cell)) & 15) == 0;
  const int64_t n_vec = aligned ? (n & ~(int64_t)3) : 0;
  if (n_vec > 0) {
    const int grid = resident_grid(c, k_move_couette<true>, 256, (n_vec / 4 + 255) / 256);
    k_move_couette<true><<<grid, 256, 0, c->stream>>>(0, n_vec, x, vx, vy, vz, cell, bounces, P);
    c->launches += 1;
  }
  if (n_vec < n) {
    const int grid = resident_grid(c, k_move_couette<false>, 256, (n - n_vec + 255) / 256);
    k_move_couette<false><<<grid, 256, 0, c->stream>>>(n_vec, n, x, vx, vy, vz, cell, bounces, P);
    c->launches += 1;
  }
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

__global__ void __launch_bounds__(256) k_fill_f32(int64_t n, float *__restrict__ dst, float value) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    dst[i] = value;
}

int launch_fill_f32(dsmc_ctx *c, int64_t n, float *dst, float value) {
  const int grid = (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->num_sms * 8);
  k_fill_f32<<<grid, 256, 0, c->stream>>>(n, dst, value);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_gather_f32(dsmc_ctx *c, int64_t n, const int32_t *perm, const float *src, float *dst) {
  const int grid = resident_grid(c, k_gather_f32, 256, (n + 255) / 256);
  k_gather_f32<<<grid, 256, 0, c->stream>>>(n, perm, src, dst);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_sample_cells(dsmc_ctx *c, int32_t K, const int32_t *cs, const float *vx, const float *vy, const float *vz,
                        double *acc) {
  const int grid = resident_grid(c, k_sample_cells, 256, ((int64_t)K + 7) / 8);
  k_sample_cells<<<grid, 256, 0, c->stream>>>(K, cs, vx, vy, vz, acc);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

}  // namespace dsmc
