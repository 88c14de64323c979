// The minimal DSMC loop around the collision step: free flight + Maxwell walls for the
// 1-D Couette layout (Q30), the gather of a per-particle array into sorted order, and the
// per-cell sampling sums behind the macroscopic fields.  Written from the paper / Q30, independent of
// oracle/.  All three are streaming kernels: coalesced loads, FP32 arithmetic (the sampling sums in FP64), grid =
// a multiple of the SM count.
//
//   k_move_couette   8 B read + 8 B written per particle (x, vx -> x, cell); vy, vz are touched only by the
//                    particles a wall re-emits.  Random numbers: Philox stream 5, counter (particle, bounce, step, 5).
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

__global__ void __launch_bounds__(256) k_move_couette(int64_t n, float *__restrict__ x, float *__restrict__ vx,
                                                     float *__restrict__ vy, float *__restrict__ vz,
                                                     int32_t *__restrict__ cell, int32_t *__restrict__ bounces,
                                                     MoveParams P) {
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
    float xx = x[p], v = vx[p], t_left = P.dt;
    float ny = 0.f, nz = 0.f;
    bool emitted = false;
    int nb = 0;
    for (;;) {
      const float xn = fmaf(v, t_left, xx);
      if (xn >= 0.f && xn <= P.L) {
        xx = xn;
        break;
      }
      if (nb == DSMC_MAX_BOUNCES) {  // give up: park the particle on the wall it was heading for
        xx = xn < 0.f ? 0.f : P.L;
        break;
      }
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
    x[p] = xx;
    cell[p] = max(0, min(P.n_cells - 1, (int)floorf(xx * P.cells_per_len)));
    if (nb) vx[p] = v;
    if (emitted) {
      vy[p] = ny;
      vz[p] = nz;
    }
    if (bounces) bounces[p] = nb;
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
  for (int64_t k = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5); k < K; k += (int64_t)gridDim.x * wpb) {
    const int a = __ldg(cs + k), b = __ldg(cs + k + 1);
    double s[7] = {0, 0, 0, 0, 0, 0, 0};
    for (int p = a + lane; p < b; p += 32) {
      const double X = vx[p], Y = vy[p], Z = vz[p];
      s[0] += X; s[1] += Y; s[2] += Z;
      s[3] += X * X; s[4] += Y * Y; s[5] += Z * Z;
      s[6] += X * Y;
    }
#pragma unroll
    for (int u = 0; u < 7; ++u) s[u] = warp_sum(s[u]);
    if (lane == 0) {
      double *o = acc + 8 * k;
      o[0] += (double)(b - a);
#pragma unroll
      for (int u = 0; u < 7; ++u) o[1 + u] += s[u];
    }
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
  const int grid = (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->num_sms * 16);
  k_move_couette<<<grid, 256, 0, c->stream>>>(n, x, vx, vy, vz, cell, bounces, P);
  c->launches += 1;
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
  const int grid = (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->num_sms * 16);
  k_gather_f32<<<grid, 256, 0, c->stream>>>(n, perm, src, dst);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_sample_cells(dsmc_ctx *c, int32_t K, const int32_t *cs, const float *vx, const float *vy, const float *vz,
                        double *acc) {
  const int grid = (int)std::min<int64_t>(((int64_t)K + 7) / 8, (int64_t)c->num_sms * 8);
  k_sample_cells<<<grid, 256, 0, c->stream>>>(K, cs, vx, vy, vz, acc);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

}  // namespace dsmc
