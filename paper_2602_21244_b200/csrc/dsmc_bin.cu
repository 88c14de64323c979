// dsmc_bin: stable counting sort of particles by cell index ("particles are sorted by
// cell index so that particles in the same cell are contiguous in memory").
//
//   k_hist     histogram of cell ids (+ range check)            4 B read / particle
//   k_scan     exclusive scan -> cell_start, scatter cursors    O(n_cells)
//   k_scatter  claim a slot in the particle's cell              4 B read + 4 B write
//   k_fixup    order each cell's ids ascending in shared memory 4 B read + 4 B write
//              (makes the result the unique stable sort, whatever order the slots were claimed in)
//   k_gather   velocities into sorted order                     4+12 B read + 12 B write
#include <algorithm>

#include "dsmc_device.cuh"
#include "dsmc_internal.h"

namespace dsmc {

__global__ void k_hist(int64_t n, int32_t K, const int32_t *__restrict__ cell, int32_t *__restrict__ counts,
                       int32_t *__restrict__ status) {
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
    int32_t c = __ldg(cell + p);
    if (c < 0 || c >= K) {
      *status = DSMC_ERR_BAD_CELL_INDEX;
    } else {
      atomicAdd(counts + c, 1);
    }
  }
}

// single CTA, 1024 threads: counts[K] -> cell_start[K+1] (exclusive), cursor[k] = cell_start[k]
__global__ void __launch_bounds__(1024) k_scan(int32_t K, int32_t *__restrict__ counts,
                                               int32_t *__restrict__ cell_start) {
  __shared__ int wsum[32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int per = (K + 1023) / 1024;
  const int lo = min(tid * per, K), hi = min(lo + per, K);
  int sum = 0;
  for (int i = lo; i < hi; ++i) sum += counts[i];
  int inc = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int w = wsum[lane], winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += t;
    }
    wsum[lane] = winc - w;
  }
  __syncthreads();
  int run = wsum[warp] + inc - sum;
  for (int i = lo; i < hi; ++i) {
    int t = counts[i];
    counts[i] = run;  // becomes the scatter cursor
    cell_start[i] = run;
    run += t;
  }
  if (tid == 1023) cell_start[K] = run;
}

__global__ void k_scatter(int64_t n, int32_t K, const int32_t *__restrict__ cell, int32_t *__restrict__ cursor,
                          int32_t *__restrict__ perm) {
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
    int32_t c = __ldg(cell + p);
    if (c >= 0 && c < K) perm[atomicAdd(cursor + c, 1)] = (int32_t)p;
  }
}

// One CTA per chunk of cells (cells whose first slot lies in [b*kChunk, (b+1)*kChunk)); one warp
// per cell sorts the cell's original ids ascending with an all-ascending bitonic network
// (partners i ^ (k-1) then i ^ j), which needs no padding for non-power-of-two sizes.
__global__ void __launch_bounds__(kThreads) k_fixup(int64_t n, int32_t K, const int32_t *__restrict__ cs,
                                                   int32_t *__restrict__ perm, int32_t *__restrict__ status) {
  __shared__ int32_t ids[kNlocMax];
  __shared__ int s_c[2];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t p_lo = (int64_t)blockIdx.x * kChunk, p_hi = min(n, p_lo + kChunk);
  if (tid == 0) {
    s_c[0] = lower_bound_cells(cs, K, p_lo);
    s_c[1] = lower_bound_cells(cs, K, p_hi);
  }
  __syncthreads();
  const int c_lo = s_c[0], c_hi = s_c[1];
  if (c_lo >= c_hi) return;
  const int q0 = cs[c_lo], q1 = cs[c_hi];
  const int n_loc = q1 - q0;
  if (n_loc > kNlocMax) {
    if (tid == 0) *status = DSMC_ERR_CELL_TOO_LARGE;
    return;
  }
  for (int q = tid; q < n_loc; q += kThreads) ids[q] = perm[q0 + q];
  __syncthreads();
  for (int c = c_lo + warp; c < c_hi; c += kThreads / 32) {
    const int a = cs[c] - q0, N = cs[c + 1] - cs[c];
    if (N < 2) continue;
    int32_t *x = ids + a;
    for (int k = 2; (k >> 1) < N; k <<= 1) {
      for (int i = lane; i < N; i += 32) {  // first sub-step of the merge: partner i ^ (k-1)
        int l = i ^ (k - 1);
        if (l > i && l < N) {
          int32_t u = x[i], v = x[l];
          if (u > v) { x[i] = v; x[l] = u; }
        }
      }
      __syncwarp();
      for (int j = k >> 2; j > 0; j >>= 1) {
        for (int i = lane; i < N; i += 32) {
          int l = i ^ j;
          if (l > i && l < N) {
            int32_t u = x[i], v = x[l];
            if (u > v) { x[i] = v; x[l] = u; }
          }
        }
        __syncwarp();
      }
    }
  }
  __syncthreads();
  for (int q = tid; q < n_loc; q += kThreads) perm[q0 + q] = ids[q];
}

__global__ void k_gather(int64_t n, const int32_t *__restrict__ perm, const float *__restrict__ vx,
                         const float *__restrict__ vy, const float *__restrict__ vz, float *__restrict__ vx_s,
                         float *__restrict__ vy_s, float *__restrict__ vz_s) {
  for (int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; s < n; s += (int64_t)gridDim.x * blockDim.x) {
    int32_t p = perm[s];
    if ((uint64_t)p >= (uint64_t)n) continue;  // only after a bad cell index (outputs unspecified)
    vx_s[s] = __ldg(vx + p);
    vy_s[s] = __ldg(vy + p);
    vz_s[s] = __ldg(vz + p);
  }
}

int launch_bin(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cell, const float *vx, const float *vy,
               const float *vz, float *vx_s, float *vy_s, float *vz_s, int32_t *perm, int32_t *cell_start) {
  cudaStream_t s = c->stream;
  if (cudaMemsetAsync(c->d_cursor, 0, sizeof(int32_t) * (size_t)(K + 1), s) != cudaSuccess) return DSMC_ERR_CUDA;
  if (n == 0) {
    return cudaMemsetAsync(cell_start, 0, sizeof(int32_t) * (size_t)(K + 1), s) == cudaSuccess ? DSMC_OK
                                                                                                : DSMC_ERR_CUDA;
  }
  const int grid = (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->num_sms * 16);
  k_hist<<<grid, 256, 0, s>>>(n, K, cell, c->d_cursor, c->d_status);
  k_scan<<<1, 1024, 0, s>>>(K, c->d_cursor, cell_start);
  k_scatter<<<grid, 256, 0, s>>>(n, K, cell, c->d_cursor, perm);
  const int chunks = (int)((n + kChunk - 1) / kChunk);
  k_fixup<<<chunks, kThreads, 0, s>>>(n, K, cell_start, perm, c->d_status);
  k_gather<<<grid, 256, 0, s>>>(n, perm, vx, vy, vz, vx_s, vy_s, vz_s);
  c->launches += 5;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

}  // namespace dsmc
