// dsmc_cell_moments / dsmc_moment_match: per-cell sums (eq. 10) and the stand-alone
// cell-wise correction (eqs. 10-11 P:L126-131 with the momentum part of P:L46; Q5).
// One warp owns one contiguous cell segment; fp32 loads, fp64 accumulation, warp shuffles,
// no global atomics.
#include <algorithm>

#include "dsmc_device.cuh"
#include "dsmc_internal.h"

namespace dsmc {

__global__ void __launch_bounds__(kThreads) k_cell_moments(int32_t K, const int32_t *__restrict__ cs,
                                                          const float *__restrict__ vx,
                                                          const float *__restrict__ vy,
                                                          const float *__restrict__ vz,
                                                          double *__restrict__ moments) {
  const int lane = threadIdx.x & 31;
  const int wpb = blockDim.x >> 5;
  for (int64_t k = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5); k < K; k += (int64_t)gridDim.x * wpb) {
    const int a = cs[k], b = cs[k + 1];
    double px = 0, py = 0, pz = 0, e = 0;
    for (int p = a + lane; p < b; p += 32) {
      double x = vx[p], y = vy[p], z = vz[p];
      px += x; py += y; pz += z;
      e += x * x + y * y + z * z;
    }
    px = warp_sum(px); py = warp_sum(py); pz = warp_sum(pz); e = warp_sum(e);
    if (lane == 0) {
      moments[4 * k + 0] = px;
      moments[4 * k + 1] = py;
      moments[4 * k + 2] = pz;
      moments[4 * k + 3] = e;
    }
  }
}

__global__ void __launch_bounds__(kThreads) k_moment_match(int32_t K, const int32_t *__restrict__ cs, float *vx,
                                                          float *vy, float *vz,
                                                          const double *__restrict__ target, uint32_t flags) {
  const int lane = threadIdx.x & 31;
  const int wpb = blockDim.x >> 5;
  for (int64_t k = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5); k < K; k += (int64_t)gridDim.x * wpb) {
    const int a = cs[k], b = cs[k + 1], N = b - a;
    if (N < 2) continue;  // Q11
    const double Et = target[4 * k + 3];
    if (flags & DSMC_F_MATCH_ENERGY_ONLY) {  // literal eq. 11
      double e = 0;
      for (int p = a + lane; p < b; p += 32) {
        double x = vx[p], y = vy[p], z = vz[p];
        e += x * x + y * y + z * z;
      }
      e = warp_sum(e);
      if (e > 0.0) {
        const double alpha = sqrt(Et / e);  // FP64: alpha = 1 + O(1e-7) is not resolvable in FP32
        for (int p = a + lane; p < b; p += 32) {
          vx[p] = (float)(alpha * vx[p]);
          vy[p] = (float)(alpha * vy[p]);
          vz[p] = (float)(alpha * vz[p]);
        }
      }
      continue;
    }
    const double utx = target[4 * k] / N, uty = target[4 * k + 1] / N, utz = target[4 * k + 2] / N;
    const double theta_t = Et - (double)N * (utx * utx + uty * uty + utz * utz);
    double px = 0, py = 0, pz = 0;
    for (int p = a + lane; p < b; p += 32) { px += vx[p]; py += vy[p]; pz += vz[p]; }
    const double upx = warp_sum(px) / N, upy = warp_sum(py) / N, upz = warp_sum(pz) / N;
    double th = 0;
    for (int p = a + lane; p < b; p += 32) {
      double x = vx[p] - upx, y = vy[p] - upy, z = vz[p] - upz;
      th += x * x + y * y + z * z;
    }
    th = warp_sum(th);
    const double alpha = (th > 0.0 && theta_t >= 0.0) ? sqrt(theta_t / th) : 1.0;
    for (int p = a + lane; p < b; p += 32) {
      vx[p] = (float)(utx + alpha * (vx[p] - upx));
      vy[p] = (float)(uty + alpha * (vy[p] - upy));
      vz[p] = (float)(utz + alpha * (vz[p] - upz));
    }
  }
}

int launch_cell_moments(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cs, const float *vx, const float *vy,
                        const float *vz, double *moments) {
  (void)n;
  const int wpb = kThreads / 32;
  const int grid = (int)std::min<int64_t>(((int64_t)K + wpb - 1) / wpb, (int64_t)c->num_sms * 32);
  k_cell_moments<<<grid, kThreads, 0, c->stream>>>(K, cs, vx, vy, vz, moments);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_moment_match(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cs, float *vx, float *vy, float *vz,
                        const double *target, uint32_t flags) {
  (void)n;
  const int wpb = kThreads / 32;
  const int grid = (int)std::min<int64_t>(((int64_t)K + wpb - 1) / wpb, (int64_t)c->num_sms * 32);
  k_moment_match<<<grid, kThreads, 0, c->stream>>>(K, cs, vx, vy, vz, target, flags);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

}  // namespace dsmc
