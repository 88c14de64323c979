// Device-side helpers of the CUDA path: Philox4x32-10, uniforms, Box-Muller, warp/block scans.
// Written for sm_100a; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dsmc {

// Philox4x32-10 (Salmon et al. SC'11): counter (c0..c3), key (k0,k1).
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                               uint32_t k1) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
    uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return make_uint4(c0, c1, c2, c3);
}

// 23-bit uniform + half step: in (0,1), exactly representable in fp32
__device__ __forceinline__ float u01(uint32_t x) { return ((float)(x >> 9) + 0.5f) * (1.0f / 8388608.0f); }

__device__ __forceinline__ uint32_t word_of(const uint4 &r, uint32_t w) {
  return w == 0 ? r.x : (w == 1 ? r.y : (w == 2 ? r.z : r.w));
}

// xi ~ N(0, I3) from one Philox block (stream 2), full-precision logf / sincospif
__device__ __forceinline__ void box_muller3(const uint4 &r, float &x0, float &x1, float &x2) {
  float rad0 = sqrtf(-2.0f * logf(u01(r.x)));
  float rad1 = sqrtf(-2.0f * logf(u01(r.z)));
  float s0, c0, s1, c1;
  sincospif(2.0f * u01(r.y), &s0, &c0);
  sincospif(2.0f * u01(r.w), &s1, &c1);
  x0 = rad0 * c0;
  x1 = rad0 * s0;
  x2 = rad1 * c1;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// In-place exclusive scan of a[0..L) in shared memory by the whole CTA (blockDim.x threads,
// multiple of 32, <= 1024).  `scratch` holds >= 33 ints.  Ends with __syncthreads().
__device__ __forceinline__ void block_excl_scan(int *a, int L, int *scratch) {
  const int nt = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int per = (L + nt - 1) / nt;
  const int lo = min(tid * per, L), hi = min(lo + per, L);
  int sum = 0;
  for (int i = lo; i < hi; ++i) sum += a[i];
  int inc = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) scratch[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int w = (lane < (nt >> 5)) ? scratch[lane] : 0;
    int winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += t;
    }
    scratch[lane] = winc - w;
  }
  __syncthreads();
  int run = scratch[warp] + inc - sum;
  for (int i = lo; i < hi; ++i) {
    int t = a[i];
    a[i] = run;
    run += t;
  }
  __syncthreads();
}

// first index c in [0, K] with cs[c] >= value (cs non-decreasing, cs[K] = n)
__device__ __forceinline__ int lower_bound_cells(const int32_t *__restrict__ cs, int K, int64_t value) {
  int lo = 0, hi = K;
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if ((int64_t)__ldg(cs + mid) < value) lo = mid + 1; else hi = mid;
  }
  return lo;
}

__device__ __forceinline__ float act_apply(int act, float z) {
  if (act == 0) return tanhf(z);
  if (act == 1) return fmaxf(z, 0.0f);
  return z / (1.0f + expf(-z));
}

}  // namespace dsmc
