// Device-side helpers of the CUDA path: Philox4x32-10, uniforms, Box-Muller, warp sums, activations.
// Written for sm_100a; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dsmc {

// Programmatic dependent launch (a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may start
// while its predecessor in the stream drains): pdl_wait() returns when the predecessor grid has completed and its
// writes are visible -- it must come before the first access to anything the predecessor touches; after
// pdl_launch_dependents() in every CTA the next kernel's CTAs may be scheduled as this grid's last wave frees SMs.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

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

__device__ __forceinline__ float act_apply(int act, float z) {
  if (act == 0) return tanhf(z);
  if (act == 1) return fmaxf(z, 0.0f);
  return z / (1.0f + expf(-z));
}

}  // namespace dsmc
