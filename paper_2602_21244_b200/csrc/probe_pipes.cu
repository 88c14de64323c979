// Pipe-throughput probe (not part of libdsmc_b200.so): MUFU.TANH / EX2 and tcgen05.ld / st per SM.
// Build + run: nvcc -gencode arch=compute_100a,code=sm_100a -O2 -o /tmp/probe_pipes paper_2602_21244_b200/csrc/probe_pipes.cu && /tmp/probe_pipes
// Its numbers (profiles/r01_pipe_probe.md) are the XU and TMEM-read ceilings quoted in DESIGN.md section 5.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1);} } while (0)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int OP>
__global__ void k_mufu(float *out, int iters) {
  float a[8];
  for (int j = 0; j < 8; ++j) a[j] = threadIdx.x * 0.001f + j;
  long long t0 = clock64();
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      if (OP == 0) asm volatile("tanh.approx.f32 %0, %0;" : "+f"(a[j]));
      else if (OP == 1) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[j]));
      else asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(a[j]));
    }
  }
  long long t1 = clock64();
  float s = 0; for (int j = 0; j < 8; ++j) s += a[j];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) out[0] = (float)(t1 - t0);
}

template <int MODE>  // 0 = ld x32, 1 = st x16, 2 = ld x32 + 32 tanh
__global__ void k_tmem(float *out, int iters) {
  __shared__ uint32_t slot;
  const int warp = threadIdx.x >> 5;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&slot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t base = slot + (((uint32_t)((warp & 3) * 32)) << 16) + (warp >> 2) * 32;
  uint32_t v[32];
  for (int j = 0; j < 32; ++j) v[j] = j;
  float acc = 0;
  __syncthreads();
  long long t0 = clock64();
  for (int i = 0; i < iters; ++i) {
    if (MODE == 0 || MODE == 2) {
      asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31]) : "r"(base));
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      if (MODE == 2) {
#pragma unroll
        for (int j = 0; j < 32; ++j) { float f = __uint_as_float(v[j]); asm volatile("tanh.approx.f32 %0, %0;" : "+f"(f)); acc += f; }
      } else acc += __uint_as_float(v[i & 31]);
    } else {
      asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(base),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
  }
  long long t1 = clock64();
  __syncthreads();
  out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
  if (threadIdx.x == 0) out[0] = (float)(t1 - t0);
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(slot) : "memory");
}

int main() {
  float *d; CK(cudaMalloc(&d, 1 << 20)); float h;
  const int it = 2000;
  for (int op = 0; op < 3; ++op) for (int nt : {128, 256, 512, 1024}) {
    if (op == 0) k_mufu<0><<<1, nt>>>(d, it); else if (op == 1) k_mufu<1><<<1, nt>>>(d, it); else k_mufu<2><<<1, nt>>>(d, it);
    CK(cudaDeviceSynchronize()); CK(cudaMemcpy(&h, d, 4, cudaMemcpyDeviceToHost));
    printf("mufu op%d threads %4d: %.2f ops/clk/SM\n", op, nt, (double)nt * it * 8 / h);
  }
  for (int mode = 0; mode < 3; ++mode) for (int nt : {128, 256, 512}) {
    if (mode == 0) k_tmem<0><<<1, nt>>>(d, it); else if (mode == 1) k_tmem<1><<<1, nt>>>(d, it); else k_tmem<2><<<1, nt>>>(d, it);
    CK(cudaDeviceSynchronize()); CK(cudaMemcpy(&h, d, 4, cudaMemcpyDeviceToHost));
    double bytes = (double)nt * it * (mode == 1 ? 64 : 128);
    printf("tmem mode%d threads %4d: %.1f B/clk/SM  (%.1f cyc/iter)\n", mode, nt, bytes / h, h / it);
  }
  return 0;
}
