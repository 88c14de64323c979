// Warp-specialised, two-slot pipeline around the tcgen05 MLP tile (plain BF16 operands).
//
// The MLP tile is bound by the XU pipe (one MUFU.TANH per hidden activation, 16 / clk / SM), not by
// the tensor pipe, so the job of this pipeline is to keep the activation warps busy: two 128-pair
// tiles ("slots") are in flight per CTA and three kinds of warps never wait for one another at a
// CTA-wide barrier, only on the mbarrier of the data they need:
//
//   IO warps   (4)  features of a tile -> A1 rows in shared memory            -> in_ready[s]
//                   ... and, after layer 3, outputs of the tile from TMEM     <- full_o[s]
//   MMA warp   (1)  one elected lane issues the UMMAs of (slot, layer) when its operand is ready and
//                   commits them to full_e[s] (layers 1, 2) or full_o[s] (layer 3)
//   ACT warps (16)  D (TMEM, fp32) -> activation -> bf16 -> A operand (TMEM)   <- full_e[s], -> a_ready[s]
//
// While the ACT warps work on slot 0 the tensor core runs slot 1's layer and vice versa.
// Tensor memory per slot: D [0,H) | A [H, H + H/2) | bias columns 8 | layer-3 output 16 (see dsmc_tc.cuh).
// The layer-3 output has its own columns and the layer-1 operand is double-buffered per slot, so the
// next tile's layer 1 never waits for the IO warps to drain the previous tile.
#pragma once
#include "dsmc_internal.h"
#include "dsmc_tc.cuh"

namespace dsmc {

constexpr int kPipeActWarps = 16, kPipeIoWarps = 4;
constexpr int kPipeThreads = (kPipeActWarps + kPipeIoWarps + 1) * 32;  // 672

template <int H>
struct PipeShape {
  static constexpr int K1 = 32;
  static constexpr int W1_BYTES = H * K1 * 2, W2_BYTES = H * H * 2, B2_BYTES = H * 16 * 2, W3_BYTES = 16 * H * 2,
                       B3_BYTES = 16 * 16 * 2;
  static constexpr int OFF_W2 = W1_BYTES, OFF_B2 = OFF_W2 + W2_BYTES, OFF_W3 = OFF_B2 + B2_BYTES,
                       OFF_B3 = OFF_W3 + W3_BYTES;
  static constexpr int BLOB_BYTES = OFF_B3 + B3_BYTES;  // the plain-BF16 prefix of the packed image
  static constexpr int A1_BYTES = 128 * K1 * 2;
  static constexpr int SMEM_BYTES = BLOB_BYTES + 4 * A1_BYTES + 128;  // A1 double-buffered per slot
  static constexpr int COL_D = 0, COL_A = H, COL_BIAS = COL_A + H / 2, COL_OUT = COL_BIAS + 8;
  static constexpr int SLOT_COLS = (COL_OUT + 16) <= 128 ? 128 : 256;
  static constexpr int TMEM_COLS = 2 * SLOT_COLS;
};

// Output layer (d_out = 1) of a 3-layer MLP in FP32, passed to the kernel by value: its weights are then constant-bank
// operands of the FMAs that form z, no load and no latency.  With a single output the third layer is a dot product per
// row, which the activation warps take in the same pass as the second activation (instead of a third tensor-core
// layer with its own commit, wake-up and read-back).
struct TcOutLayer {
  float w[128];
  float b;
};
inline TcOutLayer tc_out_layer(const MlpTcDev &net) {
  TcOutLayer o;
  for (int i = 0; i < 128; ++i) o.w[i] = i < net.H ? net.w3_host[i] : 0.f;
  o.b = net.w3_host[128];
  return o;
}

// this thread's share of z for its row: sum over the columns of column group GRP (of NQ) of w3[j] act(D[row][j]), + b3
// in group 0; d0 = tensor-memory address of the group's first D column in the thread's lane; the column indices are
// compile-time.  The caller has done tcgen05.fence::after_thread_sync.
template <int H, int NQ, int GRP, int ACT>
__device__ __forceinline__ float tc_out_partial(uint32_t d0, const TcOutLayer &W3) {
  constexpr int NC = H / (16 * NQ), C0 = GRP * (H / NQ);
  uint32_t v[2][16];
  float acc0 = GRP == 0 ? W3.b : 0.f, acc1 = 0.f;
  tc::tmem_ld16(d0, v[0]);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    tc::wait_ld();
    if (c + 1 < NC) tc::tmem_ld16(d0 + (c + 1) * 16, v[(c + 1) & 1]);
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const float z = __uint_as_float(v[c & 1][j]);
      float h;
      if (ACT == DSMC_ACT_TANH) h = tc::tanh_approx(z);
      else if (ACT == DSMC_ACT_RELU) h = fmaxf(z, 0.f);
      else h = fmaf(z, tc::tanh_approx(z), z);  // SiLU(2 y) = y + y tanh(y), y = z (the weights carry the 1/2)
      if (j & 1) acc1 = fmaf(h, W3.w[C0 + 16 * c + j], acc1);
      else acc0 = fmaf(h, W3.w[C0 + 16 * c + j], acc0);
    }
  }
  return acc0 + acc1;
}

template <int H>
struct TcPipe {
  using SH = PipeShape<H>;
  unsigned char *w, *a1;  // a1: two slots
  uint64_t *bar_w, *in_ready, *full_e, *full_o, *a_ready, *out_free;  // [2] each except bar_w
  uint32_t *tmem_slot;
  uint32_t tmem;
  uint32_t ph_in[2], ph_e[2], ph_o[2], ph_a[2], ph_of[2];  // phase bits, each role tracks the barriers it waits on

  // all threads of the CTA call; base 128-byte aligned, SH::SMEM_BYTES
  __device__ __forceinline__ void init(unsigned char *base, const void *blob, int n_act_warps, int n_io_warps) {
    w = base;
    a1 = w + SH::BLOB_BYTES;
    bar_w = reinterpret_cast<uint64_t *>(a1 + 4 * SH::A1_BYTES);
    in_ready = bar_w + 1;
    full_e = in_ready + 2;
    full_o = full_e + 2;
    a_ready = full_o + 2;
    out_free = a_ready + 2;
    tmem_slot = reinterpret_cast<uint32_t *>(out_free + 2);
    const int tid = threadIdx.x, warp = tid >> 5;
    if (tid == 0) {
      tc::mbar_init(bar_w, 1);
      for (int s = 0; s < 2; ++s) {
        tc::mbar_init(in_ready + s, n_io_warps);
        tc::mbar_init(full_e + s, 1);
        tc::mbar_init(full_o + s, 1);
        tc::mbar_init(a_ready + s, n_act_warps);
        tc::mbar_init(out_free + s, n_io_warps);
      }
      tc::mbar_fence_init();
      tc::mbar_expect_tx(bar_w, (uint32_t)SH::BLOB_BYTES);
      tc::bulk_g2s(w, blob, (uint32_t)SH::BLOB_BYTES, bar_w);  // weights staged once per CTA by the TMA engine
    }
    if (warp == 0) tc::tmem_alloc<SH::TMEM_COLS>(tmem_slot);
    tc::fence_before();
    __syncthreads();
    tc::fence_after();
    tmem = *tmem_slot;
    if (warp < 4) {  // constant bias columns (1, 1, 0, ...) of both slots' A operands
      const uint32_t one[8] = {0x3F803F80u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
      const uint32_t lane_off = ((uint32_t)(warp * 32)) << 16;
      tc::tmem_st8(tmem + lane_off + SH::COL_BIAS, one);
      tc::tmem_st8(tmem + lane_off + SH::SLOT_COLS + SH::COL_BIAS, one);
      tc::wait_st();
    }
    tc::fence_before();
    __syncthreads();
    tc::fence_after();
#pragma unroll
    for (int s = 0; s < 2; ++s) ph_in[s] = ph_e[s] = ph_o[s] = ph_a[s] = ph_of[s] = 0;
  }
  __device__ __forceinline__ void teardown() {
    tc::fence_before();
    __syncthreads();
    if ((threadIdx.x >> 5) == 0) tc::tmem_dealloc<SH::TMEM_COLS>(tmem);
  }

  __device__ __forceinline__ void warp_arrive(uint64_t *bar) {
    __syncwarp();
    if ((threadIdx.x & 31) == 0)
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc::smem_u32(bar)) : "memory");
  }

  // ---- IO warps -------------------------------------------------------------------------------
  // row r of slot s, buffer par: [x_hi | x_lo | x_hi | 1 1 0 ...] (layer 1 in split precision)
  __device__ __forceinline__ void write_a1_row(int s, int par, int r, const float (&x)[8]) {
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      hi[j] = tc::pack_bf16(x[2 * j], x[2 * j + 1]);
      lo[j] = tc::pack_bf16(x[2 * j] - __uint_as_float(hi[j] << 16), x[2 * j + 1] - __uint_as_float(hi[j] & 0xFFFF0000u));
    }
    unsigned char *a = a1 + (2 * s + par) * SH::A1_BYTES + r * 16;
    const uint4 ph = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4 *>(a) = ph;
    *reinterpret_cast<uint4 *>(a + 1 * 128 * 16) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    *reinterpret_cast<uint4 *>(a + 2 * 128 * 16) = ph;
    *reinterpret_cast<uint4 *>(a + 3 * 128 * 16) = make_uint4(0x3F803F80u, 0u, 0u, 0u);
  }
  // after the warp's rows are written
  __device__ __forceinline__ void io_publish(int s) {
    tc::fence_proxy_async();
    warp_arrive(in_ready + s);
  }
  // outputs y[0..3] of row (io_warp * 32 + lane) of slot s
  __device__ __forceinline__ void io_read_out(int s, int io_warp, float (&y)[4]) {
    tc::mbar_wait(full_o + s, ph_o[s]);
    ph_o[s] ^= 1u;
    tc::fence_after();
    uint32_t v[4];
    tc::tmem_ld4(tmem + (((uint32_t)(io_warp * 32)) << 16) + s * SH::SLOT_COLS + SH::COL_OUT, v);
    tc::wait_ld();
    tc::fence_before();
    warp_arrive(out_free + s);
    y[0] = __uint_as_float(v[0]);
    y[1] = __uint_as_float(v[1]);
    y[2] = __uint_as_float(v[2]);
    y[3] = __uint_as_float(v[3]);
  }

  // ---- MMA warp (whole warp calls; one lane issues) ---------------------------------------------
  __device__ __forceinline__ void mma_layer1(int s, int par, bool first) {
    tc::mbar_wait(in_ready + s, ph_in[s]);
    ph_in[s] ^= 1u;
    if ((threadIdx.x & 31) == 0) {
      if (first) tc::mbar_wait(bar_w, 0);
      tc::fence_after();
      constexpr uint32_t idH = tc::instr_desc(128, H);
      const uint32_t a1a = tc::smem_u32(a1 + (2 * s + par) * SH::A1_BYTES), wa = tc::smem_u32(w);
#pragma unroll
      for (int ks = 0; ks < SH::K1 / 16; ++ks)
        tc::mma_ss(tmem + s * SH::SLOT_COLS + SH::COL_D, tc::smem_desc(a1a + ks * 2 * 128 * 16, 128 * 16, 128),
                   tc::smem_desc(wa + ks * 2 * H * 16, H * 16, 128), idH, ks > 0 ? 1u : 0u);
      tc::mma_commit(full_e + s);
    }
    __syncwarp();
  }
  template <int N>
  __device__ __forceinline__ void mma_hidden(int s, uint32_t off_w, uint32_t off_b, uint64_t *done, uint32_t col_d,
                                             bool wait_out) {
    tc::mbar_wait(a_ready + s, ph_a[s]);
    ph_a[s] ^= 1u;
    if (wait_out) {  // the previous tile's outputs have been read
      tc::mbar_wait(out_free + s, ph_of[s]);
      ph_of[s] ^= 1u;
    }
    if ((threadIdx.x & 31) == 0) {
      tc::fence_after();
      constexpr uint32_t idesc = tc::instr_desc(128, N);
      const uint32_t tD = tmem + s * SH::SLOT_COLS + col_d, tA = tmem + s * SH::SLOT_COLS + SH::COL_A;
      const uint32_t wa = tc::smem_u32(w);
#pragma unroll
      for (int ks = 0; ks < H / 16; ++ks)
        tc::mma_ts(tD, tA + ks * 8, tc::smem_desc(wa + off_w + ks * 2 * N * 16, N * 16, 128), idesc, ks > 0 ? 1u : 0u);
      tc::mma_ts(tD, tmem + s * SH::SLOT_COLS + SH::COL_BIAS, tc::smem_desc(wa + off_b, N * 16, 128), idesc, 1u);
      tc::mma_commit(done);
    }
    __syncwarp();
  }
  // a hidden layer whose weights [H x H] and bias block [H x 16] sit at the given shared-memory addresses
  __device__ __forceinline__ void mma_hidden_at(int s, uint32_t w_addr, uint32_t b_addr) {
    tc::mbar_wait(a_ready + s, ph_a[s]);
    ph_a[s] ^= 1u;
    if ((threadIdx.x & 31) == 0) {
      tc::fence_after();
      constexpr uint32_t idesc = tc::instr_desc(128, H);
      const uint32_t tD = tmem + s * SH::SLOT_COLS + SH::COL_D, tA = tmem + s * SH::SLOT_COLS + SH::COL_A;
#pragma unroll
      for (int ks = 0; ks < H / 16; ++ks)
        tc::mma_ts(tD, tA + ks * 8, tc::smem_desc(w_addr + ks * 2 * H * 16, H * 16, 128), idesc, ks > 0 ? 1u : 0u);
      tc::mma_ts(tD, tmem + s * SH::SLOT_COLS + SH::COL_BIAS, tc::smem_desc(b_addr, H * 16, 128), idesc, 1u);
      tc::mma_commit(full_e + s);
    }
    __syncwarp();
  }
  __device__ __forceinline__ void mma_layer2(int s) {
    mma_hidden<H>(s, SH::OFF_W2, SH::OFF_B2, full_e + s, SH::COL_D, false);
  }
  // first: no earlier tile went through this slot
  __device__ __forceinline__ void mma_layer3(int s, bool first) {
    mma_hidden<16>(s, SH::OFF_W3, SH::OFF_B3, full_o + s, SH::COL_OUT, !first);
  }

  // ---- non-blocking issue (polling MMA warp of the fused kernel; whole warp calls, operand known ready) ----
  __device__ __forceinline__ void issue_layer1(int s, int par, bool first) {
    if ((threadIdx.x & 31) == 0) {
      if (first) tc::mbar_wait(bar_w, 0);
      tc::fence_after();
      constexpr uint32_t idH = tc::instr_desc(128, H);
      const uint32_t a1a = tc::smem_u32(a1 + (2 * s + par) * SH::A1_BYTES), wa = tc::smem_u32(w);
#pragma unroll
      for (int ks = 0; ks < SH::K1 / 16; ++ks)
        tc::mma_ss(tmem + s * SH::SLOT_COLS + SH::COL_D, tc::smem_desc(a1a + ks * 2 * 128 * 16, 128 * 16, 128),
                   tc::smem_desc(wa + ks * 2 * H * 16, H * 16, 128), idH, ks > 0 ? 1u : 0u);
      tc::mma_commit(full_e + s);
    }
    __syncwarp();
  }
  template <int N>
  __device__ __forceinline__ void issue_hidden(int s, uint32_t off_w, uint32_t off_b, uint64_t *done, uint32_t col_d) {
    if ((threadIdx.x & 31) == 0) {
      tc::fence_after();
      constexpr uint32_t idesc = tc::instr_desc(128, N);
      const uint32_t tD = tmem + s * SH::SLOT_COLS + col_d, tA = tmem + s * SH::SLOT_COLS + SH::COL_A;
      const uint32_t wa = tc::smem_u32(w);
#pragma unroll
      for (int ks = 0; ks < H / 16; ++ks)
        tc::mma_ts(tD, tA + ks * 8, tc::smem_desc(wa + off_w + ks * 2 * N * 16, N * 16, 128), idesc, ks > 0 ? 1u : 0u);
      tc::mma_ts(tD, tmem + s * SH::SLOT_COLS + SH::COL_BIAS, tc::smem_desc(wa + off_b, N * 16, 128), idesc, 1u);
      tc::mma_commit(done);
    }
    __syncwarp();
  }
  __device__ __forceinline__ void issue_layer2(int s) { issue_hidden<H>(s, SH::OFF_W2, SH::OFF_B2, full_e + s, SH::COL_D); }
  __device__ __forceinline__ void issue_layer3(int s) { issue_hidden<16>(s, SH::OFF_W3, SH::OFF_B3, full_o + s, SH::COL_OUT); }

  // ---- ACT warps: lane quadrant act_warp & 3, column group act_warp >> 2 of NQ groups -----------
  // act_body: one (slot, layer) share of this warp; the caller has observed full_e[s]
  template <int ACT, int NQ>
  __device__ __forceinline__ void act_body(int s, int act_warp) {
    tc::fence_after();
    const uint32_t base = tmem + (((uint32_t)((act_warp & 3) * 32)) << 16) + s * SH::SLOT_COLS;
    const int grp = act_warp >> 2;
    // software pipeline over 16-column chunks: the TMEM read port (64 B / clk / SM) and the XU pipe
    // (16 MUFU / clk / SM) are both needed ~1024 cycles per tile layer, so chunk c + 1 is in flight
    // while chunk c goes through the activation
    constexpr int NC = H / (16 * NQ);  // 16-column chunks per thread
    const uint32_t d0 = base + SH::COL_D + grp * (H / NQ), a0 = base + SH::COL_A + grp * (H / (2 * NQ));
    uint32_t v[2][16];
    tc::tmem_ld16(d0, v[0]);
#pragma unroll
    for (int c = 0; c < NC; ++c) {
      tc::wait_ld();
      if (c + 1 < NC) tc::tmem_ld16(d0 + (c + 1) * 16, v[(c + 1) & 1]);
      uint32_t o[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const float z0 = __uint_as_float(v[c & 1][2 * j]), z1 = __uint_as_float(v[c & 1][2 * j + 1]);
        float h0, h1;
        if (ACT == DSMC_ACT_TANH) {
          h0 = tc::tanh_approx(z0);
          h1 = tc::tanh_approx(z1);
        } else if (ACT == DSMC_ACT_RELU) {
          h0 = fmaxf(z0, 0.f);
          h1 = fmaxf(z1, 0.f);
        } else {  // SiLU(2 y) = y + y tanh(y); the packed weights already carry the factor 1/2
          h0 = fmaf(z0, tc::tanh_approx(z0), z0);
          h1 = fmaf(z1, tc::tanh_approx(z1), z1);
        }
        o[j] = tc::pack_bf16(h0, h1);
      }
      tc::tmem_st8(a0 + c * 8, o);
    }
    tc::wait_st();
    tc::fence_before();
    warp_arrive(a_ready + s);
  }
  // this warp's 32 rows hold no real pair: nothing to activate, only the hand-off (rows are independent, the
  // stale operand rows produce outputs nobody reads)
  __device__ __forceinline__ void act_skip(int s) {
    tc::fence_after();
    tc::fence_before();
    warp_arrive(a_ready + s);
  }
  template <int NQ>
  __device__ __forceinline__ void act_body(int act, int s, int act_warp) {
    if (act == DSMC_ACT_TANH) act_body<DSMC_ACT_TANH, NQ>(s, act_warp);
    else if (act == DSMC_ACT_RELU) act_body<DSMC_ACT_RELU, NQ>(s, act_warp);
    else act_body<DSMC_ACT_SILU, NQ>(s, act_warp);
  }
  // blocking form used by the fixed-schedule kernel (k_chi_batch_tc)
  __device__ __forceinline__ void act_tile(int act, int s, int act_warp) {
    tc::mbar_wait(full_e + s, ph_e[s]);
    ph_e[s] ^= 1u;
    act_body<kPipeActWarps / 4>(act, s, act_warp);
  }
};

}  // namespace dsmc
