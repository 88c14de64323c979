// BF16 tcgen05 tensor-core variant of the neural collision operators (north_star: "the MLP layers run
// as tcgen05 tensor-core GEMMs over 128-pair tiles, BF16 operands, FP32 accumulate, weights staged once
// in shared memory by TMA").  See dsmc_tc.cuh for the tile algebra and operand layouts.
//
//   k_chi_batch_tc   a10: chi for independent (E_r, b) pairs                     (BASELINE.json cfg 4)
//   k_collide_tc     a2-a9 with the VHS-NN operator (split-BF16 operands): persistent fused step; one CTA pulls
//                    chunks (dsmc_chunk.cuh) from a work counter, keeps the packed weights resident, and feeds
//                    the chunk's pairs through the tile engine 128 at a time
//   (the ab initio chi-MLP fused step is k_cells_mlp: cell teams + a tcgen05 MLP server, dsmc_cells_mlp.cu)
#include <algorithm>
#include <vector>

#include "dsmc_chunk.cuh"
#include "dsmc_tc.cuh"
#include "dsmc_tc_pipe.cuh"

namespace dsmc {

// ---------------------------------------------------------------------------------------------
// host: pack a 3-layer MLP (d_in <= 15 -> H -> H -> d_out <= 16) into the bf16 panel image
// ---------------------------------------------------------------------------------------------
static uint16_t bf16_rne(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  if ((u & 0x7F800000u) == 0x7F800000u) return (uint16_t)(u >> 16);  // inf / nan
  u += 0x7FFFu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}
static float bf16_to_float(uint16_t h) {
  const uint32_t u = (uint32_t)h << 16;
  float f;
  memcpy(&f, &u, 4);
  return f;
}
static inline size_t panel_off(int r, int k, int R) { return (size_t)(k / 8) * R * 8 + (size_t)r * 8 + (k % 8); }

int build_tc_blob(const dsmc_mlp_desc *d, void **d_blob, MlpTcDev *out, cudaStream_t s) {
  out->H = 0;
  // 2..5 hidden layers (n_layers 3..6), hidden widths <= 128 (zero-padded to H = 64 or 128: a padded unit has zero
  // weights and bias, act(0) = 0 for tanh / ReLU / SiLU, and zero weights into the next layer)
  if (d->n_layers < 3 || d->n_layers > 6) return DSMC_ERR_UNSUPPORTED_SHAPE;
  const int nh = d->n_layers - 1, d_in = d->dims[0], d_out = d->dims[d->n_layers];
  int wmax = 0;
  for (int l = 1; l <= nh; ++l) {
    if (d->dims[l] < 1 || d->dims[l] > 128) return DSMC_ERR_UNSUPPORTED_SHAPE;
    wmax = std::max(wmax, d->dims[l]);
  }
  const int H = wmax <= 64 ? 64 : 128;
  if (d_in < 1 || d_in > 8 || d_out < 1 || d_out > 16) return DSMC_ERR_UNSUPPORTED_SHAPE;
  // SiLU(z) = y + y tanh(y) with y = z / 2: the hidden layers produce y directly (exact scaling by 1/2)
  const float hs = (d->act == DSMC_ACT_SILU) ? 0.5f : 1.0f;
  // image: [W1 H x 32 | W2hi H x H | B2 H x 16 | Wout_hi 16 x H | Bout 16 x 16 | W2lo H x H | Wout_lo 16 x H |
  //         (W_l hi H x H | B_l H x 16) for the hidden layers l = 3 .. nh]; every weight w of the first part is carried
  // as bf16 hi + bf16 lo = w - hi; the plain BF16 engines stage only the part before W2lo (and the extra layers).
  const size_t n1 = (size_t)H * 32, n2 = (size_t)H * H, nb2 = (size_t)H * 16, n3 = (size_t)16 * H, nb3 = 256;
  const size_t n_main = n1 + n2 + nb2 + n3 + nb3 + n2 + n3;
  std::vector<uint16_t> blob(n_main + (size_t)(nh - 2) * (n2 + nb2), 0);
  uint16_t *w1 = blob.data(), *w2h = w1 + n1, *b2 = w2h + n2, *w3h = b2 + nb2, *b3 = w3h + n3, *w2l = b3 + nb3,
           *w3l = w2l + n2;
  auto split = [](float w, uint16_t &hi, uint16_t &lo) {
    hi = bf16_rne(w);
    lo = bf16_rne(w - bf16_to_float(hi));
  };
  const int h1 = d->dims[1], h2 = d->dims[2];
  for (int n = 0; n < h1; ++n) {
    // layer 1 always in split precision: z = W_hi x_hi + W_hi x_lo + W_lo x_hi + (b_hi + b_lo);
    // operand columns [x_hi | x_lo | x_hi | 1 1 0 ...]
    for (int k = 0; k < d_in; ++k) {
      uint16_t hi, lo;
      split(hs * d->W[0][(size_t)n * d_in + k], hi, lo);
      w1[panel_off(n, k, H)] = hi;
      w1[panel_off(n, 8 + k, H)] = hi;
      w1[panel_off(n, 16 + k, H)] = lo;
    }
    split(hs * d->b[0][n], w1[panel_off(n, 24, H)], w1[panel_off(n, 25, H)]);
  }
  for (int n = 0; n < h2; ++n) {
    for (int k = 0; k < h1; ++k) split(hs * d->W[1][(size_t)n * h1 + k], w2h[panel_off(n, k, H)], w2l[panel_off(n, k, H)]);
    split(hs * d->b[1][n], b2[panel_off(n, 0, H)], b2[panel_off(n, 1, H)]);
  }
  for (int l = 3; l <= nh; ++l) {  // hidden layers beyond the second: plain BF16 weights, split bias
    uint16_t *wl = blob.data() + n_main + (size_t)(l - 3) * (n2 + nb2), *bl = wl + n2;
    const int win = d->dims[l - 1], wout = d->dims[l];
    for (int n = 0; n < wout; ++n) {
      for (int k = 0; k < win; ++k) wl[panel_off(n, k, H)] = bf16_rne(hs * d->W[l - 1][(size_t)n * win + k]);
      split(hs * d->b[l - 1][n], bl[panel_off(n, 0, H)], bl[panel_off(n, 1, H)]);
    }
  }
  const int hl = d->dims[nh];  // width of the last hidden layer
  for (int n = 0; n < d_out; ++n) {
    for (int k = 0; k < hl; ++k) split(d->W[nh][(size_t)n * hl + k], w3h[panel_off(n, k, 16)], w3l[panel_off(n, k, 16)]);
    split(d->b[nh][n], b3[panel_off(n, 0, 16)], b3[panel_off(n, 1, 16)]);
  }
  const size_t bytes = blob.size() * sizeof(uint16_t);
  if (cudaMalloc(d_blob, bytes) != cudaSuccess) return DSMC_ERR_CUDA;
  if (cudaMemcpyAsync(*d_blob, blob.data(), bytes, cudaMemcpyHostToDevice, s) != cudaSuccess) return DSMC_ERR_CUDA;
  if (cudaStreamSynchronize(s) != cudaSuccess) return DSMC_ERR_CUDA;
  out->H = H;
  out->d_in = d_in;
  out->d_out = d_out;
  out->act = d->act;
  out->w_blob = *d_blob;
  out->blob_bytes = (uint32_t)bytes;
  out->n_hidden = nh;
  out->extra_off = (uint32_t)(n_main * sizeof(uint16_t));
  for (int k = 0; k < 129; ++k) out->w3_host[k] = 0.f;
  if (d_out == 1) {
    for (int k = 0; k < hl; ++k) out->w3_host[k] = d->W[nh][k];
    out->w3_host[128] = d->b[nh][0];
  }
  return DSMC_OK;
}

// ---------------------------------------------------------------------------------------------
// device: the tile engine.  SPLIT = false: plain BF16 operands.  SPLIT = true: activations and
// weights of layers 2 and 3 are carried as bf16 hi + bf16 lo and each layer is three BF16 UMMA
// passes (hi.hi + lo.hi + hi.lo, FP32 accumulate); used for the VHS-NN operator, whose energy-shell
// normalisation (eq. 5) amplifies operand rounding by 1 / |h_hat| (Q21).
// ---------------------------------------------------------------------------------------------
template <int H, bool SPLIT>
struct TcShape {
  static constexpr int K1 = 32;  // layer-1 operand columns: x_hi | x_lo | x_hi | (1, 1, 0 ...)
  static constexpr int W1_BYTES = H * K1 * 2, W2_BYTES = H * H * 2, B2_BYTES = H * 16 * 2, W3_BYTES = 16 * H * 2,
                       B3_BYTES = 16 * 16 * 2;
  static constexpr int OFF_W2 = W1_BYTES, OFF_B2 = OFF_W2 + W2_BYTES, OFF_W3 = OFF_B2 + B2_BYTES,
                       OFF_B3 = OFF_W3 + W3_BYTES, OFF_W2L = OFF_B3 + B3_BYTES, OFF_W3L = OFF_W2L + W2_BYTES;
  static constexpr int BLOB_BYTES = SPLIT ? OFF_W3L + W3_BYTES : OFF_W2L;
  static constexpr int A1_BYTES = 128 * K1 * 2;
  static constexpr int SMEM_BYTES = BLOB_BYTES + A1_BYTES + 64;  // + barriers, tmem slot
  // tensor memory columns: D [0, H) fp32 | A: h_hi [H, H + H/2) | bias (1,1,0..) 8 cols | h_lo H/2 cols (SPLIT)
  static constexpr int COL_D = 0, COL_A = H, COL_BIAS = COL_A + H / 2, COL_LO = COL_BIAS + 8;
  static constexpr int COLS_USED = SPLIT ? COL_LO + H / 2 : COL_LO;
  static constexpr int TMEM_COLS = COLS_USED <= 128 ? 128 : (COLS_USED <= 256 ? 256 : 512);
};

template <int H, bool SPLIT>
struct TcEngine {
  using SH = TcShape<H, SPLIT>;
  unsigned char *w, *a1;
  uint64_t *bar_w, *bar_mma;
  uint32_t *tmem_slot;
  uint32_t tmem, lane_off, phase;
  bool weights_ready;

  // base must be 128-byte aligned shared memory of SH::SMEM_BYTES; all threads call; ends synchronised
  __device__ __forceinline__ void init(unsigned char *base, const void *blob) {
    w = base;
    a1 = w + SH::BLOB_BYTES;
    bar_w = reinterpret_cast<uint64_t *>(a1 + SH::A1_BYTES);
    bar_mma = bar_w + 1;
    tmem_slot = reinterpret_cast<uint32_t *>(bar_mma + 1);
    const int tid = threadIdx.x, warp = tid >> 5;
    if (tid == 0) {
      tc::mbar_init(bar_w, 1);
      tc::mbar_init(bar_mma, 1);
      tc::mbar_fence_init();
      tc::mbar_expect_tx(bar_w, (uint32_t)SH::BLOB_BYTES);
      tc::bulk_g2s(w, blob, (uint32_t)SH::BLOB_BYTES, bar_w);  // weights staged once per CTA by the TMA engine
    }
    if (warp == 0) tc::tmem_alloc<SH::TMEM_COLS>(tmem_slot);
    tc::fence_before();
    __syncthreads();
    tc::fence_after();
    tmem = *tmem_slot;
    lane_off = ((uint32_t)((warp & 3) * 32)) << 16;
    phase = 0;
    weights_ready = false;
    if (warp < 4) {  // constant bias columns of the TMEM A operand: (1, 1, 0, ..., 0) against (b_hi, b_lo, 0, ...)
      const uint32_t one[8] = {0x3F803F80u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
      tc::tmem_st8(tmem + lane_off + SH::COL_BIAS, one);
      tc::wait_st();
    }
    tc::fence_before();
    __syncthreads();
  }

  __device__ __forceinline__ void teardown() {
    tc::fence_before();
    __syncthreads();
    if ((threadIdx.x >> 5) == 0) tc::tmem_dealloc<SH::TMEM_COLS>(tmem);
  }

  // row r of the layer-1 operand from the (up to 8) fp32 features x: [x_hi | x_lo | x_hi | 1 1 0 ...]
  __device__ __forceinline__ void write_a1_row(int r, const float (&x)[8]) {
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      hi[j] = tc::pack_bf16(x[2 * j], x[2 * j + 1]);
      const float r0 = x[2 * j] - __uint_as_float(hi[j] << 16);
      const float r1 = x[2 * j + 1] - __uint_as_float(hi[j] & 0xFFFF0000u);
      lo[j] = tc::pack_bf16(r0, r1);
    }
    const uint4 ph = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4 *>(a1 + r * 16) = ph;
    *reinterpret_cast<uint4 *>(a1 + 1 * 128 * 16 + r * 16) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    *reinterpret_cast<uint4 *>(a1 + 2 * 128 * 16 + r * 16) = ph;
    *reinterpret_cast<uint4 *>(a1 + 3 * 128 * 16 + r * 16) = make_uint4(0x3F803F80u, 0u, 0u, 0u);
  }

  // D (fp32, my lane, my half of the columns) -> act -> bf16 (hi [, lo]) -> TMEM A operand
  template <int ACT>
  __device__ __forceinline__ void epilogue() {
    const int half = threadIdx.x >> 7;
#pragma unroll
    for (int c = 0; c < H / 64; ++c) {
      const int col0 = half * (H / 2) + c * 32;
      uint32_t v[32], o[16];
      tc::tmem_ld32(tmem + lane_off + SH::COL_D + col0, v);
      tc::wait_ld();
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const float z0 = __uint_as_float(v[2 * j]), z1 = __uint_as_float(v[2 * j + 1]);
        float h0, h1;
        if (ACT == DSMC_ACT_TANH) {
          h0 = SPLIT ? tc::tanh_abs(z0) : tc::tanh_approx(z0);
          h1 = SPLIT ? tc::tanh_abs(z1) : tc::tanh_approx(z1);
        } else if (ACT == DSMC_ACT_RELU) {
          h0 = fmaxf(z0, 0.f);
          h1 = fmaxf(z1, 0.f);
        } else {  // SiLU(2 y) = y + y tanh(y); the packed weights already carry the factor 1/2
          h0 = fmaf(z0, SPLIT ? tc::tanh_abs(z0) : tc::tanh_approx(z0), z0);
          h1 = fmaf(z1, SPLIT ? tc::tanh_abs(z1) : tc::tanh_approx(z1), z1);
        }
        o[j] = tc::pack_bf16(h0, h1);
        if (SPLIT) {  // keep the residuals for the lo pass
          v[2 * j] = __float_as_uint(h0 - __uint_as_float(o[j] << 16));
          v[2 * j + 1] = __float_as_uint(h1 - __uint_as_float(o[j] & 0xFFFF0000u));
        }
      }
      tc::tmem_st16(tmem + lane_off + SH::COL_A + col0 / 2, o);
      if (SPLIT) {
#pragma unroll
        for (int j = 0; j < 16; ++j) o[j] = tc::pack_bf16(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]));
        tc::tmem_st16(tmem + lane_off + SH::COL_LO + col0 / 2, o);
      }
    }
    tc::wait_st();
    tc::fence_before();
    __syncthreads();
  }
  __device__ __forceinline__ void epilogue_act(int act) {
    if (act == DSMC_ACT_TANH) epilogue<DSMC_ACT_TANH>();
    else if (act == DSMC_ACT_RELU) epilogue<DSMC_ACT_RELU>();
    else epilogue<DSMC_ACT_SILU>();
  }

  __device__ __forceinline__ void wait_mma() {
    tc::mbar_wait(bar_mma, phase);
    phase ^= 1u;
    tc::fence_after();
  }

  // one hidden-operand layer: D[128 x N] = [h | 1] . [W | b]^T (+ lo passes), issued by one thread
  template <int N>
  __device__ __forceinline__ void issue_layer(uint32_t wh, uint32_t wb, uint32_t wl) {
    constexpr uint32_t idesc = tc::instr_desc(128, N);
    const uint32_t tD = tmem + SH::COL_D, tA = tmem + SH::COL_A;
#pragma unroll
    for (int ks = 0; ks < H / 16; ++ks)
      tc::mma_ts(tD, tA + ks * 8, tc::smem_desc(wh + ks * 2 * N * 16, N * 16, 128), idesc, ks > 0 ? 1u : 0u);
    tc::mma_ts(tD, tmem + SH::COL_BIAS, tc::smem_desc(wb, N * 16, 128), idesc, 1u);
    if (SPLIT) {
#pragma unroll
      for (int ks = 0; ks < H / 16; ++ks)
        tc::mma_ts(tD, tmem + SH::COL_LO + ks * 8, tc::smem_desc(wh + ks * 2 * N * 16, N * 16, 128), idesc, 1u);
#pragma unroll
      for (int ks = 0; ks < H / 16; ++ks)
        tc::mma_ts(tD, tA + ks * 8, tc::smem_desc(wl + ks * 2 * N * 16, N * 16, 128), idesc, 1u);
    }
    tc::mma_commit(bar_mma);
  }

  // Runs the three layers on the 128 rows staged in a1.  All threads call.  On return the outputs
  // y[r][0..15] sit in TMEM columns COL_D .. COL_D+15 of lane r (read with read_out()); the caller
  // issues tc::fence_before() after reading them and before the next run().
  __device__ __forceinline__ void run(int act) {
    tc::fence_proxy_async();  // a1 rows (generic proxy) -> visible to the tensor core (async proxy)
    __syncthreads();
    const bool issuer = threadIdx.x == 0;
    const uint32_t wa = tc::smem_u32(w);
    if (issuer) {
      if (!weights_ready) tc::mbar_wait(bar_w, 0);
      tc::fence_after();
      constexpr uint32_t idH = tc::instr_desc(128, H);
      const uint32_t a1a = tc::smem_u32(a1);
#pragma unroll
      for (int ks = 0; ks < SH::K1 / 16; ++ks)
        tc::mma_ss(tmem + SH::COL_D, tc::smem_desc(a1a + ks * 2 * 128 * 16, 128 * 16, 128),
                   tc::smem_desc(wa + ks * 2 * H * 16, H * 16, 128), idH, ks > 0 ? 1u : 0u);
      tc::mma_commit(bar_mma);
    }
    weights_ready = true;
    wait_mma();
    epilogue_act(act);
    if (issuer) {
      tc::fence_after();
      issue_layer<H>(wa + SH::OFF_W2, wa + SH::OFF_B2, wa + SH::OFF_W2L);
    }
    wait_mma();
    epilogue_act(act);
    if (issuer) {
      tc::fence_after();
      issue_layer<16>(wa + SH::OFF_W3, wa + SH::OFF_B3, wa + SH::OFF_W3L);
    }
    wait_mma();
  }

  // first four outputs of my row (threads 0..127: row = threadIdx.x)
  __device__ __forceinline__ void read_out(float (&y)[4]) {
    uint32_t v[4];
    tc::tmem_ld4(tmem + lane_off + SH::COL_D, v);
    tc::wait_ld();
    y[0] = __uint_as_float(v[0]);
    y[1] = __uint_as_float(v[1]);
    y[2] = __uint_as_float(v[2]);
    y[3] = __uint_as_float(v[3]);
  }
};

__device__ __forceinline__ unsigned char *align128(unsigned char *p) {
  return reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(p) + 127) & ~(uintptr_t)127);
}

// ---------------------------------------------------------------------------------------------
// a10: chi for independent pairs, chi = expm1(softplus(z)) = exp(z) (Q15), z = MLP(E~_n, b~).
// Persistent, warp-specialised (dsmc_tc_pipe.cuh): the k-th tile of a CTA goes through slot k & 1.
// ---------------------------------------------------------------------------------------------
// The output layer (d_out = 1) is folded into the second activation (tc_out_partial, dsmc_tc_pipe.cuh): every
// activation warp leaves the partial sum of its 32 columns in shared memory, the IO warps add the four of a row in a
// fixed order.  zs[slot][round & 1][column group][row]: double-buffered by round, so a buffer is rewritten only after
// the IO warps have published the features of the round after its last reader's (a barrier chain, not a timing guess).
template <int H, int ACT>
__device__ __forceinline__ void chi_out_tile(TcPipe<H> &pipe, int s, int act_warp, const TcOutLayer &W3, float *zrow,
                                             uint64_t *z_bar) {
  using SH = PipeShape<H>;
  constexpr int NQ = kPipeActWarps / 4;
  tc::mbar_wait(pipe.full_e + s, pipe.ph_e[s]);
  pipe.ph_e[s] ^= 1u;
  tc::fence_after();
  const int grp = act_warp >> 2, lane = threadIdx.x & 31;
  const uint32_t d0 = pipe.tmem + (((uint32_t)((act_warp & 3) * 32)) << 16) + s * SH::SLOT_COLS + SH::COL_D + grp * (H / NQ);
  float part;
  if (grp == 0) part = tc_out_partial<H, NQ, 0, ACT>(d0, W3);
  else if (grp == 1) part = tc_out_partial<H, NQ, 1, ACT>(d0, W3);
  else if (grp == 2) part = tc_out_partial<H, NQ, 2, ACT>(d0, W3);
  else part = tc_out_partial<H, NQ, 3, ACT>(d0, W3);
  zrow[grp * 128 + (act_warp & 3) * 32 + lane] = part;
  tc::fence_before();
  __syncwarp();
  if (lane == 0) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc::smem_u32(pipe.a_ready + s)) : "memory");  // D is free
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc::smem_u32(z_bar)) : "memory");
  }
}

// RAW: E, b already hold the network inputs (x0, x1) of every row (the split fused step, dsmc_cells.cu)
// DEEP: more than two hidden layers (run-time count); otherwise the layer loops fold away
template <int H, bool RAW, bool DEEP>
__global__ void __launch_bounds__(kPipeThreads, 1)
    k_chi_batch_tc(int64_t n, const float *__restrict__ E, const float *__restrict__ b, float *__restrict__ chi,
                   const MlpTcDev net, const TcOutLayer W3, float inv_bmax, float lnE_min, float inv_range) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  TcPipe<H> pipe;
  using SH = PipeShape<H>;
  float *zs = reinterpret_cast<float *>(smem_raw + SH::SMEM_BYTES);      // [2][2][4][128]
  uint64_t *z_bar = reinterpret_cast<uint64_t *>(zs + 2 * 2 * 4 * 128);  // [2], then the barrier of the extra layers
  uint64_t *x_bar = z_bar + 2;
  // hidden layers 3 .. n_hidden (W [H x H] | B [H x 16] each), behind everything else
  unsigned char *extra = smem_raw + ((SH::SMEM_BYTES + 2 * 2 * 4 * 128 * 4 + 32 + 127) & ~127);
  const int n_hidden = DEEP ? net.n_hidden : 2, n_extra = n_hidden - 2;
  constexpr uint32_t kLayerBytes = SH::W2_BYTES + SH::B2_BYTES;
  if (threadIdx.x == 0) {
    tc::mbar_init(z_bar + 0, kPipeActWarps);
    tc::mbar_init(z_bar + 1, kPipeActWarps);
    tc::mbar_init(x_bar, 1);
  }
  pipe.init(smem_raw, net.w_blob, kPipeActWarps, kPipeIoWarps);  // (fences the barrier inits, ends with CTA barriers)
  if (threadIdx.x == 0 && n_extra > 0) {
    tc::mbar_expect_tx(x_bar, (uint32_t)n_extra * kLayerBytes);
    tc::bulk_g2s(extra, reinterpret_cast<const unsigned char *>(net.w_blob) + net.extra_off, (uint32_t)n_extra * kLayerBytes, x_bar);
  }
  pdl_wait();  // the set-up above (weights, tensor memory) ran under the tail of the kernel before this one
  pdl_launch_dependents();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t n_tiles = (n + 127) / 128;
  const int64_t mine = n_tiles > blockIdx.x ? (n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const int64_t n_rounds = (mine + 1) / 2;  // two slots per round; a missing second tile runs as zeros
  if (warp < kPipeActWarps) {
    for (int64_t r = 0; r < n_rounds; ++r) {
#pragma unroll 1
      for (int l = 1; l < n_hidden; ++l) {  // every hidden activation but the last: D -> act -> bf16 A operand
        pipe.act_tile(net.act, 0, warp);
        pipe.act_tile(net.act, 1, warp);
      }
#pragma unroll 1
      for (int s = 0; s < 2; ++s) {  // the last one, with the output layer folded in
        float *zrow = zs + (size_t)((s * 2 + (int)(r & 1)) * 4) * 128;
        if (net.act == DSMC_ACT_SILU) chi_out_tile<H, DSMC_ACT_SILU>(pipe, s, warp, W3, zrow, z_bar + s);
        else if (net.act == DSMC_ACT_TANH) chi_out_tile<H, DSMC_ACT_TANH>(pipe, s, warp, W3, zrow, z_bar + s);
        else chi_out_tile<H, DSMC_ACT_RELU>(pipe, s, warp, W3, zrow, z_bar + s);
      }
    }
  } else if (warp < kPipeActWarps + kPipeIoWarps) {
    const int io_warp = warp - kPipeActWarps, row = io_warp * 32 + lane;
    auto features = [&](int s, int64_t k) {  // tile k of this CTA -> layer-1 operand buffer (s, (k >> 1) & 1)
      const int64_t p = (blockIdx.x + k * gridDim.x) * 128 + row;
      float x[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) x[j] = 0.f;
      if (RAW) {
        if (k < mine && p < n) {
          x[0] = __ldg(E + p);
          x[1] = __ldg(b + p);
        }
      } else if (k < mine && p < n) {
        const float e = (__logf(__ldg(E + p)) - lnE_min) * inv_range;
        x[0] = !(e > 0.f) ? 0.f : fminf(e, 1.f);
        const float bt = __ldg(b + p) * inv_bmax;
        x[1] = !(bt > 0.f) ? 0.f : fminf(bt, 1.f);
      }
      pipe.write_a1_row(s, (int)((k >> 1) & 1), row, x);
      pipe.io_publish(s);
    };
    if (n_rounds > 0) {
      features(0, 0);
      features(1, 1);
    }
    uint32_t phz[2] = {0u, 0u};
    for (int64_t r = 0; r < n_rounds; ++r) {
#pragma unroll 1
      for (int s = 0; s < 2; ++s) {
        const int64_t k = 2 * r + s;
        if (r + 1 < n_rounds) features(s, k + 2);  // a round ahead: off the critical path
        tc::mbar_wait(z_bar + s, phz[s]);
        phz[s] ^= 1u;
        const float *zrow = zs + (size_t)((s * 2 + (int)(r & 1)) * 4) * 128 + row;
        const float z = ((zrow[0] + zrow[128]) + zrow[256]) + zrow[384];
        const int64_t p = (blockIdx.x + k * gridDim.x) * 128 + row;
        if (k < mine && p < n) chi[p] = __expf(z);
      }
    }
  } else {
    // per round: layer 2 of both slots as their first activations end, then -- as the second activations end and free
    // the accumulators -- layer 1 of the next round's tiles
    if (n_rounds > 0) {
      pipe.mma_layer1(0, 0, true);
      pipe.mma_layer1(1, 0, false);
    }
    if (n_rounds > 0 && n_extra > 0) {
      if (lane == 0) tc::mbar_wait(x_bar, 0);  // the extra layers have landed
      __syncwarp();
    }
    for (int64_t r = 0; r < n_rounds; ++r) {
      const bool more = r + 1 < n_rounds;
      const int par = (int)((r + 1) & 1);
      pipe.mma_layer2(0);
      pipe.mma_layer2(1);
#pragma unroll 1
      for (int l = 0; l < n_extra; ++l) {
        const uint32_t wa = tc::smem_u32(extra) + (uint32_t)l * kLayerBytes;
        pipe.mma_hidden_at(0, wa, wa + SH::W2_BYTES);
        pipe.mma_hidden_at(1, wa, wa + SH::W2_BYTES);
      }
#pragma unroll 1
      for (int s = 0; s < 2; ++s) {
        tc::mbar_wait(pipe.a_ready + s, pipe.ph_a[s]);
        pipe.ph_a[s] ^= 1u;
        if (more) pipe.mma_layer1(s, par, false);
      }
    }
  }
  pipe.teardown();
}

template <int H, bool RAW>
static int launch_chi_batch_tc_h(dsmc_ctx *c, int64_t n, const float *E, const float *b, float *chi, float b_max,
                                 float lnE_min, float lnE_max, const MlpTcDev *net) {
  const float inv_range = 1.0f / (lnE_max - lnE_min);
  const int grid = (int)std::min<int64_t>((n + 127) / 128, (int64_t)c->num_sms);
  const int smem = ((PipeShape<H>::SMEM_BYTES + 2 * 2 * 4 * 128 * 4 + 32 + 127) & ~127) +
                   (net->n_hidden - 2) * (PipeShape<H>::W2_BYTES + PipeShape<H>::B2_BYTES) + 128;
  if (smem > 227 * 1024) return DSMC_ERR_UNSUPPORTED_SHAPE;
  auto kern = net->n_hidden > 2 ? k_chi_batch_tc<H, RAW, true> : k_chi_batch_tc<H, RAW, false>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return DSMC_ERR_CUDA;
  launch_pdl(kern, grid, kPipeThreads, (size_t)smem, c->stream, n, E, b, chi, *net, tc_out_layer(*net), 1.0f / b_max, lnE_min, inv_range);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_chi_batch_tc(dsmc_ctx *c, int64_t n, const float *E, const float *b, float *chi, float b_max,
                        float lnE_min, float lnE_max, const MlpTcDev *net) {
  if (net->d_in != 2 || net->d_out != 1) return DSMC_ERR_UNSUPPORTED_SHAPE;
  return net->H == 128 ? launch_chi_batch_tc_h<128, false>(c, n, E, b, chi, b_max, lnE_min, lnE_max, net)
                       : launch_chi_batch_tc_h<64, false>(c, n, E, b, chi, b_max, lnE_min, lnE_max, net);
}

// chi = exp(MLP(x0, x1)) for rows whose network inputs are given as they are (no normalisation, no clamping)
int launch_chi_rows_tc(dsmc_ctx *c, int64_t n, const float *x0, const float *x1, float *chi, const MlpTcDev *net) {
  if (net->d_in != 2 || net->d_out != 1) return DSMC_ERR_UNSUPPORTED_SHAPE;
  return net->H == 128 ? launch_chi_batch_tc_h<128, true>(c, n, x0, x1, chi, 1.f, 0.f, 1.f, net)
                       : launch_chi_batch_tc_h<64, true>(c, n, x0, x1, chi, 1.f, 0.f, 1.f, net);
}

// ---------------------------------------------------------------------------------------------
// Rows -> MLP outputs in SPLIT precision on the two-slot pipeline (the VHS-NN operator of the split fused step,
// dsmc_collide.cu): d_in <= 8 inputs per row, up to three outputs.  Layer 1 as everywhere (split operand, bias column);
// the hidden activations are carried as bf16 hi + bf16 lo in tensor memory (A_hi where the plain pipe keeps A, A_lo in
// the columns the plain pipe uses for its bias and output blocks) and layer 2 is three UMMA passes
// (hi.hi + lo.hi + hi.lo, FP32 accumulate); its bias and the whole output layer are FP32 on the CUDA cores, folded
// into the second activation (constant-bank operands): more exact than a split third tensor-core layer and no third
// hand-off.  Eq. 5 divides by |h|, so the activation is tanh_abs (3e-7), not tanh.approx.
// ---------------------------------------------------------------------------------------------
template <int ACT>
__device__ __forceinline__ float act_split(float z) {
  if (ACT == DSMC_ACT_TANH) return tc::tanh_abs(z);
  if (ACT == DSMC_ACT_RELU) return fmaxf(z, 0.f);
  return fmaf(z, tc::tanh_abs(z), z);  // SiLU(2 y) = y + y tanh(y), y = z (weights and biases carry the 1/2)
}

// first activation: D -> act -> (hi, lo) bf16 -> A_hi, A_lo of the slot
template <int H, int ACT>
__device__ __forceinline__ void act1_split(TcPipe<H> &pipe, int s, int act_warp) {
  using SH = PipeShape<H>;
  constexpr int NQ = kPipeActWarps / 4, NC = H / (16 * NQ);
  tc::mbar_wait(pipe.full_e + s, pipe.ph_e[s]);
  pipe.ph_e[s] ^= 1u;
  tc::fence_after();
  const uint32_t base = pipe.tmem + (((uint32_t)((act_warp & 3) * 32)) << 16) + s * SH::SLOT_COLS;
  const int grp = act_warp >> 2;
  const uint32_t d0 = base + SH::COL_D + grp * (H / NQ), ah = base + SH::COL_A + grp * (H / (2 * NQ)),
                 al = base + SH::COL_BIAS + grp * (H / (2 * NQ));
  uint32_t v[2][16];
  tc::tmem_ld16(d0, v[0]);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    tc::wait_ld();
    if (c + 1 < NC) tc::tmem_ld16(d0 + (c + 1) * 16, v[(c + 1) & 1]);
    uint32_t hi[8], lo[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const float h0 = act_split<ACT>(__uint_as_float(v[c & 1][2 * j])), h1 = act_split<ACT>(__uint_as_float(v[c & 1][2 * j + 1]));
      hi[j] = tc::pack_bf16(h0, h1);
      lo[j] = tc::pack_bf16(h0 - __uint_as_float(hi[j] << 16), h1 - __uint_as_float(hi[j] & 0xFFFF0000u));
    }
    tc::tmem_st8(ah + c * 8, hi);
    tc::tmem_st8(al + c * 8, lo);
  }
  tc::wait_st();
  tc::fence_before();
  pipe.warp_arrive(pipe.a_ready + s);
}

// second activation and the output layer: this thread's partial sums (its row, column group GRP) of the d_out outputs
template <int H, int GRP, int ACT>
__device__ __forceinline__ void out_split(uint32_t d0, const TcTailF32 &T, float (&y)[3]) {
  constexpr int NQ = kPipeActWarps / 4, NC = H / (16 * NQ), C0 = GRP * (H / NQ);
  uint32_t v[2][16];
  y[0] = GRP == 0 ? T.b3[0] : 0.f;
  y[1] = GRP == 0 ? T.b3[1] : 0.f;
  y[2] = GRP == 0 ? T.b3[2] : 0.f;
  tc::tmem_ld16(d0, v[0]);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    tc::wait_ld();
    if (c + 1 < NC) tc::tmem_ld16(d0 + (c + 1) * 16, v[(c + 1) & 1]);
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const float h = act_split<ACT>(__uint_as_float(v[c & 1][j]) + T.b2[C0 + 16 * c + j]);
      y[0] = fmaf(h, T.w3[0][C0 + 16 * c + j], y[0]);
      y[1] = fmaf(h, T.w3[1][C0 + 16 * c + j], y[1]);
      y[2] = fmaf(h, T.w3[2][C0 + 16 * c + j], y[2]);
    }
  }
}

template <int H, int ACT>
__device__ __forceinline__ void act2_split(TcPipe<H> &pipe, int s, int act_warp, const TcTailF32 &T, float *zrow,
                                           uint64_t *z_bar) {
  using SH = PipeShape<H>;
  constexpr int NQ = kPipeActWarps / 4;
  tc::mbar_wait(pipe.full_e + s, pipe.ph_e[s]);
  pipe.ph_e[s] ^= 1u;
  tc::fence_after();
  const int grp = act_warp >> 2, lane = threadIdx.x & 31;
  const uint32_t d0 = pipe.tmem + (((uint32_t)((act_warp & 3) * 32)) << 16) + s * SH::SLOT_COLS + SH::COL_D + grp * (H / NQ);
  float y[3];
  if (grp == 0) out_split<H, 0, ACT>(d0, T, y);
  else if (grp == 1) out_split<H, 1, ACT>(d0, T, y);
  else if (grp == 2) out_split<H, 2, ACT>(d0, T, y);
  else out_split<H, 3, ACT>(d0, T, y);
  float *zr = zrow + (grp * 128 + (act_warp & 3) * 32 + lane) * 4;  // [group][row][4]
  *reinterpret_cast<float4 *>(zr) = make_float4(y[0], y[1], y[2], 0.f);
  tc::fence_before();
  __syncwarp();
  if (lane == 0) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc::smem_u32(pipe.a_ready + s)) : "memory");  // D is free
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc::smem_u32(z_bar)) : "memory");
  }
}

template <int H>
__global__ void __launch_bounds__(kPipeThreads, 1)
    k_mlp_rows_tc_split(int64_t n, const float *__restrict__ x, int64_t x_stride, int d_in, float *__restrict__ y0,
                        float *__restrict__ y1, float *__restrict__ y2, const MlpTcDev net, const TcTailF32 T) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  using SH = PipeShape<H>;
  TcPipe<H> pipe;
  unsigned char *w2lo = smem_raw + ((SH::SMEM_BYTES + 127) & ~127);
  float *zs = reinterpret_cast<float *>(w2lo + H * H * 2);               // [2][2][4][128][4]
  uint64_t *z_bar = reinterpret_cast<uint64_t *>(zs + 2 * 2 * 4 * 128 * 4);  // [2], then the W2lo barrier
  uint64_t *w_bar = z_bar + 2;
  if (threadIdx.x == 0) {
    tc::mbar_init(z_bar + 0, kPipeActWarps);
    tc::mbar_init(z_bar + 1, kPipeActWarps);
    tc::mbar_init(w_bar, 1);
  }
  pipe.init(smem_raw, net.w_blob, kPipeActWarps, kPipeIoWarps);  // (fences the barrier inits, ends with CTA barriers)
  if (threadIdx.x == 0) {
    tc::mbar_expect_tx(w_bar, (uint32_t)(H * H * 2));
    tc::bulk_g2s(w2lo, reinterpret_cast<const unsigned char *>(net.w_blob) + SH::BLOB_BYTES, (uint32_t)(H * H * 2), w_bar);
  }
  pdl_wait();  // the set-up above ran under the tail of the kernel before this one
  pdl_launch_dependents();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t n_tiles = (n + 127) / 128;
  const int64_t mine = n_tiles > blockIdx.x ? (n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const int64_t n_rounds = (mine + 1) / 2;
  if (warp < kPipeActWarps) {
    for (int64_t r = 0; r < n_rounds; ++r) {
#pragma unroll 1
      for (int s = 0; s < 2; ++s) {
        if (net.act == DSMC_ACT_TANH) act1_split<H, DSMC_ACT_TANH>(pipe, s, warp);
        else if (net.act == DSMC_ACT_RELU) act1_split<H, DSMC_ACT_RELU>(pipe, s, warp);
        else act1_split<H, DSMC_ACT_SILU>(pipe, s, warp);
      }
#pragma unroll 1
      for (int s = 0; s < 2; ++s) {
        float *zrow = zs + (size_t)((s * 2 + (int)(r & 1)) * 4) * 128 * 4;
        if (net.act == DSMC_ACT_TANH) act2_split<H, DSMC_ACT_TANH>(pipe, s, warp, T, zrow, z_bar + s);
        else if (net.act == DSMC_ACT_RELU) act2_split<H, DSMC_ACT_RELU>(pipe, s, warp, T, zrow, z_bar + s);
        else act2_split<H, DSMC_ACT_SILU>(pipe, s, warp, T, zrow, z_bar + s);
      }
    }
  } else if (warp < kPipeActWarps + kPipeIoWarps) {
    const int io_warp = warp - kPipeActWarps, row = io_warp * 32 + lane;
    auto features = [&](int s, int64_t k) {
      const int64_t p = (blockIdx.x + k * gridDim.x) * 128 + row;
      float f[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) f[j] = (k < mine && p < n && j < d_in) ? __ldg(x + j * x_stride + p) : 0.f;
      pipe.write_a1_row(s, (int)((k >> 1) & 1), row, f);
      pipe.io_publish(s);
    };
    if (n_rounds > 0) {
      features(0, 0);
      features(1, 1);
    }
    uint32_t phz[2] = {0u, 0u};
    for (int64_t r = 0; r < n_rounds; ++r) {
#pragma unroll 1
      for (int s = 0; s < 2; ++s) {
        const int64_t k = 2 * r + s;
        if (r + 1 < n_rounds) features(s, k + 2);
        tc::mbar_wait(z_bar + s, phz[s]);
        phz[s] ^= 1u;
        const float4 *zr = reinterpret_cast<const float4 *>(zs + (size_t)((s * 2 + (int)(r & 1)) * 4) * 128 * 4) + row;
        const float4 a = zr[0], b = zr[128], c = zr[256], d = zr[384];
        const int64_t p = (blockIdx.x + k * gridDim.x) * 128 + row;
        if (k < mine && p < n) {
          y0[p] = ((a.x + b.x) + c.x) + d.x;
          y1[p] = ((a.y + b.y) + c.y) + d.y;
          y2[p] = ((a.z + b.z) + c.z) + d.z;
        }
      }
    }
  } else {
    // layer 2 in three passes: hi.hi + lo.hi + hi.lo
    auto layer2 = [&](int s) {
      tc::mbar_wait(pipe.a_ready + s, pipe.ph_a[s]);
      pipe.ph_a[s] ^= 1u;
      if (lane == 0) {
        tc::fence_after();
        constexpr uint32_t idesc = tc::instr_desc(128, H);
        const uint32_t tD = pipe.tmem + s * SH::SLOT_COLS + SH::COL_D, tAh = pipe.tmem + s * SH::SLOT_COLS + SH::COL_A,
                       tAl = pipe.tmem + s * SH::SLOT_COLS + SH::COL_BIAS;
        const uint32_t wh = tc::smem_u32(pipe.w) + SH::OFF_W2, wl = tc::smem_u32(w2lo);
#pragma unroll
        for (int ks = 0; ks < H / 16; ++ks)
          tc::mma_ts(tD, tAh + ks * 8, tc::smem_desc(wh + ks * 2 * H * 16, H * 16, 128), idesc, ks > 0 ? 1u : 0u);
#pragma unroll
        for (int ks = 0; ks < H / 16; ++ks)
          tc::mma_ts(tD, tAl + ks * 8, tc::smem_desc(wh + ks * 2 * H * 16, H * 16, 128), idesc, 1u);
#pragma unroll
        for (int ks = 0; ks < H / 16; ++ks)
          tc::mma_ts(tD, tAh + ks * 8, tc::smem_desc(wl + ks * 2 * H * 16, H * 16, 128), idesc, 1u);
        tc::mma_commit(pipe.full_e + s);
      }
      __syncwarp();
    };
    if (n_rounds > 0) {
      pipe.mma_layer1(0, 0, true);
      pipe.mma_layer1(1, 0, false);
      if (lane == 0) tc::mbar_wait(w_bar, 0);  // W2lo has landed
      __syncwarp();
    }
    for (int64_t r = 0; r < n_rounds; ++r) {
      const bool more = r + 1 < n_rounds;
      const int par = (int)((r + 1) & 1);
      layer2(0);
      layer2(1);
#pragma unroll 1
      for (int s = 0; s < 2; ++s) {
        tc::mbar_wait(pipe.a_ready + s, pipe.ph_a[s]);  // the second activation has read D
        pipe.ph_a[s] ^= 1u;
        if (more) pipe.mma_layer1(s, par, false);
      }
    }
  }
  pipe.teardown();
}

template <int H>
static int launch_mlp_rows_tc_split_h(dsmc_ctx *c, int64_t n, const float *x, int64_t x_stride, float *y0, float *y1,
                                      float *y2, const MlpTcDev *net, const TcTailF32 *tail) {
  const int grid = (int)std::min<int64_t>((n + 127) / 128, (int64_t)c->num_sms);
  const int smem = ((PipeShape<H>::SMEM_BYTES + 127) & ~127) + H * H * 2 + 2 * 2 * 4 * 128 * 16 + 64 + 128;
  auto kern = k_mlp_rows_tc_split<H>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return DSMC_ERR_CUDA;
  launch_pdl(kern, grid, kPipeThreads, (size_t)smem, c->stream, n, x, x_stride, net->d_in, y0, y1, y2, *net, *tail);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

// y[o][p] = MLP(x[0..d_in)[p])[o], o < 3, rows p < n; x: d_in arrays x + j x_stride; split-precision tensor-core path
int launch_mlp_rows_tc_split(dsmc_ctx *c, int64_t n, const float *x, int64_t x_stride, float *y0, float *y1, float *y2,
                             const MlpTcDev *net, const TcTailF32 *tail) {
  if (net->d_in < 1 || net->d_in > 8 || tail->d_out < 1 || tail->d_out > 3 || net->n_hidden != 2) return DSMC_ERR_UNSUPPORTED_SHAPE;
  return net->H == 128 ? launch_mlp_rows_tc_split_h<128>(c, n, x, x_stride, y0, y1, y2, net, tail)
                       : launch_mlp_rows_tc_split_h<64>(c, n, x, x_stride, y0, y1, y2, net, tail);
}

// ---------------------------------------------------------------------------------------------
// a2-a9 fused step, tensor-core operator.  P.op = 0: VHS-NN (eqs. 1-5), P.op = 2: chi-MLP + rotation.
// ---------------------------------------------------------------------------------------------
template <int H, bool SPLIT, class CK>
__device__ __forceinline__ void pairs_tc(const StepParams &P, const MlpTcDev &net, CK &S, TcEngine<H, SPLIT> &eng,
                                         int q0) {
  const int tid = threadIdx.x;
  const int n_pairs = S.misc[MI_NPAIRS];
  for (int t0 = 0; t0 < n_pairs; t0 += 128) {
    PairCtx c;
    const bool mine = tid < 128 && t0 + tid < n_pairs;
    if (tid < 128) {
      float x[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = 0.f;
      if (mine) {
        c = pair_setup(P, S, t0 + tid, P.op != 0);
        if (P.op == 0) {  // VHS-NN features (eqs. 1-3, Q1-Q3)
          float n0 = 0.f, n1 = 0.f, n2 = 0.f;
          if (P.flags & DSMC_F_NOISE) {
            const uint4 r = philox4x32_10((uint32_t)c.s, c.cell + P.cell_base, P.step, 2u, P.seed_lo, P.seed_hi);
            box_muller3(r, n0, n1, n2);
            n0 *= P.noise_sigma; n1 *= P.noise_sigma; n2 *= P.noise_sigma;
          }
          x[0] = c.gx * P.inv_sigma_v; x[1] = c.gy * P.inv_sigma_v; x[2] = c.gz * P.inv_sigma_v;
          if (net.d_in == 8) {
            const CellInfo &ci = S.cells[c.a];
            x[3] = sqrtf(c.g2) * P.inv_sigma_v;
            x[4] = ci.theta * P.T_coef / (float)ci.N * P.inv_T_scale;  // T = m Theta / (3 kB N)
            x[5] = n0; x[6] = n1; x[7] = n2;
          } else {
            x[3] = n0; x[4] = n1; x[5] = n2;
          }
        } else {  // chi-MLP inputs (Q15)
          const float e = (logf(P.e_coef * c.g2) - P.lnE_min) * P.inv_lnE_range;
          x[0] = !(e > 0.f) ? 0.f : fminf(e, 1.f);
          x[1] = sqrtf(c.U_b);
        }
      }
      eng.write_a1_row(tid, x);
    }
    eng.run(net.act);
    if (tid < 128) {
      float y[4];
      eng.read_out(y);
      if (mine) {
        float px = c.gx, py = c.gy, pz = c.gz, aux = 0.f;
        if (c.acc) {
          if (P.op == 0) {
            const float hn = sqrtf(y[0] * y[0] + y[1] * y[1] + y[2] * y[2]);
            aux = hn;
            if (P.flags & DSMC_F_ENERGY_SHELL) {
              if (hn >= P.shell_eps) {  // eq. 5 with the guard of Q4
                const float sc = sqrtf(c.g2) / hn;
                px = sc * y[0]; py = sc * y[1]; pz = sc * y[2];
              }
            } else {
              px = P.sigma_v * y[0]; py = P.sigma_v * y[1]; pz = P.sigma_v * y[2];
            }
          } else {
            aux = __expf(y[0]);  // chi = expm1(softplus(z)) = exp(z)
            if (c.g2 > 0.f) rotate_fast(c, aux, c.U_eps, px, py, pz);
          }
        }
        pair_commit(P, S, c, px, py, pz, aux, q0);
      }
    }
    tc::fence_before();
  }
}

template <int H, bool SPLIT, int LMAX, int AMAX, bool DEFERRED, int MINB>
__global__ void __launch_bounds__(kThreads, MINB) k_collide_tc(const StepParams P, const MlpTcDev net) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ int s_next;
  using CK = Chunk<LMAX, AMAX>;
  CK S;
  unsigned char *rest = S.carve(smem_raw);
  TcEngine<H, SPLIT> eng;
  eng.init(align128(rest), net.w_blob);
  const int n_work = DEFERRED ? *reinterpret_cast<volatile const int32_t *>(P.big) : P.n_chunks;
  for (;;) {
    if (threadIdx.x == 0) s_next = atomicAdd(P.work + (DEFERRED ? 1 : 0), 1);
    __syncthreads();
    const int w = s_next;
    __syncthreads();
    if (w >= n_work) break;
    const int chunk = DEFERRED ? P.big[1 + w] : w;
    const Team T{(int)threadIdx.x, 0};
    int q0 = 0;
    const int n_loc = chunk_begin(T, P, S, chunk, q0);
    if (n_loc == 0) continue;
    if (n_loc < 0) {
      if (threadIdx.x == 0) {
        if (DEFERRED) {
          *P.status = DSMC_ERR_CELL_TOO_LARGE;
        } else {
          const int i = atomicAdd(P.big, 1);
          P.big[1 + i] = chunk;
        }
      }
      continue;
    }
    chunk_pre_and_sort(T, P, S, n_loc);
    pairs_tc<H, SPLIT>(P, net, S, eng, q0);
    __syncthreads();
    chunk_finish(T, P, S, n_loc, q0);
    __syncthreads();
  }
  eng.teardown();
}

template <int H, bool SPLIT, int LMAX, int AMAX, bool DEFERRED, int MINB>
static int launch_tc_one(dsmc_ctx *c, const StepParams &p, const MlpTcDev &net, int grid) {
  auto kern = k_collide_tc<H, SPLIT, LMAX, AMAX, DEFERRED, MINB>;
  const size_t smem = Chunk<LMAX, AMAX>::bytes() + TcShape<H, SPLIT>::SMEM_BYTES + 256;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return DSMC_ERR_CUDA;
  kern<<<grid, kThreads, smem, c->stream>>>(p, net);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

template <int H, bool SPLIT>
static int launch_tc_pair(dsmc_ctx *c, const StepParams &p, const MlpTcDev &net) {
  constexpr int per_sm = (SPLIT && H == 128) ? 1 : 2;
  const int g_main = std::min(p.n_chunks, c->num_sms * per_sm), g_big = c->num_sms;
  int rc = launch_tc_one<H, SPLIT, kLmaxSmall, kAmaxSmall, false, per_sm>(c, p, net, g_main);
  if (rc != DSMC_OK) return rc;
  return launch_tc_one<H, SPLIT, kLmaxBig, kAmaxBig, true, 1>(c, p, net, g_big);
}

int launch_collide_tc(dsmc_ctx *c, const StepParams &p_in, const MlpTcDev *net) {
  if (p_in.op == 0 && !((net->d_in == 8 || net->d_in == 6) && net->d_out == 3 && net->n_hidden == 2)) return DSMC_ERR_UNSUPPORTED_SHAPE;
  if (p_in.op == 2 && (p_in.flags & DSMC_F_TC_ONE_KERNEL) && net->n_hidden != 2) return DSMC_ERR_UNSUPPORTED_SHAPE;
  if (p_in.op == 2 && !(net->d_in == 2 && net->d_out == 1)) return DSMC_ERR_UNSUPPORTED_SHAPE;
  // plain BF16 chi-MLP: three passes at full occupancy (dsmc_cells.cu), or, with DSMC_F_TC_ONE_KERNEL, the single kernel
  // of cell teams + MLP server (dsmc_cells_mlp.cu)
  if (p_in.op == 2 && (p_in.flags & DSMC_F_PAIR_REPLACE)) return launch_collide_replace_split(c, p_in, net);
  if (p_in.op == 2)
    return (p_in.flags & DSMC_F_TC_ONE_KERNEL) ? launch_collide_cells_mlp(c, p_in, net) : launch_collide_cells_split(c, p_in, net);
  // VHS-NN: the split form (dsmc_collide.cu) unless the one-kernel form is asked for
  if (p_in.op == 0 && (p_in.flags & DSMC_F_PAIR_REPLACE)) return launch_collide_vhs_replace_split(c, p_in, net);
  if (p_in.op == 0 && !(p_in.flags & DSMC_F_TC_ONE_KERNEL)) return launch_collide_cells_vhs_split(c, p_in, net);
  StepParams p = p_in;
  int rc = launch_chunk_map(c, p);
  if (rc != DSMC_OK) return rc;
  if (p.op == 0)  // VHS-NN: split-BF16 operands (eq. 5 conditioning, Q21)
    return net->H == 128 ? launch_tc_pair<128, true>(c, p, *net) : launch_tc_pair<64, true>(c, p, *net);
  return net->H == 128 ? launch_tc_pair<128, false>(c, p, *net) : launch_tc_pair<64, false>(c, p, *net);
}

}  // namespace dsmc
