// Fused collision step with the chi-MLP on the tensor cores, cell-team form.
//
// One persistent CTA per SM holds two kinds of warps that never meet at a CTA-wide barrier after start-up:
//
//   team warps (NTW)   the cell teams of dsmc_cells.cuh (a warp per cell of up to 256 particles, groups of 4 / 8
//                      warps on named barriers for cells of up to 1024 / 2048), each with TWO cell buffers.  After
//                      the key sort every warp owns up to 128 pair slots = one 128-row tile of the MLP: it stages the
//                      two features of every row, takes the next tile number, writes them (split BF16: hi | lo | hi)
//                      into that tile's layer-1 operand and publishes it; then it starts on its next cell in the
//                      other buffer and only afterwards sleeps until z of the first tile has been delivered into its
//                      shared memory, rotates, commits, matches and stores as in the table kernel.
//   MLP server         two independent pipelines, one per tensor-memory slot (tile t runs in slot t & 1): an MMA
//                      issue warp and NA / 2 activation warps each, around the operands of dsmc_tc_pipe.cuh.  Layer 1
//                      from shared memory (SS), layer 2 with the activations kept in tensor memory (TS); the output
//                      layer (d_out = 1) is NOT a third tensor-core layer: the warps that apply the second activation
//                      form z = b3 + sum_j w3[j] act(D[row][j]) on the CUDA cores (FP32 weights as constant-bank
//                      operands) and add their partial sums into the feeding warp's shared memory -- one hand-off
//                      (tensor core -> activation warps -> delivery warps) and its ~1300 cycles per tile are gone.
//                      Every wait is a blocking mbarrier wait on the data it needs; a slot never looks at the other
//                      one, so nothing has to be injected when one of them runs dry, and each MMA warp stops when
//                      every team warp has finished and its next tile number was never taken.
//
// Measured on cfg 5: with the activations switched off the kernel still takes 0.98 ms -- twelve
// team warps per SM (shared memory: two cell buffers each beside 82 KB of weights and operands) are latency-bound at
// ~35 000 cycles per cell -- and the server's chain per tile (activation 1, layer 2, activation 2, layer 1 of the next
// tile) is ~8 000 cycles per slot.  Both sides run at about the same pace, which is why variants of either one alone
// (lock-step rounds, an XU-pipe lock between the slots, 20 single-buffered team warps with 8 activation warps) all
// land within 4 % of one another.
#include <algorithm>

#include "dsmc_cells.cuh"
#include "dsmc_tc_pipe.cuh"

namespace dsmc {


constexpr int kMlpMaxFeeders = 32;


// Hand-offs between the team warps and the server.  Tiles are numbered by a ticket t: tile t runs in tensor-memory
// slot s = t & 1 and is the k-th tile of that slot, k = t >> 1; its layer-1 operand lives in buffer par = k & 1 of the
// slot, so its rows can be written while tile k - 1 of the slot is still in the layers (the buffer was last read by
// layer 1 of tile k - 2).  Every wait sleeps on an mbarrier; nothing spins on a lock.
struct CellsMlpCtl {
  uint64_t in_bar[2][2];               // rows of the tile in (slot, par) are written            (1 arrival)
  uint64_t op_bar[2];                  // one phase per finished layer 1 of the slot            (1 arrival)
  uint64_t done_bar[2 * kMlpMaxFeeders];  // [feeding warp][its buffer]: one phase per delivered tile (NA / 2 arrivals);
                                          // one tile in flight per barrier, so a phase parity identifies it
  float *dest[2][4];                   // where the outputs of tile k of the slot go (ring: entry k & 3 is rewritten
  int feeder[2][4];                    // for tile k + 4, after tile k has been delivered), and who waits for them
  int op_done[2];                      // finished layer 1s of the slot
  int ticket;
  int done;                            // team warps that ran out of work
  int stop_k[2];                       // per slot: the tile index at which its server warps stop (set by its MMA warp)
};

// warp-uniform test of an mbarrier phase (lanes may observe the completion at different times)
__device__ __forceinline__ bool cm_test(uint64_t *bar, uint32_t parity) {
  return __any_sync(0xffffffffu, tc::mbar_test(bar, parity));
}
__device__ __forceinline__ int cm_ld_volatile(const int *p) { return *reinterpret_cast<const volatile int *>(p); }
__device__ __forceinline__ void cm_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc::smem_u32(bar)) : "memory");
}
// one try_wait: sleeps in hardware until the phase completes or a time limit passes; true if completed
__device__ __forceinline__ bool cm_try_wait_ns(uint64_t *bar, uint32_t parity, uint32_t ns) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.b32 %0, 1, 0, p;\n\t}\n"
      : "=r"(ok)
      : "r"(tc::smem_u32(bar)), "r"(parity), "r"(ns)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ bool cm_try_wait(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.b32 %0, 1, 0, p;\n\t}\n"
      : "=r"(ok)
      : "r"(tc::smem_u32(bar)), "r"(parity), "r"(20000u)  // suspend-time hint [ns]: sleep, do not poll
      : "memory");
  return ok != 0;
}

// what a team warp sees of the server
template <int H>
struct CellsMlpFeeder {
  using SH = PipeShape<H>;
  unsigned char *a1;  // layer-1 operands: [slot][par]
  CellsMlpCtl *ctl;
  int me;             // feeding warp
  int buf;            // which of the team's two buffers the current call is about (set by CellTeam::run2)
  uint32_t ph_done;   // bit b: phase of done_bar[2 me + b] this warp waits for next

  // takes the next tile number; returns (slot | par << 1) once that layer-1 operand buffer may be written; z of the
  // tile's 128 rows will land in zbuf
  __device__ __forceinline__ int acquire(int lane, uint32_t *zbuf) {
    int sp = 0;
    if (lane == 0) {
      const int t = atomicAdd(&ctl->ticket, 1);
      const int s = t & 1, k = t >> 1, par = k & 1;
      for (;;) {  // layer 1 of tile k - 2 of this slot has read the buffer
        const int r = cm_ld_volatile(&ctl->op_done[s]);
        if (r >= k - 1) break;
        cm_try_wait(&ctl->op_bar[s], (uint32_t)r & 1u);
      }
      *reinterpret_cast<float *volatile *>(&ctl->dest[s][k & 3]) = reinterpret_cast<float *>(zbuf);
      *reinterpret_cast<volatile int *>(&ctl->feeder[s][k & 3]) = 2 * me + buf;
      sp = s | (par << 1);
    }
    return __shfl_sync(0xffffffffu, sp, 0);
  }
  // row r of the operand: [x_hi | x_lo | x_hi | 1 1 0 ...]; only the three feature words change (the rest of the
  // operand is written once when the kernel starts)
  __device__ __forceinline__ void write_row(int sp, int r, float x0, float x1) {
    const uint32_t hi = tc::pack_bf16(x0, x1);
    const uint32_t lo = tc::pack_bf16(x0 - __uint_as_float(hi << 16), x1 - __uint_as_float(hi & 0xFFFF0000u));
    unsigned char *a = a1 + (2 * (sp & 1) + (sp >> 1)) * SH::A1_BYTES + r * 16;
    *reinterpret_cast<uint32_t *>(a) = hi;
    *reinterpret_cast<uint32_t *>(a + 1 * 128 * 16) = lo;
    *reinterpret_cast<uint32_t *>(a + 2 * 128 * 16) = hi;
  }
  __device__ __forceinline__ void publish(int sp) {
    tc::fence_proxy_async();
    __syncwarp();
    if ((threadIdx.x & 31) == 0) cm_arrive(&ctl->in_bar[sp & 1][sp >> 1]);
  }
  __device__ __forceinline__ void wait(int lane) {
    while (!cm_try_wait(&ctl->done_bar[2 * me + buf], (ph_done >> buf) & 1u)) {
    }
    ph_done ^= 1u << buf;
  }
};

template <int H, int NA, int NTW, int NBUF>
__global__ void __launch_bounds__((NTW + NA + 2) * 32, 1) k_cells_mlp(const StepParams P, const CellLists Lst,
                                                                      const MlpTcDev net, const TcOutLayer W3) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  using SH = PipeShape<H>;
  using Feeder = CellsMlpFeeder<H>;
  constexpr size_t SLICE = CellTeam<32>::bytes();
  constexpr size_t TEAMS = (NBUF * NTW * SLICE + 127) & ~(size_t)127;  // NBUF cells in flight per team
  unsigned char *pipe_base = smem_raw + TEAMS;
  CellsMlpCtl *ctl = reinterpret_cast<CellsMlpCtl *>(pipe_base + SH::SMEM_BYTES);
  TcPipe<H> pipe;
  if (threadIdx.x == 0) {
    for (int s2 = 0; s2 < 2; ++s2) {
      tc::mbar_init(&ctl->in_bar[s2][0], 1);
      tc::mbar_init(&ctl->in_bar[s2][1], 1);
      tc::mbar_init(&ctl->op_bar[s2], 1);
      ctl->op_done[s2] = 0;
    }
    for (int f = 0; f < 2 * kMlpMaxFeeders; ++f) tc::mbar_init(&ctl->done_bar[f], NA / 2);
    ctl->ticket = 0;
    ctl->stop_k[0] = ctl->stop_k[1] = 0x7FFFFFFF;
    ctl->done = 0;
    tc::mbar_fence_init();
  }
  pipe.init(pipe_base, net.w_blob, NA / 2, 1);  // eight activation warps per slot; ends with CTA-wide barriers
  // constant part of the layer-1 operands (zeros and the bias column block), both slots
  for (int i = threadIdx.x; i < 4 * 128; i += (NTW + NA + 2) * 32) {
    unsigned char *a = pipe.a1 + (i >> 7) * SH::A1_BYTES + (i & 127) * 16;
#pragma unroll
    for (int j = 0; j < 3; ++j) *reinterpret_cast<uint4 *>(a + j * 128 * 16) = make_uint4(0u, 0u, 0u, 0u);
    *reinterpret_cast<uint4 *>(a + 3 * 128 * 16) = make_uint4(0x3F803F80u, 0u, 0u, 0u);
  }
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // the team warps come first (NTW is a multiple of 4): activation warp aw reads the tensor-memory lanes
  // 32 (aw & 3) .., which the hardware ties to (warp index & 3); and the scheduler prefers the higher warp indices,
  // which keeps the server ahead of the teams that feed it
  static_assert(NTW % 4 == 0, "activation warps must start at a multiple of four");
  const int tw = warp, ttid = (int)threadIdx.x;  // team warp / thread

  if (tw < NTW) {
    // ---------------- cell teams ----------------
    Feeder srv{pipe.a1, ctl, tw, 0, 0u};
    const uint32_t base_s = (uint32_t)__cvta_generic_to_shared(smem_raw);
    constexpr int G8 = NTW / 8, G4 = NTW / 4;
    {
    if (tw < 8 * G8) {  // cells of 1025..2048 particles: groups of eight warps
      const int g = tw >> 3;
      CellTeam<256, 2, Feeder> T;
      const uint32_t b0 = base_s + (uint32_t)(8 * NBUF * g * SLICE);
      T.init(b0, ttid - 256 * g, 1 + g);
      T.srv = &srv;
      if (NBUF == 2) T.run2(P, Lst.list[2], Lst.ctr + 2, Lst.work + 2, b0, b0 + (uint32_t)(8 * SLICE));
      else T.run(P, Lst.list[2], Lst.ctr + 2, Lst.work + 2);
      asm volatile("bar.sync %0, 256;" ::"r"(1 + g) : "memory");
    }
    if (tw < 4 * G4) {  // cells of 257..1024 particles: groups of four warps
      const int g = tw >> 2;
      CellTeam<128, 2, Feeder> T;
      const uint32_t b0 = base_s + (uint32_t)(4 * NBUF * g * SLICE);
      T.init(b0, ttid - 128 * g, 1 + G8 + g);
      T.srv = &srv;
      if (NBUF == 2) T.run2(P, Lst.list[1], Lst.ctr + 1, Lst.work + 1, b0, b0 + (uint32_t)(4 * SLICE));
      else T.run(P, Lst.list[1], Lst.ctr + 1, Lst.work + 1);
      asm volatile("bar.sync %0, 128;" ::"r"(1 + G8 + g) : "memory");
    }
    {
      CellTeam<32, 2, Feeder> T;
      const uint32_t b0 = base_s + (uint32_t)(NBUF * tw * SLICE);
      T.init(b0, lane, 0);
      T.srv = &srv;
      if (NBUF == 2) T.run2(P, Lst.list[0], Lst.ctr + 0, Lst.work + 0, b0, b0 + (uint32_t)SLICE);
      else T.run(P, Lst.list[0], Lst.ctr + 0, Lst.work + 0);
    }
    }
    if (lane == 0) {
      __threadfence_block();
      atomicAdd(&ctl->done, 1);
    }
  } else if (warp < NTW + NA) {
    // ---------------- MLP server: activation + delivery warps ----------------
    // Two independent pipelines, one per slot: activation warp aw serves slot (aw >> 2) & 1 (eight warps per slot: the
    // four lane quadrants x two column halves), walks that slot's tiles k = 0, 1, ... on blocking waits and never
    // looks at the other slot.  While one group waits for its tensor-core layer or delivers, the other has the XU
    // pipe to itself, so the latencies of one slot's hand-offs hide behind the other slot's activations.
    const int aw = warp - NTW;
    const int s2 = (aw >> 2) & 1, q = aw & 3, half = aw >> 3;
    const int aw_slot = q | (half << 2);  // act_body: lane quadrant = aw_slot & 3, column group = aw_slot >> 2
    constexpr int NQ = NA / 8;  // column groups per slot
    uint32_t phe = 0u;
    for (int k = 0;; ++k) {
      // ---- hidden layer 1: D -> activation -> bf16 A operand of layer 2 (tensor memory) ----
      tc::mbar_wait(pipe.full_e + s2, phe);
      phe ^= 1u;
      if (k == cm_ld_volatile(&ctl->stop_k[s2])) goto server_done;
      if (aw_slot == 0 && lane == 0) {  // the slot's layer-1 operand buffer may be rewritten
        *reinterpret_cast<volatile int *>(&ctl->op_done[s2]) = k + 1;
        __threadfence_block();
        cm_arrive(&ctl->op_bar[s2]);
      }
      __syncwarp();
      pipe.template act_body<NQ>(net.act, s2, aw_slot);
      // ---- hidden layer 2 and the output layer (d_out = 1) in one pass: z = b3 + sum_j w3[j] act(D[row][j]) on the
      // CUDA cores, so no third tensor-core layer and no hand-off for it; the two column groups of a row add their
      // partial sums into the feeding warp's (zeroed) buffer: x + y = y + x, the result does not depend on the order
      tc::mbar_wait(pipe.full_e + s2, phe);
      phe ^= 1u;
      float *dest = *reinterpret_cast<float *volatile *>(&ctl->dest[s2][k & 3]);
      const int f = cm_ld_volatile(&ctl->feeder[s2][k & 3]);
      {
        tc::fence_after();
        const uint32_t d0 = pipe.tmem + (((uint32_t)(q * 32)) << 16) + s2 * SH::SLOT_COLS + SH::COL_D + half * (H / NQ);
        float part;
        if (net.act == DSMC_ACT_SILU)
          part = half == 0 ? tc_out_partial<H, NQ, 0, DSMC_ACT_SILU>(d0, W3) : tc_out_partial<H, NQ, 1, DSMC_ACT_SILU>(d0, W3);
        else if (net.act == DSMC_ACT_TANH)
          part = half == 0 ? tc_out_partial<H, NQ, 0, DSMC_ACT_TANH>(d0, W3) : tc_out_partial<H, NQ, 1, DSMC_ACT_TANH>(d0, W3);
        else
          part = half == 0 ? tc_out_partial<H, NQ, 0, DSMC_ACT_RELU>(d0, W3) : tc_out_partial<H, NQ, 1, DSMC_ACT_RELU>(d0, W3);
        tc::fence_before();
        asm volatile("red.shared.add.f32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(dest + q * 32 + lane)), "f"(part)
                     : "memory");
      }
      __syncwarp();
      if (lane == 0) {
        __threadfence_block();
        asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc::smem_u32(pipe.a_ready + s2)) : "memory");  // D may be overwritten
        cm_arrive(&ctl->done_bar[f]);  // this warp's share of z is in the feeding warp's shared memory
      }
    }
  } else {
    // ---------------- MLP server: one MMA issue warp per slot ----------------
    const int s2 = warp - NTW - NA;
    uint32_t pa = 0u;
    for (int k = 0;; ++k) {
      // rows of tile t = 2 k + s2: wait for them; stop when nobody has taken that number and nobody will
      const int t = 2 * k + s2;
      uint64_t *bar = &ctl->in_bar[s2][k & 1];
      const uint32_t par = (uint32_t)(k >> 1) & 1u;
      bool stop = false;
      for (;;) {
        if (cm_try_wait_ns(bar, par, 2000u)) break;
        int st = 0;
        if (lane == 0) {
          const int d = cm_ld_volatile(&ctl->done);      // read first: once every team warp has finished ...
          const int tk = cm_ld_volatile(&ctl->ticket);   // ... no tile number is taken any more
          st = (d == NTW && tk <= t) ? 1 : 0;
        }
        if (__shfl_sync(0xffffffffu, st, 0)) {
          stop = true;
          break;
        }
      }
      if (stop) {
        if (lane == 0) {
          *reinterpret_cast<volatile int *>(&ctl->stop_k[s2]) = k;
          __threadfence_block();
        }
        __syncwarp();
        pipe.issue_layer1(s2, k & 1, k == 0);  // an empty one: it wakes the slot's activation warps, which then stop
        break;
      }
      pipe.issue_layer1(s2, k & 1, k == 0);
      tc::mbar_wait(pipe.a_ready + s2, pa);
      pa ^= 1u;
      pipe.issue_layer2(s2);
      tc::mbar_wait(pipe.a_ready + s2, pa);  // the second activation has read D: the next tile's layer 1 may go
      pa ^= 1u;
    }
  }
server_done:
  pipe.teardown();
}

void launch_cell_lists(dsmc_ctx *c, const StepParams &p, CellLists &L);  // dsmc_cells.cu

template <int H, int NA, int NTW, int NBUF>
static int launch_cells_mlp_one(dsmc_ctx *c, const StepParams &p, const CellLists &L, const MlpTcDev &net,
                               const TcOutLayer &w3) {
  auto kern = k_cells_mlp<H, NA, NTW, NBUF>;
  const size_t smem = ((NBUF * NTW * CellTeam<32>::bytes() + 127) & ~(size_t)127) + PipeShape<H>::SMEM_BYTES +
                      sizeof(CellsMlpCtl) + 128;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return DSMC_ERR_CUDA;
  kern<<<c->num_sms, (NTW + NA + 2) * 32, smem, c->stream>>>(p, L, net, w3);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

// op 2 (ab initio chi-MLP), plain BF16 operands
int launch_collide_cells_mlp(dsmc_ctx *c, const StepParams &p, const MlpTcDev *net) {
  if (p.op != 2 || net->d_in != 2 || net->d_out != 1 || (net->H != 64 && net->H != 128))
    return DSMC_ERR_UNSUPPORTED_SHAPE;
  CellLists L;
  launch_cell_lists(c, p, L);
  const TcOutLayer w3 = tc_out_layer(*net);
  if (net->H == 128) return launch_cells_mlp_one<128, 16, 12, 2>(c, p, L, *net, w3);
  return launch_cells_mlp_one<64, 16, 12, 2>(c, p, L, *net, w3);
}

}  // namespace dsmc
