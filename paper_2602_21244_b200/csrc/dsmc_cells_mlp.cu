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
//   MLP server         NA activation warps + one MMA warp around the two-slot tcgen05 pipeline of dsmc_tc_pipe.cuh:
//                      layer 1 from shared memory (SS), layers 2 and 3 with the activations kept in tensor memory (TS).
//                      Tile t runs in slot t & 1; a ROUND is the two tiles 2 r, 2 r + 1 and both kinds of server warps
//                      walk the rounds in a fixed order on blocking mbarrier waits (a wake-up costs ~60 cycles, a poll
//                      ~150: measured, profiles/r02_*).  The first four activation warps deliver the layer-3 outputs.
//                      The MMA warp fills slot 1 with an empty tile when nobody feeds it (so that a tile in slot 0 is
//                      never held back), and stops the server when every team warp has finished.
//
// The server is bound by the XU pipe (one MUFU per hidden activation); the team warps exist to keep its two slots
// full, so their own latencies (HBM loads, waiting for z) cost nothing as long as enough tiles are in flight.
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
  uint64_t out_bar[2];                 // one phase per delivered tile of the slot              (4 arrivals)
  uint64_t done_bar[2 * kMlpMaxFeeders];  // [feeding warp][its buffer]: one phase per delivered tile (4 arrivals);
                                          // one tile in flight per barrier, so a phase parity identifies it
  float *dest[2][4];                   // where the outputs of tile k of the slot go (ring: entry k & 3 is rewritten
  int feeder[2][4];                    // for tile k + 4, after tile k has been delivered), and who waits for them
  int op_done[2];                      // finished layer 1s of the slot
  int ticket;
  int done;                            // team warps that ran out of work
  int poison;                          // the round after the last one with real tiles (set by the last team warp)
  float scratch[128];                  // outputs of empty tiles
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

template <int H, int NA, int NTW>
__global__ void __launch_bounds__((NTW + NA + 1) * 32, 1) k_cells_mlp(const StepParams P, const CellLists Lst,
                                                                      const MlpTcDev net) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  using SH = PipeShape<H>;
  using Feeder = CellsMlpFeeder<H>;
  constexpr size_t SLICE = CellTeam<32>::bytes();
  constexpr size_t TEAMS = (2 * NTW * SLICE + 127) & ~(size_t)127;  // two buffers per team
  unsigned char *pipe_base = smem_raw + TEAMS;
  CellsMlpCtl *ctl = reinterpret_cast<CellsMlpCtl *>(pipe_base + SH::SMEM_BYTES);
  TcPipe<H> pipe;
  if (threadIdx.x == 0) {
    for (int s2 = 0; s2 < 2; ++s2) {
      tc::mbar_init(&ctl->in_bar[s2][0], 1);
      tc::mbar_init(&ctl->in_bar[s2][1], 1);
      tc::mbar_init(&ctl->op_bar[s2], 1);
      tc::mbar_init(&ctl->out_bar[s2], 4);
      ctl->op_done[s2] = 0;
    }
    for (int f = 0; f < 2 * kMlpMaxFeeders; ++f) tc::mbar_init(&ctl->done_bar[f], 4);
    ctl->ticket = 0;
    ctl->poison = 0x7FFFFFFF;
    ctl->done = 0;
    tc::mbar_fence_init();
  }
  pipe.init(pipe_base, net.w_blob, NA, 1);  // one feeding warp per tile; ends with CTA-wide barriers
  // constant part of the layer-1 operands (zeros and the bias column block), both slots
  for (int i = threadIdx.x; i < 4 * 128; i += (NTW + NA + 1) * 32) {
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
      T.init(base_s + (uint32_t)(16 * g * SLICE), ttid - 256 * g, 1 + g);
      T.srv = &srv;
      T.run2(P, Lst.list[2], Lst.ctr + 2, Lst.ctr + 4 + 2, base_s + (uint32_t)(16 * g * SLICE), base_s + (uint32_t)((16 * g + 8) * SLICE));
      asm volatile("bar.sync %0, 256;" ::"r"(1 + g) : "memory");
    }
    if (tw < 4 * G4) {  // cells of 257..1024 particles: groups of four warps
      const int g = tw >> 2;
      CellTeam<128, 2, Feeder> T;
      T.init(base_s + (uint32_t)(8 * g * SLICE), ttid - 128 * g, 1 + G8 + g);
      T.srv = &srv;
      T.run2(P, Lst.list[1], Lst.ctr + 1, Lst.ctr + 4 + 1, base_s + (uint32_t)(8 * g * SLICE), base_s + (uint32_t)((8 * g + 4) * SLICE));
      asm volatile("bar.sync %0, 128;" ::"r"(1 + G8 + g) : "memory");
    }
    {
      CellTeam<32, 2, Feeder> T;
      T.init(base_s + (uint32_t)(2 * tw * SLICE), lane, 0);
      T.srv = &srv;
      T.run2(P, Lst.list[0], Lst.ctr + 0, Lst.ctr + 4 + 0, base_s + (uint32_t)(2 * tw * SLICE), base_s + (uint32_t)((2 * tw + 1) * SLICE));
    }
    }
    if (lane == 0) {
      __threadfence_block();
      atomicAdd(&ctl->done, 1);
    }
  } else if (warp < NTW + NA) {
    // ---------------- MLP server: activation + delivery warps ----------------
    // Fixed order, blocking waits (as in k_chi_batch_tc): round r = tiles 2 r (slot 0) and 2 r + 1 (slot 1).
    const int aw = warp - NTW;
    uint32_t phe[2] = {0u, 0u}, pho[2] = {0u, 0u};
    bool pend1 = false;  // slot 1 of the previous round is still to be delivered
    // rows 32 aw .. 32 aw + 31 of the layer-3 output of tile (slot s2, round rr) -> the feeding warp (aw < 4)
    auto deliver = [&](int s2, int rr) {
      tc::mbar_wait(pipe.full_o + s2, pho[s2]);
      pho[s2] ^= 1u;
      tc::fence_after();
      uint32_t v[4];
      tc::tmem_ld4(pipe.tmem + (((uint32_t)(aw * 32)) << 16) + s2 * SH::SLOT_COLS + SH::COL_OUT, v);
      tc::wait_ld();
      tc::fence_before();
      float *dest = *reinterpret_cast<float *volatile *>(&ctl->dest[s2][rr & 3]);
      const int f = cm_ld_volatile(&ctl->feeder[s2][rr & 3]);
      dest[aw * 32 + lane] = __uint_as_float(v[0]);
      __syncwarp();
      if (lane == 0) {
        __threadfence_block();
        cm_arrive(&ctl->out_bar[s2]);  // the output columns may be overwritten (layer 3 of the next round)
        cm_arrive(&ctl->done_bar[f]);  // z is in the feeding warp's shared memory
      }
    };
    // Order of a round: act(0, L1), [deliver slot 1 of the previous round], act(1, L1), act(0, L2), act(1, L2),
    // deliver slot 0.  Slot 1's layer 3 is issued only when act(1, L2) ends, so its delivery waits until the next
    // activation is done rather than hold up four of the activation warps.
    for (int r = 0;; ++r) {
#pragma unroll
      for (int layer = 0; layer < 2; ++layer) {
#pragma unroll
        for (int s2 = 0; s2 < 2; ++s2) {
          if (layer == 0 && s2 == 0 && aw < 4 && r >= 1) {
            // the next round normally stands ready (its layer 1 was issued early); if it does not, slot 1 of the last
            // round is delivered while waiting: a submitted tile never depends on further tiles being fed
            while (!cm_test(pipe.full_e + 0, phe[0])) {
              if (pend1 && cm_test(pipe.full_o + 1, pho[1])) {
                deliver(1, r - 1);
                pend1 = false;
              }
            }
          } else {
            tc::mbar_wait(pipe.full_e + s2, phe[s2]);
          }
          phe[s2] ^= 1u;
          if (layer == 0 && s2 == 0 && r == cm_ld_volatile(&ctl->poison)) {
            if (aw < 4 && pend1) deliver(1, r - 1);
            goto server_done;
          }
          if (layer == 0 && aw == 0 && lane == 0) {  // the slot's layer-1 operand buffer may be rewritten
            *reinterpret_cast<volatile int *>(&ctl->op_done[s2]) = r + 1;
            __threadfence_block();
            cm_arrive(&ctl->op_bar[s2]);
          }
          __syncwarp();
          pipe.template act_body<NA / 4>(net.act, s2, aw);
          if (layer == 0 && s2 == 0 && aw < 4 && pend1) {
            deliver(1, r - 1);
            pend1 = false;
          }
        }
      }
      if (aw < 4) {
        deliver(0, r);
        pend1 = true;
      }
    }
  } else {
    // ---------------- MLP server: MMA issue warp ----------------
    // layer 3 of both slots goes out before the warp waits for the rows of the next round, so every submitted tile
    // is delivered whatever the team warps do next
    uint32_t pa[2] = {0u, 0u};
    // Rows of tile 2 r + s2.  0: they are there.  1: nobody has taken that tile number and either every team warp has
    // finished or slot 1 has waited long enough while slot 0 holds a real tile: the warp takes the number itself and the
    // round runs with an empty tile in slot 1 (stale operand, outputs to nobody).  2 (slot 0 only): no tile will ever
    // come: stop.
    auto rows = [&](int s2, int r) -> int {
      const int t = 2 * r + s2;
      uint64_t *bar = &ctl->in_bar[s2][r & 1];
      const uint32_t par = (uint32_t)(r >> 1) & 1u;
      for (int it = 0;; ++it) {
        if (__any_sync(0xffffffffu, tc::mbar_test(bar, par))) return 0;
        int act = 0;
        if (lane == 0 && cm_ld_volatile(&ctl->ticket) == t) {
          const bool all_done = cm_ld_volatile(&ctl->done) == NTW;  // then no number is taken any more
          if (s2 == 0) {
            if (all_done && cm_ld_volatile(&ctl->ticket) == t) act = 2;
          } else if ((all_done || it > 8) && atomicCAS(&ctl->ticket, t, t + 1) == t) {
            *reinterpret_cast<float *volatile *>(&ctl->dest[s2][r & 3]) = ctl->scratch;
            *reinterpret_cast<volatile int *>(&ctl->feeder[s2][r & 3]) = 2 * kMlpMaxFeeders - 1;
            __threadfence_block();
            cm_arrive(bar);
            act = 1;
          }
        }
        act = __shfl_sync(0xffffffffu, act, 0);
        if (act) return act;
      }
    };
    bool first = true;
    if (rows(0, 0) == 2) {
      *reinterpret_cast<volatile int *>(&ctl->poison) = 0;
      __threadfence_block();
    }
    pipe.issue_layer1(0, 0, first);  // (an empty one when stopping: it wakes the activation warps)
    first = false;
    if (cm_ld_volatile(&ctl->poison) != 0) {
      rows(1, 0);
      pipe.issue_layer1(1, 0, false);
      for (int r = 0;; ++r) {
        // are the rows of the next round there already?  (asked now, while the activation warps work, because the
        // answer takes ~150 cycles; normally they are, and the round ends without looking again)
        const bool early0 = __any_sync(0xffffffffu, tc::mbar_test(&ctl->in_bar[0][(r + 1) & 1], (uint32_t)((r + 1) >> 1) & 1u));
        const bool early1 = __any_sync(0xffffffffu, tc::mbar_test(&ctl->in_bar[1][(r + 1) & 1], (uint32_t)((r + 1) >> 1) & 1u));
#pragma unroll
        for (int s2 = 0; s2 < 2; ++s2) {
          tc::mbar_wait(pipe.a_ready + s2, pa[s2]);
          pa[s2] ^= 1u;
          pipe.issue_layer2(s2);
        }
        bool stop = false;
#pragma unroll
        for (int s2 = 0; s2 < 2; ++s2) {
          tc::mbar_wait(pipe.a_ready + s2, pa[s2]);
          pa[s2] ^= 1u;
          if (r >= 1) tc::mbar_wait(&ctl->out_bar[s2], (uint32_t)(r - 1) & 1u);  // previous round delivered
          pipe.issue_layer3(s2);
          // slot 0's next layer 1 goes out ahead of slot 1's layer 3 when its rows are there (the usual case): the
          // activation warps then find work the moment they finish act(1, L2).  Otherwise it waits until both layer 3s
          // are out, so that every submitted tile is delivered whatever the team warps do next.
          if (s2 == (early0 ? 0 : 1)) {
            stop = !early0 && rows(0, r + 1) == 2;
            if (stop) {
              *reinterpret_cast<volatile int *>(&ctl->poison) = r + 1;
              __threadfence_block();
            }
            pipe.issue_layer1(0, (r + 1) & 1, false);
          }
        }
        if (stop) break;
        if (!early1) rows(1, r + 1);
        pipe.issue_layer1(1, (r + 1) & 1, false);
      }
    }
  }
server_done:
  pipe.teardown();
}

void launch_cell_lists(dsmc_ctx *c, const StepParams &p, CellLists &L);  // dsmc_cells.cu

template <int H, int NA, int NTW>
static int launch_cells_mlp_one(dsmc_ctx *c, const StepParams &p, const CellLists &L, const MlpTcDev &net) {
  auto kern = k_cells_mlp<H, NA, NTW>;
  const size_t smem = ((2 * NTW * CellTeam<32>::bytes() + 127) & ~(size_t)127) + PipeShape<H>::SMEM_BYTES +
                      sizeof(CellsMlpCtl) + 128;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return DSMC_ERR_CUDA;
  kern<<<c->num_sms, (NTW + NA + 1) * 32, smem, c->stream>>>(p, L, net);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

// op 2 (ab initio chi-MLP), plain BF16 operands
int launch_collide_cells_mlp(dsmc_ctx *c, const StepParams &p, const MlpTcDev *net) {
  if (p.op != 2 || net->d_in != 2 || net->d_out != 1 || (net->H != 64 && net->H != 128))
    return DSMC_ERR_UNSUPPORTED_SHAPE;
  CellLists L;
  launch_cell_lists(c, p, L);
  if (net->H == 128) return launch_cells_mlp_one<128, 16, 12>(c, p, L, *net);
  return launch_cells_mlp_one<64, 16, 12>(c, p, L, *net);
}

}  // namespace dsmc
