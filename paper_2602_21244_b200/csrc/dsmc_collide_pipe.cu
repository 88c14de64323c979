// Fused collision step with the chi-MLP on the tensor cores, warp-specialised (plain BF16 operands).
//
// One persistent CTA per SM.  Three kinds of warps, no CTA-wide barrier after start-up:
//
//   chunk groups (NG x 8 warps)  each group pulls chunks (dsmc_chunk.cuh) from the work counter and runs
//       the whole per-chunk path on its own shared-memory chunk: load, cell moments, Philox pairing keys
//       + sort (ALU work), then its pairs 128 at a time through the MLP server, then matching + store.
//       The two halves of a group (4 warps each) feed one tile each: features -> A1 rows of a free slot,
//       wait for the slot's layer-3 output, rotate + commit.
//   ACT warps (8)   MLP server, activation stage: whichever slot has a finished layer 1 / 2 in TMEM gets
//       D -> tanh/SiLU -> bf16 -> A operand (dsmc_tc_pipe.cuh act_body)
//   MMA warp (1)    MLP server, issue stage: a small state machine per slot issues layer 1 when a half
//       group has published its rows, layers 2 and 3 when the ACT warps have published the operand
//
// The ALU-bound chunk phases of one group overlap the XU/TMEM-bound MLP phases of the other, and the two
// TMEM slots keep the ACT warps busy while a UMMA of the other slot is in flight.  A slot is owned by one
// half group from acquire (before its rows are written) to release (after its outputs are read), so no
// operand or accumulator is ever reused while in flight.
#include <algorithm>

#include "dsmc_chunk.cuh"
#include "dsmc_tc_pipe.cuh"

namespace dsmc {

constexpr int kFuseActWarps = 8;
constexpr int fuse_threads(int ng) { return ng * kThreads + kFuseActWarps * 32 + 32; }

struct FuseCtl {
  int lock[2];     // slot ownership: 0 free, 1 taken
  int use_cnt[2];  // completed + current uses of the slot (parity of its full_o phase)
  int done;        // chunk groups that ran out of work
  int next[2];     // per group: chunk handed out by the work counter
  int slot_of[4];  // per half group: slot | phase parity << 1
};

__device__ __forceinline__ void half_sync(int id) { asm volatile("bar.sync %0, 128;" ::"r"(id) : "memory"); }
__device__ __forceinline__ int ld_volatile(const int *p) { return *reinterpret_cast<const volatile int *>(p); }

// the pairs of one chunk through the MLP server; called by all 256 threads of a group
template <int H, class CK>
__device__ __forceinline__ void pairs_pipe(const Team &T, int g, const StepParams &P, CK &S, TcPipe<H> &pipe,
                                           FuseCtl *ctl, int q0) {
  using SH = PipeShape<H>;
  const int hg = T.tid >> 7, r = T.tid & 127, hw = (T.tid >> 5) & 3;
  const int n_pairs = S.misc[MI_NPAIRS];
  const int bar_id = 3 + 2 * g + hg, me = 2 * g + hg;
  for (int t0 = hg * 128; t0 < n_pairs; t0 += 256) {
    const bool mine = t0 + r < n_pairs;
    PairCtx c;
    float x[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) x[k] = 0.f;
    if (mine) {  // chi-MLP inputs (Q15)
      c = pair_setup(P, S, t0 + r, true);
      const float e = (__logf(P.e_coef * c.g2) - P.lnE_min) * P.inv_lnE_range;
      x[0] = !(e > 0.f) ? 0.f : fminf(e, 1.f);
      x[1] = sqrtf(c.U_b);
    }
    if (r == 0) {  // take a free slot
      int s = -1;
      while (s < 0) {
        if (atomicCAS(&ctl->lock[0], 0, 1) == 0) s = 0;
        else if (atomicCAS(&ctl->lock[1], 0, 1) == 0) s = 1;
        else __nanosleep(64);
      }
      __threadfence_block();
      const int n = ld_volatile(&ctl->use_cnt[s]);
      *reinterpret_cast<volatile int *>(&ctl->use_cnt[s]) = n + 1;
      *reinterpret_cast<volatile int *>(&ctl->slot_of[me]) = s | ((n & 1) << 1);
    }
    half_sync(bar_id);
    const int sv = ld_volatile(&ctl->slot_of[me]);
    const int s = sv & 1;
    pipe.write_a1_row(s, 0, r, x);
    pipe.io_publish(s);
    tc::mbar_wait(pipe.full_o + s, (uint32_t)(sv >> 1));
    tc::fence_after();
    uint32_t v[4];
    tc::tmem_ld4(pipe.tmem + (((uint32_t)(hw * 32)) << 16) + s * SH::SLOT_COLS + SH::COL_OUT, v);
    tc::wait_ld();
    tc::fence_before();
    half_sync(bar_id);
    if (r == 0) {
      __threadfence_block();
      atomicExch(&ctl->lock[s], 0);
    }
    if (mine) {
      float px = c.gx, py = c.gy, pz = c.gz, chi = 0.f;
      if (c.acc) {
        chi = __expf(__uint_as_float(v[0]));  // chi = expm1(softplus(z)) = exp(z)
        if (c.g2 > 0.f) rotate_fast(c, chi, c.U_eps, px, py, pz);
      }
      pair_commit(P, S, c, px, py, pz, chi, q0);
    }
  }
}

template <int LMAX, int AMAX>
constexpr size_t chunk_region_bytes() {
  return (Chunk<LMAX, AMAX>::bytes() + 127) & ~(size_t)127;
}

template <int H, int LMAX, int AMAX, int NG, bool DEFERRED>
__global__ void __launch_bounds__(fuse_threads(NG), 1) k_collide_pipe(const StepParams P, const MlpTcDev net) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  using CK = Chunk<LMAX, AMAX>;
  unsigned char *base = smem_raw;  // dynamic shared memory starts 128-byte aligned (no static __shared__ here)
  unsigned char *pipe_base = base + NG * chunk_region_bytes<LMAX, AMAX>();
  FuseCtl *ctl = reinterpret_cast<FuseCtl *>(pipe_base + PipeShape<H>::SMEM_BYTES);
  TcPipe<H> pipe;
  if (threadIdx.x == 0) {
    ctl->lock[0] = ctl->lock[1] = 0;
    ctl->use_cnt[0] = ctl->use_cnt[1] = 0;
    ctl->done = 0;
  }
  pipe.init(pipe_base, net.w_blob, kFuseActWarps, 4);  // ends with CTA-wide barriers
  const int warp = threadIdx.x >> 5;

  if (warp < NG * 8) {
    // ---------------- chunk group ----------------
    const int g = warp >> 3;
    const Team T{(int)threadIdx.x - g * kThreads, 1 + g};
    CK S;
    S.carve(base + g * chunk_region_bytes<LMAX, AMAX>());
    const int n_work = DEFERRED ? ld_volatile(P.big) : P.n_chunks;
    for (;;) {
      if (T.tid == 0) *reinterpret_cast<volatile int *>(&ctl->next[g]) = atomicAdd(P.work + (DEFERRED ? 1 : 0), 1);
      T.sync();
      const int w = ld_volatile(&ctl->next[g]);
      T.sync();
      if (w >= n_work) break;
      const int chunk = DEFERRED ? P.big[1 + w] : w;
      int q0 = 0;
      const int n_loc = chunk_begin(T, P, S, chunk, q0);
      if (n_loc == 0) continue;
      if (n_loc < 0) {
        if (T.tid == 0) {
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
      pairs_pipe<H>(T, g, P, S, pipe, ctl, q0);
      T.sync();
      chunk_finish(T, P, S, n_loc, q0);
      T.sync();
    }
    if (T.tid == 0) {
      __threadfence_block();
      atomicAdd(&ctl->done, 1);
    }
  } else if (warp < NG * 8 + kFuseActWarps) {
    // ---------------- MLP server: activation warps ----------------
    const int aw = warp - NG * 8;
    uint32_t ph0 = 0, ph1 = 0;
    for (;;) {
      bool any = false;
      if (tc::mbar_test(pipe.full_e + 0, ph0)) {
        ph0 ^= 1u;
        pipe.template act_body<kFuseActWarps / 4>(net.act, 0, aw);
        any = true;
      }
      if (tc::mbar_test(pipe.full_e + 1, ph1)) {
        ph1 ^= 1u;
        pipe.template act_body<kFuseActWarps / 4>(net.act, 1, aw);
        any = true;
      }
      if (!any) {
        if (ld_volatile(&ctl->done) == NG) break;
        __nanosleep(32);
      }
    }
  } else {
    // ---------------- MLP server: MMA issue warp ----------------
    uint32_t pin0 = 0, pin1 = 0, pa0 = 0, pa1 = 0;
    int st0 = 0, st1 = 0;  // 0: wait rows -> layer 1; 1: wait operand -> layer 2; 2: wait operand -> layer 3
    bool first = true;
    for (;;) {
      bool any = false;
      if (st0 == 0) {
        if (tc::mbar_test(pipe.in_ready + 0, pin0)) { pin0 ^= 1u; pipe.issue_layer1(0, first); first = false; st0 = 1; any = true; }
      } else if (tc::mbar_test(pipe.a_ready + 0, pa0)) {
        pa0 ^= 1u;
        if (st0 == 1) { pipe.issue_layer2(0); st0 = 2; } else { pipe.issue_layer3(0); st0 = 0; }
        any = true;
      }
      if (st1 == 0) {
        if (tc::mbar_test(pipe.in_ready + 1, pin1)) { pin1 ^= 1u; pipe.issue_layer1(1, first); first = false; st1 = 1; any = true; }
      } else if (tc::mbar_test(pipe.a_ready + 1, pa1)) {
        pa1 ^= 1u;
        if (st1 == 1) { pipe.issue_layer2(1); st1 = 2; } else { pipe.issue_layer3(1); st1 = 0; }
        any = true;
      }
      if (!any) {
        if (ld_volatile(&ctl->done) == NG) break;
        __nanosleep(32);
      }
    }
  }
  pipe.teardown();
}

template <int H, int LMAX, int AMAX, int NG, bool DEFERRED>
static int launch_pipe_one(dsmc_ctx *c, const StepParams &p, const MlpTcDev &net, int grid) {
  auto kern = k_collide_pipe<H, LMAX, AMAX, NG, DEFERRED>;
  const size_t smem = NG * chunk_region_bytes<LMAX, AMAX>() + PipeShape<H>::SMEM_BYTES + sizeof(FuseCtl) + 256;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return DSMC_ERR_CUDA;
  kern<<<grid, fuse_threads(NG), smem, c->stream>>>(p, net);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

template <int H>
static int launch_pipe_h(dsmc_ctx *c, const StepParams &p, const MlpTcDev &net) {
  const int g_main = std::max(1, std::min((p.n_chunks + 1) / 2, c->num_sms));
  int rc = launch_pipe_one<H, kLmaxSmall, kAmaxSmall, 2, false>(c, p, net, g_main);
  if (rc != DSMC_OK) return rc;
  return launch_pipe_one<H, kLmaxBig, kAmaxBig, 1, true>(c, p, net, c->num_sms);
}

// op 2 (ab initio chi-MLP), plain BF16: chunk map, main pass, deferred pass
int launch_collide_pipe(dsmc_ctx *c, const StepParams &p_in, const MlpTcDev *net) {
  if (p_in.op != 2 || net->d_in != 2 || net->d_out != 1) return DSMC_ERR_UNSUPPORTED_SHAPE;
  StepParams p = p_in;
  int rc = launch_chunk_map(c, p);
  if (rc != DSMC_OK) return rc;
  return net->H == 128 ? launch_pipe_h<128>(c, p, *net) : launch_pipe_h<64>(c, p, *net);
}

}  // namespace dsmc
