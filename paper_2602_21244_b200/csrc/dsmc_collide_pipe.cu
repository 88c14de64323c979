// Fused collision step with the chi-MLP on the tensor cores, warp-specialised (plain BF16 operands).
//
// One persistent CTA per SM.  Three kinds of warps, no CTA-wide barrier after start-up:
//
//   chunk groups (NG teams of NT threads: 5 x 128 on 704-slot chunks, 4 x 128 on 1024-slot chunks, 1 x 256 on
//       the rest)  each group pulls chunks (dsmc_chunk.cuh) from a work counter and owns NBUF shared-memory
//       chunk buffers (NBUF = 1 as launched: shared memory goes to more groups rather than to double buffers).
//       Stage A of a chunk: load, cell moments, Philox pairing keys + sort, then its pairs are SUBMITTED 128 at a time to the MLP server (features -> A1 rows of a free
//       slot; U_eps and the acceptance bit are parked in the chunk).  Stage B: when the server has delivered
//       chi for all tiles of the chunk, rotate + commit, matching, store.  With NBUF = 2 a group runs stage A
//       of its next chunk while the server works on the previous one, so the ALU-bound chunk work and the
//       XU/TMEM-bound MLP overlap inside every group.
//   MLP server = ACT warps (8) + MMA warp (1)
//       MMA warp: a state machine per slot issues layer 1 when a half group has published its rows, layers
//       2 and 3 when the ACT warps have published the operand (dsmc_tc_pipe.cuh).
//       ACT warps: whichever slot has a finished layer 1 / 2 in TMEM gets D -> tanh/SiLU -> bf16 -> A operand;
//       the first four also DELIVER a finished layer 3: z of the 128 rows -> the chunk's shared memory, bump
//       the chunk's tile counter, free the slot.  The server never waits for a chunk group.
//
// A slot is owned by one tile from acquire (before its rows are written) to delivery, so no operand or
// accumulator is reused while in flight.
#include <algorithm>

#include "dsmc_chunk.cuh"
#include "dsmc_tc_pipe.cuh"

namespace dsmc {

constexpr int fuse_threads(int ng, int nt, int na) { return ng * nt + na * 32 + 32; }  // groups + ACT warps + MMA warp
enum { MI_NLOC = 5, MI_Q0 = 6 };  // per-buffer chunk state parked in misc[] between stage A and stage B

struct FuseCtl {
  int lock[2];           // slot ownership: 0 free, 1 taken
  int outcnt[2];         // delivery warps done with the slot's outputs
  float *dest[2];        // where the slot's 128 outputs go (chunk shared memory)
  int *done_ctr[2];      // the chunk's delivered-tile counter
  int n_valid[2];        // rows of the slot that are real pairs
  int done;              // chunk groups that ran out of work
  int next[6];           // per group: chunk handed out by the work counter
  int slot_of[12];       // per 128-row feeder: slot taken for the tile being submitted
  int tiles_done[6][2];  // [group][buffer]
};

__device__ __forceinline__ void half_sync(int id) { asm volatile("bar.sync %0, 128;" ::"r"(id) : "memory"); }
__device__ __forceinline__ int ld_volatile(const int *p) { return *reinterpret_cast<const volatile int *>(p); }

// stage A, last part: all pairs of the chunk go to the MLP server; called by all threads of a group
template <int H, int NG, class TM, class CK>
__device__ __forceinline__ void submit_pairs(const TM &T, int g, int b, const StepParams &P, CK &S, TcPipe<H> &pipe,
                                             FuseCtl *ctl) {
  const int hg = T.tid >> 7, r = T.tid & 127;
  const int n_pairs = S.misc[MI_NPAIRS];
  constexpr int NH = TM::kN / 128;  // 128-row feeders per team
  const int me = NH * g + hg, bar_id = 1 + NG + me;
  float *zbuf = reinterpret_cast<float *>(S.key);  // keys are dead after the sort: z of pair t lands in key[t]
  for (int t0 = hg * 128; t0 < n_pairs; t0 += TM::kN) {
    const bool mine = t0 + r < n_pairs;
    float x[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) x[k] = 0.f;
    if (mine) {  // chi-MLP inputs (Q15); U_eps (> 0) and the acceptance bit (sign) wait in cnt[t]
      const PairCtx c = pair_setup(P, S, t0 + r, true);
      const float e = (__logf(P.e_coef * c.g2) - P.lnE_min) * P.inv_lnE_range;
      x[0] = !(e > 0.f) ? 0.f : fminf(e, 1.f);
      x[1] = sqrtf(c.U_b);
      S.cnt[t0 + r] = __float_as_int(c.acc ? c.U_eps : -c.U_eps);
    }
    if (r == 0) {  // take a free slot and say where its outputs go
      int s = -1;
      while (s < 0) {
        if (atomicCAS(&ctl->lock[0], 0, 1) == 0) s = 0;
        else if (atomicCAS(&ctl->lock[1], 0, 1) == 0) s = 1;
        else __nanosleep(64);
      }
      __threadfence_block();
      *reinterpret_cast<float *volatile *>(&ctl->dest[s]) = zbuf + t0;
      *reinterpret_cast<int *volatile *>(&ctl->done_ctr[s]) = &ctl->tiles_done[g][b];
      *reinterpret_cast<volatile int *>(&ctl->n_valid[s]) = min(128, n_pairs - t0);
      *reinterpret_cast<volatile int *>(&ctl->slot_of[me]) = s;
    }
    half_sync(bar_id);
    const int s = ld_volatile(&ctl->slot_of[me]);
    pipe.write_a1_row(s, 0, r, x);
    pipe.io_publish(s);
    half_sync(bar_id);  // slot_of[me] may be overwritten by the next tile only after everyone has read it
  }
}

// stage B, first part: chi has been delivered for every tile; rotate and commit all pairs of the chunk
template <class TM, class CK>
__device__ __forceinline__ void finish_pairs(const TM &T, const StepParams &P, CK &S, const int *tiles_done, int q0) {
  const int n_pairs = S.misc[MI_NPAIRS];
  const int n_tiles = (n_pairs + 127) >> 7;
  if (T.tid == 0)
    while (ld_volatile(tiles_done) < n_tiles) __nanosleep(64);
  T.sync();
  for (int t = T.tid; t < n_pairs; t += TM::kN) {
    PairCtx c = pair_load(P, S, t);
    const float ue = __int_as_float(S.cnt[t]);
    c.acc = ue > 0.f;
    c.U_eps = fabsf(ue);
    float px = c.gx, py = c.gy, pz = c.gz, chi = 0.f;
    if (c.acc) {
      chi = __expf(__uint_as_float(S.key[t]));  // chi = expm1(softplus(z)) = exp(z)
      if (c.g2 > 0.f) rotate_fast(c, chi, c.U_eps, px, py, pz);
    }
    pair_commit(P, S, c, px, py, pz, chi, q0);
  }
}

template <int LMAX, int AMAX>
constexpr size_t chunk_region_bytes() {
  return (Chunk<LMAX, AMAX>::bytes() + 127) & ~(size_t)127;
}

// SRC: 0 = every chunk (work counter 0), 1 = deferred list P.big (counter 1), 2 = second list P.big2 (counter 2).
// DST: where a chunk that does not fit this footprint goes (1 = P.big, 2 = P.big2, 0 = DSMC_ERR_CELL_TOO_LARGE).
template <int H, int LMAX, int AMAX, int NG, int NT, int NA, int NBUF, int SRC, int DST>
__global__ void __launch_bounds__(fuse_threads(NG, NT, NA), 1) k_collide_pipe(const StepParams P, const MlpTcDev net) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  using CK = Chunk<LMAX, AMAX>;
  constexpr size_t REGION = chunk_region_bytes<LMAX, AMAX>();
  unsigned char *base = smem_raw;  // dynamic shared memory starts 128-byte aligned (no static __shared__ here)
  unsigned char *pipe_base = base + NG * NBUF * REGION;
  FuseCtl *ctl = reinterpret_cast<FuseCtl *>(pipe_base + PipeShape<H>::SMEM_BYTES);
  TcPipe<H> pipe;
  if (threadIdx.x == 0) {
    ctl->lock[0] = ctl->lock[1] = 0;
    ctl->outcnt[0] = ctl->outcnt[1] = 0;
    ctl->done = 0;
  }
  pipe.init(pipe_base, net.w_blob, NA, 4);  // ends with CTA-wide barriers
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  constexpr int GW = NG * NT / 32;  // warps of the chunk groups
  if (warp < GW) {
    // ---------------- chunk group ----------------
    const int g = warp / (NT / 32);
    const TeamT<NT> T{(int)threadIdx.x - g * NT, 1 + g};
    const int32_t *src_list = SRC == 1 ? P.big : P.big2;
    const int n_work = SRC == 0 ? P.n_chunks : ld_volatile(src_list);
    bool more = true, have0 = false, have1 = false;
    int b = 0;
    for (;;) {
      // ---- stage A on buffer b ----
      bool got = false;
      CK S;
      S.carve(base + (size_t)(g * NBUF + b) * REGION);
      if (more) {
        if (T.tid == 0) {
          *reinterpret_cast<volatile int *>(&ctl->next[g]) = atomicAdd(P.work + SRC, 1);
          *reinterpret_cast<volatile int *>(&ctl->tiles_done[g][b]) = 0;
        }
        T.sync();
        const int w = ld_volatile(&ctl->next[g]);
        T.sync();
        if (w >= n_work) {
          more = false;
        } else {
          const int chunk = SRC == 0 ? w : src_list[1 + w];
          int q0 = 0;
          const int n_loc = chunk_begin(T, P, S, chunk, q0);
          if (n_loc < 0 && T.tid == 0) {
            if (DST == 0) {
              *P.status = DSMC_ERR_CELL_TOO_LARGE;
            } else {
              int32_t *dst_list = DST == 1 ? P.big : P.big2;
              const int i = atomicAdd(dst_list, 1);
              dst_list[1 + i] = chunk;
            }
          }
          if (n_loc > 0) {
            if (T.tid == 0) {
              S.misc[MI_NLOC] = n_loc;
              S.misc[MI_Q0] = q0;
            }
            chunk_pre_and_sort(T, P, S, n_loc);
            submit_pairs<H, NG>(T, g, b, P, S, pipe, ctl);
            got = true;
          }
        }
      }
      if (b == 0) have0 = got; else have1 = got;
      // ---- stage B on the other buffer (the same one when NBUF == 1) ----
      const int ob = NBUF == 2 ? (b ^ 1) : b;
      if (ob == 0 ? have0 : have1) {
        CK So;
        So.carve(base + (size_t)(g * NBUF + ob) * REGION);
        T.sync();  // misc[] written by thread 0, halves done submitting
        const int n_loc = So.misc[MI_NLOC], q0 = So.misc[MI_Q0];
        finish_pairs(T, P, So, &ctl->tiles_done[g][ob], q0);
        T.sync();
        chunk_finish(T, P, So, n_loc, q0);
        T.sync();
        if (ob == 0) have0 = false; else have1 = false;
      }
      if (!more && !have0 && !have1) break;
      if (NBUF == 2) b ^= 1;
    }
    if (T.tid == 0) {
      __threadfence_block();
      atomicAdd(&ctl->done, 1);
    }
  } else if (warp < GW + NA) {
    // ---------------- MLP server: activation + delivery warps ----------------
    using SH = PipeShape<H>;
    const int aw = warp - GW;
    uint32_t ph0 = 0, ph1 = 0, po0 = 0, po1 = 0;
    auto deliver = [&](int s) {  // aw < 4: rows 32 aw .. 32 aw + 31 of the slot's layer-3 output -> the chunk
      tc::fence_after();
      uint32_t v[4];
      tc::tmem_ld4(pipe.tmem + (((uint32_t)(aw * 32)) << 16) + s * SH::SLOT_COLS + SH::COL_OUT, v);
      tc::wait_ld();
      tc::fence_before();
      float *dest = *reinterpret_cast<float *volatile *>(&ctl->dest[s]);
      const int row = aw * 32 + lane;
      if (row < ld_volatile(&ctl->n_valid[s])) dest[row] = __uint_as_float(v[0]);
      __syncwarp();
      if (lane == 0) {
        __threadfence_block();
        if (atomicAdd(&ctl->outcnt[s], 1) == 3) {  // last of the four: count the tile, free the slot
          int *ctr = *reinterpret_cast<int *volatile *>(&ctl->done_ctr[s]);
          atomicExch(&ctl->outcnt[s], 0);
          atomicAdd(ctr, 1);
          __threadfence_block();
          atomicExch(&ctl->lock[s], 0);
        }
      }
    };
    for (;;) {
      bool any = false;
      if (tc::mbar_test(pipe.full_e + 0, ph0)) {
        ph0 ^= 1u;
        pipe.template act_body<NA / 4>(net.act, 0, aw);
        any = true;
      }
      if (tc::mbar_test(pipe.full_e + 1, ph1)) {
        ph1 ^= 1u;
        pipe.template act_body<NA / 4>(net.act, 1, aw);
        any = true;
      }
      if (aw < 4) {
        if (tc::mbar_test(pipe.full_o + 0, po0)) { po0 ^= 1u; deliver(0); any = true; }
        if (tc::mbar_test(pipe.full_o + 1, po1)) { po1 ^= 1u; deliver(1); any = true; }
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
        if (tc::mbar_test(pipe.in_ready + 0, pin0)) { pin0 ^= 1u; pipe.issue_layer1(0, 0, first); first = false; st0 = 1; any = true; }
      } else if (tc::mbar_test(pipe.a_ready + 0, pa0)) {
        pa0 ^= 1u;
        if (st0 == 1) { pipe.issue_layer2(0); st0 = 2; } else { pipe.issue_layer3(0); st0 = 0; }
        any = true;
      }
      if (st1 == 0) {
        if (tc::mbar_test(pipe.in_ready + 1, pin1)) { pin1 ^= 1u; pipe.issue_layer1(1, 0, first); first = false; st1 = 1; any = true; }
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

template <int H, int LMAX, int AMAX, int NG, int NT, int NA, int NBUF, int SRC, int DST>
static int launch_pipe_one(dsmc_ctx *c, const StepParams &p, const MlpTcDev &net, int grid) {
  auto kern = k_collide_pipe<H, LMAX, AMAX, NG, NT, NA, NBUF, SRC, DST>;
  const size_t smem = NG * NBUF * chunk_region_bytes<LMAX, AMAX>() + PipeShape<H>::SMEM_BYTES + sizeof(FuseCtl) + 128;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return DSMC_ERR_CUDA;
  kern<<<grid, fuse_threads(NG, NT, NA), smem, c->stream>>>(p, net);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

template <int H>
static int launch_pipe_h(dsmc_ctx *c, const StepParams &p, const MlpTcDev &net) {
  // three footprints, as in the table path: 704-slot chunks on five 128-thread groups per SM, 1024-slot chunks
  // on four, then any legal chunk on one 256-thread group
  const int g0 = std::max(1, std::min((p.n_chunks + 4) / 5, c->num_sms));
  int rc = launch_pipe_one<H, 704, kAmaxSmall, 5, 128, 8, 1, 0, 1>(c, p, net, g0);  // (6 groups + 4 ACT warps: slower)
  if (rc != DSMC_OK) return rc;
  rc = launch_pipe_one<H, 1024, kAmaxSmall, 4, 128, 8, 1, 1, 2>(c, p, net, c->num_sms);
  if (rc != DSMC_OK) return rc;
  return launch_pipe_one<H, kLmaxBig, kAmaxBig, 1, 256, 8, 1, 2, 0>(c, p, net, c->num_sms);
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
