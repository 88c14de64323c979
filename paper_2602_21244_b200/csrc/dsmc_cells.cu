// Fused collision step, chi-table operator, "cell team" form (the north_star kernel).
//
// One TEAM owns one cell from its first HBM read to its last HBM write: a warp for cells of up to 256 particles,
// the 128 threads of a CTA for up to 1024, a 256-thread CTA for up to DSMC_MAX_CELL_PARTICLES = 2048.  A thread
// holds at most 8 particles and 8 pairing keys in registers, so every phase is a short, fully unrolled loop whose
// trip count is uniform over the team, and the warp teams synchronise with __syncwarp only (no CTA barrier on the
// path of a small cell).
//
//   load      12 B / particle, coalesced, straight into registers; the pre-collision sums (eq. 10) are
//             taken from those registers about a pivot (mean of the cell's first 32 particles), then the
//             velocities go to shared memory (SoA)
//   keys      one Philox block per 4 slots (stream 0, DESIGN "RNG addressing"); bucket = top L bits of the key,
//             L = ceil(log2 N); one shared-memory atomic per key returns its arrival index
//   scan      exclusive prefix of the bucket counts; every counter becomes (bucket start | members << 16)
//   place     a key alone in its bucket has its final rank (56-61 % of them); the others write their
//             COMPOSITE (key << L | slot: the order of (key, slot) inside a bucket, in 32 bits) at bucket start
//             + arrival index
//   rank      ... and count the smaller composites of their bucket: pi = the unique ascending order of
//             (key << 32 | slot) (Q7); pairs are (pi[2s], pi[2s+1])
//   pairs     two pair slots per thread (they share one Philox block of stream 1): gather, table lookup
//             (one 16 B fetch from the L2-resident quad table through the TEX pipe), rotation by (chi, eps) (Q16),
//             centre-of-mass update (eqs. 6-8) written back to shared memory
//   finish    post-collision sums from shared memory into registers, matching coefficients (eqs. 10-11, P:L46,
//             Q5) in FP32 (alpha - 1 = del / (1 + sqrt(1 + del)): no cancellation), v <- v + (alpha - 1) v + B
//             applied to the registers, 12 B / particle stored
//
// Work distribution: k_cell_lists sorts the cells that have pairs to collide into three lists by size; the
// CTAs of k_cells are persistent and draw list entries from a counter (the next entry is fetched while the
// current cell is processed).  Results depend only on (seed, step, cell, slot).
#include <algorithm>

#include "dsmc_cells.cuh"

namespace dsmc {

// ---------------------------------------------------------------------------------------------
// cell lists: (cell, first slot, N, M) of every cell with M > 0, by size class
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_cell_lists(int32_t K, const int32_t *__restrict__ cs,
                                                    const int32_t *__restrict__ pairs_count, int32_t pairs_per_cell,
                                                    int4 *__restrict__ list0, int4 *__restrict__ list1,
                                                    int4 *__restrict__ list2, int32_t *__restrict__ ctr,
                                                    int32_t *__restrict__ ctr_other, int32_t *__restrict__ status) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  pdl_wait();  // (cell_start may come from the kernel before this one: dsmc_bin's last)
  pdl_launch_dependents();
  if (c < 8) ctr_other[c] = 0;  // the counters of the next launch (this launch's list lengths were zeroed by the previous one)
  if (c < 4) ctr[4 + c] = 0;    // this launch's work counters (nobody reads them before this kernel has completed)
  int cls = -1;
  int4 item = make_int4(0, 0, 0, 0);
  if (c < K) {
    const int gs = __ldg(cs + c), N = __ldg(cs + c + 1) - gs;
    int M = N >> 1;
    const int req = pairs_count ? __ldg(pairs_count + c) : pairs_per_cell;
    if (req >= 0 && req < M) M = req;
    if (N > kMaxCell) {
      *status = DSMC_ERR_CELL_TOO_LARGE;
    } else if (N >= 2 && M > 0) {
      cls = N <= 256 ? 0 : (N <= 1024 ? 1 : 2);
      item = make_int4(c, gs, N, M);
    }
  }
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const unsigned m = __ballot_sync(0xffffffffu, cls == k);
    if (m == 0) continue;
    int base = 0;
    if (lane == __ffs(m) - 1) base = atomicAdd(ctr + k, __popc(m));
    base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
    if (cls == k) {
      int4 *list = k == 0 ? list0 : (k == 1 ? list1 : list2);
      list[base + __popc(m & ((1u << lane) - 1u))] = item;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// kernels
// ---------------------------------------------------------------------------------------------
// main kernel: 128-thread CTAs.  First the cells of 257..1024 particles, one per CTA at a time; then the cells of
// up to 256 particles, one per warp at a time.  Both forms use the same shared-memory footprint.
// OP 0: the whole step with the chi table.  OP 3 / 4: first / second pass of the split chi-MLP step (below).
template <int OP>
__global__ void __launch_bounds__(128, 8) k_cells(const StepParams P, const CellLists Lst) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  pdl_wait();
  pdl_launch_dependents();
  {
    CellTeam<128, OP> T;
    T.init((uint32_t)__cvta_generic_to_shared(smem_raw), threadIdx.x, 0);
    T.run(P, Lst.list[1], Lst.ctr + 1, Lst.work + 1);
  }
  __syncthreads();
  {
    CellTeam<32, OP> T;
    T.init((uint32_t)__cvta_generic_to_shared(smem_raw) + (threadIdx.x >> 5) * (uint32_t)CellTeam<32>::bytes(), threadIdx.x & 31, 0);
    T.run(P, Lst.list[0], Lst.ctr + 0, Lst.work + 0);
  }
}

// cells of 1025..2048 particles: one 256-thread CTA per cell at a time
template <int OP>
__global__ void __launch_bounds__(256, 2) k_cells_big(const StepParams P, const CellLists Lst) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  pdl_wait();
  pdl_launch_dependents();
  CellTeam<256, OP> T;
  T.init((uint32_t)__cvta_generic_to_shared(smem_raw), threadIdx.x, 0);
  T.run(P, Lst.list[2], Lst.ctr + 2, Lst.work + 2);
}

// cell lists of this step (alternating counter sets: this launch zeroes the set of the next step)
void launch_cell_lists(dsmc_ctx *c, const StepParams &p, CellLists &L) {
  const size_t K = (size_t)c->max_cells;
  for (int k = 0; k < 3; ++k) L.list[k] = c->d_cell_list + k * K;
  const int e = (int)(c->list_epoch & 1);
  c->list_epoch += 1;
  L.ctr = c->d_list_ctr + 8 * e;
  L.work = L.ctr + 4;
  launch_pdl(k_cell_lists, (p.n_cells + 255) / 256, 256, 0, c->stream, p.n_cells, p.cell_start, p.pairs_count,
             p.pairs_per_cell, L.list[0], L.list[1], L.list[2], L.ctr, c->d_list_ctr + 8 * (1 - e), p.status);
  c->launches += 1;
}

// REUSE: walk the lists the previous pass of this step made (same cells, same pair counts) with a fresh set of work
// counters -- the other epoch's, which k_cell_lists zeroed and nobody has used since -- instead of building them again
template <int OP, bool REUSE = false>
static int launch_cells_pass(dsmc_ctx *c, const StepParams &p) {
  CellLists L;
  if (REUSE) {
    const size_t K = (size_t)c->max_cells;
    const int e = (int)((c->list_epoch - 1) & 1);  // the epoch of the lists just made
    for (int k = 0; k < 3; ++k) L.list[k] = c->d_cell_list + k * K;
    L.ctr = c->d_list_ctr + 8 * e;
    L.work = c->d_list_ctr + 8 * (1 - e) + 4;
  } else {
    launch_cell_lists(c, p, L);
  }
  {
    auto kern = k_cells<OP>;
    const size_t smem = CellTeam<128>::bytes();
    static_assert(CellTeam<128>::bytes() == 4 * CellTeam<32>::bytes(), "the two team forms share one footprint");
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
      return DSMC_ERR_CUDA;
    launch_pdl(kern, c->num_sms * 8, 128, smem, c->stream, p, L);
  }
  {
    auto kern = k_cells_big<OP>;
    const size_t smem = CellTeam<256>::bytes();
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
      return DSMC_ERR_CUDA;
    launch_pdl(kern, c->num_sms * 2, 256, smem, c->stream, p, L);
  }
  c->launches += 2;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_collide_cells(dsmc_ctx *c, const StepParams &p) { return launch_cells_pass<0>(c, p); }

// chi-MLP step on the tensor cores, SPLIT form: three passes at full occupancy instead of one kernel in which twelve
// team warps and the MLP server share an SM (dsmc_cells_mlp.cu; measured: that kernel's team side alone needs 0.98 ms
// on cfg 5).
//   pass 1 (OP 3)  load, key sort -> pairing (stored, 2 B / particle), pair gather -> the two network inputs of every
//                  pair (8 B / pair)
//   pass 2         k_chi_batch_tc on the pair arrays (rows = pair slots): chi, 4 B / pair
//   pass 3 (OP 4)  load, pre-collision sums, stored pairing, gather, acceptance, rotation by (chi, eps), commit,
//                  matching, store
// Everything random is regenerated from (seed, step, cell, slot) in both passes; results do not depend on the launch
// geometry.  The pair arrays and the stored pairing live in the radix sort's first ping-pong buffer (16 B / particle,
// idle while a collision step runs; 8 B / particle needed).
int launch_collide_cells_split(dsmc_ctx *c, const StepParams &p_in, const MlpTcDev *net) {
  if (p_in.op != 2 || net->d_in != 2 || net->d_out != 1 || (net->H != 64 && net->H != 128))
    return DSMC_ERR_UNSUPPORTED_SHAPE;
  StepParams p = p_in;
  const int64_t np = (p.n / 2 + 4) & ~(int64_t)3;  // pair index = first slot of the cell / 2 + pair slot < n / 2 + 1
  float *base = reinterpret_cast<float *>(c->d_bin_rec[0]);
  p.feat0 = base;
  p.feat1 = base + np;
  p.chi_pair = base + 2 * np;
  p.pi_g = reinterpret_cast<uint16_t *>(base + 3 * np);
  int rc = launch_cells_pass<3>(c, p);
  if (rc != DSMC_OK) return rc;
  rc = launch_chi_rows_tc(c, p.n / 2 + 1, p.feat0, p.feat1, p.chi_pair, net);
  if (rc != DSMC_OK) return rc;
  return launch_cells_pass<4, true>(c, p);
}

// VHS-NN operator on the tensor cores, split form on the cell-team kernels (default for DSMC_F_BF16_TC;
// DSMC_F_TC_ONE_KERNEL keeps the chunk kernel with its own engine, k_collide_tc): OP 5 (pairing + the 8 or 6 network inputs of
// every pair, eqs. 1-3), k_mlp_rows_tc_split (split-precision batch, dsmc_collide_tc.cu), OP 6 (stored pairing, outputs
// -> eq. 5 -> eqs. 6-8, matching, store).  Pair arrays: inputs in the radix sort's record buffer (16 B / particle),
// outputs and the stored pairing in its two cell-id buffers.
int launch_collide_cells_vhs_split(dsmc_ctx *c, const StepParams &p_in, const MlpTcDev *net) {
  const TcTailF32 *tail = &c->tc_tail[0];
  if (p_in.op != 0 || !((net->d_in == 8 || net->d_in == 6) && net->d_out == 3) || tail->d_out != 3)
    return DSMC_ERR_UNSUPPORTED_SHAPE;
  StepParams p = p_in;
  const int64_t np = (p.n / 2 + 4) & ~(int64_t)3;
  p.feat0 = reinterpret_cast<float *>(c->d_bin_rec[0]);
  p.split_np = np;
  p.split_din = net->d_in;
  p.out3[0] = reinterpret_cast<float *>(c->d_bin_cell[0]);
  p.out3[1] = p.out3[0] + np;
  p.out3[2] = reinterpret_cast<float *>(c->d_bin_cell[1]);
  p.pi_g = reinterpret_cast<uint16_t *>(p.out3[2] + np);
  int rc = launch_cells_pass<5>(c, p);
  if (rc != DSMC_OK) return rc;
  rc = launch_mlp_rows_tc_split(c, p.n / 2 + 1, p.feat0, np, p.out3[0], p.out3[1], p.out3[2], net, tail);
  if (rc != DSMC_OK) return rc;
  return launch_cells_pass<6, true>(c, p);
}

}  // namespace dsmc
