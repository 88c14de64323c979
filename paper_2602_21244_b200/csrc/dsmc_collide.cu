// Fused neural DSMC collision step (FP32 CUDA-core variant and the chi-table variant).
//
// One CTA owns a "chunk": the run of whole cells whose first slot lies in
// [b*kChunk, (b+1)*kChunk) of the cell-sorted arrays.  The chunk is a single contiguous range of
// particles, loaded once into shared memory (12 B read / particle), processed entirely on chip
// and stored once (12 B write / particle):
//
//   S1 load            S2 pre-collision cell moments (eq. 10; warp per cell, fp64 sums)
//   S3 pairing keys    Philox(seed; slot, cell, step, stream 0); bucket = mulhi(key, N_k)
//   S4 bucket scan + placement + in-bucket ranking  -> pi = argsort of (key, slot), bit-exact
//   S5 pair loop       operator (f_theta MLP | chi table | chi MLP) -> energy shell / rotation
//                      -> centre-of-mass update (eqs. 5-8)
//   S6 post moments + moment matching (eqs. 10-11)      S7 store
//
// The pairing is the unique ascending order of the 64-bit keys (key<<32 | slot); because
// mulhi(key, N) is monotone in key, sorting by bucket and then ranking inside each (tiny) bucket
// gives exactly that order in O(N) work with one thread per particle, independent of cell sizes.
#include <algorithm>

#include "dsmc_device.cuh"
#include "dsmc_internal.h"

namespace dsmc {

struct CellInfo {
  int32_t cell;     // global cell id
  int32_t start;    // first local slot
  int32_t N, M;     // particles, pairs
  int32_t pair_off; // first pair index of this cell in the chunk's pair list
  int32_t collided; // any pair collided
  float ux, uy, uz; // pre-collision mean velocity
  float theta;      // pre-collision sum |v-u|^2
  float e_pre;      // pre-collision sum |v|^2
  float T;          // m theta / (3 kB N)
};

// shared-memory carve-up (bytes) for the chunk state
struct ChunkSmem {
  float *vx, *vy, *vz;
  uint32_t *key;
  int *cnt;
  uint16_t *ord, *pi, *lc, *pairs;
  CellInfo *cells;
  int *misc;  // [0] c_lo [1] c_hi [2] n_act [3] n_pairs, [8..40] scan scratch
  float *mlp; // 2 x dmax x TP floats (only when an MLP runs)
};

__host__ __device__ inline size_t chunk_smem_bytes(int mlp_floats) {
  size_t b = 0;
  b += sizeof(float) * 3 * kNlocMax;
  b += sizeof(uint32_t) * kNlocMax;
  b += sizeof(int) * (kNlocMax + 4);
  b += sizeof(uint16_t) * (3 * kNlocMax + kNlocMax / 2 + 8);
  b += sizeof(CellInfo) * kActMax;
  b += sizeof(int) * 48;
  b += sizeof(float) * (size_t)mlp_floats;
  return b + 64;
}

__device__ __forceinline__ ChunkSmem carve(unsigned char *base) {
  ChunkSmem s;
  float *f = reinterpret_cast<float *>(base);
  s.vx = f; s.vy = f + kNlocMax; s.vz = f + 2 * kNlocMax;
  s.key = reinterpret_cast<uint32_t *>(f + 3 * kNlocMax);
  s.cnt = reinterpret_cast<int *>(s.key + kNlocMax);
  s.cells = reinterpret_cast<CellInfo *>(s.cnt + kNlocMax + 4);
  s.misc = reinterpret_cast<int *>(s.cells + kActMax);
  s.mlp = reinterpret_cast<float *>((reinterpret_cast<uintptr_t>(s.misc + 48) + 15) & ~(uintptr_t)15);
  return s;
}

// ---------------------------------------------------------------------------------------------
// S1-S4: load, pre-moments, pairing.  Returns n_loc (0 = nothing to do).  All threads call.
// u16 arrays live after the MLP buffer so the float buffers stay 16-byte aligned.
// ---------------------------------------------------------------------------------------------
__device__ int chunk_prepare(const StepParams &P, ChunkSmem &S, int &q0_out) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t p_lo = (int64_t)blockIdx.x * kChunk, p_hi = min(P.n, p_lo + (int64_t)kChunk);
  if (tid == 0) {
    S.misc[0] = lower_bound_cells(P.cell_start, P.n_cells, p_lo);
    S.misc[1] = lower_bound_cells(P.cell_start, P.n_cells, p_hi);
    S.misc[2] = 0;
    S.misc[3] = 0;
  }
  __syncthreads();
  const int c_lo = S.misc[0], c_hi = S.misc[1];
  if (c_lo >= c_hi) return 0;
  const int q0 = P.cell_start[c_lo], q1 = P.cell_start[c_hi];
  const int n_loc = q1 - q0;
  q0_out = q0;
  if (n_loc <= 0) return 0;
  if (n_loc > kNlocMax) {
    if (tid == 0) *P.status = DSMC_ERR_CELL_TOO_LARGE;
    return 0;
  }
  // S1: one coalesced read of the chunk
  for (int q = tid; q < n_loc; q += kThreads) {
    S.vx[q] = P.vx[q0 + q];
    S.vy[q] = P.vy[q0 + q];
    S.vz[q] = P.vz[q0 + q];
    S.cnt[q] = 0;
    S.lc[q] = 0xFFFFu;
  }
  __syncthreads();
  // S2: warp per cell -- fp64 sums, centred second pass
  for (int c = c_lo + warp; c < c_hi; c += kThreads / 32) {
    const int gs = P.cell_start[c], N = P.cell_start[c + 1] - gs;
    if (N < 2) continue;
    if (N > kMaxCell) {
      if (lane == 0) *P.status = DSMC_ERR_CELL_TOO_LARGE;
      continue;
    }
    const int ls = gs - q0;
    int a = 0;
    if (lane == 0) a = atomicAdd(&S.misc[2], 1);
    a = __shfl_sync(0xffffffffu, a, 0);
    double sx = 0, sy = 0, sz = 0, e = 0;
    for (int q = ls + lane; q < ls + N; q += 32) {
      double x = S.vx[q], y = S.vy[q], z = S.vz[q];
      sx += x; sy += y; sz += z;
      e += x * x + y * y + z * z;
      S.lc[q] = (uint16_t)a;
    }
    sx = warp_sum(sx); sy = warp_sum(sy); sz = warp_sum(sz); e = warp_sum(e);
    const double ux = sx / N, uy = sy / N, uz = sz / N;
    double th = 0;
    for (int q = ls + lane; q < ls + N; q += 32) {
      double x = S.vx[q] - ux, y = S.vy[q] - uy, z = S.vz[q] - uz;
      th += x * x + y * y + z * z;
    }
    th = warp_sum(th);
    if (lane == 0) {
      CellInfo ci;
      ci.cell = c; ci.start = ls; ci.N = N;
      int M = N >> 1;
      if (P.pairs_per_cell >= 0 && P.pairs_per_cell < M) M = P.pairs_per_cell;
      ci.M = M; ci.pair_off = 0; ci.collided = 0;
      ci.ux = (float)ux; ci.uy = (float)uy; ci.uz = (float)uz;
      ci.theta = (float)th; ci.e_pre = (float)e;
      ci.T = (float)((double)P.mass * th / (3.0 * 1.380649e-23 * (double)N));
      S.cells[a] = ci;
    }
  }
  __syncthreads();
  const int n_act = S.misc[2];
  if (n_act == 0) return -n_loc;  // nothing collides; caller skips the store too
  // pair offsets: exclusive scan of M over the active cells (reuse key[] as scratch ints)
  int *poff = reinterpret_cast<int *>(S.key);
  for (int a = tid; a < n_act; a += kThreads) poff[a] = S.cells[a].M;
  __syncthreads();
  block_excl_scan(poff, n_act, S.misc + 8);
  for (int a = tid; a < n_act; a += kThreads) S.cells[a].pair_off = poff[a];
  if (tid == 0) S.misc[3] = poff[n_act - 1] + S.cells[n_act - 1].M;
  __syncthreads();
  // S3: one pairing key per slot; bucket counts
  for (int q = tid; q < n_loc; q += kThreads) {
    const int a = S.lc[q];
    if (a == 0xFFFF) {  // single-particle cell: occupies its own bucket so offsets stay aligned
      S.cnt[q] = 1;
      continue;
    }
    const CellInfo &ci = S.cells[a];
    const uint32_t p = (uint32_t)(q - ci.start);
    const uint4 r = philox4x32_10(p >> 2, (uint32_t)ci.cell, P.step, 0u, P.seed_lo, P.seed_hi);
    const uint32_t k = word_of(r, p & 3u);
    S.key[q] = k;
    atomicAdd(&S.cnt[ci.start + (int)__umulhi(k, (uint32_t)ci.N)], 1);
    if ((p & 1u) == 0 && (int)(p >> 1) < ci.M) S.pairs[ci.pair_off + (p >> 1)] = (uint16_t)q;
  }
  __syncthreads();
  // S4: bucket starts, placement, in-bucket ranking
  block_excl_scan(S.cnt, n_loc, S.misc + 8);
  for (int q = tid; q < n_loc; q += kThreads) {
    const int a = S.lc[q];
    if (a == 0xFFFF) {
      atomicAdd(&S.cnt[q], 1);
      continue;
    }
    const CellInfo &ci = S.cells[a];
    const int bkt = ci.start + (int)__umulhi(S.key[q], (uint32_t)ci.N);
    S.ord[atomicAdd(&S.cnt[bkt], 1)] = (uint16_t)q;  // cnt[bkt] ends as the bucket's end
  }
  __syncthreads();
  for (int q = tid; q < n_loc; q += kThreads) {
    const int a = S.lc[q];
    if (a == 0xFFFF) continue;
    const CellInfo &ci = S.cells[a];
    const uint32_t k = S.key[q];
    const int bkt = ci.start + (int)__umulhi(k, (uint32_t)ci.N);
    const int b0 = bkt > 0 ? S.cnt[bkt - 1] : 0, b1 = S.cnt[bkt];
    int rank = 0;
    for (int t = b0; t < b1; ++t) {
      const int o = S.ord[t];
      const uint32_t ko = S.key[o];
      rank += (ko < k || (ko == k && o < q)) ? 1 : 0;
    }
    S.pi[b0 + rank] = (uint16_t)(q - ci.start);
  }
  __syncthreads();
  return n_loc;
}

// ---------------------------------------------------------------------------------------------
// Per-pair physics shared by the operator variants
// ---------------------------------------------------------------------------------------------
struct PairCtx {
  int a, s, i, j;   // active cell, pair slot, local particle indices
  float gx, gy, gz, g2, g;
  bool acc;
  float U_b, U_eps;
};

__device__ __forceinline__ PairCtx pair_setup(const StepParams &P, const ChunkSmem &S, int t) {
  PairCtx c;
  const int q = S.pairs[t];
  c.a = S.lc[q];
  const CellInfo &ci = S.cells[c.a];
  c.s = (q - ci.start) >> 1;
  c.i = ci.start + S.pi[q];
  c.j = ci.start + S.pi[q + 1];
  c.gx = S.vx[c.i] - S.vx[c.j];  // eq. 1
  c.gy = S.vy[c.i] - S.vy[c.j];
  c.gz = S.vz[c.i] - S.vz[c.j];
  c.g2 = c.gx * c.gx + c.gy * c.gy + c.gz * c.gz;
  c.g = sqrtf(c.g2);
  c.acc = true;
  c.U_b = 0.f; c.U_eps = 0.f;
  if (P.op != 0 || ((P.flags & DSMC_F_ACCEPT) && P.cap != nullptr)) {
    const uint4 r = philox4x32_10((uint32_t)c.s, (uint32_t)ci.cell, P.step, 1u, P.seed_lo, P.seed_hi);
    c.U_b = u01(r.y);
    c.U_eps = u01(r.z);
    if ((P.flags & DSMC_F_ACCEPT) && P.cap != nullptr) {
      const float cap = __ldg(P.cap + ci.cell);
      const float w = (P.op == 0) ? P.vhs_c * powf(c.g, P.vhs_e) : c.g;  // sigma_T(g) g  |  g
      c.acc = u01(r.x) * cap < w;
    }
  }
  return c;
}

__device__ __forceinline__ void pair_commit(const StepParams &P, ChunkSmem &S, const PairCtx &c, float px, float py,
                                            float pz, float aux, int q0) {
  const CellInfo &ci = S.cells[c.a];
  if (c.acc) {  // eqs. 6-8
    const float cx = 0.5f * (S.vx[c.i] + S.vx[c.j]);
    const float cy = 0.5f * (S.vy[c.i] + S.vy[c.j]);
    const float cz = 0.5f * (S.vz[c.i] + S.vz[c.j]);
    S.vx[c.i] = cx + 0.5f * px; S.vy[c.i] = cy + 0.5f * py; S.vz[c.i] = cz + 0.5f * pz;
    S.vx[c.j] = cx - 0.5f * px; S.vy[c.j] = cy - 0.5f * py; S.vz[c.j] = cz - 0.5f * pz;
    S.cells[c.a].collided = 1;
  }
  const int64_t d = (int64_t)q0 + ci.start + c.s;
  if (P.dump.pair_i) P.dump.pair_i[d] = c.i - ci.start;
  if (P.dump.pair_j) P.dump.pair_j[d] = c.j - ci.start;
  if (P.dump.accepted) P.dump.accepted[d] = c.acc ? 1 : 0;
  if (P.dump.gprime) { P.dump.gprime[3 * d] = px; P.dump.gprime[3 * d + 1] = py; P.dump.gprime[3 * d + 2] = pz; }
  if (P.dump.aux) P.dump.aux[d] = aux;
}

// rotation of g by deflection chi and azimuth eps (Q16)
__device__ __forceinline__ void rotate(const PairCtx &c, float chi, float eps_over_pi, float &px, float &py,
                                       float &pz) {
  float sc, cc, se, ce;
  sincosf(chi, &sc, &cc);
  sincospif(eps_over_pi, &se, &ce);
  const float gperp = sqrtf(c.gy * c.gy + c.gz * c.gz);
  if (gperp <= 1e-30f * c.g) {
    px = c.gx * cc;
    py = fabsf(c.gx) * sc * ce;
    pz = fabsf(c.gx) * sc * se;
    return;
  }
  const float inv = 1.0f / gperp;
  px = c.gx * cc + gperp * sc * se;
  py = c.gy * cc + sc * (c.g * c.gz * ce - c.gx * c.gy * se) * inv;
  pz = c.gz * cc - sc * (c.g * c.gy * ce + c.gx * c.gz * se) * inv;
}

// bilinear chi(E~, b~) from the L2-resident table, both coordinates clamped (Q13)
__device__ __forceinline__ float chi_table(const ChiTableDev &T, float lnE, float bt) {
  float tE = (lnE - T.lnE_min) * T.inv_dlnE;
  float tB = bt * (float)(T.nB - 1);
  tE = !(tE > 0.f) ? 0.f : fminf(tE, (float)(T.nE - 1));
  tB = !(tB > 0.f) ? 0.f : fminf(tB, (float)(T.nB - 1));
  const int iE = min((int)tE, T.nE - 2), iB = min((int)tB, T.nB - 2);
  const float fE = tE - (float)iE, fB = tB - (float)iB;
  const float *r0 = T.chi + (size_t)iE * T.nB + iB;
  const float c00 = __ldg(r0), c01 = __ldg(r0 + 1), c10 = __ldg(r0 + T.nB), c11 = __ldg(r0 + T.nB + 1);
  return (1.f - fE) * ((1.f - fB) * c00 + fB * c01) + fE * ((1.f - fB) * c10 + fB * c11);
}

// ---------------------------------------------------------------------------------------------
// FP32 MLP over a tile of TP pairs.  X = buf[0] holds features [k][TP]; result left in the
// returned buffer as [o][TP].  Thread (tp = tid % (TP/4), to = tid / (TP/4)) owns 4 pairs x
// outputs {to, to + n_to, ...}.
// ---------------------------------------------------------------------------------------------
template <int TP>
__device__ float *mlp_tile_fp32(const MlpDev &net, float *buf) {
  constexpr int NTP = TP / 4, NTO = kThreads / NTP, MAXM = 256 / NTO > 8 ? 8 : 256 / NTO;
  const int tid = threadIdx.x, tp = tid % NTP, to = tid / NTP;
  float *in = buf, *out = buf + net.dmax * TP;
  for (int l = 0; l < net.n_layers; ++l) {
    const int Din = net.dims[l], Dout = net.dims[l + 1];
    const float *__restrict__ Wt = net.Wt[l];
    const bool hidden = (l + 1 < net.n_layers);
    for (int m0 = 0; m0 * NTO < Dout; m0 += MAXM) {
      float acc[MAXM][4];
#pragma unroll
      for (int m = 0; m < MAXM; ++m) {
        const int o = to + NTO * (m0 + m);
        const float b = o < Dout ? __ldg(net.b[l] + o) : 0.f;
        acc[m][0] = b; acc[m][1] = b; acc[m][2] = b; acc[m][3] = b;
      }
      for (int k = 0; k < Din; ++k) {
        const float4 x = *reinterpret_cast<const float4 *>(in + k * TP + 4 * tp);
#pragma unroll
        for (int m = 0; m < MAXM; ++m) {
          const int o = to + NTO * (m0 + m);
          if (NTO * (m0 + m) < Dout) {  // CTA-uniform
            const float w = o < Dout ? __ldg(Wt + k * Dout + o) : 0.f;
            acc[m][0] = fmaf(w, x.x, acc[m][0]);
            acc[m][1] = fmaf(w, x.y, acc[m][1]);
            acc[m][2] = fmaf(w, x.z, acc[m][2]);
            acc[m][3] = fmaf(w, x.w, acc[m][3]);
          }
        }
      }
#pragma unroll
      for (int m = 0; m < MAXM; ++m) {
        const int o = to + NTO * (m0 + m);
        if (o < Dout) {
          float4 y;
          y.x = hidden ? act_apply(net.act, acc[m][0]) : acc[m][0];
          y.y = hidden ? act_apply(net.act, acc[m][1]) : acc[m][1];
          y.z = hidden ? act_apply(net.act, acc[m][2]) : acc[m][2];
          y.w = hidden ? act_apply(net.act, acc[m][3]) : acc[m][3];
          *reinterpret_cast<float4 *>(out + o * TP + 4 * tp) = y;
        }
      }
    }
    __syncthreads();
    float *t = in; in = out; out = t;
  }
  return in;
}

// S6 + S7: post-collision moments, moment matching, single coalesced store
__device__ void chunk_finish(const StepParams &P, ChunkSmem &S, int n_loc, int q0) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n_act = S.misc[2];
  if (P.flags & DSMC_F_MOMENT_MATCH) {
    for (int a = warp; a < n_act; a += kThreads / 32) {
      const CellInfo ci = S.cells[a];
      if (!ci.collided) continue;
      const int ls = ci.start, N = ci.N;
      if (P.flags & DSMC_F_MATCH_ENERGY_ONLY) {  // literal eq. 11
        double e = 0;
        for (int q = ls + lane; q < ls + N; q += 32) {
          double x = S.vx[q], y = S.vy[q], z = S.vz[q];
          e += x * x + y * y + z * z;
        }
        e = warp_sum(e);
        if (e > 0.0) {
          const float alpha = (float)sqrt((double)ci.e_pre / e);
          for (int q = ls + lane; q < ls + N; q += 32) { S.vx[q] *= alpha; S.vy[q] *= alpha; S.vz[q] *= alpha; }
        }
        continue;
      }
      double sx = 0, sy = 0, sz = 0;
      for (int q = ls + lane; q < ls + N; q += 32) { sx += S.vx[q]; sy += S.vy[q]; sz += S.vz[q]; }
      const double ux = warp_sum(sx) / N, uy = warp_sum(sy) / N, uz = warp_sum(sz) / N;
      double th = 0;
      for (int q = ls + lane; q < ls + N; q += 32) {
        double x = S.vx[q] - ux, y = S.vy[q] - uy, z = S.vz[q] - uz;
        th += x * x + y * y + z * z;
      }
      th = warp_sum(th);
      const double alpha = th > 0.0 ? sqrt((double)ci.theta / th) : 1.0;
      for (int q = ls + lane; q < ls + N; q += 32) {
        S.vx[q] = (float)((double)ci.ux + alpha * (S.vx[q] - ux));
        S.vy[q] = (float)((double)ci.uy + alpha * (S.vy[q] - uy));
        S.vz[q] = (float)((double)ci.uz + alpha * (S.vz[q] - uz));
      }
    }
    __syncthreads();
  }
  for (int q = tid; q < n_loc; q += kThreads) {
    P.vx[q0 + q] = S.vx[q];
    P.vy[q0 + q] = S.vy[q];
    P.vz[q0 + q] = S.vz[q];
  }
}

// ---------------------------------------------------------------------------------------------
// kernels
// ---------------------------------------------------------------------------------------------
template <int TP>
__global__ void __launch_bounds__(kThreads) k_collide_fp32(const StepParams P, const MlpDev net, int mlp_floats) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  ChunkSmem S = carve(smem_raw);
  uint16_t *u16 = reinterpret_cast<uint16_t *>(S.mlp + mlp_floats);
  S.ord = u16; S.pi = u16 + kNlocMax; S.lc = u16 + 2 * kNlocMax; S.pairs = u16 + 3 * kNlocMax;
  int q0 = 0;
  const int n_loc = chunk_prepare(P, S, q0);
  if (n_loc <= 0) return;
  const int tid = threadIdx.x;
  const int n_pairs = S.misc[3];

  if (P.op == 1) {  // chi table: one thread per pair, no tile
    for (int t = tid; t < n_pairs; t += kThreads) {
      PairCtx c = pair_setup(P, S, t);
      float px = c.gx, py = c.gy, pz = c.gz, chi = 0.f;
      if (c.acc) {
        const float lnE = logf(P.e_coef * c.g2);  // E~ = ln(m g^2 / (4 kB))
        chi = chi_table(P.table, lnE, sqrtf(c.U_b));
        if (c.g > 0.f) rotate(c, chi, 2.0f * c.U_eps, px, py, pz);
      }
      pair_commit(P, S, c, px, py, pz, chi, q0);
    }
    __syncthreads();
  } else {
    const int d0 = net.dims[0];
    for (int t0 = 0; t0 < n_pairs; t0 += TP) {
      PairCtx c;
      const bool mine = tid < TP && t0 + tid < n_pairs;
      if (tid < TP) {
        float x[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (mine) {
          c = pair_setup(P, S, t0 + tid);
          const CellInfo &ci = S.cells[c.a];
          if (P.op == 0) {  // VHS-NN features (eqs. 1-3, Q1-Q3)
            float n0 = 0.f, n1 = 0.f, n2 = 0.f;
            if (P.flags & DSMC_F_NOISE) {
              const uint4 r = philox4x32_10((uint32_t)c.s, (uint32_t)ci.cell, P.step, 2u, P.seed_lo, P.seed_hi);
              box_muller3(r, n0, n1, n2);
              n0 *= P.noise_sigma; n1 *= P.noise_sigma; n2 *= P.noise_sigma;
            }
            x[0] = c.gx * P.inv_sigma_v; x[1] = c.gy * P.inv_sigma_v; x[2] = c.gz * P.inv_sigma_v;
            if (d0 == 8) {
              x[3] = c.g * P.inv_sigma_v; x[4] = ci.T * P.inv_T_scale;
              x[5] = n0; x[6] = n1; x[7] = n2;
            } else {
              x[3] = n0; x[4] = n1; x[5] = n2;
            }
          } else {  // chi-MLP inputs (Q15)
            const float lnE = logf(P.e_coef * c.g2);
            float e = (lnE - P.lnE_min) * P.inv_lnE_range;
            x[0] = !(e > 0.f) ? 0.f : fminf(e, 1.f);
            x[1] = sqrtf(c.U_b);
          }
        }
        for (int k = 0; k < d0; ++k) S.mlp[k * TP + tid] = x[k];
      }
      __syncthreads();
      const float *out = mlp_tile_fp32<TP>(net, S.mlp);
      if (mine) {
        float px = c.gx, py = c.gy, pz = c.gz, aux = 0.f;
        if (c.acc) {
          if (P.op == 0) {
            const float hx = out[tid], hy = out[TP + tid], hz = out[2 * TP + tid];
            const float hn = sqrtf(hx * hx + hy * hy + hz * hz);
            aux = hn;
            if (P.flags & DSMC_F_ENERGY_SHELL) {
              if (hn >= P.shell_eps) {  // eq. 5 with the guard of Q4
                const float sc = c.g / hn;
                px = sc * hx; py = sc * hy; pz = sc * hz;
              }
            } else {
              px = P.sigma_v * hx; py = P.sigma_v * hy; pz = P.sigma_v * hz;
            }
          } else {
            const float z = out[tid];
            const float y = fmaxf(z, 0.f) + log1pf(expf(-fabsf(z)));  // softplus
            aux = expm1f(y);                                           // chi
            if (c.g > 0.f) rotate(c, aux, 2.0f * c.U_eps, px, py, pz);
          }
        }
        pair_commit(P, S, c, px, py, pz, aux, q0);
      }
      __syncthreads();
    }
  }
  chunk_finish(P, S, n_loc, q0);
}

int launch_collide(dsmc_ctx *c, const StepParams &p, const MlpDev *net) {
  const int chunks = (int)((p.n + kChunk - 1) / kChunk);
  MlpDev nd{};
  int mlp_floats = 0, TP = 64;
  if (p.op != 1) {
    nd = *net;
    TP = nd.dmax <= 128 ? 64 : 32;
    mlp_floats = 2 * nd.dmax * TP;
  }
  const size_t smem = chunk_smem_bytes(mlp_floats);
  cudaError_t e;
  if (TP == 64) {
    e = cudaFuncSetAttribute(k_collide_fp32<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return DSMC_ERR_CUDA;
    k_collide_fp32<64><<<chunks, kThreads, smem, c->stream>>>(p, nd, mlp_floats);
  } else {
    e = cudaFuncSetAttribute(k_collide_fp32<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return DSMC_ERR_CUDA;
    k_collide_fp32<32><<<chunks, kThreads, smem, c->stream>>>(p, nd, mlp_floats);
  }
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------
// a10: chi for independent pairs (BASELINE.json cfg 4)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_chi_batch_table(int64_t n, const float *__restrict__ E,
                                                        const float *__restrict__ b, float *__restrict__ chi,
                                                        ChiTableDev T, float inv_bmax) {
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x)
    chi[p] = chi_table(T, logf(__ldg(E + p)), __ldg(b + p) * inv_bmax);
}

template <int TP>
__global__ void __launch_bounds__(kThreads) k_chi_batch_mlp(int64_t n, const float *__restrict__ E,
                                                           const float *__restrict__ b, float *__restrict__ chi,
                                                           const MlpDev net, float inv_bmax, float lnE_min,
                                                           float inv_range) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float *buf = reinterpret_cast<float *>(smem_raw);
  const int tid = threadIdx.x;
  const int64_t n_tiles = (n + TP - 1) / TP;
  for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int64_t p = tile * TP + tid;
    if (tid < TP) {
      float x0 = 0.f, x1 = 0.f;
      if (p < n) {
        float e = (logf(__ldg(E + p)) - lnE_min) * inv_range;
        x0 = !(e > 0.f) ? 0.f : fminf(e, 1.f);
        float bt = __ldg(b + p) * inv_bmax;
        x1 = !(bt > 0.f) ? 0.f : fminf(bt, 1.f);
      }
      buf[tid] = x0;
      buf[TP + tid] = x1;
    }
    __syncthreads();
    const float *out = mlp_tile_fp32<TP>(net, buf);
    if (tid < TP && p < n) {
      const float z = out[tid];
      chi[p] = expm1f(fmaxf(z, 0.f) + log1pf(expf(-fabsf(z))));
    }
    __syncthreads();
  }
}

int launch_chi_batch(dsmc_ctx *c, int64_t n, const float *E, const float *b, float *chi, int mode, float b_max,
                     float lnE_min, float lnE_max, const MlpDev *net) {
  if (mode == 0) {
    const int grid = (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->num_sms * 16);
    k_chi_batch_table<<<grid, 256, 0, c->stream>>>(n, E, b, chi, c->table, 1.0f / b_max);
  } else {
    const MlpDev nd = *net;
    const float inv_range = 1.0f / (lnE_max - lnE_min);
    if (nd.dmax <= 128) {
      const size_t smem = sizeof(float) * 2 * nd.dmax * 64;
      cudaFuncSetAttribute(k_chi_batch_mlp<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      const int grid = (int)std::min<int64_t>((n + 63) / 64, (int64_t)c->num_sms * 2);
      k_chi_batch_mlp<64><<<grid, kThreads, smem, c->stream>>>(n, E, b, chi, nd, 1.0f / b_max, lnE_min, inv_range);
    } else {
      const size_t smem = sizeof(float) * 2 * nd.dmax * 32;
      cudaFuncSetAttribute(k_chi_batch_mlp<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      const int grid = (int)std::min<int64_t>((n + 31) / 32, (int64_t)c->num_sms * 2);
      k_chi_batch_mlp<32><<<grid, kThreads, smem, c->stream>>>(n, E, b, chi, nd, 1.0f / b_max, lnE_min, inv_range);
    }
  }
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

}  // namespace dsmc
