// Chunk machinery shared by every variant of the fused collision kernel (product code only).
//
// A "chunk" is the run of whole cells whose first slot lies in [b*kChunk, (b+1)*kChunk) of the
// cell-sorted arrays: one contiguous particle range, owned by one CTA, read from HBM once
// (12 B / particle), processed entirely in shared memory and written once (12 B / particle).
//
//   begin     chunk -> cell range (precomputed map), cell discovery, one coalesced load
//   pre       per 256-particle segment (one warp each): pivoted FP32 sums for eq. 10,
//             Philox pairing keys (one block per 4 slots), bucket counts
//   sort      exclusive scan of the bucket counts, placement, in-bucket ranking -> pi, the unique
//             ascending order of (key << 32 | slot); pairs are (pi[2s], pi[2s+1])   (Q7)
//   [pairs]   operator specific: table / FP32 MLP / tcgen05 MLP           (caller)
//   finish    post-collision segment sums, moment matching folded into the store as one FMA per
//             component: v <- alpha v + B, B = u_pre - alpha u_post (eqs. 10-11, Q5)
//
// Cell sums are accumulated in FP32 about a pivot near the cell mean (mean of the first 32 particles
// before the collisions, u_pre after them), 8 values per lane, and combined across lanes in FP32 and across
// segments in FP64 in a fixed order, so results do not depend on scheduling.
#pragma once
#include "dsmc_device.cuh"
#include "dsmc_internal.h"

namespace dsmc {

constexpr int kSeg = 128;  // particles per segment = one warp pass of 32 Philox blocks (measured: 256 leaves warps idle, 64 half-fills the key loop)
constexpr int kWarps = kThreads / 32;

struct __align__(16) CellInfo {
  float ux, uy, uz, theta;  // pre-collision mean, sum |v-u|^2; chunk_finish overwrites: Bx, By, Bz, alpha - 1
  int32_t cell;             // global cell id
  int32_t pair_off;         // first entry of this cell in pairs[]
  uint16_t start, N, M, seg0;
  int32_t collided;
  int32_t pad[3];
};
static_assert(sizeof(CellInfo) == 48, "CellInfo layout");

enum { MI_NACT = 0, MI_NSEG = 1, MI_NPAIRS = 2, MI_SCAN = 8 /* .. +40 */ };

// REPLACE_: pairs drawn with replacement (DSMC_F_PAIR_REPLACE) -- a compile-time variant so that the default
// (matching) path carries none of its code.
// PACK2N: the key sort uses 2 N buckets per cell, two 16-bit counters per int of cnt (shorter in-bucket ranking loops:
// fused table step 0.476 -> 0.468 ms; the latency-bound groups of the tensor-core kernel lose 2 % to the extra
// arithmetic, so only the table kernels switch it on)
template <int LMAX_, int AMAX_, bool REPLACE_ = false, bool PACK2N_ = false>
struct Chunk {
  static constexpr int LMAX = LMAX_, AMAX = AMAX_;
  static constexpr bool REPLACE = REPLACE_, PACK2N = PACK2N_;
  static constexpr int SMAX = (LMAX / kSeg + AMAX + 2 + 3) & ~3;  // multiple of 4: keeps every array 16-byte aligned
  float4 *v;        // [LMAX] velocities (x, y, z, unused)
  float4 *part;     // [SMAX] segment partial sums
  CellInfo *cells;  // [AMAX]
  uint32_t *key;    // [LMAX]
  int *cnt;         // [LMAX + 4]
  uint32_t *pairs;  // [LMAX / 2] position of the pair's first member | active cell << 16
  uint32_t *segs;   // [SMAX] active cell | piece << 16
  int *misc;        // [64]
  uint16_t *ord, *pi;  // [LMAX]

  static constexpr size_t bytes() {
    return sizeof(float4) * LMAX + sizeof(float4) * SMAX + sizeof(CellInfo) * AMAX + 4 * LMAX + 4 * (LMAX + 4) +
           4 * (LMAX / 2) + 4 * SMAX + 4 * 64 + 2 * 2 * LMAX + 16;
  }
  __device__ __forceinline__ unsigned char *carve(unsigned char *base) {
    v = reinterpret_cast<float4 *>(base);
    part = v + LMAX;
    cells = reinterpret_cast<CellInfo *>(part + SMAX);
    key = reinterpret_cast<uint32_t *>(cells + AMAX);
    cnt = reinterpret_cast<int *>(key + LMAX);
    pairs = reinterpret_cast<uint32_t *>(cnt + LMAX + 4);
    segs = pairs + LMAX / 2;
    misc = reinterpret_cast<int *>(segs + SMAX);
    ord = reinterpret_cast<uint16_t *>(misc + 64);
    pi = ord + LMAX;
    static_assert(LMAX % 8 == 0 && (sizeof(CellInfo) * AMAX) % 16 == 0, "chunk arrays must stay 16-byte aligned");
    return reinterpret_cast<unsigned char *>(pi + LMAX);
  }
};

// A team = the kThreads threads that own one chunk: the whole CTA (bar 0) in the one-chunk-per-CTA
// kernels, or one of several 256-thread groups of a warp-specialised CTA (named barrier bar > 0).
template <int NT>
struct TeamT {
  static constexpr int kN = NT, kW = NT / 32;
  int tid;  // 0 .. NT-1 within the team
  int bar;  // hardware barrier id
  __device__ __forceinline__ void sync() const {
    asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(NT) : "memory");
  }
};
using Team = TeamT<kThreads>;

// Exclusive scan of a[0..L) in shared memory by the whole team.  a is 16-byte aligned and has room for
// L rounded up to 4.  Each thread owns eight consecutive elements per pass (two 16 B accesses),
// scans it in registers, warp totals go through one shuffle scan.  `scratch` holds >= kWarps + 1 ints.
// Ends with T.sync().
// PACKED: every int holds two 16-bit counts (low half first); the scan runs over the 2 L halves and each half ends
// as its own exclusive prefix (values stay below 65536).
template <class TM, bool PACKED = false>
__device__ __forceinline__ void block_excl_scan_coalesced(const TM &T, int *a, int L, int *scratch) {
  const int tid = T.tid, lane = tid & 31, warp = tid >> 5;
  int carry = 0;
  for (int base = 0; base < L; base += 8 * TM::kN) {  // eight consecutive elements per thread and pass
    const int i = base + 8 * tid;
    int x[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) x[u] = 0;
    if (i < L) {
      const int4 lo = *reinterpret_cast<const int4 *>(a + i);
      x[0] = lo.x; x[1] = lo.y; x[2] = lo.z; x[3] = lo.w;
      if (i + 4 < L) {
        const int4 hi = *reinterpret_cast<const int4 *>(a + i + 4);
        x[4] = hi.x; x[5] = hi.y; x[6] = hi.z; x[7] = hi.w;
      }
#pragma unroll
      for (int u = 1; u < 8; ++u)
        if (i + u >= L) x[u] = 0;
    }
    int tot = 0;
    int lo16[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {  // x[u] <- exclusive prefix inside the thread
      lo16[u] = PACKED ? (x[u] & 0xFFFF) : 0;
      const int t = PACKED ? lo16[u] + (int)((uint32_t)x[u] >> 16) : x[u];
      x[u] = tot;
      tot += t;
    }
    int inc = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) scratch[warp] = inc;
    T.sync();
    int off = carry, all = 0;
#pragma unroll
    for (int w = 0; w < TM::kW; ++w) {
      const int sw = scratch[w];
      off += (w < warp) ? sw : 0;
      all += sw;
    }
    const int e0 = off + inc - tot;
    if (PACKED) {
#pragma unroll
      for (int u = 0; u < 8; ++u) x[u] = ((e0 + x[u]) | ((e0 + x[u] + lo16[u]) << 16)) - e0;  // the stores below add e0 back
    }
    if (i < L) {
      *reinterpret_cast<int4 *>(a + i) = make_int4(e0 + x[0], e0 + x[1], e0 + x[2], e0 + x[3]);
      if (i + 4 < L) *reinterpret_cast<int4 *>(a + i + 4) = make_int4(e0 + x[4], e0 + x[5], e0 + x[6], e0 + x[7]);
    }
    carry += all;
    T.sync();
  }
}

__device__ __forceinline__ float warp_sum_f(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Four warp sums for the price of six shuffles (instead of twenty): the butterfly halves the number of values a
// lane carries in each of its first two steps.  Returns the total of a in lanes 0-7, b in 8-15, c in 16-23, d in
// 24-31 (lane >> 3 selects the component).
__device__ __forceinline__ float warp_sum4_t(float a, float b, float c, float d, int lane) {
  const bool up = lane & 16;
  float k0 = up ? c : a, k1 = up ? d : b;
  k0 += __shfl_xor_sync(0xffffffffu, up ? a : c, 16);
  k1 += __shfl_xor_sync(0xffffffffu, up ? b : d, 16);
  const bool up2 = lane & 8;
  float k = up2 ? k1 : k0;
  k += __shfl_xor_sync(0xffffffffu, up2 ? k0 : k1, 8);
  k += __shfl_xor_sync(0xffffffffu, k, 4);
  k += __shfl_xor_sync(0xffffffffu, k, 2);
  k += __shfl_xor_sync(0xffffffffu, k, 1);
  return k;
}

// ---------------------------------------------------------------------------------------------
// begin: returns n_loc > 0 when there is work, 0 when the chunk has nothing to collide (nothing
// to store either), -1 when the chunk does not fit this variant (caller defers it).
// ---------------------------------------------------------------------------------------------
template <class TM, class CK>
__device__ int chunk_begin(const TM &T, const StepParams &P, CK &S, int chunk, int &q0_out) {
  const int tid = T.tid;
  const int4 meta = __ldg(P.chunk_meta + chunk);  // (first cell, end cell, first slot, end slot): one load
  const int c_lo = meta.x, c_hi = meta.y, q0 = meta.z;
  if (c_lo >= c_hi) return 0;
  const int n_loc = meta.w - q0;
  q0_out = q0;
  if (n_loc <= 0) return 0;
  if (n_loc > CK::LMAX) return -1;
  // one coalesced read of the chunk, asynchronously (global -> shared without registers) so that its latency
  // overlaps the cell discovery below
  {
    const uint32_t sv = (uint32_t)__cvta_generic_to_shared(S.v);
    for (int q = tid; q < n_loc; q += TM::kN) {
      const uint32_t d = sv + 16u * (uint32_t)q;
      asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(P.vx + q0 + q) : "memory");
      asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d + 4u), "l"(P.vy + q0 + q) : "memory");
      asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d + 8u), "l"(P.vz + q0 + q) : "memory");
    }
  }
  for (int q = 4 * tid; q < n_loc; q += 4 * TM::kN) *reinterpret_cast<int4 *>(S.cnt + q) = make_int4(0, 0, 0, 0);
  if (tid < 8) S.misc[tid] = 0;
  T.sync();
  // cell discovery (order of the active list is irrelevant to the results)
  for (int c = c_lo + tid; c < c_hi; c += TM::kN) {
    const int gs = __ldg(P.cell_start + c), N = __ldg(P.cell_start + c + 1) - gs;
    if (N == 1) S.cnt[gs - q0] = 1;  // lone particle (low half = its first bucket): keeps bucket positions aligned with slots
    if (N < 2) continue;
    const int a = atomicAdd(&S.misc[MI_NACT], 1);
    if (a >= CK::AMAX) continue;
    int M = N >> 1;
    const int req = P.pairs_count ? __ldg(P.pairs_count + c) : P.pairs_per_cell;
    if (req >= 0 && req < M) M = req;
    const int nseg = (N + kSeg - 1) / kSeg;
    const int seg0 = atomicAdd(&S.misc[MI_NSEG], nseg);
    CellInfo ci;
    ci.ux = ci.uy = ci.uz = ci.theta = 0.f;
    ci.cell = c;
    ci.pair_off = atomicAdd(&S.misc[MI_NPAIRS], M);
    ci.start = (uint16_t)(gs - q0);
    ci.N = (uint16_t)N;
    ci.M = (uint16_t)M;
    ci.seg0 = (uint16_t)seg0;
    ci.collided = (M > 0 && !(P.flags & DSMC_F_ACCEPT)) ? 1 : 0;
    ci.pad[0] = ci.pad[1] = ci.pad[2] = 0;
    S.cells[a] = ci;
    for (int i = 0; i < nseg; ++i) S.segs[seg0 + i] = (uint32_t)a | ((uint32_t)i << 16);
  }
  asm volatile("cp.async.wait_all;" ::: "memory");
  T.sync();
  if (S.misc[MI_NACT] > CK::AMAX) return -1;
  if (S.misc[MI_NACT] == 0) return 0;
  return n_loc;
}

// pre-collision segment sums + pairing keys + bucket counts; then cell finalisation + sort
template <class TM, class CK>
__device__ void chunk_pre_and_sort(const TM &T, const StepParams &P, CK &S, int n_loc) {
  const int tid = T.tid, lane = tid & 31, warp = tid >> 5;
  const int n_act = S.misc[MI_NACT], n_seg = S.misc[MI_NSEG];
  for (int sg = warp; sg < n_seg; sg += TM::kW) {
    const uint32_t e = S.segs[sg];
    const int a = e & 0xFFFFu, piece = e >> 16;
    const CellInfo &ci = S.cells[a];
    const int start = ci.start, N = ci.N, M = ci.M, pair_off = ci.pair_off;
    const uint32_t cell = (uint32_t)ci.cell + P.cell_base;
    const int lo = start + piece * kSeg, hi = min(lo + kSeg, start + N);
    // pivot = mean of the cell's first (up to) 32 particles: identical in every warp that works on this cell,
    // and close enough to the cell mean that Theta = sum d^2 - N |mean d|^2 loses no digits to cancellation
    float4 pv;
    {
      const int m = min(N, 32);
      const float4 f = lane < m ? S.v[start + lane] : make_float4(0.f, 0.f, 0.f, 0.f);
      const float im = 1.0f / (float)m;
      const float t = warp_sum4_t(f.x, f.y, f.z, 0.f, lane) * im;
      pv.x = __shfl_sync(0xffffffffu, t, 0);
      pv.y = __shfl_sync(0xffffffffu, t, 8);
      pv.z = __shfl_sync(0xffffffffu, t, 16);
      pv.w = 0.f;
      if (lane == 0 && piece == 0) {  // parked in the cell record until the finalisation below replaces it by u
        S.cells[a].ux = pv.x;
        S.cells[a].uy = pv.y;
        S.cells[a].uz = pv.z;
      }
    }
    float sx = 0.f, sy = 0.f, sz = 0.f, s2 = 0.f;
#pragma unroll
    for (int r = 0; r < kSeg / 32; ++r) {  // the segment's four rows: loads issued together
      const int q = lo + lane + 32 * r;
      if (q < hi) {
        const float4 v = S.v[q];
        const float dx = v.x - pv.x, dy = v.y - pv.y, dz = v.z - pv.z;
        sx += dx; sy += dy; sz += dz;
        s2 = fmaf(dx, dx, s2); s2 = fmaf(dy, dy, s2); s2 = fmaf(dz, dz, s2);
      }
    }
    {
      const float t = warp_sum4_t(sx, sy, sz, s2, lane);
      if ((lane & 7) == 0) reinterpret_cast<float *>(&S.part[sg])[lane >> 3] = t;
    }
    if (CK::REPLACE) {  // no matching to build: pair list only, and clear the change accumulators
      for (int q = lo + lane; q < hi; q += 32) {
        reinterpret_cast<float *>(S.key)[q] = 0.f;
        reinterpret_cast<float *>(S.cnt)[q] = 0.f;
        reinterpret_cast<float *>(S.ord)[q] = 0.f;
      }
      const int s_hi = min(M, (piece + 1) * (kSeg / 2));
      for (int s = piece * (kSeg / 2) + lane; s < s_hi; s += 32)
        S.pairs[pair_off + s] = (uint32_t)(start + 2 * s) | ((uint32_t)a << 16);
      continue;
    }
    // pairing keys: Philox block blk serves slots 4 blk .. 4 blk + 3 of the cell (stream 0)
    const int b_hi = min((piece + 1) * (kSeg / 4), (N + 3) >> 2);
    for (int blk = piece * (kSeg / 4) + lane; blk < b_hi; blk += 32) {
      const uint4 r = philox4x32_10((uint32_t)blk, cell, P.step, 0u, P.seed_lo, P.seed_hi);
      const uint32_t k[4] = {r.x, r.y, r.z, r.w};
      const int p = 4 * blk;
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        if (p + w < N) {
          S.key[start + p + w] = k[w];
          if (CK::PACK2N) {
            const int b2 = (int)__umulhi(k[w], 2u * (uint32_t)N);  // 2 N buckets per cell, two 16-bit counters per int
            atomicAdd(&S.cnt[start + (b2 >> 1)], (b2 & 1) ? 0x10000 : 1);
          } else {
            atomicAdd(&S.cnt[start + (int)__umulhi(k[w], (uint32_t)N)], 1);
          }
        }
      }
      const int s = p >> 1;
      if (s < M) S.pairs[pair_off + s] = (uint32_t)(start + p) | ((uint32_t)a << 16);
      if (s + 1 < M) S.pairs[pair_off + s + 1] = (uint32_t)(start + p + 2) | ((uint32_t)a << 16);
    }
  }
  T.sync();
  // cell finalisation: u = pivot + mean(d), Theta = sum d^2 - N |mean(d)|^2   (eq. 10)
  for (int a = tid; a < n_act; a += TM::kN) {
    CellInfo &ci = S.cells[a];
    const int N = ci.N, nseg = (N + kSeg - 1) / kSeg;
    double sx = 0, sy = 0, sz = 0, s2 = 0;
    for (int i = 0; i < nseg; ++i) {
      const float4 p = S.part[ci.seg0 + i];
      sx += p.x; sy += p.y; sz += p.z; s2 += p.w;
    }
    const double inv = 1.0 / N;
    const double dx = sx * inv, dy = sy * inv, dz = sz * inv;
    ci.ux = (float)((double)ci.ux + dx);  // pivot + mean(d)
    ci.uy = (float)((double)ci.uy + dy);
    ci.uz = (float)((double)ci.uz + dz);
    ci.theta = (float)fmax(s2 - N * (dx * dx + dy * dy + dz * dz), 0.0);  // a cold cell may round below zero
  }
  if (CK::REPLACE) {  // pairs are drawn, not matched: nothing to sort
    T.sync();
    return;
  }
  block_excl_scan_coalesced<TM, CK::PACK2N>(T, S.cnt, n_loc, S.misc + MI_SCAN);
  // placement, one warp per segment (cell constants in registers): cnt[bucket] ends as the bucket's end
  for (int sg = warp; sg < n_seg; sg += TM::kW) {
    const uint32_t e = S.segs[sg];
    const CellInfo &ci = S.cells[e & 0xFFFFu];
    const int start = ci.start, N = ci.N, piece = e >> 16;
    const int lo = start + piece * kSeg, hi = min(lo + kSeg, start + N);
#pragma unroll
    for (int r = 0; r < kSeg / 32; ++r) {
      const int q = lo + lane + 32 * r;
      if (q >= hi) continue;
      if (CK::PACK2N) {
        const int b2 = (int)__umulhi(S.key[q], 2u * (uint32_t)N);
        const uint32_t old = (uint32_t)atomicAdd(&S.cnt[start + (b2 >> 1)], (b2 & 1) ? 0x10000 : 1);
        S.ord[(b2 & 1) ? (old >> 16) : (old & 0xFFFFu)] = (uint16_t)q;
      } else {
        const int bkt = start + (int)__umulhi(S.key[q], (uint32_t)N);
        S.ord[atomicAdd(&S.cnt[bkt], 1)] = (uint16_t)q;
      }
    }
  }
  T.sync();
  // in-bucket ranking by (key, slot): buckets hold ~1 particle on average (~0.5 with PACK2N).  The first bucket of a cell
  // begins at the cell's first slot, every other one where the previous bucket ends.
  for (int sg = warp; sg < n_seg; sg += TM::kW) {
    const uint32_t e = S.segs[sg];
    const CellInfo &ci = S.cells[e & 0xFFFFu];
    const int start = ci.start, N = ci.N, piece = e >> 16;
    const int lo = start + piece * kSeg, hi = min(lo + kSeg, start + N);
    for (int q = lo + lane; q < hi; q += 32) {
      const uint32_t k = S.key[q];
      int b0, b1;
      if (CK::PACK2N) {
        const int b2 = 2 * start + (int)__umulhi(k, 2u * (uint32_t)N);  // bucket index in 16-bit units
        const uint16_t *c16 = reinterpret_cast<const uint16_t *>(S.cnt);
        b0 = b2 > 2 * start ? c16[b2 - 1] : start;
        b1 = c16[b2];
      } else {
        const int bkt = start + (int)__umulhi(k, (uint32_t)N);
        b0 = bkt > start ? S.cnt[bkt - 1] : start;
        b1 = S.cnt[bkt];
      }
      int rank = 0;
      if (b1 - b0 > 1) {
#pragma unroll 1
        for (int t = b0; t < b1; ++t) {
          const int o = S.ord[t];
          const uint32_t ko = S.key[o];
          rank += (ko < k || (ko == k && o < q)) ? 1 : 0;
        }
      }
      S.pi[b0 + rank] = (uint16_t)q;
    }
  }
  T.sync();
}

// ---------------------------------------------------------------------------------------------
// Per-pair helpers
// ---------------------------------------------------------------------------------------------
struct PairCtx {
  int a, s, i, j, start;  // active cell, pair slot, local particle indices, cell's first slot
  uint32_t cell;
  float4 vi, vj;
  float gx, gy, gz, g2;
  bool acc;
  float U_b, U_eps;
};

// the two members of pair t (from the matching, or drawn with replacement), their velocities and relative
// velocity (eq. 1)
template <class CK>
__device__ __forceinline__ PairCtx pair_load(const StepParams &P, const CK &S, int t) {
  PairCtx c;
  const uint32_t e = S.pairs[t];
  const int pos = e & 0xFFFFu;
  c.a = e >> 16;
  const CellInfo &ci = S.cells[c.a];
  c.start = ci.start;
  c.cell = (uint32_t)ci.cell;
  c.s = (pos - c.start) >> 1;
  if (CK::REPLACE) {  // stream 4: i = mulhi(R0, N), j = mulhi(R1, N - 1) + (j >= i)
    const uint4 r = philox4x32_10((uint32_t)c.s, c.cell + P.cell_base, P.step, 4u, P.seed_lo, P.seed_hi);
    const int N = ci.N;
    const int i = (int)__umulhi(r.x, (uint32_t)N);
    int j = (int)__umulhi(r.y, (uint32_t)(N - 1));
    j += (j >= i) ? 1 : 0;
    c.i = c.start + i;
    c.j = c.start + j;
  } else {
    c.i = S.pi[pos];
    c.j = S.pi[pos + 1];
  }
  c.vi = S.v[c.i];
  c.vj = S.v[c.j];
  c.gx = c.vi.x - c.vj.x;  // eq. 1
  c.gy = c.vi.y - c.vj.y;
  c.gz = c.vi.z - c.vj.z;
  c.g2 = fmaf(c.gx, c.gx, fmaf(c.gy, c.gy, c.gz * c.gz));
  c.acc = true;
  c.U_b = 0.f;
  c.U_eps = 0.f;
  return c;
}

template <class CK>
__device__ __forceinline__ PairCtx pair_setup(const StepParams &P, const CK &S, int t, bool need_randoms) {
  PairCtx c = pair_load(P, S, t);
  const bool accept = (P.flags & DSMC_F_ACCEPT) && P.cap != nullptr;
  if (need_randoms || accept) {
    // stream 1: one block per two pair slots, (U_b, U_eps) = words 2(s&1), 2(s&1)+1 of block s>>1
    const uint4 r = philox4x32_10((uint32_t)c.s >> 1, c.cell + P.cell_base, P.step, 1u, P.seed_lo, P.seed_hi);
    c.U_b = u01((c.s & 1) ? r.z : r.x);
    c.U_eps = u01((c.s & 1) ? r.w : r.y);
    if (accept) {  // stream 3: U_acc = word s&3 of block s>>2
      const uint4 ra = philox4x32_10((uint32_t)c.s >> 2, c.cell + P.cell_base, P.step, 3u, P.seed_lo, P.seed_hi);
      const float cap = __ldg(P.cap + c.cell);
      const float g = sqrtf(c.g2);
      const float w = (P.op == 0) ? P.vhs_c * powf(g, P.vhs_e) : g;  // sigma_T(g) g  |  g
      c.acc = u01(word_of(ra, (uint32_t)c.s & 3u)) * cap < w;
    }
  }
  return c;
}

template <class CK>
__device__ __forceinline__ void pair_commit(const StepParams &P, CK &S, const PairCtx &c, float px, float py,
                                            float pz, float aux, int q0) {
  if (c.acc && CK::REPLACE) {
    // batch semantics: v_i' - v_i = (g' - g) / 2 = -(v_j' - v_j) (eqs. 6-8) is added to the particle's change;
    // S.v keeps the pre-collision velocities until chunk_finish applies the sums
    float *dx = reinterpret_cast<float *>(S.key), *dy = reinterpret_cast<float *>(S.cnt),
          *dz = reinterpret_cast<float *>(S.ord);
    const float hx = 0.5f * (px - c.gx), hy = 0.5f * (py - c.gy), hz = 0.5f * (pz - c.gz);
    atomicAdd(dx + c.i, hx); atomicAdd(dy + c.i, hy); atomicAdd(dz + c.i, hz);
    atomicAdd(dx + c.j, -hx); atomicAdd(dy + c.j, -hy); atomicAdd(dz + c.j, -hz);
    if (P.flags & DSMC_F_ACCEPT) S.cells[c.a].collided = 1;
  } else if (c.acc) {  // eqs. 6-8
    const float cx = 0.5f * (c.vi.x + c.vj.x), cy = 0.5f * (c.vi.y + c.vj.y), cz = 0.5f * (c.vi.z + c.vj.z);
    S.v[c.i] = make_float4(fmaf(0.5f, px, cx), fmaf(0.5f, py, cy), fmaf(0.5f, pz, cz), 0.f);
    S.v[c.j] = make_float4(fmaf(-0.5f, px, cx), fmaf(-0.5f, py, cy), fmaf(-0.5f, pz, cz), 0.f);
    if (P.flags & DSMC_F_ACCEPT) S.cells[c.a].collided = 1;
  }
  if (P.dump_any) {
    const int64_t d = (int64_t)q0 + c.start + c.s;
    if (P.dump.pair_i) P.dump.pair_i[d] = c.i - c.start;
    if (P.dump.pair_j) P.dump.pair_j[d] = c.j - c.start;
    if (P.dump.accepted) P.dump.accepted[d] = c.acc ? 1 : 0;
    if (P.dump.gprime) { P.dump.gprime[3 * d] = px; P.dump.gprime[3 * d + 1] = py; P.dump.gprime[3 * d + 2] = pz; }
    if (P.dump.aux) P.dump.aux[d] = aux;
  }
}

// Rotation of g by deflection chi and azimuth eps = 2 pi U_eps (Q16).  MUFU sin/cos on
// arguments inside [-pi, pi] (abs. error 2^-21.4): eps is taken as 2 pi (U - 1/2) with both signs flipped.
__device__ __forceinline__ void rotate_fast(const PairCtx &c, float chi, float U_eps, float &px, float &py,
                                            float &pz) {
  float sc, cc, se, ce;
  __sincosf(chi, &sc, &cc);
  __sincosf(6.283185307179586f * (U_eps - 0.5f), &se, &ce);
  se = -se;
  ce = -ce;
  const float gp2 = fmaf(c.gy, c.gy, c.gz * c.gz);
  const float g = c.g2 * rsqrtf(c.g2);
  if (gp2 <= 1e-30f * c.g2 * 1e-30f) {  // g_perp <= 1e-30 g
    px = c.gx * cc;
    py = fabsf(c.gx) * sc * ce;
    pz = fabsf(c.gx) * sc * se;
    return;
  }
  const float inv = rsqrtf(gp2), gperp = gp2 * inv;
  const float sci = sc * inv;
  px = fmaf(c.gx, cc, gperp * sc * se);
  py = fmaf(c.gy, cc, sci * (g * c.gz * ce - c.gx * c.gy * se));
  pz = fmaf(c.gz, cc, -sci * (g * c.gy * ce + c.gx * c.gz * se));
}

// table coordinate t_E = (ln x - lnE_min) (nE-1)/(lnE_max-lnE_min) from x = E_r/k_B, with the exponent
// and mantissa of x handled separately (MUFU.LG2 only sees [1,2), abs. error 2^-22)
__device__ __forceinline__ float table_tE(const ChiTableDev &T, float x) {
  const int xi = __float_as_int(x);
  const float e = (float)((xi >> 23) - 127);
  const float m = __int_as_float((xi & 0x007FFFFF) | 0x3F800000);
  return fmaf(__log2f(m), T.c1, fmaf(e, T.c1, T.c0));
}

// bilinear chi(E~, b~) from the L2-resident quad table, coordinates clamped (Q13).
// quad[iE (nB-1) + iB] = (chi[iE][iB], chi[iE][iB+1], chi[iE+1][iB], chi[iE+1][iB+1]): one 16 B load.
__device__ __forceinline__ float chi_table_t(const ChiTableDev &T, float tE, float tB) {
  tE = fminf(fmaxf(tE, 0.f), (float)(T.nE - 1));
  tB = fminf(fmaxf(tB, 0.f), (float)(T.nB - 1));
  const int iE = min((int)tE, T.nE - 2), iB = min((int)tB, T.nB - 2);
  const float fE = tE - (float)iE, fB = tB - (float)iB;
  const float4 q = __ldg(T.quad + (size_t)iE * (T.nB - 1) + iB);
  const float lo = fmaf(fB, q.y - q.x, q.x), hi = fmaf(fB, q.w - q.z, q.z);
  return fmaf(fE, hi - lo, lo);
}

// ---------------------------------------------------------------------------------------------
// finish: post-collision sums, matching coefficients, single coalesced store
// ---------------------------------------------------------------------------------------------
template <class TM, class CK>
__device__ void chunk_finish(const TM &T, const StepParams &P, CK &S, int n_loc, int q0) {
  const int tid = T.tid, lane = tid & 31, warp = tid >> 5;
  const int n_act = S.misc[MI_NACT], n_seg = S.misc[MI_NSEG];
  constexpr bool replace = CK::REPLACE;
  if (P.flags & DSMC_F_MOMENT_MATCH) {
    for (int sg = warp; sg < n_seg; sg += TM::kW) {
      const uint32_t e = S.segs[sg];
      const int a = e & 0xFFFFu, piece = e >> 16;
      const CellInfo &ci = S.cells[a];
      if (!ci.collided) continue;
      const int lo = ci.start + piece * kSeg, hi = min(lo + kSeg, (int)ci.start + (int)ci.N);
      const float ux = ci.ux, uy = ci.uy, uz = ci.uz;
      float sx = 0.f, sy = 0.f, sz = 0.f, s2 = 0.f;
#pragma unroll
      for (int r = 0; r < kSeg / 32; ++r) {
        const int q = lo + lane + 32 * r;
        if (q < hi) {
          float4 v = S.v[q];
          if (replace) {  // with-replacement selection: apply the accumulated changes (this thread owns slot q)
            v.x += reinterpret_cast<const float *>(S.key)[q];
            v.y += reinterpret_cast<const float *>(S.cnt)[q];
            v.z += reinterpret_cast<const float *>(S.ord)[q];
            S.v[q] = v;
          }
          const float dx = v.x - ux, dy = v.y - uy, dz = v.z - uz;
          sx += dx; sy += dy; sz += dz;
          s2 = fmaf(dx, dx, s2); s2 = fmaf(dy, dy, s2); s2 = fmaf(dz, dz, s2);
        }
      }
      const float t = warp_sum4_t(sx, sy, sz, s2, lane);
      if ((lane & 7) == 0) reinterpret_cast<float *>(&S.part[sg])[lane >> 3] = t;
    }
    T.sync();
    for (int a = tid; a < n_act; a += TM::kN) {
      CellInfo &ci = S.cells[a];
      double alpha = 1.0, bx = 0.0, by = 0.0, bz = 0.0;
      if (ci.collided) {
        const int N = ci.N, nseg = (N + kSeg - 1) / kSeg;
        double sx = 0, sy = 0, sz = 0, s2 = 0;
        for (int i = 0; i < nseg; ++i) {
          const float4 p = S.part[ci.seg0 + i];
          sx += p.x; sy += p.y; sz += p.z; s2 += p.w;
        }
        const double inv = 1.0 / N;
        const double dx = sx * inv, dy = sy * inv, dz = sz * inv;  // u_post - u_pre
        const double th_post = s2 - N * (dx * dx + dy * dy + dz * dz);
        const double ux = ci.ux, uy = ci.uy, uz = ci.uz;
        if (P.flags & DSMC_F_MATCH_ENERGY_ONLY) {  // literal eq. 11: v <- v sqrt(E_pre / E_post)
          const double px = ux + dx, py = uy + dy, pz = uz + dz;
          const double e_pre = (double)ci.theta + N * (ux * ux + uy * uy + uz * uz);
          const double e_post = th_post + N * (px * px + py * py + pz * pz);
          if (e_post > 0.0) alpha = sqrt(e_pre / e_post);
        } else {  // v <- u_pre + alpha (v - u_post)
          if (th_post > 0.0) alpha = sqrt((double)ci.theta / th_post);
          bx = ux - alpha * (ux + dx);
          by = uy - alpha * (uy + dy);
          bz = uz - alpha * (uz + dz);
        }
      }
      // alpha is 1 + O(1e-7): FP32 cannot resolve it (spacing 6e-8 .. 1.2e-7 around 1, a biased correction that
      // showed as a -2.6e-8 per step energy drift), so the store applies v + (alpha - 1) v + B with alpha - 1 in FP32
      ci.ux = (float)bx; ci.uy = (float)by; ci.uz = (float)bz; ci.theta = (float)(alpha - 1.0);
    }
    T.sync();
    // store, one warp per segment: v <- v + (alpha - 1) v + B with the cell's coefficients in registers.  Cells in
    // which nothing collided (and particles of cells with N < 2) are unchanged and not written.
    for (int sg = warp; sg < n_seg; sg += TM::kW) {
      const uint32_t e = S.segs[sg];
      const CellInfo &ci = S.cells[e & 0xFFFFu];
      if (!ci.collided) continue;
      const float4 co = *reinterpret_cast<const float4 *>(&ci);
      const int piece = e >> 16;
      const int lo = ci.start + piece * kSeg, hi = min(lo + kSeg, (int)ci.start + (int)ci.N);
#pragma unroll
      for (int r = 0; r < kSeg / 32; ++r) {
        const int q = lo + lane + 32 * r;
        if (q < hi) {
          const float4 v = S.v[q];
          P.vx[q0 + q] = fmaf(co.w, v.x, v.x + co.x);
          P.vy[q0 + q] = fmaf(co.w, v.y, v.y + co.y);
          P.vz[q0 + q] = fmaf(co.w, v.z, v.z + co.z);
        }
      }
    }
  } else {
    for (int sg = warp; sg < n_seg; sg += TM::kW) {
      const uint32_t e = S.segs[sg];
      const CellInfo &ci = S.cells[e & 0xFFFFu];
      if (!ci.collided) continue;
      const int piece = e >> 16;
      const int lo = ci.start + piece * kSeg, hi = min(lo + kSeg, (int)ci.start + (int)ci.N);
      for (int q = lo + lane; q < hi; q += 32) {
        float4 v = S.v[q];
        if (replace) {
          v.x += reinterpret_cast<const float *>(S.key)[q];
          v.y += reinterpret_cast<const float *>(S.cnt)[q];
          v.z += reinterpret_cast<const float *>(S.ord)[q];
        }
        P.vx[q0 + q] = v.x;
        P.vy[q0 + q] = v.y;
        P.vz[q0 + q] = v.z;
      }
    }
  }
}

}  // namespace dsmc
