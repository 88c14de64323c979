// The cell team: everything one team of NT threads does to one cell of the fused collision step
// (dsmc_cells.cu holds the description of the phases and the kernels).  Product code only.
#pragma once
#include "dsmc_device.cuh"
#include "dsmc_internal.h"

namespace dsmc {

constexpr int kRankWin = 4;   // bucket members compared without a loop

struct CellLists {
  int4 *list[3];  // (cell, first slot, N, M) by size class: N <= 256, <= 1024, <= 2048
  int32_t *ctr;   // [0..2] entries of each list
  int32_t *work;  // [0..2] work counters of the kernels that walk the lists
};

// Four warp sums for the price of six shuffles: returns the total of a in lanes 0-7, b in 8-15, c in 16-23, d in 24-31.
__device__ __forceinline__ float warp_sum4(float a, float b, float c, float d, int lane) {
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

// packed FP32 pairs (FADD2 / FFMA2 on sm_100a): two rows of a thread's particles per instruction
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(f32x2 v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ float hsum2(f32x2 v) { float a, b; upk2(v, a, b); return a + b; }

// MUFU wrappers with flush-to-zero (no denormal pre-scaling code around them)
__device__ __forceinline__ float mufu_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_sqrt(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_sin(float x) { float y; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_cos(float x) { float y; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// table coordinate t_E = (ln x - lnE_min) (nE-1)/(lnE_max-lnE_min) from x = E_r/k_B, exponent and mantissa of x
// handled separately (MUFU.LG2 only sees [1,2), abs. error 2^-22)
__device__ __forceinline__ float cells_tE(const ChiTableDev &T, float x) {
  const int xi = __float_as_int(x);
  const float e = (float)((xi >> 23) - 127);
  const float m = __int_as_float((xi & 0x007FFFFF) | 0x3F800000);
  return fmaf(mufu_lg2(m), T.c1, fmaf(e, T.c1, T.c0));
}

// bilinear chi(E~, b~) from the L2-resident quad table, coordinates clamped (Q13)
__device__ __forceinline__ float cells_chi(const ChiTableDev &T, float tE, float tB) {
  tE = fminf(fmaxf(tE, 0.f), T.fE1);
  tB = fminf(fmaxf(tB, 0.f), T.fB1);
  const int iE = min((int)tE, T.nE - 2), iB = min((int)tB, T.nB - 2);
  const float fE = tE - (float)iE, fB = tB - (float)iB;
  const float4 q = T.tex ? tex1Dfetch<float4>(T.tex, iE * (T.nB - 1) + iB) : __ldg(T.quad + (size_t)iE * (T.nB - 1) + iB);
  const float lo = fmaf(fB, q.y - q.x, q.x), hi = fmaf(fB, q.w - q.z, q.z);
  return fmaf(fE, hi - lo, lo);
}

// Rotation of g by deflection chi and azimuth eps (Q16); eps in [-pi, pi) (the azimuth is uniform, so
// 2 pi (U - 1/2) serves as 2 pi U with both signs flipped), MUFU sin / cos.
__device__ __forceinline__ void cells_rotate(float gx, float gy, float gz, float g2, float chi, float eps, float &px,
                                             float &py, float &pz) {
  const float sc = mufu_sin(chi), cc = mufu_cos(chi);
  const float se = -mufu_sin(eps), ce = -mufu_cos(eps);
  const float gp2 = fmaf(gy, gy, gz * gz);
  const float g = g2 * mufu_rsqrt(g2);
  const float inv = mufu_rsqrt(gp2), gperp = gp2 * inv;
  const float sci = sc * inv;
  px = fmaf(gx, cc, gperp * sc * se);
  py = fmaf(gy, cc, sci * (g * gz * ce - gx * gy * se));
  pz = fmaf(gz, cc, -sci * (g * gy * ce + gx * gz * se));
  if (__builtin_expect(gp2 <= 1e-30f * g2 * 1e-30f, 0)) {  // g_perp <= 1e-30 g: the other two axes
    px = gx * cc;
    py = fabsf(gx) * sc * ce;
    pz = fabsf(gx) * sc * se;
  }
}

// Philox4x32-10 with the round keys as constant-bank operands (StepParams::rk): per round two 32 x 32 -> 64 bit
// products and two three-input xors.
__device__ __forceinline__ uint4 cells_philox(const StepParams &P, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    c0 = (uint32_t)(p1 >> 32) ^ c1 ^ P.rk[2 * r];
    c2 = (uint32_t)(p0 >> 32) ^ c3 ^ P.rk[2 * r + 1];
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
  }
  return make_uint4(c0, c1, c2, c3);
}

// In-bucket rank of composite e: the number of smaller composites among the first min(m, 4) members of its bucket
// (shared address addr), added to rank.  Straight-line predicated code: one predicate per member position, one
// predicated load, one compare, one predicated add each.
__device__ __forceinline__ void cells_rank4(uint32_t &rank, uint32_t addr, uint32_t e, uint32_t m) {
  asm volatile(
      "{\n\t.reg .pred q1, q2, q3, p;\n\t.reg .u32 v0, v1, v2, v3;\n\t"
      "setp.gt.u32 q1, %3, 1;\n\t"
      "setp.gt.u32 q2, %3, 2;\n\t"
      "setp.gt.u32 q3, %3, 3;\n\t"
      "mov.u32 v0, %2;\n\t"  // a member that is not there compares as e itself: not smaller
      "mov.u32 v1, %2;\n\t"
      "mov.u32 v2, %2;\n\t"
      "mov.u32 v3, %2;\n\t"
      "@q1 ld.shared.u32 v0, [%1];\n\t"
      "@q1 ld.shared.u32 v1, [%1+4];\n\t"
      "@q2 ld.shared.u32 v2, [%1+8];\n\t"
      "@q3 ld.shared.u32 v3, [%1+12];\n\t"
      "setp.lt.u32 p, v0, %2;\n\t"
      "@p add.u32 %0, %0, 1;\n\t"
      "setp.lt.u32 p, v1, %2;\n\t"
      "@p add.u32 %0, %0, 1;\n\t"
      "setp.lt.u32 p, v2, %2;\n\t"
      "@p add.u32 %0, %0, 1;\n\t"
      "setp.lt.u32 p, v3, %2;\n\t"
      "@p add.u32 %0, %0, 1;\n\t}"
      : "+r"(rank)
      : "r"(addr), "r"(e), "r"(m)
      : "memory");
}

// Placement of one key (straight-line predicated code).  bo = bucket | arrival index << 16; the bucket's counter
// holds (start | members << 16).  A key alone in its bucket is ranked: pi[start] = its byte offset.  Otherwise its
// composite goes to K2[start + arrival index] and the counter word is returned for the ranking (0 = nothing to rank).
__device__ __forceinline__ uint32_t cells_place(uint32_t bo, int p, int N, uint32_t comp, uint32_t cnt_s, uint32_t k2_s,
                                                uint32_t pi_s) {
  uint32_t out;
  asm volatile(
      "{\n\t.reg .pred qv, q1, qm;\n\t.reg .u32 w, b0, m, a, t;\n\t.reg .u16 h;\n\t"
      "setp.lt.s32 qv, %2, %3;\n\t"
      "and.b32 a, %1, 0xffff;\n\t"
      "mad.lo.u32 a, a, 4, %5;\n\t"
      "mov.u32 w, 0;\n\t"
      "@qv ld.shared.u32 w, [a];\n\t"
      "shr.u32 m, w, 16;\n\t"
      "and.b32 b0, w, 0xffff;\n\t"
      "setp.eq.u32 q1, m, 1;\n\t"
      "setp.gt.u32 qm, m, 1;\n\t"
      "mad.lo.u32 t, b0, 2, %7;\n\t"
      "shl.b32 a, %2, 2;\n\t"
      "cvt.u16.u32 h, a;\n\t"
      "@q1 st.shared.u16 [t], h;\n\t"
      "shr.u32 t, %1, 16;\n\t"
      "add.u32 t, t, b0;\n\t"
      "mad.lo.u32 t, t, 4, %6;\n\t"
      "@qm st.shared.u32 [t], %4;\n\t"
      "selp.u32 %0, w, 0, qm;\n\t}"
      : "=r"(out)
      : "r"(bo), "r"(p), "r"(N), "r"(comp), "r"(cnt_s), "r"(k2_s), "r"(pi_s)
      : "memory");
  return out;
}

// OP 0: chi from the table.  OP 2: chi-MLP through the CTA's tensor-core MLP server (SRV, dsmc_cells_mlp.cu).
struct NoServer {
  int buf;
  __device__ int acquire(int, uint32_t *) { return 0; }
  __device__ void write_row(int, int, float, float) {}
  __device__ void publish(int) {}
  __device__ void wait(int) {}
};

template <int NT, int OP = 0, class SRV = NoServer>
struct CellTeam {
  static constexpr int C = 8 * NT;  // slots: a thread holds 8 particles / 8 keys / 8 bucket counters
  static constexpr int NW = NT / 32;
  float *X, *Y, *Z;   // [C] velocities of the cell
  uint32_t *cnt;      // [C] bucket counters, then (bucket start | members << 16)
  uint32_t *K2;       // [C] composites of the keys that share a bucket, in bucket order
  uint16_t *pi;       // [C] BYTE OFFSETS (4 slot) of the particles in ascending (key, slot) order
  float4 *part;       // [2][8] per-warp partial sums, before / after the collisions (NT > 32)
  int *misc;          // [0..7] warp totals of the scan, [8..11] next list entry, [12] any pair accepted
  int tid, bar;
  SRV *srv;

  static constexpr size_t bytes() { return (size_t)C * (12 + 4 + 4 + 2) + 3 * NT; }  // + part, misc (320 B, NT > 32)

  // base_s: shared-space address of the team's block.  It is made opaque to the compiler, which otherwise rebuilds
  // it from the special registers (6-8 instructions) in front of most shared-memory accesses instead of keeping it.
  __device__ __forceinline__ void init(uint32_t base_s, int tid_, int bar_) {
    tid = tid_;
    bar = bar_;
    asm volatile("" : "+r"(base_s));
    unsigned char *base = reinterpret_cast<unsigned char *>(__cvta_shared_to_generic(base_s));
    X = reinterpret_cast<float *>(base);
    Y = X + C;
    Z = Y + C;
    cnt = reinterpret_cast<uint32_t *>(Z + C);
    K2 = cnt + C;
    pi = reinterpret_cast<uint16_t *>(K2 + C);
    part = reinterpret_cast<float4 *>(pi + C);
    misc = reinterpret_cast<int *>(part + 16);
  }
  __device__ __forceinline__ void sync() const {
    if (NT == 32)
      __syncwarp();
    else
      asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(NT) : "memory");
  }

  // the list entry of index idx (thread 0 only); N = 0 when the list is exhausted
  __device__ __forceinline__ int4 entry(const int4 *list, int n_items, int idx) const {
    return idx < n_items ? __ldg(list + idx) : make_int4(0, 0, 0, 0);
  }
  __device__ __forceinline__ int4 share(int4 it) const {  // thread 0's entry to the whole team
    if (NT == 32) {
      it.x = __shfl_sync(0xffffffffu, it.x, 0);
      it.y = __shfl_sync(0xffffffffu, it.y, 0);
      it.z = __shfl_sync(0xffffffffu, it.z, 0);
      it.w = __shfl_sync(0xffffffffu, it.w, 0);
      return it;
    }
    return *reinterpret_cast<const int4 *>(misc + 8);
  }

  __device__ void run(const StepParams &P, const int4 *__restrict__ list, const int32_t *n_items_ptr, int32_t *work) {
    const int n_items = __ldg(n_items_ptr);
    int4 item = make_int4(0, 0, 0, 0);
    if (tid == 0) {
      item = entry(list, n_items, atomicAdd(work, 1));
      if (NT > 32) *reinterpret_cast<int4 *>(misc + 8) = item;
    }
    if (NT > 32) sync();
    item = share(item);
    if (NT > 32) sync();
    while (item.z > 0) item = cell(P, item, list, n_items, work);
  }

  // OP 2: two cells in flight per team, one in each of its two buffers: while the server works on the tile(s) of one
  // cell the team loads, sorts and submits the next one
  __device__ void run2(const StepParams &P, const int4 *__restrict__ list, const int32_t *n_items_ptr, int32_t *work,
                       uint32_t base0, uint32_t base1) {
    const int n_items = __ldg(n_items_ptr);
    const int t = tid, br = bar;
    init(base0, t, br);
    int4 item = make_int4(0, 0, 0, 0);
    if (tid == 0) {
      item = entry(list, n_items, atomicAdd(work, 1));
      if (NT > 32) *reinterpret_cast<int4 *>(misc + 8) = item;
    }
    if (NT > 32) sync();
    item = share(item);
    if (NT > 32) sync();
    int4 prev = make_int4(0, 0, 0, 0);
    int b = 0;
    while (item.z > 0 || prev.z > 0) {
      int4 nxt = make_int4(0, 0, 0, 0);
      if (item.z > 0) {
        init(b ? base1 : base0, t, br);
        srv->buf = b;
        nxt = cell<1>(P, item, list, n_items, work);
      }
      if (prev.z > 0) {
        init(b ? base0 : base1, t, br);
        srv->buf = b ^ 1;
        cell<2>(P, prev, list, n_items, work);
      }
      prev = item;
      item = nxt;
      b ^= 1;
    }
  }

  // team sums of (a, b, c, d): per-warp butterfly, then (NT > 32) the warps' partials through shared memory in a
  // fixed order.  `slot` selects the partial-sum buffer; contains one team barrier when NT > 32.
  __device__ __forceinline__ void team_sum4(float &a, float &b, float &c, float &d, int slot) const {
    const int lane = tid & 31, warp = tid >> 5;
    const float t = warp_sum4(a, b, c, d, lane);
    if (NT == 32) {
      a = __shfl_sync(0xffffffffu, t, 0);
      b = __shfl_sync(0xffffffffu, t, 8);
      c = __shfl_sync(0xffffffffu, t, 16);
      d = __shfl_sync(0xffffffffu, t, 24);
    } else {
      if ((lane & 7) == 0) reinterpret_cast<float *>(&part[8 * slot + warp])[lane >> 3] = t;
      sync();
      a = b = c = d = 0.f;
#pragma unroll
      for (int w = 0; w < NW; ++w) {
        const float4 p = part[8 * slot + w];
        a += p.x; b += p.y; c += p.z; d += p.w;
      }
    }
  }

  // Pairs of the cell: the thread owns pair slots 2 dp, 2 dp + 1, dp = tid + NT r, r = 0, 1 (one Philox block of
  // stream 1 serves both).  STAGE 0: chi from the table, rotation, commit.  STAGE 1 (chi-MLP): features of every pair
  // slot -> row ((2 r + k) 32 + lane) of the warp's tile in the MLP server's layer-1 operand; eps (or a sentinel for
  // a pair that does not collide) parked in cnt[].  STAGE 2: chi = exp(z) from the delivered outputs, rotation, commit.
  template <int STAGE>
  __device__ __forceinline__ bool pairs_phase(const StepParams &P, const int4 item, uint32_t cell_ctr, bool accept,
                                              int slot, float tfeat = 0.f) {
    const int lane = tid & 31, warp = tid >> 5;
    const int gs = item.y, M = item.w;
    bool any_acc = false;
    const float nBm1 = P.table.fB1;
    const char *Xb = reinterpret_cast<const char *>(X);
    float *park = reinterpret_cast<float *>(cnt) + 128 * warp;  // STAGE 1 -> 2: eps per row (cnt is dead by now)
    float *stage = reinterpret_cast<float *>(K2) + 256 * warp;  // STAGE 1: features [2][128]; STAGE 2: z [128]
    const float *zbuf = stage;
#pragma unroll 1
    for (int r = 0; r < 2; ++r) {  // not unrolled: the body is the largest piece of code of the kernel
      const int dp = tid + NT * r;
      const int s0 = 2 * dp;
      if (s0 < M) {
        const uint2 w2 = *reinterpret_cast<const uint2 *>(pi + 4 * dp);
        const bool v1 = s0 + 1 < M;
        uint32_t oi[2] = {w2.x & 0xFFFFu, w2.y & 0xFFFFu};
        uint32_t oj[2] = {w2.x >> 16, w2.y >> 16};
        if (!v1) { oi[1] = oi[0]; oj[1] = oj[0]; }
        float Ub[2] = {0.f, 0.f}, eps[2] = {0.f, 0.f}, Ua[2] = {0.f, 0.f}, cap = 0.f;
        if (STAGE != 2) {
          if (STAGE < 5) {  // (the VHS-NN stages 5, 6 draw no impact parameter and no azimuth)
            const uint4 rr = cells_philox(P, (uint32_t)dp, cell_ctr, P.step, 1u);
            // U_b = ((x >> 9) + 1/2) 2^-23 built from the float 1.f + (x >> 9) 2^-23; eps = 2 pi (U_eps - 1/2) likewise
            Ub[0] = __uint_as_float((rr.x >> 9) | 0x3F800000u) - 0.99999994f;
            Ub[1] = __uint_as_float((rr.z >> 9) | 0x3F800000u) - 0.99999994f;
            eps[0] = fmaf(__uint_as_float((rr.y >> 9) | 0x3F800000u) - 1.5f, 6.2831855f, 3.7450704e-7f);
            eps[1] = fmaf(__uint_as_float((rr.w >> 9) | 0x3F800000u) - 1.5f, 6.2831855f, 3.7450704e-7f);
          }
          if (accept) {  // stream 3: U_acc of pair slot s = word s & 3 of block s >> 2
            const uint4 ra = cells_philox(P, (uint32_t)dp >> 1, cell_ctr, P.step, 3u);
            Ua[0] = u01((dp & 1) ? ra.z : ra.x);
            Ua[1] = u01((dp & 1) ? ra.w : ra.y);
            cap = __ldg(P.cap + item.x);
          }
        }
        float vix[2], viy[2], viz[2], vjx[2], vjy[2], vjz[2];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const float *pi_ = reinterpret_cast<const float *>(Xb + oi[k]), *pj_ = reinterpret_cast<const float *>(Xb + oj[k]);
          vix[k] = pi_[0]; viy[k] = pi_[C]; viz[k] = pi_[2 * C];
          vjx[k] = pj_[0]; vjy[k] = pj_[C]; vjz[k] = pj_[2 * C];
        }
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const bool valid = k == 0 || v1;
          const int row = (2 * r + k) * 32 + lane;
          const float gx = vix[k] - vjx[k], gy = viy[k] - vjy[k], gz = viz[k] - vjz[k];  // eq. 1
          const float g2 = fmaf(gx, gx, fmaf(gy, gy, gz * gz));
          bool acc = valid;
          if (STAGE != 2) {
            // ab initio: constant cross-section, U g_max < g; VHS-NN: U (sigma g)_max < sigma_T(g) g
            if (accept) acc = valid && (Ua[k] * cap < (STAGE >= 5 ? P.vhs_c * powf(sqrtf(g2), P.vhs_e) : sqrtf(g2)));
          }
          if (STAGE == 5) {  // VHS-NN inputs (eqs. 1-3, Q1-Q3) -> pair arrays feat0 + k split_np
            if (valid) {
              float n0 = 0.f, n1 = 0.f, n2 = 0.f;
              if (P.flags & DSMC_F_NOISE) {
                const uint4 rn = cells_philox(P, (uint32_t)(s0 + k), cell_ctr, P.step, 2u);
                box_muller3(rn, n0, n1, n2);
                n0 *= P.noise_sigma; n1 *= P.noise_sigma; n2 *= P.noise_sigma;
              }
              float *f = P.feat0 + (int64_t)(gs >> 1) + s0 + k;
              const int64_t np = P.split_np;
              f[0] = gx * P.inv_sigma_v; f[np] = gy * P.inv_sigma_v; f[2 * np] = gz * P.inv_sigma_v;
              if (P.split_din == 8) {
                f[3 * np] = sqrtf(g2) * P.inv_sigma_v;
                f[4 * np] = tfeat;
                f[5 * np] = n0; f[6 * np] = n1; f[7 * np] = n2;
              } else {
                f[3 * np] = n0; f[4 * np] = n1; f[5 * np] = n2;
              }
            }
            continue;
          }
          if (STAGE == 1 || STAGE == 3) {  // chi-MLP inputs (Q15): ((E~ - E~min) / (E~max - E~min) clamped to [0, 1], b~)
            const float e = (0.6931471806f * mufu_lg2(P.e_coef * g2) - P.lnE_min) * P.inv_lnE_range;
            const float x0 = !(e > 0.f) ? 0.f : fminf(e, 1.f), x1 = mufu_sqrt(Ub[k]);
            if (STAGE == 1) {
              stage[row] = x0;
              stage[128 + row] = x1;
              park[row] = acc ? eps[k] : 1e30f;
            } else if (valid) {  // split form: the inputs go to the pair arrays, the rest is redone by the second pass
              const int64_t pp = (int64_t)(gs >> 1) + s0 + k;
              P.feat0[pp] = x0;
              P.feat1[pp] = x1;
            }
            continue;
          }
          float px = gx, py = gy, pz = gz, chi = 0.f;
          if (STAGE == 2) {
            eps[k] = park[row];
            acc = valid && eps[k] < 1e29f;
          }
          if (acc && STAGE == 6) {  // VHS-NN: outputs of the batch kernel -> eq. 5 (guard Q4) -> eqs. 6-8
            const int64_t pp = (int64_t)(gs >> 1) + s0 + k;
            const float h0 = __ldg(P.out3[0] + pp), h1 = __ldg(P.out3[1] + pp), h2 = __ldg(P.out3[2] + pp);
            const float hn = sqrtf(h0 * h0 + h1 * h1 + h2 * h2);
            chi = hn;  // (dumped as aux)
            if (P.flags & DSMC_F_ENERGY_SHELL) {
              if (hn >= P.shell_eps) {
                const float sc = sqrtf(g2) / hn;
                px = sc * h0; py = sc * h1; pz = sc * h2;
              }
            } else {
              px = P.sigma_v * h0; py = P.sigma_v * h1; pz = P.sigma_v * h2;
            }
            const float hx = px - gx, hy = py - gy, hz = pz - gz;
            float *qi = reinterpret_cast<float *>(const_cast<char *>(Xb) + oi[k]);
            float *qj = reinterpret_cast<float *>(const_cast<char *>(Xb) + oj[k]);
            qi[0] = fmaf(0.5f, hx, vix[k]); qi[C] = fmaf(0.5f, hy, viy[k]); qi[2 * C] = fmaf(0.5f, hz, viz[k]);
            qj[0] = fmaf(-0.5f, hx, vjx[k]); qj[C] = fmaf(-0.5f, hy, vjy[k]); qj[2 * C] = fmaf(-0.5f, hz, vjz[k]);
            any_acc = true;
          } else if (acc) {
            if (STAGE == 2) {
              chi = __expf(zbuf[row]);  // chi = expm1(softplus(z)) = exp(z)
            } else if (STAGE == 4) {
              chi = __ldg(P.chi_pair + (int64_t)(gs >> 1) + s0 + k);  // split form: chi of the batch kernel
            } else {
              // E~ = ln(m g^2 / (4 kB)), b~ = sqrt(U_b)
              chi = cells_chi(P.table, cells_tE(P.table, P.e_coef * g2), mufu_sqrt(Ub[k]) * nBm1);
            }
            if (g2 > 0.f) cells_rotate(gx, gy, gz, g2, chi, eps[k], px, py, pz);
            // eqs. 6-8 as v_i + (g' - g) / 2, v_j - (g' - g) / 2
            const float hx = px - gx, hy = py - gy, hz = pz - gz;
            float *qi = reinterpret_cast<float *>(const_cast<char *>(Xb) + oi[k]);
            float *qj = reinterpret_cast<float *>(const_cast<char *>(Xb) + oj[k]);
            qi[0] = fmaf(0.5f, hx, vix[k]); qi[C] = fmaf(0.5f, hy, viy[k]); qi[2 * C] = fmaf(0.5f, hz, viz[k]);
            qj[0] = fmaf(-0.5f, hx, vjx[k]); qj[C] = fmaf(-0.5f, hy, vjy[k]); qj[2 * C] = fmaf(-0.5f, hz, vjz[k]);
            any_acc = true;
          }
          if (P.dump_any && valid) {
            const int64_t d = (int64_t)gs + s0 + k;
            if (P.dump.pair_i) P.dump.pair_i[d] = (int32_t)(oi[k] >> 2);
            if (P.dump.pair_j) P.dump.pair_j[d] = (int32_t)(oj[k] >> 2);
            if (P.dump.accepted) P.dump.accepted[d] = acc ? 1 : 0;
            if (P.dump.gprime) { P.dump.gprime[3 * d] = px; P.dump.gprime[3 * d + 1] = py; P.dump.gprime[3 * d + 2] = pz; }
            if (P.dump.aux) P.dump.aux[d] = chi;
          }
        }
      } else if (STAGE == 1) {  // rows of pair slots that do not exist: defined inputs, nothing to collide
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          stage[(2 * r + k) * 32 + lane] = 0.f;
          stage[128 + (2 * r + k) * 32 + lane] = 0.f;
          park[(2 * r + k) * 32 + lane] = 1e30f;
        }
      }
    }
    return any_acc;
  }

  // one cell; returns the team's next list entry.  HALF 0: the whole cell.  OP 2 only: HALF 1 = up to the publication
  // of the warp's tile (returns the next entry), HALF 2 = from the delivery of z to the store: between the two the
  // team works on another cell in its other buffer (run2).
  template <int HALF = 0>
  __device__ __forceinline__ int4 cell(const StepParams &P, const int4 item, const int4 *__restrict__ list, int n_items,
                                       int32_t *work) {
    const int lane = tid & 31, warp = tid >> 5;
    const int gs = item.y, N = item.z, M = item.w;
    const uint32_t cell_ctr = (uint32_t)item.x + P.cell_base;
    const int Lb = 32 - __clz(N - 1);  // bucket = top Lb bits of the key; 2^Lb >= N buckets
    const int NB = 1 << Lb;
    const bool accept = (P.flags & DSMC_F_ACCEPT) && P.cap != nullptr;
    const float fN = (float)N, invN = 1.0f / fN;
    float ux = 0.f, uy = 0.f, uz = 0.f, theta = 0.f;
    int4 next = make_int4(0, 0, 0, 0);
    float *state = NT == 32 ? reinterpret_cast<float *>(part) : reinterpret_cast<float *>(misc + 16);
    if (HALF != 2) {
    int next_idx = 0;
    if (tid == 0) {
      next_idx = atomicAdd(work, 1);  // consumed after the loads below have landed
      if (NT > 32) misc[12] = 0;
    }
    // bucket counters: thread t owns [4 t, 4 t + 4) and [4 NT + 4 t, 4 NT + 4 t + 4): conflict-free 16-byte accesses
    if (4 * tid < NB) *reinterpret_cast<uint4 *>(cnt + 4 * tid) = make_uint4(0u, 0u, 0u, 0u);
    if (4 * (tid + NT) < NB) *reinterpret_cast<uint4 *>(cnt + 4 * (tid + NT)) = make_uint4(0u, 0u, 0u, 0u);
    // ---- load (12 B / particle) + pre-collision sums about the pivot (eq. 10) ----
    {
      const float *__restrict__ gx = P.vx + gs, *__restrict__ gy = P.vy + gs, *__restrict__ gz = P.vz + gs;
      float x[8], y[8], z[8];
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int q = tid + NT * r;
        x[r] = y[r] = z[r] = 0.f;
        if (q < N) {
          x[r] = __ldcs(gx + q);
          y[r] = __ldcs(gy + q);
          z[r] = __ldcs(gz + q);
        }
      }
      float pvx, pvy, pvz;
      {
        const int m32 = min(N, 32);
        float a = x[0], b = y[0], c = z[0];  // NT == 32: the first row is the cell's first 32 particles
        if (NT > 32) {
          a = b = c = 0.f;
          if (lane < m32) {
            a = __ldcs(gx + lane);
            b = __ldcs(gy + lane);
            c = __ldcs(gz + lane);
          }
        }
        const float t = warp_sum4(a, b, c, 0.f, lane) * (1.0f / (float)m32);
        pvx = __shfl_sync(0xffffffffu, t, 0);
        pvy = __shfl_sync(0xffffffffu, t, 8);
        pvz = __shfl_sync(0xffffffffu, t, 16);
      }
      // rows beyond the cell stand at the pivot (d = 0), so the sums need no predicates; two rows per instruction
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int q = tid + NT * r;
        if (q < N) {
          X[q] = x[r];
          Y[q] = y[r];
          Z[q] = z[r];
        } else {
          x[r] = pvx;
          y[r] = pvy;
          z[r] = pvz;
        }
      }
      float sx, sy, sz, s2;
      {
        const f32x2 px2 = pk2(pvx, pvx), py2 = pk2(pvy, pvy), pz2 = pk2(pvz, pvz);
        f32x2 ax = pk2(0.f, 0.f), ay = ax, az = ax, a2 = ax;
#pragma unroll
        for (int r = 0; r < 8; r += 2) {
          const f32x2 dx = sub2(pk2(x[r], x[r + 1]), px2), dy = sub2(pk2(y[r], y[r + 1]), py2),
                      dz = sub2(pk2(z[r], z[r + 1]), pz2);
          ax = add2(ax, dx); ay = add2(ay, dy); az = add2(az, dz);
          a2 = fma2(dx, dx, a2); a2 = fma2(dy, dy, a2); a2 = fma2(dz, dz, a2);
        }
        sx = hsum2(ax); sy = hsum2(ay); sz = hsum2(az); s2 = hsum2(a2);
      }
      team_sum4(sx, sy, sz, s2, 0);
      if (NT == 32) sync();  // counters zeroed before the first atomic (NT > 32: the barrier inside team_sum4)
      // u = pivot + mean(d); Theta = sum d^2 - N |mean d|^2: the pivot lies within a fraction of a thermal speed of
      // the mean, so the subtraction loses no digits
      const float mx = sx * invN, my = sy * invN, mz = sz * invN;
      ux = pvx + mx;
      uy = pvy + my;
      uz = pvz + mz;
      theta = fmaxf(s2 - fN * fmaf(mx, mx, fmaf(my, my, mz * mz)), 0.f);
    }
    if (tid == 0) next = entry(list, n_items, next_idx);
    if (OP == 4 || OP == 6) {  // split form, second pass: the pairing was made (and stored) by the first pass
      const uint16_t *__restrict__ gp = P.pi_g + gs;
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int q = tid + NT * r;
        if (q < N) pi[q] = __ldg(gp + q);
      }
    } else {
    // ---- pairing keys (stream 0: block blk serves slots 4 blk .. 4 blk + 3) and bucket counts ----
    // per key: comp = key << Lb | slot (the (key, slot) order inside a bucket), bo = bucket | arrival index << 16
    uint32_t comp[8], bo[8];
    {
      const int sh = 32 - Lb;
#pragma unroll
      for (int r2 = 0; r2 < 2; ++r2) {
        const int blk = tid + NT * r2;
        if (4 * blk < N) {
          const uint4 r = cells_philox(P, (uint32_t)blk, cell_ctr, P.step, 0u);
          const uint32_t k[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
          for (int w = 0; w < 4; ++w) {
            const int p = 4 * blk + w;
            comp[4 * r2 + w] = (k[w] << Lb) | (uint32_t)p;
            bo[4 * r2 + w] = k[w] >> sh;
            if (p < N) bo[4 * r2 + w] |= atomicAdd(&cnt[k[w] >> sh], 1u) << 16;
          }
        }
      }
    }
    sync();
    // ---- exclusive scan of the bucket counts: counter -> (start | members << 16) ----
    {
      uint4 v[2];
      v[0] = v[1] = make_uint4(0u, 0u, 0u, 0u);
      if (4 * tid < NB) v[0] = *reinterpret_cast<const uint4 *>(cnt + 4 * tid);
      if (4 * (tid + NT) < NB) v[1] = *reinterpret_cast<const uint4 *>(cnt + 4 * (tid + NT));
      // both blocks of a thread in one packed warp scan (two 16-bit running sums per word)
      const uint32_t pk = (v[0].x + v[0].y + v[0].z + v[0].w) | ((v[1].x + v[1].y + v[1].z + v[1].w) << 16);
      uint32_t inc = pk;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
      }
      uint32_t exc = inc - pk, all;
      if (NT == 32) {
        all = __shfl_sync(0xffffffffu, inc, 31);
      } else {
        if (lane == 31) misc[warp] = (int)inc;
        sync();
        all = 0;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
          const uint32_t t = (uint32_t)misc[w];
          exc += (w < warp) ? t : 0u;
          all += t;
        }
      }
      // block 0 of every thread precedes block 1 of thread 0
      const uint32_t base[2] = {exc & 0xFFFFu, (exc >> 16) + (all & 0xFFFFu)};
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        uint4 o;
        o.x = base[u] | (v[u].x << 16);
        o.y = (base[u] + v[u].x) | (v[u].y << 16);
        o.z = (base[u] + v[u].x + v[u].y) | (v[u].z << 16);
        o.w = (base[u] + v[u].x + v[u].y + v[u].z) | (v[u].w << 16);
        if (4 * (tid + NT * u) < NB) *reinterpret_cast<uint4 *>(cnt + 4 * (tid + NT * u)) = o;
      }
    }
    sync();
    // ---- placement: a key alone in its bucket is ranked; the others line up in their bucket ----
    // afterwards bo = (bucket start | members << 16) for the keys that still have to be ranked, 0 otherwise
    const uint32_t slot_mask = (uint32_t)NB - 1u;
    const uint32_t cnt_s = (uint32_t)__cvta_generic_to_shared(cnt), k2s = (uint32_t)__cvta_generic_to_shared(K2),
                   pi_s = (uint32_t)__cvta_generic_to_shared(pi);
#pragma unroll
    for (int j = 0; j < 8; ++j)
      bo[j] = cells_place(bo[j], 4 * (tid + NT * (j >> 2)) + (j & 3), N, comp[j], cnt_s, k2s, pi_s);
    sync();
    // ---- in-bucket ranking by composite = (key, slot) order ----
    {
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const uint32_t b0 = bo[j] & 0xFFFFu, m = bo[j] >> 16, e = comp[j];
        uint32_t rank = b0;
        cells_rank4(rank, k2s + 4u * b0, e, m);
        if (m > (uint32_t)kRankWin) {
#pragma unroll 1
          for (uint32_t t = kRankWin; t < m; ++t) rank += (K2[b0 + t] < e) ? 1u : 0u;
        }
        if (m > 1u) pi[rank] = (uint16_t)(4u * (e & slot_mask));
      }
    }
    }  // OP != 4, 6
    if (NT > 32 && tid == 0) *reinterpret_cast<int4 *>(misc + 8) = next;
    sync();
    if (OP == 3 || OP == 5) {  // split form, first pass: the pairing goes to HBM for the second pass
      uint16_t *__restrict__ gp = P.pi_g + gs;
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int q = tid + NT * r;
        if (q < N) gp[q] = pi[q];
      }
    }
    }  // HALF != 2
    // ---- pairs: thread owns pair slots 2 dp, 2 dp + 1 (one Philox block of stream 1 serves both) ----
    bool any_acc;
    if (OP == 2) {
      // chi-MLP on the tensor cores: every warp sends the features of its (up to) 128 pair slots to the CTA's MLP
      // server as one tile, waits for z, then rotates and commits
      if (HALF != 2) {
        // (the features are staged in the warp's own shared memory first, so that the server never waits for them)
        pairs_phase<1>(P, item, cell_ctr, accept, 0);
        __syncwarp();
        const float *st = reinterpret_cast<const float *>(K2) + 256 * warp;
        float f0[4], f1[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          f0[u] = st[32 * u + lane];
          f1[u] = st[128 + 32 * u + lane];
        }
        // (the same words then receive z: the server ADDS the partial sums of its column groups into them)
        __syncwarp();
#pragma unroll
        for (int u = 0; u < 4; ++u) reinterpret_cast<float *>(K2 + 256 * warp)[32 * u + lane] = 0.f;
        const int slot = srv->acquire(lane, K2 + 256 * warp);
#pragma unroll
        for (int u = 0; u < 4; ++u) srv->write_row(slot, 32 * u + lane, f0[u], f1[u]);
        srv->publish(slot);
      }
      if (HALF == 1) {  // the cell's pre-collision state waits in its buffer
        if (tid == 0) *reinterpret_cast<float4 *>(state) = make_float4(ux, uy, uz, theta);
        return share(next);
      }
      if (HALF == 2) {
        sync();
        const float4 st4 = *reinterpret_cast<const float4 *>(state);
        ux = st4.x; uy = st4.y; uz = st4.z; theta = st4.w;
      }
      srv->wait(lane);
      any_acc = pairs_phase<2>(P, item, cell_ctr, accept, 0);
    } else if (OP == 3) {
      any_acc = pairs_phase<3>(P, item, cell_ctr, accept, 0);
    } else if (OP == 4) {
      any_acc = pairs_phase<4>(P, item, cell_ctr, accept, 0);
    } else if (OP == 5) {  // VHS-NN split form: T_cell = m Theta / (3 kB N) is one of the network inputs
      any_acc = pairs_phase<5>(P, item, cell_ctr, accept, 0, theta * P.T_coef * invN * P.inv_T_scale);
    } else if (OP == 6) {
      any_acc = pairs_phase<6>(P, item, cell_ctr, accept, 0);
    } else {
      any_acc = pairs_phase<0>(P, item, cell_ctr, accept, 0);
    }
    bool collided = OP != 3 && OP != 5;  // (first pass of the split forms: nothing is committed, nothing to store)
    if (accept) {
      collided = __any_sync(0xffffffffu, any_acc);
      if (NT > 32 && collided && lane == 0) misc[12] = 1;
    }
    sync();
    if (NT > 32 && accept) collided = misc[12] != 0;
    next = share(next);
    // ---- finish: post-collision sums, matching coefficients, store (12 B / particle) ----
    if (collided) {  // team-uniform
      float *__restrict__ ox = P.vx + gs, *__restrict__ oy = P.vy + gs, *__restrict__ oz = P.vz + gs;
      float x[8], y[8], z[8];
#pragma unroll
      for (int r = 0; r < 8; ++r) {  // rows beyond the cell stand at u_pre: no contribution to the sums
        const int q = tid + NT * r;
        x[r] = ux; y[r] = uy; z[r] = uz;
        if (q < N) {
          x[r] = X[q];
          y[r] = Y[q];
          z[r] = Z[q];
        }
      }
      float am1 = 0.f, Bx = 0.f, By = 0.f, Bz = 0.f;
      if (P.flags & DSMC_F_MOMENT_MATCH) {
        float sx, sy, sz, s2;
        {
          const f32x2 ux2 = pk2(ux, ux), uy2 = pk2(uy, uy), uz2 = pk2(uz, uz);
          f32x2 ax = pk2(0.f, 0.f), ay = ax, az = ax, a2 = ax;
#pragma unroll
          for (int r = 0; r < 8; r += 2) {
            const f32x2 dx = sub2(pk2(x[r], x[r + 1]), ux2), dy = sub2(pk2(y[r], y[r + 1]), uy2),
                        dz = sub2(pk2(z[r], z[r + 1]), uz2);
            ax = add2(ax, dx); ay = add2(ay, dy); az = add2(az, dz);
            a2 = fma2(dx, dx, a2); a2 = fma2(dy, dy, a2); a2 = fma2(dz, dz, a2);
          }
          sx = hsum2(ax); sy = hsum2(ay); sz = hsum2(az); s2 = hsum2(a2);
        }
        team_sum4(sx, sy, sz, s2, 1);
        const float dx = sx * invN, dy = sy * invN, dz = sz * invN;  // u_post - u_pre
        const float th_post = s2 - fN * fmaf(dx, dx, fmaf(dy, dy, dz * dz));
        if (P.flags & DSMC_F_MATCH_ENERGY_ONLY) {  // literal eq. 11: v <- v sqrt(E_pre / E_post)
          const float qx = ux + dx, qy = uy + dy, qz = uz + dz;
          const float e_pre = theta + fN * fmaf(ux, ux, fmaf(uy, uy, uz * uz));
          const float e_post = th_post + fN * fmaf(qx, qx, fmaf(qy, qy, qz * qz));
          if (e_post > 0.f) {
            const float del = (e_pre - e_post) / e_post;  // alpha - 1 = sqrt(1 + del) - 1 without cancellation
            am1 = del / (1.0f + sqrtf(1.0f + del));
          }
        } else {  // v <- u_pre + alpha (v - u_post)
          if (th_post > 0.f) {
            const float del = (theta - th_post) / th_post;
            am1 = del / (1.0f + sqrtf(1.0f + del));
          }
          // B = u_pre - alpha (u_pre + d) = -(alpha - 1) u_pre - alpha d
          Bx = -fmaf(am1, ux, fmaf(am1, dx, dx));
          By = -fmaf(am1, uy, fmaf(am1, dy, dy));
          Bz = -fmaf(am1, uz, fmaf(am1, dz, dz));
        }
      }
      // alpha is 1 + O(1e-7), which FP32 cannot resolve: the store applies v + (alpha - 1) v + B
      {
        const f32x2 a2 = pk2(am1, am1), bx2 = pk2(Bx, Bx), by2 = pk2(By, By), bz2 = pk2(Bz, Bz);
#pragma unroll
        for (int r = 0; r < 8; r += 2) {
          float o0, o1;
          const f32x2 vx2 = pk2(x[r], x[r + 1]), vy2 = pk2(y[r], y[r + 1]), vz2 = pk2(z[r], z[r + 1]);
          const int q0 = tid + NT * r, q1 = q0 + NT;
          upk2(fma2(a2, vx2, add2(vx2, bx2)), o0, o1);
          if (q0 < N) __stcs(ox + q0, o0);
          if (q1 < N) __stcs(ox + q1, o1);
          upk2(fma2(a2, vy2, add2(vy2, by2)), o0, o1);
          if (q0 < N) __stcs(oy + q0, o0);
          if (q1 < N) __stcs(oy + q1, o1);
          upk2(fma2(a2, vz2, add2(vz2, bz2)), o0, o1);
          if (q0 < N) __stcs(oz + q0, o0);
          if (q1 < N) __stcs(oz + q1, o1);
        }
      }
    }
    return next;
  }
};

}  // namespace dsmc
