// The cell team: everything one team of NT threads does to one cell of the fused collision step
// (dsmc_cells.cu holds the description of the phases and the kernels).  Product code only.
#pragma once
#include "dsmc_device.cuh"
#include "dsmc_internal.h"

namespace dsmc {

constexpr int kCellsXB = 0;   // 1: twice as many key buckets (2^(L+1)): fewer shared buckets, longer scan
constexpr int kRankWin = 4;   // bucket members compared without a loop

struct CellLists {
  int4 *list[3];  // (cell, first slot, N, M) by size class: N <= 256, <= 1024, <= 2048
  int32_t *ctr;   // [0..2] entries of each list, [4..6] work counters
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

// table coordinate t_E = (ln x - lnE_min) (nE-1)/(lnE_max-lnE_min) from x = E_r/k_B, exponent and mantissa of x
// handled separately (MUFU.LG2 only sees [1,2), abs. error 2^-22)
__device__ __forceinline__ float cells_tE(const ChiTableDev &T, float x) {
  const int xi = __float_as_int(x);
  const float e = (float)((xi >> 23) - 127);
  const float m = __int_as_float((xi & 0x007FFFFF) | 0x3F800000);
  return fmaf(__log2f(m), T.c1, fmaf(e, T.c1, T.c0));
}

// bilinear chi(E~, b~) from the L2-resident quad table, coordinates clamped (Q13)
__device__ __forceinline__ float cells_chi(const ChiTableDev &T, float tE, float tB) {
  tE = fminf(fmaxf(tE, 0.f), (float)(T.nE - 1));
  tB = fminf(fmaxf(tB, 0.f), (float)(T.nB - 1));
  const int iE = min((int)tE, T.nE - 2), iB = min((int)tB, T.nB - 2);
  const float fE = tE - (float)iE, fB = tB - (float)iB;
  const float4 q = __ldg(T.quad + (size_t)iE * (T.nB - 1) + iB);
  const float lo = fmaf(fB, q.y - q.x, q.x), hi = fmaf(fB, q.w - q.z, q.z);
  return fmaf(fE, hi - lo, lo);
}

// Rotation of g by deflection chi and azimuth eps = 2 pi U_eps (Q16).  MUFU sin/cos on arguments inside
// [-pi, pi]: eps is taken as 2 pi (U - 1/2) with both signs flipped.
__device__ __forceinline__ void cells_rotate(float gx, float gy, float gz, float g2, float chi, float U_eps,
                                             float &px, float &py, float &pz) {
  float sc, cc, se, ce;
  __sincosf(chi, &sc, &cc);
  __sincosf(6.283185307179586f * (U_eps - 0.5f), &se, &ce);
  se = -se;
  ce = -ce;
  const float gp2 = fmaf(gy, gy, gz * gz);
  const float g = g2 * rsqrtf(g2);
  if (gp2 <= 1e-30f * g2 * 1e-30f) {  // g_perp <= 1e-30 g
    px = gx * cc;
    py = fabsf(gx) * sc * ce;
    pz = fabsf(gx) * sc * se;
    return;
  }
  const float inv = rsqrtf(gp2), gperp = gp2 * inv;
  const float sci = sc * inv;
  px = fmaf(gx, cc, gperp * sc * se);
  py = fmaf(gy, cc, sci * (g * gz * ce - gx * gy * se));
  pz = fmaf(gz, cc, -sci * (g * gy * ce + gx * gz * se));
}

template <int NT, int XB>
struct CellTeam {
  static constexpr int C = 8 * NT;     // slots: a thread holds 8 particles / 8 keys
  static constexpr int CPT = 8 << XB;  // bucket counters per thread
  static constexpr int NW = NT / 32;
  float *X, *Y, *Z;   // [C] velocities of the cell
  uint32_t *cnt;      // [C << XB] bucket counters, then (bucket start | members << 16)
  uint32_t *K2;       // [C] composites of the keys that share a bucket, in bucket order
  uint16_t *pi;       // [C] slots in ascending (key, slot) order
  float4 *part;       // [2][8] per-warp partial sums, before / after the collisions (NT > 32)
  int *misc;          // [0..7] warp totals of the scan, [8..11] next list entry, [12] any pair accepted
  int tid, bar;

  static constexpr size_t bytes() { return (size_t)C * (12 + (4 << XB) + 4 + 2) + 3 * NT; }  // + part, misc (320 B, NT > 32)

  __device__ __forceinline__ void init(unsigned char *base, int tid_, int bar_) {
    tid = tid_;
    bar = bar_;
    X = reinterpret_cast<float *>(base);
    Y = X + C;
    Z = Y + C;
    cnt = reinterpret_cast<uint32_t *>(Z + C);
    K2 = cnt + (C << XB);
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

  // one cell; returns the team's next list entry
  __device__ __forceinline__ int4 cell(const StepParams &P, const int4 item, const int4 *__restrict__ list, int n_items,
                                       int32_t *work) {
    const int lane = tid & 31, warp = tid >> 5;
    const int gs = item.y, N = item.z, M = item.w;
    const uint32_t cell_ctr = (uint32_t)item.x + P.cell_base;
    const int Lb = 32 - __clz(N - 1) + XB;  // bucket = top Lb bits of the key; 2^(Lb - XB) >= N
    const int NB = 1 << Lb;
    const bool accept = (P.flags & DSMC_F_ACCEPT) && P.cap != nullptr;
    int next_idx = 0;
    if (tid == 0) {
      next_idx = atomicAdd(work, 1);  // consumed after the loads below have landed
      if (NT > 32) misc[12] = 0;
    }
    if (CPT * tid < NB) {
#pragma unroll
      for (int u = 0; u < CPT / 4; ++u) *reinterpret_cast<uint4 *>(cnt + CPT * tid + 4 * u) = make_uint4(0u, 0u, 0u, 0u);
    }
    // ---- load (12 B / particle) + pre-collision sums about the pivot (eq. 10) ----
    float ux, uy, uz, theta;
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
      float sx = 0.f, sy = 0.f, sz = 0.f, s2 = 0.f;
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int q = tid + NT * r;
        if (q < N) {
          const float dx = x[r] - pvx, dy = y[r] - pvy, dz = z[r] - pvz;
          sx += dx; sy += dy; sz += dz;
          s2 = fmaf(dx, dx, s2); s2 = fmaf(dy, dy, s2); s2 = fmaf(dz, dz, s2);
          X[q] = x[r];
          Y[q] = y[r];
          Z[q] = z[r];
        }
      }
      const float t = warp_sum4(sx, sy, sz, s2, lane);
      double dsx, dsy, dsz, ds2;
      if (NT == 32) {
        dsx = __shfl_sync(0xffffffffu, t, 0);
        dsy = __shfl_sync(0xffffffffu, t, 8);
        dsz = __shfl_sync(0xffffffffu, t, 16);
        ds2 = __shfl_sync(0xffffffffu, t, 24);
        sync();  // counters zeroed before the first atomic
      } else {
        if ((lane & 7) == 0) reinterpret_cast<float *>(&part[warp])[lane >> 3] = t;
        sync();
        dsx = dsy = dsz = ds2 = 0.0;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
          const float4 p = part[w];
          dsx += p.x; dsy += p.y; dsz += p.z; ds2 += p.w;
        }
      }
      const double inv = 1.0 / N;
      const double dx = dsx * inv, dy = dsy * inv, dz = dsz * inv;
      ux = (float)((double)pvx + dx);  // pivot + mean(d)
      uy = (float)((double)pvy + dy);
      uz = (float)((double)pvz + dz);
      theta = (float)fmax(ds2 - N * (dx * dx + dy * dy + dz * dz), 0.0);
    }
    int4 next = make_int4(0, 0, 0, 0);
    if (tid == 0) next = entry(list, n_items, next_idx);
    // ---- pairing keys (stream 0: block blk serves slots 4 blk .. 4 blk + 3) and bucket counts ----
    uint32_t comp[8], bo[8];
    {
      const int sh = 32 - Lb;
#pragma unroll
      for (int r2 = 0; r2 < 2; ++r2) {
        const int blk = tid + NT * r2;
#pragma unroll
        for (int w = 0; w < 4; ++w) bo[4 * r2 + w] = 0xFFFFFFFFu;
        if (4 * blk < N) {
          const uint4 r = philox4x32_10((uint32_t)blk, cell_ctr, P.step, 0u, P.seed_lo, P.seed_hi);
          const uint32_t k[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
          for (int w = 0; w < 4; ++w) {
            const int p = 4 * blk + w;
            if (p < N) {
              const uint32_t b = k[w] >> sh;
              const uint32_t old = atomicAdd(&cnt[b], 1u);
              comp[4 * r2 + w] = (k[w] << Lb) | (uint32_t)p;
              bo[4 * r2 + w] = b | (old << 16);
            }
          }
        }
      }
    }
    sync();
    // ---- exclusive scan of the bucket counts: counter -> (start | members << 16) ----
    {
      uint32_t c[CPT];
      const bool act = CPT * tid < NB;
#pragma unroll
      for (int u = 0; u < CPT / 4; ++u) {
        uint4 v = make_uint4(0u, 0u, 0u, 0u);
        if (act) v = *reinterpret_cast<const uint4 *>(cnt + CPT * tid + 4 * u);
        c[4 * u] = v.x; c[4 * u + 1] = v.y; c[4 * u + 2] = v.z; c[4 * u + 3] = v.w;
      }
      uint32_t tot = 0;
#pragma unroll
      for (int j = 0; j < CPT; ++j) {
        const uint32_t t = c[j];
        c[j] = tot | (t << 16);
        tot += t;
      }
      uint32_t inc = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
      }
      uint32_t base = inc - tot;
      if (NT > 32) {
        if (lane == 31) misc[warp] = (int)inc;
        sync();
#pragma unroll
        for (int w = 0; w < NW; ++w) base += (w < warp) ? (uint32_t)misc[w] : 0u;
      }
      if (act) {
#pragma unroll
        for (int u = 0; u < CPT / 4; ++u)
          *reinterpret_cast<uint4 *>(cnt + CPT * tid + 4 * u) =
              make_uint4(c[4 * u] + base, c[4 * u + 1] + base, c[4 * u + 2] + base, c[4 * u + 3] + base);
      }
    }
    sync();
    // ---- placement: a key alone in its bucket is ranked; the others line up in their bucket ----
    const uint32_t slot_mask = (uint32_t)NB - 1u;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      if (bo[j] != 0xFFFFFFFFu) {
        const uint32_t w = cnt[bo[j] & 0xFFFFu], old = bo[j] >> 16;
        const uint32_t b0 = w & 0xFFFFu;
        if ((w >> 16) == 1u) {
          pi[b0] = (uint16_t)(comp[j] & slot_mask);
          bo[j] = 0xFFFFFFFFu;
        } else {
          K2[b0 + old] = comp[j];
          bo[j] = w;
        }
      }
    }
    sync();
    // ---- in-bucket ranking by composite = (key, slot) order ----
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      if (bo[j] != 0xFFFFFFFFu) {
        const uint32_t b0 = bo[j] & 0xFFFFu, m = bo[j] >> 16, e = comp[j];
        uint32_t rank = 0;
#pragma unroll
        for (int t = 0; t < kRankWin; ++t)
          if ((uint32_t)t < m) rank += (K2[b0 + t] < e) ? 1u : 0u;
        if (m > (uint32_t)kRankWin) {
#pragma unroll 1
          for (uint32_t t = kRankWin; t < m; ++t) rank += (K2[b0 + t] < e) ? 1u : 0u;
        }
        pi[b0 + rank] = (uint16_t)(e & slot_mask);
      }
    }
    if (NT > 32 && tid == 0) *reinterpret_cast<int4 *>(misc + 8) = next;
    sync();
    // ---- pairs: thread owns pair slots 2 dp, 2 dp + 1 (one Philox block of stream 1 serves both) ----
    bool any_acc = false;
    {
      const float nBm1 = (float)(P.table.nB - 1);
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        const int dp = tid + NT * r;
        const int s0 = 2 * dp;
        if (s0 < M) {
          const uint2 w2 = *reinterpret_cast<const uint2 *>(pi + 4 * dp);
          const bool v1 = s0 + 1 < M;
          int pi_[2] = {(int)(w2.x & 0xFFFFu), (int)(w2.y & 0xFFFFu)};
          int pj_[2] = {(int)(w2.x >> 16), (int)(w2.y >> 16)};
          if (!v1) { pi_[1] = pi_[0]; pj_[1] = pj_[0]; }
          const uint4 rr = philox4x32_10((uint32_t)dp, cell_ctr, P.step, 1u, P.seed_lo, P.seed_hi);
          const float Ub[2] = {u01(rr.x), u01(rr.z)}, Ue[2] = {u01(rr.y), u01(rr.w)};
          float Ua[2] = {0.f, 0.f}, cap = 0.f;
          if (accept) {  // stream 3: U_acc of pair slot s = word s & 3 of block s >> 2
            const uint4 ra = philox4x32_10((uint32_t)dp >> 1, cell_ctr, P.step, 3u, P.seed_lo, P.seed_hi);
            Ua[0] = u01((dp & 1) ? ra.z : ra.x);
            Ua[1] = u01((dp & 1) ? ra.w : ra.y);
            cap = __ldg(P.cap + item.x);
          }
          float vix[2], viy[2], viz[2], vjx[2], vjy[2], vjz[2];
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            vix[k] = X[pi_[k]]; viy[k] = Y[pi_[k]]; viz[k] = Z[pi_[k]];
            vjx[k] = X[pj_[k]]; vjy[k] = Y[pj_[k]]; vjz[k] = Z[pj_[k]];
          }
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            const bool valid = k == 0 || v1;
            const float gx = vix[k] - vjx[k], gy = viy[k] - vjy[k], gz = viz[k] - vjz[k];  // eq. 1
            const float g2 = fmaf(gx, gx, fmaf(gy, gy, gz * gz));
            bool acc = valid;
            if (accept) acc = valid && (Ua[k] * cap < sqrtf(g2));  // constant cross-section: U g_max < g
            float px = gx, py = gy, pz = gz, chi = 0.f;
            if (acc) {
              // E~ = ln(m g^2 / (4 kB)), b~ = sqrt(U_b)
              float sb;
              asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(sb) : "f"(Ub[k]));
              chi = cells_chi(P.table, cells_tE(P.table, P.e_coef * g2), sb * nBm1);
              if (g2 > 0.f) cells_rotate(gx, gy, gz, g2, chi, Ue[k], px, py, pz);
              // eqs. 6-8
              const float cx = 0.5f * (vix[k] + vjx[k]), cy = 0.5f * (viy[k] + vjy[k]), cz = 0.5f * (viz[k] + vjz[k]);
              X[pi_[k]] = fmaf(0.5f, px, cx); Y[pi_[k]] = fmaf(0.5f, py, cy); Z[pi_[k]] = fmaf(0.5f, pz, cz);
              X[pj_[k]] = fmaf(-0.5f, px, cx); Y[pj_[k]] = fmaf(-0.5f, py, cy); Z[pj_[k]] = fmaf(-0.5f, pz, cz);
              any_acc = true;
            }
            if (P.dump_any && valid) {
              const int64_t d = (int64_t)gs + s0 + k;
              if (P.dump.pair_i) P.dump.pair_i[d] = pi_[k];
              if (P.dump.pair_j) P.dump.pair_j[d] = pj_[k];
              if (P.dump.accepted) P.dump.accepted[d] = acc ? 1 : 0;
              if (P.dump.gprime) { P.dump.gprime[3 * d] = px; P.dump.gprime[3 * d + 1] = py; P.dump.gprime[3 * d + 2] = pz; }
              if (P.dump.aux) P.dump.aux[d] = chi;
            }
          }
        }
      }
    }
    bool collided = true;
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
      for (int r = 0; r < 8; ++r) {
        const int q = tid + NT * r;
        x[r] = y[r] = z[r] = 0.f;
        if (q < N) {
          x[r] = X[q];
          y[r] = Y[q];
          z[r] = Z[q];
        }
      }
      float am1 = 0.f, Bx = 0.f, By = 0.f, Bz = 0.f;
      if (P.flags & DSMC_F_MOMENT_MATCH) {
        float sx = 0.f, sy = 0.f, sz = 0.f, s2 = 0.f;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
          const int q = tid + NT * r;
          if (q < N) {
            const float dx = x[r] - ux, dy = y[r] - uy, dz = z[r] - uz;
            sx += dx; sy += dy; sz += dz;
            s2 = fmaf(dx, dx, s2); s2 = fmaf(dy, dy, s2); s2 = fmaf(dz, dz, s2);
          }
        }
        const float t = warp_sum4(sx, sy, sz, s2, lane);
        double dsx, dsy, dsz, ds2;
        if (NT == 32) {
          dsx = __shfl_sync(0xffffffffu, t, 0);
          dsy = __shfl_sync(0xffffffffu, t, 8);
          dsz = __shfl_sync(0xffffffffu, t, 16);
          ds2 = __shfl_sync(0xffffffffu, t, 24);
        } else {
          if ((lane & 7) == 0) reinterpret_cast<float *>(&part[8 + warp])[lane >> 3] = t;
          sync();
          dsx = dsy = dsz = ds2 = 0.0;
#pragma unroll
          for (int w = 0; w < NW; ++w) {
            const float4 p = part[8 + w];
            dsx += p.x; dsy += p.y; dsz += p.z; ds2 += p.w;
          }
        }
        const double inv = 1.0 / N;
        const double dx = dsx * inv, dy = dsy * inv, dz = dsz * inv;  // u_post - u_pre
        const double th_post = ds2 - N * (dx * dx + dy * dy + dz * dz);
        double alpha = 1.0, bx = 0.0, by = 0.0, bz = 0.0;
        if (P.flags & DSMC_F_MATCH_ENERGY_ONLY) {  // literal eq. 11: v <- v sqrt(E_pre / E_post)
          const double qx = ux + dx, qy = uy + dy, qz = uz + dz;
          const double e_pre = (double)theta + N * ((double)ux * ux + (double)uy * uy + (double)uz * uz);
          const double e_post = th_post + N * (qx * qx + qy * qy + qz * qz);
          if (e_post > 0.0) alpha = sqrt(e_pre / e_post);
        } else {  // v <- u_pre + alpha (v - u_post)
          if (th_post > 0.0) alpha = sqrt((double)theta / th_post);
          bx = ux - alpha * (ux + dx);
          by = uy - alpha * (uy + dy);
          bz = uz - alpha * (uz + dz);
        }
        // alpha is 1 + O(1e-7), which FP32 cannot resolve: the store applies v + (alpha - 1) v + B
        am1 = (float)(alpha - 1.0);
        Bx = (float)bx; By = (float)by; Bz = (float)bz;
      }
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int q = tid + NT * r;
        if (q < N) {
          __stcs(ox + q, fmaf(am1, x[r], x[r] + Bx));
          __stcs(oy + q, fmaf(am1, y[r], y[r] + By));
          __stcs(oz + q, fmaf(am1, z[r], z[r] + Bz));
        }
      }
    }
    return next;
  }
};

}  // namespace dsmc
