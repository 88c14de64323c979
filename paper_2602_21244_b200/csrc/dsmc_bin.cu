// dsmc_bin: stable counting sort of particles by cell index ("particles are sorted by
// cell index so that particles in the same cell are contiguous in memory").
//
// Random-order input makes a one-shot scatter/gather move 32-64 B of DRAM per 4-byte element, so
// the sort is a least-significant-digit radix sort over the cell id (<= 9 bits per pass, 2 passes
// for 80 000 cells) that carries the whole particle record along: every pass reads its input
// once, coalesced, reorders one 4096-particle tile in shared memory and writes runs of
// consecutive records.  Each pass is stable, so equal cells keep ascending particle ids and the
// result is the unique stable sort (bit-exact against the oracle).
//
//   per pass   k_tile_hist   digit histogram of every tile            -> hist[tile][digit], group sums
//              k_prefix      exclusive prefix over (digit, tile)       in place
//              k_downsweep   stable in-tile ranking (warp match + per-warp digit counters),
//                            reorder in shared memory, write runs
//   finally    k_cell_start  CSR offsets from the boundaries of the sorted cell ids
//
// Algorithmic traffic (2 passes): 4+16+20 B and 4+20+20 B per particle, +8 B for the offsets.
#include <algorithm>

#include "dsmc_device.cuh"
#include "dsmc_internal.h"

namespace dsmc {

constexpr int kBinThreads = 512;
constexpr int kBinWarps = kBinThreads / 32;
constexpr int kBinItems = kBinTile / kBinThreads;  // 8 per thread, 256 consecutive per warp
static_assert(kBinItems == 8, "tile / threads");

struct BinPass {
  int shift, mask, R;  // digit = (cell >> shift) & mask, R = number of digit values (<= 512)
};

__device__ __forceinline__ int bin_digit(int c, const BinPass &ps) { return (c >> ps.shift) & ps.mask; }

// ---------------------------------------------------------------------------------------------
// k_tile_hist: hist[t][d] = number of items of tile t with digit d; group[g][d] += the same.
// FIRST pass also range-checks the cell ids (bad ids are dropped here and in the down-sweep).
// ---------------------------------------------------------------------------------------------
template <bool FIRST>
__global__ void __launch_bounds__(kBinThreads) k_tile_hist(int64_t n, int32_t K, const int32_t *__restrict__ cell,
                                                          BinPass ps, int tiles_per_group,
                                                          int32_t *__restrict__ hist, int32_t *__restrict__ group,
                                                          int32_t *__restrict__ status) {
  __shared__ int h[kBinMaxRadix];
  const int tid = threadIdx.x;
  const int t = blockIdx.x;
  h[tid] = 0;
  __syncthreads();
  const int64_t base = (int64_t)t * kBinTile;
#pragma unroll
  for (int r = 0; r < kBinItems; ++r) {
    const int64_t i = base + r * kBinThreads + tid;
    if (i < n) {
      const int c = __ldg(cell + i);
      if (FIRST && (c < 0 || c >= K)) {
        *status = DSMC_ERR_BAD_CELL_INDEX;
      } else {
        atomicAdd(&h[bin_digit(c, ps)], 1);
      }
    }
  }
  __syncthreads();
  if (tid < ps.R) {
    const int x = h[tid];
    hist[(size_t)t * kBinMaxRadix + tid] = x;
    if (x) atomicAdd(&group[(size_t)(t / tiles_per_group) * kBinMaxRadix + tid], x);
  }
}

// ---------------------------------------------------------------------------------------------
// k_prefix: hist[t][d] <- number of items with a smaller digit, or the same digit in an earlier
// tile.  One CTA per group of consecutive tiles; thread d owns digit d.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBinThreads) k_prefix(int n_tiles, int n_groups, int tiles_per_group, BinPass ps,
                                                       int32_t *__restrict__ hist,
                                                       const int32_t *__restrict__ group) {
  __shared__ int scratch[kBinWarps + 1];
  const int d = threadIdx.x, lane = d & 31, warp = d >> 5;
  const int g = blockIdx.x;
  int before = 0, total = 0;
  if (d < ps.R) {
    for (int gg = 0; gg < n_groups; ++gg) {
      const int x = __ldg(group + (size_t)gg * kBinMaxRadix + d);
      before += gg < g ? x : 0;
      total += x;
    }
  }
  // exclusive scan of `total` over the digits (block scan, 512 threads)
  int inc = total;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += y;
  }
  if (lane == 31) scratch[warp] = inc;
  __syncthreads();
  int woff = 0;
#pragma unroll
  for (int w = 0; w < kBinWarps; ++w) woff += (w < warp) ? scratch[w] : 0;
  int run = woff + inc - total + before;
  if (d >= ps.R) return;
  const int t0 = g * tiles_per_group, t1 = min(t0 + tiles_per_group, n_tiles);
  int t = t0;
  for (; t + 8 <= t1; t += 8) {
    int x[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) x[u] = hist[(size_t)(t + u) * kBinMaxRadix + d];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      hist[(size_t)(t + u) * kBinMaxRadix + d] = run;
      run += x[u];
    }
  }
  for (; t < t1; ++t) {
    const int x = hist[(size_t)t * kBinMaxRadix + d];
    hist[(size_t)t * kBinMaxRadix + d] = run;
    run += x;
  }
}

// ---------------------------------------------------------------------------------------------
// k_downsweep: one CTA per tile.  Warp w owns items [256 w, 256 w + 256) of the tile and walks
// them in index order, 32 at a time: lanes with the same digit find one another with
// match.any, the first of them bumps the warp's private counter of that digit, so
// rank = (items of this digit in earlier warps) + (earlier rounds) + (earlier lanes): stable.
// ---------------------------------------------------------------------------------------------
struct BinIo {
  // FIRST pass input
  const int32_t *cell;
  const float *vx, *vy, *vz;
  // later-pass input / not-LAST output: records (idx, vx, vy, vz) and their cell ids
  const float4 *rec_in;
  const int32_t *cell_in;
  float4 *rec_out;
  int32_t *cell_out;
  // LAST pass output
  float *vx_s, *vy_s, *vz_s;
  int32_t *perm, *cell_sorted;
};

template <bool FIRST, bool LAST>
__global__ void __launch_bounds__(kBinThreads, 2) k_downsweep(int64_t n, int32_t K, BinPass ps, BinIo io,
                                                              const int32_t *__restrict__ hist) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4 *srec = reinterpret_cast<float4 *>(smem_raw);                    // [tile]
  int32_t *scell = reinterpret_cast<int32_t *>(srec + kBinTile);          // [tile]
  int32_t *tile_off = scell + kBinTile;                                   // [R]
  int32_t *gdst = tile_off + kBinMaxRadix;                                // [R]
  uint16_t *wc = reinterpret_cast<uint16_t *>(gdst + kBinMaxRadix);       // [warps][R]
  __shared__ int scratch[kBinWarps + 1];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int t = blockIdx.x;
  const int64_t base = (int64_t)t * kBinTile + warp * (32 * kBinItems);
  const int32_t *cin = FIRST ? io.cell : io.cell_in;

  for (int i = tid; i < kBinWarps * kBinMaxRadix / 2; i += kBinThreads) reinterpret_cast<uint32_t *>(wc)[i] = 0u;
  int c[kBinItems];
#pragma unroll
  for (int r = 0; r < kBinItems; ++r) {
    const int64_t i = base + r * 32 + lane;
    c[r] = i < n ? __ldg(cin + i) : -1;
    if (FIRST && c[r] >= K) c[r] = -1;  // dropped (status already set by k_tile_hist)
  }
  __syncthreads();
  uint16_t *mywc = wc + warp * kBinMaxRadix;
  int lr[kBinItems];
#pragma unroll
  for (int r = 0; r < kBinItems; ++r) {
    const int d = c[r] >= 0 ? bin_digit(c[r], ps) : 0xFFFF;
    const uint32_t m = __match_any_sync(0xffffffffu, d);
    const int rk = __popc(m & ((1u << lane) - 1u));
    int old = 0;
    if (rk == 0 && c[r] >= 0) {
      old = mywc[d];
      mywc[d] = (uint16_t)(old + __popc(m));
    }
    old = __shfl_sync(0xffffffffu, old, __ffs(m) - 1);
    lr[r] = old + rk;
    __syncwarp();
  }
  __syncthreads();
  // per digit: exclusive scan of the warp counters over the warps, tile count, then over digits
  int cnt = 0;
  if (tid < ps.R) {
#pragma unroll
    for (int w = 0; w < kBinWarps; ++w) {
      const int x = wc[w * kBinMaxRadix + tid];
      wc[w * kBinMaxRadix + tid] = (uint16_t)cnt;
      cnt += x;
    }
  }
  int inc = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += y;
  }
  if (lane == 31) scratch[warp] = inc;
  __syncthreads();
  int woff = 0;
#pragma unroll
  for (int w = 0; w < kBinWarps; ++w) woff += (w < warp) ? scratch[w] : 0;
  if (tid == kBinThreads - 1) scratch[kBinWarps] = woff + inc;  // items kept in this tile
  if (tid < ps.R) {
    const int off = woff + inc - cnt;
    tile_off[tid] = off;
    gdst[tid] = __ldg(hist + (size_t)t * kBinMaxRadix + tid) - off;
  }
  __syncthreads();
  // payload -> sorted position in shared memory
  float4 rec[kBinItems];
#pragma unroll
  for (int r = 0; r < kBinItems; ++r) {
    const int64_t i = base + r * 32 + lane;
    if (c[r] >= 0) {
      if (FIRST) {
        rec[r] = make_float4(__int_as_float((int)i), __ldg(io.vx + i), __ldg(io.vy + i), __ldg(io.vz + i));
      } else {
        rec[r] = __ldg(io.rec_in + i);
      }
    }
  }
#pragma unroll
  for (int r = 0; r < kBinItems; ++r) {
    if (c[r] >= 0) {
      const int d = bin_digit(c[r], ps);
      const int pos = tile_off[d] + mywc[d] + lr[r];
      srec[pos] = rec[r];
      scell[pos] = c[r];
    }
  }
  __syncthreads();
  const int kept = scratch[kBinWarps];
  for (int pos = tid; pos < kept; pos += kBinThreads) {
    const int cc = scell[pos];
    const int64_t dst = (int64_t)gdst[bin_digit(cc, ps)] + pos;
    const float4 rr = srec[pos];
    if (LAST) {
      io.perm[dst] = __float_as_int(rr.x);
      io.vx_s[dst] = rr.y;
      io.vy_s[dst] = rr.z;
      io.vz_s[dst] = rr.w;
      io.cell_sorted[dst] = cc;
    } else {
      io.rec_out[dst] = rr;
      io.cell_out[dst] = cc;
    }
  }
}

// cell_start[c] = first sorted slot whose cell id is >= c (CSR offsets; covers empty cells)
__global__ void __launch_bounds__(256) k_cell_start(int64_t n, int32_t K, const int32_t *__restrict__ cell_sorted,
                                                   int32_t *__restrict__ cell_start) {
  const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (s > n) return;
  int prev = s > 0 ? __ldg(cell_sorted + s - 1) : -1;
  int cur = s < n ? __ldg(cell_sorted + s) : K;
  prev = max(-1, min(prev, K));
  cur = max(-1, min(cur, K));
  for (int cc = prev + 1; cc <= cur; ++cc) cell_start[cc] = (int32_t)s;
}

template <bool FIRST, bool LAST>
static void launch_downsweep(int n_tiles, cudaStream_t s, int64_t n, int32_t K, const BinPass &ps, const BinIo &io,
                             const int32_t *hist) {
  auto kern = k_downsweep<FIRST, LAST>;
  const size_t smem = (size_t)kBinTile * 20 + 2 * 4 * kBinMaxRadix + 2 * kBinWarps * kBinMaxRadix;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  kern<<<n_tiles, kBinThreads, smem, s>>>(n, K, ps, io, hist);
}

int bin_num_passes(int32_t K) {
  int bits = 1;
  while ((int64_t(1) << bits) < (int64_t)K) ++bits;
  return (bits + 8) / 9;
}

int launch_bin(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cell, const float *vx, const float *vy,
               const float *vz, float *vx_s, float *vy_s, float *vz_s, int32_t *perm, int32_t *cell_start) {
  cudaStream_t s = c->stream;
  if (n == 0) {
    return cudaMemsetAsync(cell_start, 0, sizeof(int32_t) * (size_t)(K + 1), s) == cudaSuccess ? DSMC_OK
                                                                                                : DSMC_ERR_CUDA;
  }
  int bits = 1;
  while ((int64_t(1) << bits) < (int64_t)K) ++bits;
  const int passes = (bits + 8) / 9;
  const int dbits = (bits + passes - 1) / passes;
  const int n_tiles = (int)((n + kBinTile - 1) / kBinTile);
  const int n_groups = std::min(n_tiles, c->num_sms);
  const int tpg = (n_tiles + n_groups - 1) / n_groups;
  const int groups = (n_tiles + tpg - 1) / tpg;
  for (int p = 0; p < passes; ++p) {
    BinPass ps;
    ps.shift = p * dbits;
    ps.mask = (1 << dbits) - 1;
    ps.R = (p == passes - 1) ? (int)((((int64_t)K - 1) >> ps.shift) + 1) : (1 << dbits);
    if (ps.R > kBinMaxRadix) return DSMC_ERR_INVALID_ARG;
    const bool first = p == 0, last = p == passes - 1;
    BinIo io{};
    io.cell = cell; io.vx = vx; io.vy = vy; io.vz = vz;
    io.rec_in = c->d_bin_rec[(p + 1) & 1];
    io.cell_in = c->d_bin_cell[(p + 1) & 1];
    io.rec_out = c->d_bin_rec[p & 1];
    io.cell_out = c->d_bin_cell[p & 1];
    io.vx_s = vx_s; io.vy_s = vy_s; io.vz_s = vz_s; io.perm = perm;
    io.cell_sorted = c->d_bin_cell[p & 1];
    if (cudaMemsetAsync(c->d_bin_group, 0, sizeof(int32_t) * (size_t)groups * kBinMaxRadix, s) != cudaSuccess)
      return DSMC_ERR_CUDA;
    if (first)
      k_tile_hist<true><<<n_tiles, kBinThreads, 0, s>>>(n, K, cell, ps, tpg, c->d_bin_hist, c->d_bin_group, c->d_status);
    else
      k_tile_hist<false><<<n_tiles, kBinThreads, 0, s>>>(n, K, io.cell_in, ps, tpg, c->d_bin_hist, c->d_bin_group,
                                                         c->d_status);
    k_prefix<<<groups, kBinThreads, 0, s>>>(n_tiles, groups, tpg, ps, c->d_bin_hist, c->d_bin_group);
    if (first && last) launch_downsweep<true, true>(n_tiles, s, n, K, ps, io, c->d_bin_hist);
    else if (first) launch_downsweep<true, false>(n_tiles, s, n, K, ps, io, c->d_bin_hist);
    else if (last) launch_downsweep<false, true>(n_tiles, s, n, K, ps, io, c->d_bin_hist);
    else launch_downsweep<false, false>(n_tiles, s, n, K, ps, io, c->d_bin_hist);
    c->launches += 3;
    if (last) {
      k_cell_start<<<(int)((n + 1 + 255) / 256), 256, 0, s>>>(n, K, io.cell_sorted, cell_start);
      c->launches += 1;
    }
  }
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

}  // namespace dsmc
