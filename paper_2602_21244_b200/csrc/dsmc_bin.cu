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
//   finally    k_cell_tile_sums, k_cell_scan   CSR offsets = prefix sum of the per-cell counts the last down-sweep
//                            accumulates (one atomic per run of equal cells; the sorted cell ids are never written)
//
// Algorithmic traffic (2 passes): 4+16+20 B and 4+20+16 B per particle.
#include <algorithm>

#include "dsmc_device.cuh"
#include "dsmc_internal.h"

namespace dsmc {

constexpr int kBinThreads = 512;
constexpr int kBinWarps = kBinThreads / 32;
constexpr int kBinItems = kBinTile / kBinThreads;  // 8 per thread, 256 consecutive per warp
static_assert(kBinItems == 8, "tile / threads");
constexpr int kHistTiles = 4;  // tiles per k_tile_hist CTA

struct BinPass {
  int shift, mask, R;  // digit = (cell >> shift) & mask, R = number of digit values (<= 512)
};

__device__ __forceinline__ int bin_digit(int c, const BinPass &ps) { return (c >> ps.shift) & ps.mask; }

// ---------------------------------------------------------------------------------------------
// k_tile_hist: hist[t][d] = number of items of tile t with digit d; group[g][d] += the same.
// One CTA covers kHistTiles consecutive tiles (same group) so that 32 loads per thread are in
// flight before the first shared-memory atomic.  FIRST pass also range-checks the cell ids (bad
// ids are dropped here and in the down-sweep).
// ---------------------------------------------------------------------------------------------
template <bool FIRST>
__global__ void __launch_bounds__(kBinThreads) k_tile_hist(int64_t n, int32_t K, int n_tiles,
                                                          const int32_t *__restrict__ cell, BinPass ps,
                                                          int tiles_per_group, int32_t *__restrict__ hist,
                                                          int32_t *__restrict__ group,
                                                          int32_t *__restrict__ status) {
  __shared__ int h[kHistTiles][kBinMaxRadix];
  const int tid = threadIdx.x;
  const int t0 = blockIdx.x * kHistTiles;
  if (!FIRST) pdl_wait();  // (the first kernel of the chain is launched the ordinary way)
  pdl_launch_dependents();
#pragma unroll
  for (int k = 0; k < kHistTiles; ++k) h[k][tid] = 0;
  int c[kHistTiles][kBinItems];
#pragma unroll
  for (int k = 0; k < kHistTiles; ++k) {
    const int64_t base = (int64_t)(t0 + k) * kBinTile;
#pragma unroll
    for (int r = 0; r < kBinItems; ++r) {
      const int64_t i = base + r * kBinThreads + tid;
      c[k][r] = i < n ? __ldg(cell + i) : -1;
    }
  }
  __syncthreads();
  bool bad = false;
#pragma unroll
  for (int k = 0; k < kHistTiles; ++k) {
#pragma unroll
    for (int r = 0; r < kBinItems; ++r) {
      const int cc = c[k][r];
      const int64_t i = (int64_t)(t0 + k) * kBinTile + r * kBinThreads + tid;
      if (FIRST && i < n && (cc < 0 || cc >= K)) bad = true;
      // later passes re-check the range too: when the first pass dropped bad ids, the tail of the ping-pong buffers
      // behind the kept records is stale, and a stale id must never index outside the digit tables
      if (cc >= 0 && cc < K) atomicAdd(&h[k][bin_digit(cc, ps)], 1);
    }
  }
  if (FIRST && bad) *status = DSMC_ERR_BAD_CELL_INDEX;
  __syncthreads();
  if (tid < ps.R) {
    int sum = 0;
#pragma unroll
    for (int k = 0; k < kHistTiles; ++k) {
      if (t0 + k < n_tiles) {
        const int x = h[k][tid];
        hist[(size_t)(t0 + k) * kBinMaxRadix + tid] = x;
        sum += x;
      }
    }
    if (sum) atomicAdd(&group[(size_t)(t0 / tiles_per_group) * kBinMaxRadix + tid], sum);
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
  pdl_wait();
  pdl_launch_dependents();
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
  // the walk is a chain of L2 / DRAM round trips (one CTA per SM, nothing else to run): eighteen loads in flight per
  // trip, predicated at the end of the group, so that a group of 36 tiles takes two trips (it was 4 trips of 8 and a
  // serial remainder of 4: the remainder alone was a quarter of the kernel)
  constexpr int kWalk = 18;
  for (int t = t0; t < t1; t += kWalk) {
    int x[kWalk];
#pragma unroll
    for (int u = 0; u < kWalk; ++u) x[u] = t + u < t1 ? hist[(size_t)(t + u) * kBinMaxRadix + d] : 0;
#pragma unroll
    for (int u = 0; u < kWalk; ++u) {
      if (t + u < t1) hist[(size_t)(t + u) * kBinMaxRadix + d] = run;
      run += x[u];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// k_downsweep: one CTA per tile.  The tile's cell ids and payload are staged in shared memory by
// bulk async copies (cp.async.bulk + mbarrier) issued by one thread at kernel start, so the HBM
// reads overlap the ranking.  Warp w owns items [256 w, 256 w + 256) of the tile and walks them in
// index order, 32 at a time: lanes with the same digit find one another with match.any, the first
// of them bumps the warp's private counter of that digit, so
// rank = (items of this digit in earlier warps) + (earlier rounds) + (earlier lanes): stable.
// The copy-out walks the sorted positions and gathers through the inverse permutation, writing
// runs of consecutive records.
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
  int32_t *perm;
  int32_t *cell_count;  // [n_cells + 1], zeroed: particles per cell, counted by the LAST pass
  int32_t bulk_ok;  // FIRST-pass inputs are 16-byte aligned
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE;\n"
      "bra WAIT_LOOP;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// global -> shared bulk copy; bytes > 0 and a multiple of 16, both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

template <bool FIRST, bool LAST>
__global__ void __launch_bounds__(kBinThreads, 2) k_downsweep(int64_t n, int32_t K, BinPass ps, BinIo io,
                                                              const int32_t *__restrict__ hist,
                                                              int32_t *__restrict__ group, int group_rows) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  // staging (unsorted, tile order): cell ids, then (FIRST) vx | vy | vz, else records
  int32_t *scell = reinterpret_cast<int32_t *>(smem_raw);                 // [tile]
  float *sv = reinterpret_cast<float *>(scell + kBinTile);                // FIRST: [3][tile]
  float4 *srec = reinterpret_cast<float4 *>(scell + kBinTile);            // else:  [tile]
  unsigned char *after = smem_raw + (size_t)kBinTile * (FIRST ? 16 : 20);
  int32_t *tile_off = reinterpret_cast<int32_t *>(after);                 // [R]
  int32_t *gdst = tile_off + kBinMaxRadix;                                // [R]
  uint16_t *wc = reinterpret_cast<uint16_t *>(gdst + kBinMaxRadix);       // [warps][R]
  uint16_t *inv = wc + kBinWarps * kBinMaxRadix;                          // [tile] sorted pos -> tile index
  __shared__ int scratch[kBinWarps + 1];
  __shared__ __align__(8) uint64_t bar[2];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int t = blockIdx.x;
  pdl_wait();
  pdl_launch_dependents();
  const int64_t tbase = (int64_t)t * kBinTile;
  const int cnt_tile = (int)min((int64_t)kBinTile, n - tbase);
  const int32_t *cin = FIRST ? io.cell : io.cell_in;
  const bool bulk = !FIRST || io.bulk_ok;
  const int n_bulk = bulk ? (cnt_tile & ~3) : 0;  // 4-byte arrays: whole 16-byte units only

  if (tid == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if (n_bulk > 0) {
      mbar_expect_tx(&bar[0], (uint32_t)n_bulk * 4u);
      bulk_g2s(scell, cin + tbase, (uint32_t)n_bulk * 4u, &bar[0]);
    } else {
      mbar_expect_tx(&bar[0], 0u);
    }
    if (FIRST) {
      if (n_bulk > 0) {
        mbar_expect_tx(&bar[1], (uint32_t)n_bulk * 12u);
        bulk_g2s(sv, io.vx + tbase, (uint32_t)n_bulk * 4u, &bar[1]);
        bulk_g2s(sv + kBinTile, io.vy + tbase, (uint32_t)n_bulk * 4u, &bar[1]);
        bulk_g2s(sv + 2 * kBinTile, io.vz + tbase, (uint32_t)n_bulk * 4u, &bar[1]);
      } else {
        mbar_expect_tx(&bar[1], 0u);
      }
    } else {
      mbar_expect_tx(&bar[1], (uint32_t)cnt_tile * 16u);
      bulk_g2s(srec, io.rec_in + tbase, (uint32_t)cnt_tile * 16u, &bar[1]);
    }
  }
  // the group sums of this pass have been consumed by k_prefix: leave them zero for the next pass / the next call (no
  // memset between the kernels: every boundary in this chain of short kernels costs microseconds)
  if (t < group_rows) group[(size_t)t * kBinMaxRadix + tid] = 0;
  for (int i = tid; i < kBinWarps * kBinMaxRadix / 2; i += kBinThreads) reinterpret_cast<uint32_t *>(wc)[i] = 0u;
  // items the bulk copies do not cover (ragged tail, or unaligned caller arrays)
  for (int j = n_bulk + tid; j < cnt_tile; j += kBinThreads) {
    scell[j] = __ldg(cin + tbase + j);
    if (FIRST) {
      sv[j] = __ldg(io.vx + tbase + j);
      sv[kBinTile + j] = __ldg(io.vy + tbase + j);
      sv[2 * kBinTile + j] = __ldg(io.vz + tbase + j);
    }
  }
  __syncthreads();
  mbar_wait(&bar[0], 0);

  uint16_t *mywc = wc + warp * kBinMaxRadix;
  const int nbits = __popc((unsigned)ps.mask);
  const int jbase = warp * (32 * kBinItems) + lane;
  int c[kBinItems], lr[kBinItems];
#pragma unroll
  for (int r = 0; r < kBinItems; ++r) {
    const int j = jbase + r * 32;
    c[r] = j < cnt_tile ? scell[j] : -1;
    if (c[r] >= K) c[r] = -1;  // dropped (status already set by k_tile_hist); later passes: stale tail, see k_tile_hist
  }
#pragma unroll
  for (int r = 0; r < kBinItems; ++r) {
    const int d = c[r] >= 0 ? bin_digit(c[r], ps) : 0xFFFF;
    // lanes with the same digit: one ballot per digit bit (MATCH.ANY takes time in proportion to the number of
    // distinct values in the warp, and with 512 digits nearly all 32 are distinct: it was the top stall of the pass)
    // (later passes see fewer distinct digits per warp -- their input is ordered by the lower digits -- and there
    // match.any is the faster of the two: measured 153 against 158 us)
    uint32_t m;
    if (FIRST) {
      m = __ballot_sync(0xffffffffu, c[r] >= 0);
      m = c[r] >= 0 ? m : ~m;
#pragma unroll
      for (int b = 0; b < 9; ++b) {
        if (b < nbits) {
          const bool bit = (d >> b) & 1;
          const uint32_t bal = __ballot_sync(0xffffffffu, bit);
          m &= bit ? bal : ~bal;
        }
      }
    } else {
      m = __match_any_sync(0xffffffffu, d);
    }
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
#pragma unroll
  for (int r = 0; r < kBinItems; ++r) {
    if (c[r] >= 0) {
      const int d = bin_digit(c[r], ps);
      inv[tile_off[d] + mywc[d] + lr[r]] = (uint16_t)(jbase + r * 32);
    }
  }
  __syncthreads();
  mbar_wait(&bar[1], 0);
  const int kept = scratch[kBinWarps];
  // two positions per trip: their (inv -> staged record) load chains overlap (four need more than the 64
  // registers two CTAs per SM leave: measured no better than one)
#pragma unroll 2
  for (int pos = tid; pos < kept; pos += kBinThreads) {
    const int j = inv[pos];
    const int cc = scell[j];
    const int64_t dst = (int64_t)gdst[bin_digit(cc, ps)] + pos;
    float4 rr;
    if (FIRST) {
      rr = make_float4(__int_as_float((int)(tbase + j)), sv[j], sv[kBinTile + j], sv[2 * kBinTile + j]);
    } else {
      rr = srec[j];
    }
    if (LAST) {
      io.perm[dst] = __float_as_int(rr.x);
      io.vx_s[dst] = rr.y;
      io.vy_s[dst] = rr.z;
      io.vz_s[dst] = rr.w;
      // particles per cell: the 32 consecutive sorted positions of a warp hold a few runs of equal cell ids (the
      // tile arrives ordered by the lower digits), one atomic per run
      const uint32_t m = __match_any_sync(__activemask(), cc);
      if (lane == __ffs(m) - 1) atomicAdd(io.cell_count + cc, __popc(m));
    } else {
      io.rec_out[dst] = rr;
      io.cell_out[dst] = cc;
    }
  }
}

// cell_start = exclusive prefix sum of the per-cell counts (CSR offsets; entry n_cells = particles kept).  Two
// launches: sums of 4096-count tiles, then every CTA adds up the tiles before its own and scans its tile.
constexpr int kScanThreads = 256, kScanItems = 16, kScanTile = kScanThreads * kScanItems;

__global__ void __launch_bounds__(kScanThreads) k_cell_tile_sums(int32_t n, const int32_t *__restrict__ count,
                                                                int32_t *__restrict__ tile_sums) {
  __shared__ int ws[kScanThreads / 32];
  const int base = blockIdx.x * kScanTile;
  pdl_wait();
  pdl_launch_dependents();
  int sum = 0;
#pragma unroll
  for (int r = 0; r < kScanItems; ++r) {
    const int i = base + r * kScanThreads + threadIdx.x;
    sum += i < n ? __ldg(count + i) : 0;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = sum;
  __syncthreads();
  if (threadIdx.x == 0) {
    int t = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) t += ws[w];
    tile_sums[blockIdx.x] = t;
  }
}

__global__ void __launch_bounds__(kScanThreads) k_cell_scan(int32_t n, int32_t *__restrict__ count,
                                                           const int32_t *__restrict__ tile_sums,
                                                           int32_t *__restrict__ cell_start) {
  __shared__ int ws[kScanThreads / 32];
  __shared__ int sc[kScanTile];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int base = blockIdx.x * kScanTile;
  pdl_wait();
  pdl_launch_dependents();
  // tiles before this one
  int before = 0;
  for (int t = tid; t < (int)blockIdx.x; t += kScanThreads) before += __ldg(tile_sums + t);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) before += __shfl_xor_sync(0xffffffffu, before, o);
  if (lane == 0) ws[warp] = before;
  // stage the tile (coalesced), then every thread owns kScanItems consecutive counts
#pragma unroll
  for (int r = 0; r < kScanItems; ++r) {
    const int i = base + r * kScanThreads + tid;
    int cnt_i = 0;
    if (i < n) {
      cnt_i = count[i];
      count[i] = 0;  // left zero for the next call (k_cell_tile_sums has read it already)
    }
    sc[r * kScanThreads + tid] = cnt_i;
  }
  __syncthreads();
  before = 0;
#pragma unroll
  for (int w = 0; w < kScanThreads / 32; ++w) before += ws[w];
  int loc[kScanItems], sum = 0;
#pragma unroll
  for (int r = 0; r < kScanItems; ++r) {
    loc[r] = sum;
    sum += sc[tid * kScanItems + r];
  }
  int inc = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += y;
  }
  __syncthreads();  // ws and sc are read by everyone above
  if (lane == 31) ws[warp] = inc;
  __syncthreads();
  int woff = 0;
#pragma unroll
  for (int w = 0; w < kScanThreads / 32; ++w) woff += (w < warp) ? ws[w] : 0;
  const int mine = before + woff + inc - sum;
#pragma unroll
  for (int r = 0; r < kScanItems; ++r) sc[tid * kScanItems + r] = mine + loc[r];
  __syncthreads();
#pragma unroll
  for (int r = 0; r < kScanItems; ++r) {
    const int i = base + r * kScanThreads + tid;
    if (i < n) cell_start[i] = sc[r * kScanThreads + tid];
  }
}

template <bool FIRST, bool LAST>
static void launch_downsweep(int n_tiles, cudaStream_t s, int64_t n, int32_t K, const BinPass &ps, const BinIo &io,
                             const int32_t *hist, int32_t *group, int group_rows) {
  auto kern = k_downsweep<FIRST, LAST>;
  const size_t smem = (size_t)kBinTile * (FIRST ? 16 : 20) + 2 * 4 * kBinMaxRadix + 2 * kBinWarps * kBinMaxRadix +
                      2 * kBinTile + 128;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  launch_pdl(kern, n_tiles, kBinThreads, smem, s, n, K, ps, io, hist, group, group_rows);
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
  // (d_cell_count and d_bin_group are zero on entry: zeroed once when the workspace is made, and every call leaves them
  // zero -- k_cell_scan clears the counts it has read, the down-sweeps clear the group sums)
  int bits = 1;
  while ((int64_t(1) << bits) < (int64_t)K) ++bits;
  const int passes = (bits + 8) / 9;
  const int dbits = (bits + passes - 1) / passes;
  const int n_tiles = (int)((n + kBinTile - 1) / kBinTile);
  const int n_groups = std::min(n_tiles, c->num_sms);
  const int tpg = (((n_tiles + n_groups - 1) / n_groups) + kHistTiles - 1) / kHistTiles * kHistTiles;
  const int groups = (n_tiles + tpg - 1) / tpg;
  const int hist_grid = (n_tiles + kHistTiles - 1) / kHistTiles;
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
    io.cell_count = c->d_cell_count;
    io.bulk_ok = ((reinterpret_cast<uintptr_t>(cell) | reinterpret_cast<uintptr_t>(vx) |
                   reinterpret_cast<uintptr_t>(vy) | reinterpret_cast<uintptr_t>(vz)) & 15) == 0;
    if (first)
      k_tile_hist<true><<<hist_grid, kBinThreads, 0, s>>>(n, K, n_tiles, cell, ps, tpg, c->d_bin_hist,
                                                          c->d_bin_group, c->d_status);
    else
      launch_pdl(k_tile_hist<false>, hist_grid, kBinThreads, 0, s, n, K, n_tiles, io.cell_in, ps, tpg, c->d_bin_hist,
                 c->d_bin_group, c->d_status);
    launch_pdl(k_prefix, groups, kBinThreads, 0, s, n_tiles, groups, tpg, ps, c->d_bin_hist, c->d_bin_group);
    if (first && last) launch_downsweep<true, true>(n_tiles, s, n, K, ps, io, c->d_bin_hist, c->d_bin_group, groups);
    else if (first) launch_downsweep<true, false>(n_tiles, s, n, K, ps, io, c->d_bin_hist, c->d_bin_group, groups);
    else if (last) launch_downsweep<false, true>(n_tiles, s, n, K, ps, io, c->d_bin_hist, c->d_bin_group, groups);
    else launch_downsweep<false, false>(n_tiles, s, n, K, ps, io, c->d_bin_hist, c->d_bin_group, groups);
    c->launches += 3;
    if (last) {
      const int n_scan = K + 1, scan_tiles = (n_scan + kScanTile - 1) / kScanTile;
      launch_pdl(k_cell_tile_sums, scan_tiles, kScanThreads, 0, s, n_scan, c->d_cell_count, c->d_cell_tile_sums);
      launch_pdl(k_cell_scan, scan_tiles, kScanThreads, 0, s, n_scan, c->d_cell_count, c->d_cell_tile_sums, cell_start);
      c->launches += 2;
    }
  }
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

}  // namespace dsmc
