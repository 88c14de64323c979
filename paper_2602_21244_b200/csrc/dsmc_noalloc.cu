// dsmc_bin_noalloc: the cell sort of dsmc_bin for callers that cannot allocate device memory -- code under
// CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No context: the radix sort's workspace
// (tile histograms, group sums, the record and cell-id buffers between the two passes, per-cell counts, scan tile sums,
// a status word) lives in ONE file-scope device array of fixed size, so the call allocates nothing and frees nothing.
//
// Limits (fixed at build time): n <= DSMC_NOALLOC_MAX_PARTICLES = 2^20, n_cells <= DSMC_NOALLOC_MAX_CELLS = 2^17 (two
// radix passes).  The array is 22.5 MB (22 545 152 bytes); every GPU that loads the library holds it until the process exits.
//
// The kernels are the ones dsmc_bin launches (launch_bin, dsmc_bin.cu), handed workspace pointers into the array.  In
// HOST code the array's name is a host-side stand-in, not a device address, so its address is taken once per device
// with cudaGetSymbolAddress (device current) and only that pointer ever reaches a kernel.
//
// Every call shares the array and the array keeps the last call's contents: the status word is cleared on the caller's
// stream at the start of the call; the per-cell counts and the group sums start at zero because the array is
// zero-initialised when the module loads and the kernels that consume them leave them zero (as in dsmc_bin).  Calls that overlap on the
// GPU (two streams, two threads, or a dsmc_bin_noalloc graph replayed concurrently with itself) RACE on the array.
#include <mutex>

#include "dsmc_internal.h"

namespace dsmc {

constexpr int64_t kNaMaxParticles = DSMC_NOALLOC_MAX_PARTICLES;
constexpr int32_t kNaMaxCells = DSMC_NOALLOC_MAX_CELLS;
constexpr size_t na_align(size_t b) { return (b + 255) & ~(size_t)255; }
constexpr size_t kNaTiles = (size_t)((kNaMaxParticles + kBinTile - 1) / kBinTile);
// layout [bytes]
constexpr size_t kNaOffStatus = 0;
constexpr size_t kNaOffHist = na_align(kNaOffStatus + sizeof(int32_t));
constexpr size_t kNaOffGroup = na_align(kNaOffHist + sizeof(int32_t) * kNaTiles * kBinMaxRadix);
constexpr size_t kNaOffRec = na_align(kNaOffGroup + sizeof(int32_t) * kNaTiles * kBinMaxRadix);  // groups <= tiles
constexpr size_t kNaOffCell = na_align(kNaOffRec + sizeof(float4) * (size_t)kNaMaxParticles);
constexpr size_t kNaOffCount = na_align(kNaOffCell + sizeof(int32_t) * (size_t)kNaMaxParticles);
constexpr size_t kNaOffSums = na_align(kNaOffCount + sizeof(int32_t) * ((size_t)kNaMaxCells + 1));
constexpr size_t kNaBytes = na_align(kNaOffSums + sizeof(int32_t) * ((size_t)kNaMaxCells / 4096 + 2));
static_assert(kNaBytes < (size_t)24 << 20, "the scratch array is meant to stay modest");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNaBytes];

struct NaDevice {
  bool ready;
  int rc;
  unsigned char *scratch;  // DEVICE address of g_noalloc_scratch on this device (cudaGetSymbolAddress)
  int num_sms;
};
static NaDevice g_na_dev[64];
static std::mutex g_na_mutex;

// once per device, with that device current
static int na_setup(int dev, NaDevice **out) {
  if (dev < 0 || dev >= 64) return DSMC_ERR_INVALID_ARG;
  std::lock_guard<std::mutex> lock(g_na_mutex);
  NaDevice &d = g_na_dev[dev];
  if (!d.ready) {
    d.rc = DSMC_OK;
    void *ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_noalloc_scratch) != cudaSuccess || ptr == nullptr) d.rc = DSMC_ERR_CUDA;
    if (d.rc == DSMC_OK && cudaDeviceGetAttribute(&d.num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
      d.rc = DSMC_ERR_CUDA;
    d.scratch = static_cast<unsigned char *>(ptr);
    d.ready = d.rc == DSMC_OK;  // a failed set-up is tried again by the next call
    if (d.rc != DSMC_OK) {
      cudaGetLastError();
      return d.rc;
    }
  }
  *out = &d;
  return DSMC_OK;
}

}  // namespace dsmc

using namespace dsmc;

extern "C" int dsmc_noalloc_setup(void) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return DSMC_ERR_CUDA;
  NaDevice *d = nullptr;
  return na_setup(dev, &d);
}

extern "C" int dsmc_bin_noalloc(void *stream, int64_t n, int32_t K, const int32_t *cell, const float *vx, const float *vy,
                                const float *vz, float *vx_s, float *vy_s, float *vz_s, int32_t *perm,
                                int32_t *cell_start, int32_t *status_dev) {
  if (n < 0 || K <= 0 || !cell_start) return DSMC_ERR_INVALID_ARG;
  if (n > kNaMaxParticles || K > kNaMaxCells) return DSMC_ERR_NOALLOC_LIMIT;
  if (n > 0 && (!cell || !vx || !vy || !vz || !vx_s || !vy_s || !vz_s || !perm)) return DSMC_ERR_INVALID_ARG;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return DSMC_ERR_CUDA;
  NaDevice *d = nullptr;
  int rc = na_setup(dev, &d);
  if (rc != DSMC_OK) return rc;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  unsigned char *w = d->scratch;
  // a context on the stack whose workspace pointers lead into the array: launch_bin touches nothing else of it
  dsmc_ctx c{};
  c.device = dev;
  c.stream = s;
  c.num_sms = d->num_sms;
  c.max_particles = kNaMaxParticles;
  c.max_cells = kNaMaxCells;
  c.d_status = reinterpret_cast<int32_t *>(w + kNaOffStatus);
  c.d_bin_hist = reinterpret_cast<int32_t *>(w + kNaOffHist);
  c.d_bin_group = reinterpret_cast<int32_t *>(w + kNaOffGroup);
  c.d_bin_rec[0] = reinterpret_cast<float4 *>(w + kNaOffRec);  // two passes at most: buffer 1 of each pair is never used
  c.d_bin_cell[0] = reinterpret_cast<int32_t *>(w + kNaOffCell);
  c.d_cell_count = reinterpret_cast<int32_t *>(w + kNaOffCount);
  c.d_cell_tile_sums = reinterpret_cast<int32_t *>(w + kNaOffSums);
  if (bin_num_passes(K) > 2) return DSMC_ERR_NOALLOC_LIMIT;
  if (cudaMemsetAsync(c.d_status, 0, sizeof(int32_t), s) != cudaSuccess) return DSMC_ERR_CUDA;
  rc = launch_bin(&c, n, K, cell, vx, vy, vz, vx_s, vy_s, vz_s, perm, cell_start);
  if (rc != DSMC_OK) return rc;
  if (status_dev &&
      cudaMemcpyAsync(status_dev, c.d_status, sizeof(int32_t), cudaMemcpyDeviceToDevice, s) != cudaSuccess)
    return DSMC_ERR_CUDA;
  return DSMC_OK;
}
