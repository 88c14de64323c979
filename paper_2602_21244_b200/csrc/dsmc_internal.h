// Internal declarations shared by the translation units of libdsmc_b200.so (product code only;
// nothing here is seen by, or shared with, oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/dsmc.h"

namespace dsmc {

constexpr int kChunk = 512;                           // chunk granularity (particles)
constexpr int kMaxCell = DSMC_MAX_CELL_PARTICLES;     // largest resident cell
constexpr int kNlocMax = kChunk + kMaxCell;           // most particles one CTA can own (deferred variant)
constexpr int kLmaxSmall = 1536, kAmaxSmall = 64;     // small-footprint variant: 4 CTAs / SM
constexpr int kLmaxBig = kNlocMax, kAmaxBig = kChunk / 2;  // deferred variant: any legal chunk
constexpr int kThreads = 256;
constexpr int kBinTile = 4096;      // particles per radix-sort tile (dsmc_bin)
constexpr int kBinMaxRadix = 512;   // digit values per pass
constexpr float kBoltzmann = 1.380649e-23f;

// MLP staged on the device: Wt[l] is W[l] transposed, [in][out] row-major (fp32).
struct MlpDev {
  int n_layers;
  int dims[8];
  int act;
  int dmax;
  const float *Wt[7];
  const float *b[7];
};

// BF16 tensor-core image of an MLP with 2..5 hidden layers of width <= H (in <= 8 -> H -> ... -> H -> out <= 16), see
// dsmc_collide_tc.cu; more than two hidden layers: plain-BF16 batch path only (chi-MLP)
struct MlpTcDev {
  int H;                      // 64 or 128, 0 = not available
  int d_in, d_out, act;
  const void *w_blob;         // bf16 weights and biases (hi + lo parts) in UMMA K-major core-matrix layout
  uint32_t blob_bytes;
  int n_hidden;               // hidden layers (2..5); widths below H are zero-padded to H
  uint32_t extra_off;         // byte offset in w_blob of the hidden layers 3..n_hidden: (W [H x H] | B [H x 16]) each, plain BF16
  float w3_host[129];         // HOST copy of the FP32 output layer when d_out = 1: w[0..H), bias at [128]
};

// FP32 tail of a 3-layer MLP with up to three outputs (the VHS-NN operator on the split tensor-core path): bias of
// the second hidden layer (already scaled by 1/2 for SiLU, like the packed weights) and the whole output layer.
// Passed to the batch kernel by value: constant-bank operands.
struct TcTailF32 {
  float b2[128];
  float w3[3][128];
  float b3[3];
  int d_out;
};

struct ChiTableDev {
  const float4 *quad;  // [(nE-1)(nB-1)] the four nodes around each grid cell (one 16 B load per lookup)
  int nE, nB;
  float lnE_min, inv_dlnE;  // inv_dlnE = (nE-1)/(lnE_max-lnE_min)
  float c0, c1;             // t_E = c0 + c1 log2(E_r/k_B): c1 = ln2 inv_dlnE, c0 = -lnE_min inv_dlnE
  float fE1, fB1;           // nE - 1, nB - 1 as floats
  cudaTextureObject_t tex;  // the quad table as a linear float4 texture (0 = none): gathers through the TEX pipe
                            // leave the LSU pipe to the shared-memory traffic (measured, profiles/r02_probes.md)
};

struct StepParams {
  // common
  int64_t n;
  int32_t n_cells;
  const int32_t *cell_start;
  float *vx, *vy, *vz;
  const float *cap;  // sigma_cr_max / cr_max or nullptr
  uint32_t seed_lo, seed_hi, step;
  uint32_t rk[20];     // Philox round keys (seed_lo + r W0, seed_hi + r W1), r = 0..9: constant-bank operands
  uint32_t cell_base;  // RNG cell coordinate of local cell 0
  uint32_t flags;
  int32_t pairs_per_cell;
  const int32_t *pairs_count;  // per-cell request or nullptr
  int32_t op;  // 0 = VHS-NN, 1 = ab initio table, 2 = ab initio MLP
  float mass;
  // VHS-NN
  float inv_sigma_v, sigma_v, inv_T_scale, noise_sigma, shell_eps;
  float T_coef;        // m / (3 kB): T_cell = T_coef Theta / N
  float vhs_c, vhs_e;  // sigma_T(g) g = vhs_c * g^vhs_e
  // ab initio
  float lnE_min, inv_lnE_range;
  float e_coef;  // m / (4 kB)
  ChiTableDev table;
  dsmc_pair_dump dump;
  int32_t dump_any;
  int32_t *status;
  // split form of the chi-MLP step (dsmc_cells.cu): per pair (index = first slot of the cell / 2 + pair slot) the two
  // network inputs and chi; per particle the pairing permutation as 16-bit byte offsets
  float *feat0, *feat1, *chi_pair;
  uint16_t *pi_g;
  float *out3[3];       // VHS-NN split form: the three network outputs per pair
  int64_t split_np;     // VHS-NN split form: stride between the input arrays feat0 + k split_np, k < split_din
  int32_t split_din;
  int32_t split_stage;  // chunk kernels (with-replacement selection): 0 = whole step, 3 = network inputs only, 4 = chi from chi_pair
  // chunk decomposition (filled by launch_chunk_map)
  int32_t n_chunks;
  const int32_t *chunk_first;  // [n_chunks + 1]
  const int4 *chunk_meta;      // [n_chunks] (first cell, end cell, first slot, end slot)
  int32_t *big;                // [0] = count, [1..] deferred chunk ids
  int32_t *big2;               // second-level deferred list (chunks that did not fit the middle footprint)
  int32_t *work;               // [0], [1]: next chunk / next deferred entry (persistent kernels)
};

}  // namespace dsmc

namespace dsmc {
// launch with programmatic stream serialisation: the kernel calls pdl_wait() before it touches its predecessor's data
template <class... KArgs, class... Args>
static inline cudaError_t launch_pdl(void (*kern)(KArgs...), int grid, int block, size_t smem, cudaStream_t s, Args... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)block);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

}  // namespace dsmc

struct dsmc_ctx {
  int device;
  cudaStream_t stream;
  cudaStream_t side_stream;  // dsmc_step_host: perm / cell_start go back to the host while the collide kernels run
  cudaEvent_t ev_bin, ev_side;
  int64_t max_particles;
  int32_t max_cells;
  int32_t *d_status;
  // dsmc_bin workspace: tile histograms, group sums, ping-pong record / cell-id buffers
  int32_t *d_bin_hist;   // [tiles][kBinMaxRadix]
  int32_t *d_bin_group;  // [num_sms][kBinMaxRadix]
  float4 *d_bin_rec[2];  // (idx, vx, vy, vz) between passes
  int32_t *d_bin_cell[2];
  int32_t *d_cell_count;      // [max_cells + 1] particles per cell (dsmc_bin)
  int32_t *d_cell_tile_sums;  // [(max_cells + 1) / 4096 + 1]
  int32_t *d_chunk_first;  // [max_particles / kChunk + 2]
  int4 *d_chunk_meta;      // [max_particles / kChunk + 2]
  int32_t *d_big;          // [max_particles / kChunk + 2]
  int32_t *d_big2;         // [max_particles / kChunk + 2]
  int32_t *d_work;         // [4] work counters of the persistent kernels ([0] main pass, [1] deferred pass)
  int4 *d_cell_list;       // [3][max_cells] cell lists of the cell-team kernels (dsmc_cells.cu)
  int32_t *d_list_ctr;     // [2][8] list lengths and work counters, alternating between steps
  int64_t list_epoch;
  int64_t launches;
  int num_sms;
  // operators
  bool has_mlp[2];
  dsmc::MlpDev mlp[2];
  dsmc::MlpTcDev mlp_tc[2];
  float *d_weights[2];
  dsmc::TcTailF32 tc_tail[2];  // HOST copies, filled by dsmc_set_mlp when the tensor-core image exists
  void *d_tc_blob[2];
  bool has_table;
  dsmc::ChiTableDev table;
  float *d_table;
  // dsmc_step_host staging
  int32_t *h_cell;
  float *h_v[3], *h_vs[3];
  int32_t *h_perm, *h_cell_start;
  float *h_x[2];  // dsmc_couette_run: positions (unsorted / sorted)
  int32_t *h_counts;  // dsmc_couette_run, NTC: candidate counts, remainders, count / acceptance caps [cells]
  double *h_rem;
  float *h_cap[2];
  int64_t host_cap_n;
  int32_t host_cap_cells;
};

namespace dsmc {
// launchers (each returns a DSMC_* status and bumps ctx->launches)
int bin_num_passes(int32_t K);
int launch_bin(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cell, const float *vx, const float *vy,
               const float *vz, float *vx_s, float *vy_s, float *vz_s, int32_t *perm, int32_t *cell_start);
int launch_cell_moments(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cs, const float *vx, const float *vy,
                        const float *vz, double *moments);
int launch_moment_match(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cs, float *vx, float *vy, float *vz,
                        const double *target, uint32_t flags);
int launch_chunk_map(dsmc_ctx *c, StepParams &p);
int launch_collide(dsmc_ctx *c, const StepParams &p, const MlpDev *net);
int launch_collide_cells(dsmc_ctx *c, const StepParams &p);
int launch_collide_cells_mlp(dsmc_ctx *c, const StepParams &p, const MlpTcDev *net);
int launch_collide_cells_split(dsmc_ctx *c, const StepParams &p, const MlpTcDev *net);
int launch_collide_replace_split(dsmc_ctx *c, const StepParams &p, const MlpTcDev *net);  // dsmc_collide.cu
int launch_collide_cells_vhs_split(dsmc_ctx *c, const StepParams &p, const MlpTcDev *net);  // dsmc_cells.cu
int launch_collide_vhs_replace_split(dsmc_ctx *c, const StepParams &p, const MlpTcDev *net);  // dsmc_collide.cu
int launch_chi_rows_tc(dsmc_ctx *c, int64_t n, const float *x0, const float *x1, float *chi, const MlpTcDev *net);
int launch_mlp_rows_tc_split(dsmc_ctx *c, int64_t n, const float *x, int64_t x_stride, float *y0, float *y1, float *y2,
                             const MlpTcDev *net, const TcTailF32 *tail);  // chi-MLP on tcgen05 (dsmc_cells_mlp.cu)  // cell-team form, chi-table operator (dsmc_cells.cu)
int launch_collide_tc(dsmc_ctx *c, const StepParams &p, const MlpTcDev *net);
int launch_chi_batch(dsmc_ctx *c, int64_t n, const float *E, const float *b, float *chi, int mode, float b_max,
                     float lnE_min, float lnE_max, const MlpDev *net);
int launch_chi_batch_tc(dsmc_ctx *c, int64_t n, const float *E, const float *b, float *chi, float b_max,
                        float lnE_min, float lnE_max, const MlpTcDev *net);
int launch_chi_exact(dsmc_ctx *c, int64_t n, const float *E_over_k, const float *b, float *chi, double eps_over_k,
                     double sigma, int take_abs);
int launch_table_node_coords(dsmc_ctx *c, int nE, int nB, double lnE_min, double lnE_max, float *E, float *b);
int launch_cap_and_quad(dsmc_ctx *c, int nE, int nB, float *table_dev, float4 *quad_dev);
int launch_chi_table_lj(dsmc_ctx *c, int nE, int nB, double lnE_min, double lnE_max, double b_max, double eps_over_k,
                        double sigma, float *table_dev, float4 *quad_dev);
int launch_move_couette(dsmc_ctx *c, int64_t n, float *x, float *vx, float *vy, float *vz, int32_t *cell,
                        int32_t *bounces, const dsmc_couette_params *g, uint64_t seed, uint32_t step);
int launch_ntc_counts(dsmc_ctx *c, int32_t K, const int32_t *cs, const float *cap, double coef, double *remainder,
                      int32_t *counts);
int launch_fill_f32(dsmc_ctx *c, int64_t n, float *dst, float value);
int launch_gather_f32(dsmc_ctx *c, int64_t n, const int32_t *perm, const float *src, float *dst);
int launch_sample_cells(dsmc_ctx *c, int32_t K, const int32_t *cs, const float *vx, const float *vy, const float *vz,
                        double *acc);
// host-side packing of the tensor-core weight image (dsmc_collide_tc.cu)
int build_tc_blob(const dsmc_mlp_desc *d, void **d_blob, MlpTcDev *out, cudaStream_t s);
}  // namespace dsmc
