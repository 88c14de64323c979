// C-ABI entry points of libdsmc_b200.so (see include/dsmc.h): context management, operator
// staging, argument checks, and dispatch to the kernel launchers.  No compute happens here.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <utility>
#include <vector>

#include "dsmc_internal.h"

using namespace dsmc;

#define CK(x)                                  \
  do {                                         \
    if ((x) != cudaSuccess) return DSMC_ERR_CUDA; \
  } while (0)

// the quad table as a linear texture (cell-team kernel: gathers on the TEX pipe); 0 when it cannot be made
static void make_table_texture(dsmc_ctx *c, size_t n_quads) {
  if (c->table.tex) cudaDestroyTextureObject(c->table.tex);
  c->table.tex = 0;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, c->device) != cudaSuccess || n_quads > (size_t)prop.maxTexture1DLinear) return;
  cudaResourceDesc rd;
  memset(&rd, 0, sizeof(rd));
  rd.resType = cudaResourceTypeLinear;
  rd.res.linear.devPtr = c->d_table;
  rd.res.linear.desc = cudaCreateChannelDesc<float4>();
  rd.res.linear.sizeInBytes = n_quads * sizeof(float4);
  cudaTextureDesc td;
  memset(&td, 0, sizeof(td));
  td.readMode = cudaReadModeElementType;
  cudaTextureObject_t t = 0;
  if (cudaCreateTextureObject(&t, &rd, &td, nullptr) == cudaSuccess) c->table.tex = t;
  else cudaGetLastError();
}

extern "C" {

static int create_impl(dsmc_ctx *c, int device, int64_t max_particles, int32_t max_cells) {
  c->device = device;
  c->stream = 0;
  c->max_particles = max_particles;
  c->max_cells = max_cells;
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, device));
  c->num_sms = prop.multiProcessorCount;
  CK(cudaMalloc(&c->d_status, sizeof(int32_t)));
  CK(cudaMemset(c->d_status, 0, sizeof(int32_t)));
  {
    const size_t np = (size_t)(max_particles > 0 ? max_particles : 1);
    const size_t tiles = (np + kBinTile - 1) / kBinTile;
    const int passes = bin_num_passes(max_cells > 0 ? max_cells : 1);
    if (passes > 3) return DSMC_ERR_INVALID_ARG;
    CK(cudaMalloc(&c->d_bin_hist, sizeof(int32_t) * tiles * kBinMaxRadix));
    CK(cudaMalloc(&c->d_bin_group, sizeof(int32_t) * (size_t)c->num_sms * kBinMaxRadix));
    CK(cudaMalloc(&c->d_cell_count, sizeof(int32_t) * ((size_t)(max_cells > 0 ? max_cells : 1) + 1)));
    // both are kept zero between calls by the kernels that consume them (no memsets inside dsmc_bin)
    CK(cudaMemset(c->d_bin_group, 0, sizeof(int32_t) * (size_t)c->num_sms * kBinMaxRadix));
    CK(cudaMemset(c->d_cell_count, 0, sizeof(int32_t) * ((size_t)(max_cells > 0 ? max_cells : 1) + 1)));
    CK(cudaMalloc(&c->d_cell_tile_sums, sizeof(int32_t) * ((size_t)(max_cells > 0 ? max_cells : 1) / 4096 + 2)));
    for (int i = 0; i < 2; ++i) {
      CK(cudaMalloc(&c->d_bin_cell[i], sizeof(int32_t) * (np + 16)));  // (+ slack: the VHS-NN split form keeps its outputs here)
      // (buffer 0 always exists: the split tensor-core steps keep their pair arrays there, up to 16 B / particle + 128 B)
      if (i == 0 || i < passes - 1) CK(cudaMalloc(&c->d_bin_rec[i], sizeof(float4) * (np + 16)));
    }
  }
  const size_t n_chunks = (size_t)(max_particles / kChunk + 2);
  CK(cudaMalloc(&c->d_chunk_first, sizeof(int32_t) * n_chunks));
  CK(cudaMalloc(&c->d_big, sizeof(int32_t) * (n_chunks + 1)));
  CK(cudaMalloc(&c->d_chunk_meta, sizeof(int4) * n_chunks));
  CK(cudaMalloc(&c->d_big2, sizeof(int32_t) * (n_chunks + 1)));
  CK(cudaMalloc(&c->d_work, sizeof(int32_t) * 4));
  CK(cudaMalloc(&c->d_cell_list, sizeof(int4) * 3 * (size_t)(max_cells > 0 ? max_cells : 1)));
  CK(cudaMalloc(&c->d_list_ctr, sizeof(int32_t) * 32));
  CK(cudaMemset(c->d_list_ctr, 0, sizeof(int32_t) * 32));
  return DSMC_OK;
}

int dsmc_destroy(dsmc_ctx *c);

int dsmc_create(dsmc_ctx **out, int device, int64_t max_particles, int32_t max_cells) {
  if (!out || max_particles < 0 || max_cells < 0 || max_particles >= (int64_t(1) << 31)) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(device));
  dsmc_ctx *c = new (std::nothrow) dsmc_ctx();
  if (!c) return DSMC_ERR_CUDA;
  memset(c, 0, sizeof(*c));
  const int rc = create_impl(c, device, max_particles, max_cells);
  if (rc != DSMC_OK) {  // frees whatever was allocated before the failure
    c->device = device;
    dsmc_destroy(c);
    cudaGetLastError();
    return rc;
  }
  *out = c;
  return DSMC_OK;
}

int dsmc_destroy(dsmc_ctx *c) {
  if (!c) return DSMC_OK;
  cudaSetDevice(c->device);
  cudaStreamSynchronize(c->stream);
  cudaFree(c->d_status);
  cudaFree(c->d_bin_hist);
  cudaFree(c->d_bin_group);
  cudaFree(c->d_cell_count);
  cudaFree(c->d_cell_tile_sums);
  for (int i = 0; i < 2; ++i) { cudaFree(c->d_bin_rec[i]); cudaFree(c->d_bin_cell[i]); }
  cudaFree(c->d_chunk_first);
  cudaFree(c->d_big);
  cudaFree(c->d_chunk_meta);
  cudaFree(c->d_big2);
  cudaFree(c->d_work);
  cudaFree(c->d_cell_list);
  cudaFree(c->d_list_ctr);
  for (int s = 0; s < 2; ++s) {
    cudaFree(c->d_weights[s]);
    cudaFree(c->d_tc_blob[s]);
  }
  if (c->table.tex) cudaDestroyTextureObject(c->table.tex);
  cudaFree(c->d_table);
  cudaFree(c->h_cell);
  for (int a = 0; a < 3; ++a) { cudaFree(c->h_v[a]); cudaFree(c->h_vs[a]); }
  cudaFree(c->h_perm);
  cudaFree(c->h_cell_start);
  cudaFree(c->h_x[0]);
  cudaFree(c->h_x[1]);
  cudaFree(c->h_counts);
  cudaFree(c->h_rem);
  cudaFree(c->h_cap[0]);
  cudaFree(c->h_cap[1]);
  if (c->side_stream) {
    cudaStreamDestroy(c->side_stream);
    cudaEventDestroy(c->ev_bin);
    cudaEventDestroy(c->ev_side);
  }
  delete c;
  return DSMC_OK;
}

int dsmc_set_stream(dsmc_ctx *c, void *cuda_stream) {
  if (!c) return DSMC_ERR_INVALID_ARG;
  c->stream = (cudaStream_t)cuda_stream;
  return DSMC_OK;
}

int dsmc_sync_status(dsmc_ctx *c) {
  if (!c) return DSMC_ERR_INVALID_ARG;
  int32_t st = 0;
  CK(cudaMemcpyAsync(&st, c->d_status, sizeof(st), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  if (st != 0) CK(cudaMemsetAsync(c->d_status, 0, sizeof(int32_t), c->stream));
  return st;
}

const char *dsmc_strerror(int s) {
  switch (s) {
    case DSMC_OK: return "ok";
    case DSMC_ERR_INVALID_ARG: return "invalid argument";
    case DSMC_ERR_BAD_CELL_INDEX: return "cell index out of range";
    case DSMC_ERR_CELL_TOO_LARGE: return "cell has more particles than DSMC_MAX_CELL_PARTICLES";
    case DSMC_ERR_NOT_CONFIGURED: return "operator (MLP or chi table) not set";
    case DSMC_ERR_CUDA: return "CUDA runtime error";
    case DSMC_ERR_UNSUPPORTED_SHAPE: return "MLP shape not supported by the requested path";
    case DSMC_ERR_NOALLOC_LIMIT: return "size beyond the fixed scratch array of the no-allocation entry point (DSMC_NOALLOC_MAX_*)";
    default: return "unknown status";
  }
}

int64_t dsmc_launch_count(const dsmc_ctx *c) { return c ? c->launches : 0; }

int dsmc_set_mlp(dsmc_ctx *c, int slot, const dsmc_mlp_desc *d) {
  if (!c || !d || slot < 0 || slot > 1 || !d->W || !d->b) return DSMC_ERR_INVALID_ARG;
  if (d->n_layers < 2 || d->n_layers > 6) return DSMC_ERR_UNSUPPORTED_SHAPE;
  if (d->act < 0 || d->act > 2) return DSMC_ERR_INVALID_ARG;
  int dmax = 0;
  size_t total = 0;
  for (int l = 0; l <= d->n_layers; ++l) {
    if (d->dims[l] < 1 || d->dims[l] > 256) return DSMC_ERR_UNSUPPORTED_SHAPE;
    dmax = d->dims[l] > dmax ? d->dims[l] : dmax;
    if (l < d->n_layers) total += (size_t)d->dims[l] * d->dims[l + 1] + d->dims[l + 1];
  }
  if (slot == 0 && (!(d->dims[0] == 8 || d->dims[0] == 6) || d->dims[d->n_layers] != 3)) return DSMC_ERR_UNSUPPORTED_SHAPE;
  if (slot == 1 && (d->dims[0] != 2 || d->dims[d->n_layers] != 1)) return DSMC_ERR_UNSUPPORTED_SHAPE;
  for (int l = 0; l < d->n_layers; ++l)
    if (!d->W[l] || !d->b[l]) return DSMC_ERR_INVALID_ARG;
  // stage transposed fp32 weights: Wt[l][in][out].  The new image is built completely before the old one is released,
  // so a failure leaves the slot as it was.
  std::vector<float> host((total + 3) & ~size_t(3));
  MlpDev m{};
  m.n_layers = d->n_layers;
  m.act = d->act;
  m.dmax = (dmax + 3) & ~3;
  CK(cudaSetDevice(c->device));
  float *wnew = nullptr;
  CK(cudaMalloc(&wnew, sizeof(float) * host.size()));
  size_t off = 0;
  for (int l = 0; l < d->n_layers; ++l) {
    const int din = d->dims[l], dout = d->dims[l + 1];
    m.dims[l] = din;
    m.dims[l + 1] = dout;
    m.Wt[l] = wnew + off;
    for (int i = 0; i < din; ++i)
      for (int o = 0; o < dout; ++o) host[off + (size_t)i * dout + o] = d->W[l][(size_t)o * din + i];
    off += (size_t)din * dout;
    m.b[l] = wnew + off;
    for (int o = 0; o < dout; ++o) host[off + o] = d->b[l][o];
    off += dout;
  }
  if (cudaMemcpy(wnew, host.data(), sizeof(float) * host.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
    cudaFree(wnew);
    return DSMC_ERR_CUDA;
  }
  // tensor-core image when the shape allows it
  void *blob_new = nullptr;
  MlpTcDev tc_new;
  memset(&tc_new, 0, sizeof(tc_new));
  const int rc = build_tc_blob(d, &blob_new, &tc_new, c->stream);
  if (rc != DSMC_OK && rc != DSMC_ERR_UNSUPPORTED_SHAPE) {
    cudaFree(wnew);
    cudaFree(blob_new);
    return rc;
  }
  CK(cudaStreamSynchronize(c->stream));  // no kernel still reads the old images
  cudaFree(c->d_weights[slot]);
  cudaFree(c->d_tc_blob[slot]);
  c->d_weights[slot] = wnew;
  c->d_tc_blob[slot] = blob_new;
  c->mlp[slot] = m;
  c->mlp_tc[slot] = tc_new;
  memset(&c->tc_tail[slot], 0, sizeof(c->tc_tail[slot]));
  if (tc_new.H != 0 && d->n_layers == 3 && d->dims[3] <= 3) {
    dsmc::TcTailF32 &t = c->tc_tail[slot];
    const int H = d->dims[2];  // width of the second hidden layer (units beyond it are zero padding)
    const float hs = d->act == DSMC_ACT_SILU ? 0.5f : 1.0f;
    t.d_out = d->dims[3];
    for (int k = 0; k < H; ++k) t.b2[k] = hs * d->b[1][k];
    for (int o = 0; o < t.d_out; ++o) {
      for (int k = 0; k < H; ++k) t.w3[o][k] = d->W[2][(size_t)o * H + k];
      t.b3[o] = d->b[2][o];
    }
  }
  c->has_mlp[slot] = true;
  return DSMC_OK;
}

// makes `tnew` (device, 4 (nE-1)(nB-1) floats in quad layout, ownership passes to the context) the context's table
static void install_quad_table(dsmc_ctx *c, int32_t nE, int32_t nB, float lnE_min, float lnE_max, float *tnew) {
  if (c->table.tex) cudaDestroyTextureObject(c->table.tex);
  c->table.tex = 0;
  cudaFree(c->d_table);
  c->d_table = tnew;
  c->table.quad = reinterpret_cast<const float4 *>(c->d_table);
  c->table.nE = nE;
  c->table.nB = nB;
  c->table.lnE_min = lnE_min;
  const double inv = (double)(nE - 1) / ((double)lnE_max - (double)lnE_min);
  c->table.inv_dlnE = (float)inv;
  c->table.c1 = (float)(0.6931471805599453 * inv);
  c->table.c0 = (float)(-(double)lnE_min * inv);
  c->table.fE1 = (float)(nE - 1);
  c->table.fB1 = (float)(nB - 1);
  make_table_texture(c, (size_t)(nE - 1) * (nB - 1));
  c->has_table = true;
}

int dsmc_set_chi_table(dsmc_ctx *c, const float *chi_host, int32_t nE, int32_t nB, float lnE_min, float lnE_max) {
  if (!c || !chi_host || nE < 2 || nB < 2 || !(lnE_max > lnE_min)) return DSMC_ERR_INVALID_ARG;
  for (size_t i = 0; i < (size_t)nE * nB; ++i)
    if (!isfinite(chi_host[i])) return DSMC_ERR_INVALID_ARG;  // a non-finite node would poison every pair near it
  CK(cudaSetDevice(c->device));
  // device layout: the 2x2 nodes of every grid cell side by side, so a lookup is one 16-byte load
  const size_t nq = (size_t)(nE - 1) * (nB - 1);
  std::vector<float> quad(4 * nq);
  for (int iE = 0; iE + 1 < nE; ++iE)
    for (int iB = 0; iB + 1 < nB; ++iB) {
      float *q = &quad[4 * ((size_t)iE * (nB - 1) + iB)];
      q[0] = chi_host[(size_t)iE * nB + iB];
      q[1] = chi_host[(size_t)iE * nB + iB + 1];
      q[2] = chi_host[(size_t)(iE + 1) * nB + iB];
      q[3] = chi_host[(size_t)(iE + 1) * nB + iB + 1];
    }
  // the new table is on the device before the old one is released: a failure leaves the context as it was
  float *tnew = nullptr;
  CK(cudaMalloc(&tnew, sizeof(float) * quad.size()));
  if (cudaMemcpy(tnew, quad.data(), sizeof(float) * quad.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
    cudaFree(tnew);
    return DSMC_ERR_CUDA;
  }
  CK(cudaStreamSynchronize(c->stream));
  install_quad_table(c, nE, nB, lnE_min, lnE_max, tnew);
  return DSMC_OK;
}

static int check_sorted_args(dsmc_ctx *c, int64_t n, int32_t K, const void *cs, const void *x, const void *y,
                             const void *z) {
  if (!c || n < 0 || K < 0 || n >= (int64_t(1) << 31) || n > c->max_particles) return DSMC_ERR_INVALID_ARG;
  if (n == 0 || K == 0) return 1;  // nothing to do
  if (!cs || !x || !y || !z) return DSMC_ERR_INVALID_ARG;
  return DSMC_OK;
}

int dsmc_bin(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cell, const float *vx, const float *vy,
             const float *vz, float *vx_s, float *vy_s, float *vz_s, int32_t *perm, int32_t *cell_start) {
  if (!c || n < 0 || K < 0 || n >= (int64_t(1) << 31) || K > c->max_cells || n > c->max_particles)
    return DSMC_ERR_INVALID_ARG;
  if (!cell_start) return DSMC_ERR_INVALID_ARG;
  if (n > 0 && (!cell || !vx || !vy || !vz || !vx_s || !vy_s || !vz_s || !perm)) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  return launch_bin(c, n, K, cell, vx, vy, vz, vx_s, vy_s, vz_s, perm, cell_start);
}

int dsmc_cell_moments(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cs, const float *vx, const float *vy,
                      const float *vz, double *moments) {
  if (!c || n < 0 || K < 0) return DSMC_ERR_INVALID_ARG;
  if (K == 0) return DSMC_OK;
  if (!cs || !moments || (n > 0 && (!vx || !vy || !vz))) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  return launch_cell_moments(c, n, K, cs, vx, vy, vz, moments);
}

int dsmc_moment_match(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cs, float *vx, float *vy, float *vz,
                      const double *target, uint32_t flags) {
  int rc = check_sorted_args(c, n, K, cs, vx, vy, vz);
  if (rc != DSMC_OK) return rc == 1 ? DSMC_OK : rc;
  if (!target) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  return launch_moment_match(c, n, K, cs, vx, vy, vz, target, flags);
}

static void fill_common(StepParams &p, dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cs, float *vx, float *vy,
                        float *vz, const float *cap, uint64_t seed, uint32_t step, const dsmc_pair_dump *dump) {
  memset(&p, 0, sizeof(p));
  p.n = n; p.n_cells = K; p.cell_start = cs;
  p.vx = vx; p.vy = vy; p.vz = vz;
  p.cap = cap;
  p.seed_lo = (uint32_t)(seed & 0xFFFFFFFFu);
  p.seed_hi = (uint32_t)(seed >> 32);
  p.step = step;
  for (uint32_t r = 0; r < 10; ++r) {
    p.rk[2 * r] = p.seed_lo + r * 0x9E3779B9u;
    p.rk[2 * r + 1] = p.seed_hi + r * 0xBB67AE85u;
  }
  if (dump) p.dump = *dump;
  p.dump_any = (dump && (dump->pair_i || dump->pair_j || dump->accepted || dump->gprime || dump->aux)) ? 1 : 0;
  p.status = c->d_status;
}

int dsmc_collide_vhs_nn(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cs, float *vx, float *vy, float *vz,
                        const float *sigma_cr_max, const dsmc_vhs_params *prm, uint64_t seed, uint32_t step,
                        const dsmc_pair_dump *dump) {
  if (!prm) return DSMC_ERR_INVALID_ARG;
  int rc = check_sorted_args(c, n, K, cs, vx, vy, vz);
  if (rc != DSMC_OK) return rc == 1 ? DSMC_OK : rc;
  if (!c->has_mlp[0]) return DSMC_ERR_NOT_CONFIGURED;
  if (!(prm->sigma_v > 0.f) || !(prm->T_scale > 0.f) || !(prm->mass > 0.f)) return DSMC_ERR_INVALID_ARG;
  StepParams p;
  fill_common(p, c, n, K, cs, vx, vy, vz, sigma_cr_max, seed, step, dump);
  p.flags = prm->flags;
  p.pairs_per_cell = prm->pairs_per_cell;
  p.pairs_count = prm->pairs_count;
  p.op = 0;
  p.cell_base = (uint32_t)prm->cell_base;
  p.mass = prm->mass;
  p.sigma_v = prm->sigma_v;
  p.inv_sigma_v = 1.0f / prm->sigma_v;
  p.inv_T_scale = 1.0f / prm->T_scale;
  p.T_coef = (float)((double)prm->mass / (3.0 * 1.380649e-23));
  p.noise_sigma = prm->noise_sigma;
  p.shell_eps = prm->shell_eps;
  if ((prm->flags & DSMC_F_ACCEPT) && sigma_cr_max) {
    // sigma_T(g) g = pi d^2 (2 kB T_ref / (m_r g^2))^(omega-1/2) / Gamma(5/2-omega) * g, m_r = m/2
    const double mr = 0.5 * (double)prm->mass, kB = 1.380649e-23;
    p.vhs_c = (float)(M_PI * (double)prm->d_ref * prm->d_ref * pow(2.0 * kB * prm->T_ref / mr, prm->omega - 0.5) /
                      tgamma(2.5 - prm->omega));
    p.vhs_e = (float)(2.0 - 2.0 * (double)prm->omega);
  }
  CK(cudaSetDevice(c->device));
  if (prm->flags & DSMC_F_BF16_TC) {
    if (c->mlp_tc[0].H == 0) return DSMC_ERR_UNSUPPORTED_SHAPE;
    return launch_collide_tc(c, p, &c->mlp_tc[0]);
  }
  return launch_collide(c, p, &c->mlp[0]);
}

int dsmc_collide_abinitio(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cs, float *vx, float *vy, float *vz,
                          const float *cr_max, const dsmc_abinitio_params *prm, uint64_t seed, uint32_t step,
                          const dsmc_pair_dump *dump) {
  if (!prm) return DSMC_ERR_INVALID_ARG;
  int rc = check_sorted_args(c, n, K, cs, vx, vy, vz);
  if (rc != DSMC_OK) return rc == 1 ? DSMC_OK : rc;
  if (prm->chi_mode != 0 && prm->chi_mode != 1) return DSMC_ERR_INVALID_ARG;
  if (prm->chi_mode == 0 && !c->has_table) return DSMC_ERR_NOT_CONFIGURED;
  if (prm->chi_mode == 1 && !c->has_mlp[1]) return DSMC_ERR_NOT_CONFIGURED;
  if (!(prm->mass > 0.f)) return DSMC_ERR_INVALID_ARG;
  if (prm->chi_mode == 1 && !(prm->lnE_max > prm->lnE_min)) return DSMC_ERR_INVALID_ARG;
  StepParams p;
  fill_common(p, c, n, K, cs, vx, vy, vz, cr_max, seed, step, dump);
  p.flags = prm->flags & ~(uint32_t)(DSMC_F_NOISE | DSMC_F_ENERGY_SHELL);
  p.pairs_per_cell = prm->pairs_per_cell;
  p.pairs_count = prm->pairs_count;
  p.op = prm->chi_mode == 0 ? 1 : 2;
  p.cell_base = (uint32_t)prm->cell_base;
  p.mass = prm->mass;
  p.e_coef = (float)((double)prm->mass / (4.0 * 1.380649e-23));
  p.lnE_min = prm->lnE_min;
  p.inv_lnE_range = prm->chi_mode == 1 ? 1.0f / (prm->lnE_max - prm->lnE_min) : 0.f;
  p.table = c->table;
  CK(cudaSetDevice(c->device));
  if (prm->chi_mode == 1 && (prm->flags & DSMC_F_BF16_TC)) {
    if (c->mlp_tc[1].H == 0) return DSMC_ERR_UNSUPPORTED_SHAPE;
    return launch_collide_tc(c, p, &c->mlp_tc[1]);
  }
  return launch_collide(c, p, prm->chi_mode == 1 ? &c->mlp[1] : nullptr);
}

int dsmc_chi_batch(dsmc_ctx *c, int64_t n, const float *E_over_k, const float *b, float *chi, int32_t chi_mode,
                   float b_max, float lnE_min, float lnE_max, uint32_t flags) {
  if (!c || n < 0 || (chi_mode != 0 && chi_mode != 1) || !(b_max > 0.f)) return DSMC_ERR_INVALID_ARG;
  if (n == 0) return DSMC_OK;
  if (!E_over_k || !b || !chi) return DSMC_ERR_INVALID_ARG;
  if (chi_mode == 0 && !c->has_table) return DSMC_ERR_NOT_CONFIGURED;
  if (chi_mode == 1 && !c->has_mlp[1]) return DSMC_ERR_NOT_CONFIGURED;
  if (chi_mode == 1 && !(lnE_max > lnE_min)) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  if (chi_mode == 1 && (flags & DSMC_F_BF16_TC)) {
    if (c->mlp_tc[1].H == 0) return DSMC_ERR_UNSUPPORTED_SHAPE;
    return launch_chi_batch_tc(c, n, E_over_k, b, chi, b_max, lnE_min, lnE_max, &c->mlp_tc[1]);
  }
  return launch_chi_batch(c, n, E_over_k, b, chi, chi_mode, b_max, lnE_min, lnE_max, &c->mlp[1]);
}

static int ensure_host_staging(dsmc_ctx *c, int64_t n, int32_t K) {
  if (n <= c->host_cap_n && K <= c->host_cap_cells) return DSMC_OK;
  // every pointer is nulled as it is freed: a failure below leaves nothing dangling for dsmc_destroy or the next call
  auto drop = [](auto *&p) {
    cudaFree(p);
    p = nullptr;
  };
  drop(c->h_cell);
  for (int a = 0; a < 3; ++a) {
    drop(c->h_v[a]);
    drop(c->h_vs[a]);
  }
  drop(c->h_perm);
  drop(c->h_cell_start);
  drop(c->h_x[0]);
  drop(c->h_x[1]);
  drop(c->h_counts);
  drop(c->h_rem);
  drop(c->h_cap[0]);
  drop(c->h_cap[1]);
  c->host_cap_n = 0;
  c->host_cap_cells = 0;
  CK(cudaMalloc(&c->h_cell, sizeof(int32_t) * (size_t)n));
  for (int a = 0; a < 3; ++a) {
    CK(cudaMalloc(&c->h_v[a], sizeof(float) * (size_t)n));
    CK(cudaMalloc(&c->h_vs[a], sizeof(float) * (size_t)n));
  }
  CK(cudaMalloc(&c->h_perm, sizeof(int32_t) * (size_t)n));
  for (int a = 0; a < 2; ++a) CK(cudaMalloc(&c->h_x[a], sizeof(float) * (size_t)n));
  CK(cudaMalloc(&c->h_cell_start, sizeof(int32_t) * (size_t)(K + 1)));
  CK(cudaMalloc(&c->h_counts, sizeof(int32_t) * (size_t)K));
  CK(cudaMalloc(&c->h_rem, sizeof(double) * (size_t)K));
  for (int a = 0; a < 2; ++a) CK(cudaMalloc(&c->h_cap[a], sizeof(float) * (size_t)K));
  c->host_cap_n = n;
  c->host_cap_cells = K;
  return DSMC_OK;
}

int dsmc_build_chi_table_lj(dsmc_ctx *c, int32_t nE, int32_t nB, float lnE_min, float lnE_max, float b_max,
                            float eps_over_k, float sigma, float *chi_out) {
  if (!c || nE < 2 || nB < 2 || !(lnE_max > lnE_min) || !(b_max > 0.f) || !(eps_over_k > 0.f) || !(sigma > 0.f))
    return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  CK(cudaStreamSynchronize(c->stream));
  const size_t nq = (size_t)(nE - 1) * (nB - 1), nn = (size_t)nE * nB;
  float *nodes = nullptr, *tnew = nullptr;
  CK(cudaMalloc(&tnew, sizeof(float) * 4 * nq));
  if (cudaMalloc(&nodes, sizeof(float) * nn) != cudaSuccess) {
    cudaFree(tnew);
    return DSMC_ERR_CUDA;
  }
  int rc = launch_chi_table_lj(c, nE, nB, (double)lnE_min, (double)lnE_max, (double)b_max, (double)eps_over_k,
                               (double)sigma, nodes, reinterpret_cast<float4 *>(tnew));
  if (rc == DSMC_OK && chi_out &&
      cudaMemcpyAsync(chi_out, nodes, sizeof(float) * nn, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess)
    rc = DSMC_ERR_CUDA;
  if (cudaStreamSynchronize(c->stream) != cudaSuccess) rc = DSMC_ERR_CUDA;
  cudaFree(nodes);
  if (rc != DSMC_OK) {  // the installed table (if any) stays
    cudaFree(tnew);
    return rc;
  }
  install_quad_table(c, nE, nB, lnE_min, lnE_max, tnew);
  return DSMC_OK;
}

int dsmc_build_chi_table_mlp(dsmc_ctx *c, int32_t nE, int32_t nB, float lnE_min, float lnE_max, uint32_t flags,
                             float *chi_out) {
  if (!c || nE < 2 || nB < 2 || !(lnE_max > lnE_min) || (flags & ~(uint32_t)DSMC_F_BF16_TC)) return DSMC_ERR_INVALID_ARG;
  if (!c->has_mlp[1]) return DSMC_ERR_NOT_CONFIGURED;
  if ((flags & DSMC_F_BF16_TC) && c->mlp_tc[1].H == 0) return DSMC_ERR_UNSUPPORTED_SHAPE;
  CK(cudaSetDevice(c->device));
  CK(cudaStreamSynchronize(c->stream));
  const size_t nq = (size_t)(nE - 1) * (nB - 1), nn = (size_t)nE * nB;
  float *nodes = nullptr, *tnew = nullptr, *coord = nullptr;
  CK(cudaMalloc(&tnew, sizeof(float) * 4 * nq));
  if (cudaMalloc(&nodes, sizeof(float) * nn) != cudaSuccess || cudaMalloc(&coord, sizeof(float) * 2 * nn) != cudaSuccess) {
    cudaFree(tnew);
    cudaFree(nodes);
    return DSMC_ERR_CUDA;
  }
  // node coordinates as a pair batch (E_r / k_B = exp(lnE_i), b = j / (nB - 1) with b_max = 1), the chi-MLP on them
  // through the same kernels dsmc_chi_batch uses, then the cap (Q23) and the quad layout
  int rc = launch_table_node_coords(c, nE, nB, (double)lnE_min, (double)lnE_max, coord, coord + nn);
  if (rc == DSMC_OK)
    rc = (flags & DSMC_F_BF16_TC)
             ? launch_chi_batch_tc(c, (int64_t)nn, coord, coord + nn, nodes, 1.f, lnE_min, lnE_max, &c->mlp_tc[1])
             : launch_chi_batch(c, (int64_t)nn, coord, coord + nn, nodes, 1, 1.f, lnE_min, lnE_max, &c->mlp[1]);
  if (rc == DSMC_OK) rc = launch_cap_and_quad(c, nE, nB, nodes, reinterpret_cast<float4 *>(tnew));
  if (rc == DSMC_OK && chi_out &&
      cudaMemcpyAsync(chi_out, nodes, sizeof(float) * nn, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess)
    rc = DSMC_ERR_CUDA;
  if (cudaStreamSynchronize(c->stream) != cudaSuccess) rc = DSMC_ERR_CUDA;
  cudaFree(nodes);
  cudaFree(coord);
  if (rc != DSMC_OK) {  // the installed table (if any) stays
    cudaFree(tnew);
    return rc;
  }
  install_quad_table(c, nE, nB, lnE_min, lnE_max, tnew);
  return DSMC_OK;
}

int dsmc_chi_exact_batch(dsmc_ctx *c, int64_t n, const float *E_over_k, const float *b, float *chi, float eps_over_k,
                         float sigma, uint32_t flags) {
  if (!c || n < 0 || !(eps_over_k > 0.f) || !(sigma > 0.f)) return DSMC_ERR_INVALID_ARG;
  if (n == 0) return DSMC_OK;
  if (!E_over_k || !b || !chi) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  return launch_chi_exact(c, n, E_over_k, b, chi, (double)eps_over_k, (double)sigma, (flags & DSMC_F_CHI_ABS) ? 1 : 0);
}

int dsmc_step_host_submit(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cell_h, const float *vx_h,
                          const float *vy_h, const float *vz_h, float *vx_out_h, float *vy_out_h, float *vz_out_h,
                          int32_t *perm_h, int32_t *cell_start_h, const dsmc_vhs_params *vhs,
                          const dsmc_abinitio_params *abi, uint64_t seed, uint32_t step) {
  if (!c || n <= 0 || K <= 0 || K > c->max_cells || (!vhs && !abi) || (vhs && abi)) return DSMC_ERR_INVALID_ARG;
  if (!cell_h || !vx_h || !vy_h || !vz_h || !vx_out_h || !vy_out_h || !vz_out_h) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  int rc = ensure_host_staging(c, n, K);
  if (rc != DSMC_OK) return rc;
  cudaStream_t s = c->stream;
  const float *src[3] = {vx_h, vy_h, vz_h};
  float *dst[3] = {vx_out_h, vy_out_h, vz_out_h};
  CK(cudaMemcpyAsync(c->h_cell, cell_h, sizeof(int32_t) * (size_t)n, cudaMemcpyHostToDevice, s));
  for (int a = 0; a < 3; ++a) CK(cudaMemcpyAsync(c->h_v[a], src[a], sizeof(float) * (size_t)n, cudaMemcpyHostToDevice, s));
  rc = dsmc_bin(c, n, K, c->h_cell, c->h_v[0], c->h_v[1], c->h_v[2], c->h_vs[0], c->h_vs[1], c->h_vs[2], c->h_perm,
                c->h_cell_start);
  if (rc != DSMC_OK) return rc;
  // perm and cell_start are final once the bin is done: they travel back on a side stream under the collide kernels
  const bool side = perm_h || cell_start_h;
  if (side) {
    if (!c->side_stream) {
      CK(cudaStreamCreateWithFlags(&c->side_stream, cudaStreamNonBlocking));
      CK(cudaEventCreateWithFlags(&c->ev_bin, cudaEventDisableTiming));
      CK(cudaEventCreateWithFlags(&c->ev_side, cudaEventDisableTiming));
    }
    CK(cudaEventRecord(c->ev_bin, s));
    CK(cudaStreamWaitEvent(c->side_stream, c->ev_bin, 0));
    if (perm_h)
      CK(cudaMemcpyAsync(perm_h, c->h_perm, sizeof(int32_t) * (size_t)n, cudaMemcpyDeviceToHost, c->side_stream));
    if (cell_start_h)
      CK(cudaMemcpyAsync(cell_start_h, c->h_cell_start, sizeof(int32_t) * (size_t)(K + 1), cudaMemcpyDeviceToHost,
                         c->side_stream));
  }
  if (vhs)
    rc = dsmc_collide_vhs_nn(c, n, K, c->h_cell_start, c->h_vs[0], c->h_vs[1], c->h_vs[2], nullptr, vhs, seed, step,
                             nullptr);
  else
    rc = dsmc_collide_abinitio(c, n, K, c->h_cell_start, c->h_vs[0], c->h_vs[1], c->h_vs[2], nullptr, abi, seed,
                               step, nullptr);
  if (rc != DSMC_OK) {
    if (side) cudaStreamSynchronize(c->side_stream);  // the copies into the caller's buffers must not outlive the call
    return rc;
  }
  for (int a = 0; a < 3; ++a) CK(cudaMemcpyAsync(dst[a], c->h_vs[a], sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost, s));
  if (side) {  // join the side stream before the final synchronisation
    CK(cudaEventRecord(c->ev_side, c->side_stream));
    CK(cudaStreamWaitEvent(s, c->ev_side, 0));
  }
  return DSMC_OK;
}

int dsmc_step_host(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cell_h, const float *vx_h, const float *vy_h,
                   const float *vz_h, float *vx_out_h, float *vy_out_h, float *vz_out_h, int32_t *perm_h,
                   int32_t *cell_start_h, const dsmc_vhs_params *vhs, const dsmc_abinitio_params *abi,
                   uint64_t seed, uint32_t step) {
  const int rc = dsmc_step_host_submit(c, n, K, cell_h, vx_h, vy_h, vz_h, vx_out_h, vy_out_h, vz_out_h, perm_h,
                                       cell_start_h, vhs, abi, seed, step);
  if (rc != DSMC_OK) {
    if (c) cudaStreamSynchronize(c->stream);  // copies into the caller's buffers must not outlive a failed call
    return rc;
  }
  return dsmc_sync_status(c);
}

int dsmc_ntc_counts(dsmc_ctx *c, int32_t K, const int32_t *cs, const float *sigma_cr_max, double coef,
                    double *remainder, int32_t *counts) {
  if (!c || K < 0 || !(coef >= 0.0)) return DSMC_ERR_INVALID_ARG;
  if (K == 0) return DSMC_OK;
  if (!cs || !sigma_cr_max || !remainder || !counts) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  return launch_ntc_counts(c, K, cs, sigma_cr_max, coef, remainder, counts);
}

int dsmc_move_couette(dsmc_ctx *c, int64_t n, float *x, float *vx, float *vy, float *vz, int32_t *cell,
                      int32_t *bounces, const dsmc_couette_params *g, uint64_t seed, uint32_t step) {
  if (!c || n < 0 || !g || !(g->L > 0.f) || !(g->dt >= 0.f) || !(g->rt_wall > 0.f) || g->n_cells <= 0 ||
      !(g->accommodation >= 0.f && g->accommodation <= 1.f))
    return DSMC_ERR_INVALID_ARG;
  if (n == 0) return DSMC_OK;
  if (!x || !vx || !vy || !vz || !cell) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  return launch_move_couette(c, n, x, vx, vy, vz, cell, bounces, g, seed, step);
}

int dsmc_gather_f32(dsmc_ctx *c, int64_t n, const int32_t *perm, const float *src, float *dst) {
  if (!c || n < 0) return DSMC_ERR_INVALID_ARG;
  if (n == 0) return DSMC_OK;
  if (!perm || !src || !dst || src == dst) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  return launch_gather_f32(c, n, perm, src, dst);
}

int dsmc_sample_cells(dsmc_ctx *c, int64_t n, int32_t K, const int32_t *cs, const float *vx, const float *vy,
                      const float *vz, double *acc) {
  if (!c || n < 0 || K < 0) return DSMC_ERR_INVALID_ARG;
  if (K == 0) return DSMC_OK;
  if (!cs || !acc || (n > 0 && (!vx || !vy || !vz))) return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  return launch_sample_cells(c, K, cs, vx, vy, vz, acc);
}

int dsmc_couette_run(dsmc_ctx *c, int64_t n, float *x, float *vx, float *vy, float *vz,
                     const dsmc_couette_params *g, const dsmc_vhs_params *vhs, const dsmc_abinitio_params *abi,
                     uint64_t seed, uint32_t step0, int32_t n_steps, int32_t sample_from, double *acc) {
  if (!c || n <= 0 || n > c->max_particles || !g || g->n_cells <= 0 || g->n_cells > c->max_cells || n_steps < 0 ||
      (!vhs && !abi) || (vhs && abi) || !x || !vx || !vy || !vz)
    return DSMC_ERR_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  const int32_t K = g->n_cells;
  int rc = ensure_host_staging(c, n, K);
  if (rc != DSMC_OK) return rc;
  cudaStream_t s = c->stream;
  const size_t bytes = sizeof(float) * (size_t)n;
  // state lives in (h_x[0], h_v) before the move / bin and in (h_x[1], h_vs) after it
  float *user[4] = {x, vx, vy, vz};
  float *sorted[4] = {c->h_x[1], c->h_vs[0], c->h_vs[1], c->h_vs[2]};
  float *unsorted[4] = {c->h_x[0], c->h_v[0], c->h_v[1], c->h_v[2]};
  for (int a = 0; a < 4; ++a) CK(cudaMemcpyAsync(unsorted[a], user[a], bytes, cudaMemcpyDeviceToDevice, s));
  // NTC rate control: per-cell candidate counts every step, uniform caps
  const bool ntc = g->ntc_coef > 0.f;
  dsmc_vhs_params pv;
  dsmc_abinitio_params pa;
  const float *cap = nullptr;
  if (vhs) pv = *vhs;
  if (abi) pa = *abi;
  if (ntc) {
    if (!(g->sigma_cr_max > 0.f)) return DSMC_ERR_INVALID_ARG;
    const float cap_accept =
        vhs ? g->sigma_cr_max : (float)((double)g->sigma_cr_max / (M_PI * (double)abi->b_max * (double)abi->b_max));
    rc = launch_fill_f32(c, K, c->h_cap[0], g->sigma_cr_max);
    if (rc == DSMC_OK) rc = launch_fill_f32(c, K, c->h_cap[1], cap_accept);
    if (rc != DSMC_OK) return rc;
    CK(cudaMemsetAsync(c->h_rem, 0, sizeof(double) * (size_t)K, s));
    pv.pairs_count = pa.pairs_count = c->h_counts;
    if ((vhs ? vhs->flags : abi->flags) & DSMC_F_ACCEPT) cap = c->h_cap[1];
  }
  for (int32_t k = 0; k < n_steps; ++k) {
    const uint32_t step = step0 + (uint32_t)k;
    rc = dsmc_move_couette(c, n, unsorted[0], unsorted[1], unsorted[2], unsorted[3], c->h_cell, nullptr, g, seed,
                           step);
    if (rc != DSMC_OK) return rc;
    rc = dsmc_bin(c, n, K, c->h_cell, unsorted[1], unsorted[2], unsorted[3], sorted[1], sorted[2], sorted[3],
                  c->h_perm, c->h_cell_start);
    if (rc != DSMC_OK) return rc;
    rc = dsmc_gather_f32(c, n, c->h_perm, unsorted[0], sorted[0]);
    if (rc != DSMC_OK) return rc;
    if (ntc) {
      rc = dsmc_ntc_counts(c, K, c->h_cell_start, c->h_cap[0], (double)g->ntc_coef, c->h_rem, c->h_counts);
      if (rc != DSMC_OK) return rc;
    }
    if (vhs)
      rc = dsmc_collide_vhs_nn(c, n, K, c->h_cell_start, sorted[1], sorted[2], sorted[3], cap, &pv, seed, step,
                               nullptr);
    else
      rc = dsmc_collide_abinitio(c, n, K, c->h_cell_start, sorted[1], sorted[2], sorted[3], cap, &pa, seed, step,
                                 nullptr);
    if (rc != DSMC_OK) return rc;
    if (acc && k >= sample_from) {
      rc = dsmc_sample_cells(c, n, K, c->h_cell_start, sorted[1], sorted[2], sorted[3], acc);
      if (rc != DSMC_OK) return rc;
    }
    for (int a = 0; a < 4; ++a) std::swap(sorted[a], unsorted[a]);  // this step's output is the next step's input
  }
  for (int a = 0; a < 4; ++a) CK(cudaMemcpyAsync(user[a], unsorted[a], bytes, cudaMemcpyDeviceToDevice, s));
  return dsmc_sync_status(c);
}

}  // extern "C"
