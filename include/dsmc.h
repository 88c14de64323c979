/*
 * dsmc.h -- C ABI of the B200-native neural DSMC collision step.
 *
 * Method: Roohi, Shoja-sani, Stefanov, "Physics Constrained Neural Collision Operators for
 * Variable Hard Sphere Surrogates and Ab Initio Angle Prediction in DSMC" (arxiv 2602.21244).
 * Citations "P:L<n>" are line numbers of the paper text; "Q<n>" are the readings
 * listed in DESIGN.md.  One call = one stage of the per-step collision path:
 *
 *   dsmc_bin               sort particles by cell index
 *   dsmc_collide_vhs_nn    fused step with the VHS-surrogate MLP (eqs. 1-11)
 *   dsmc_collide_abinitio  fused step with chi(E,b) by table or MLP + rotation
 *   dsmc_cell_moments      per-cell momentum / energy sums (eq. 10)
 *   dsmc_moment_match      cell-wise correction on its own (eqs. 10-11)
 *   dsmc_chi_batch         chi for independent (E_r, b) pairs
 *   dsmc_chi_exact_batch   chi by the deflection-integral quadrature itself (eq. 16), LJ 12-6
 *   dsmc_build_chi_table_lj  the chi table generated on the device by that quadrature
 *   dsmc_build_chi_table_mlp the chi table generated on the device by the chi-MLP
 *   dsmc_step_host         bin + fused step on HOST buffers (copies inside), for end-to-end timing
 *   dsmc_ntc_counts        NTC candidate counts with carried remainder
 *   dsmc_move_couette, dsmc_gather_f32, dsmc_sample_cells, dsmc_couette_run
 *                          the minimal DSMC loop around the step for the 1-D Couette layout
 *
 * Conventions
 *   - Plain C, no C++/torch types.  Every function returns an int status (0 = DSMC_OK).
 *   - Unless marked HOST, array arguments are DEVICE pointers owned by the caller; the library
 *     never allocates, frees or retains them.  Arrays need only their natural alignment.
 *   - Work is enqueued asynchronously on the context's stream (dsmc_set_stream; default stream
 *     0).  Argument errors detectable on the host are returned immediately and nothing is
 *     launched.  Data errors found on the device (cell index out of range, cell larger than
 *     DSMC_MAX_CELL_PARTICLES) set a sticky status word returned (and cleared) by
 *     dsmc_sync_status(), which synchronises the stream; outputs of such a call are unspecified.
 *   - One context per device and stream; a context is not thread-safe.
 *   - There is no CPU fallback: every stage runs in this library's sm_100a kernels.
 *
 * Random numbers: Philox4x32-10, key = seed, counter =
 * (index, cell, step, stream); stream 0 = pairing keys (slot p uses word p&3 of block p>>2),
 * stream 1 = (U_b, U_eps) of pair slot s (words 2(s&1), 2(s&1)+1 of block s>>1), stream 2 = Box-Muller
 * normals of pair slot s, stream 3 = U_acc of pair slot s (word s&3 of block s>>2, drawn only with
 * DSMC_F_ACCEPT); cell = local cell index + cell_base;
 * u = ((x>>9)+0.5) 2^-23.  Results therefore depend only on (seed, step, cell, slot): runs are bit-reproducible and a
 * run sharded by cell ranges is bit-identical to the unsharded one.  One exception: with DSMC_F_PAIR_REPLACE the
 * velocity changes of a particle that sits in several pairs are added with shared-memory floating-point atomics,
 * whose order is not fixed; those results are reproducible to rounding only (a few ulp of the change).
 */
#ifndef DSMC_H
#define DSMC_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DSMC_OK 0
#define DSMC_ERR_INVALID_ARG (-1)
#define DSMC_ERR_BAD_CELL_INDEX (-2)
#define DSMC_ERR_CELL_TOO_LARGE (-3)
#define DSMC_ERR_NOT_CONFIGURED (-4)
#define DSMC_ERR_CUDA (-5)
#define DSMC_ERR_UNSUPPORTED_SHAPE (-6)
#define DSMC_ERR_NOALLOC_LIMIT (-7) /* dsmc_bin_noalloc: n or n_cells beyond the fixed scratch array */

/* largest cell the SMEM-resident fused step accepts */
#define DSMC_MAX_CELL_PARTICLES 2048

typedef struct dsmc_ctx dsmc_ctx;

/* Create a context on CUDA device `device` sized for at most max_particles / max_cells.
 * Owns: scan scratch, staged weights, the chi table copy, the status word. */
int dsmc_create(dsmc_ctx **out, int device, int64_t max_particles, int32_t max_cells);
int dsmc_destroy(dsmc_ctx *ctx);
/* Borrow a cudaStream_t (e.g. torch's current stream); NULL = default stream. */
int dsmc_set_stream(dsmc_ctx *ctx, void *cuda_stream);
/* Synchronise the stream; return and clear the sticky device status. */
int dsmc_sync_status(dsmc_ctx *ctx);
const char *dsmc_strerror(int status);
/* Number of kernels this context has launched so far (bench bookkeeping). */
int64_t dsmc_launch_count(const dsmc_ctx *ctx);

/* ---- operators ------------------------------------------------------------------------- */
typedef enum { DSMC_ACT_TANH = 0, DSMC_ACT_RELU = 1, DSMC_ACT_SILU = 2 } dsmc_act;

/* h^(l) = act(W^(l) h^(l-1) + b^(l)), last layer linear.
 * W, b: HOST pointers, fp32, W[l] row-major [dims[l+1]][dims[l]]; copied during the call. */
typedef struct {
  int32_t n_layers; /* linear layers, 2..6 */
  int32_t dims[8];  /* dims[0] = inputs, dims[n_layers] = outputs; every dim <= 256 */
  int32_t act;      /* dsmc_act of the hidden layers */
  const float *const *W;
  const float *const *b;
} dsmc_mlp_desc;

/* slot 0: VHS-surrogate f_theta (eqs. 3-4): dims[0] = 8 (g/sigma_v (3), |g|/sigma_v,
 *         T_cell/T_scale, sigma_xi*xi (3); BASELINE.json form, Q2-Q3) or 6 (g/sigma_v (+) xi,
 *         the paper's eq. 3 as read in Q1); dims[n_layers] = 3.
 * slot 1: chi-MLP: dims[0] = 2 ((E~-E~min)/(E~max-E~min), b~), output 1,
 *         chi = expm1(softplus(z)) (Q15).
 * The BF16 tensor-core paths (DSMC_F_BF16_TC) take at most 8 inputs and hidden widths <= 128 (any widths: narrower
 * layers are zero-padded on the device to 64 or 128).  chi-MLP (slot 1): 2 to 5 hidden layers (n_layers 3..6), e.g. the
 * paper's five hidden layers of decreasing width; VHS-NN (slot 0) and every DSMC_F_TC_ONE_KERNEL form: exactly 2 hidden
 * layers.  Other shapes run only on the FP32 path (DSMC_ERR_UNSUPPORTED_SHAPE otherwise). */
int dsmc_set_mlp(dsmc_ctx *ctx, int slot, const dsmc_mlp_desc *desc);

/* chi table: chi_host HOST fp32 [nE][nB] row-major, node (iE,iB) at
 * E~ = lnE_min + iE (lnE_max-lnE_min)/(nE-1) with E~ = ln(E_r/k_B [K]), b~ = iB/(nB-1).
 * Lookups clamp both coordinates to the grid (Q13).  Copied during the call.  Every node must be finite
 * (DSMC_ERR_INVALID_ARG otherwise): cap nodes on the orbiting singularity as dsmc_build_chi_table_lj does (64 pi, Q23). */
int dsmc_set_chi_table(dsmc_ctx *ctx, const float *chi_host, int32_t nE, int32_t nB, float lnE_min,
                       float lnE_max);

/* ---- a1: binning ---------------------------------------------------------------
 * Stable counting sort of n particles by cell[p] in [0, n_cells).  Outputs: cell_start
 * [n_cells+1] (CSR offsets), perm[n] (sorted slot -> original particle id; ties keep the
 * original order, so the result is unique), and the velocities gathered into sorted order.
 * n == 0: cell_start is zero-filled.  Bad index: sticky DSMC_ERR_BAD_CELL_INDEX. */
int dsmc_bin(dsmc_ctx *ctx, int64_t n, int32_t n_cells, const int32_t *cell, const float *vx,
             const float *vy, const float *vz, float *vx_s, float *vy_s, float *vz_s, int32_t *perm,
             int32_t *cell_start);

/* ---- a1 without any allocation --------------------------------------------------------------------------
 * The same sort as dsmc_bin (same kernels, bit-identical outputs) for callers that cannot call cudaMalloc: code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it.  No context: the workspace is one file-scope
 * device array of fixed size (22.5 MB; every GPU that loads the library holds it until the process exits), so the call
 * allocates and frees NOTHING (no cudaMalloc / cudaFree / allocating library routine; it enqueues memsets, kernels and
 * one 4-byte device-to-device copy on `stream`, a cudaStream_t passed as void *, and returns without synchronising).
 * Runs on the CURRENT device.  Limits: n <= DSMC_NOALLOC_MAX_PARTICLES and n_cells <= DSMC_NOALLOC_MAX_CELLS,
 * otherwise DSMC_ERR_NOALLOC_LIMIT (nothing is enqueued).  All arrays are caller-owned DEVICE pointers as in dsmc_bin.
 * status_dev: optional DEVICE int32 that receives DSMC_OK or DSMC_ERR_BAD_CELL_INDEX when the call's work completes
 * (there is no context to hold a sticky status).
 * SHARED STATE: every call on a device uses the same array, which keeps the previous call's contents (what must start
 * at zero is cleared by the call itself).  Calls that overlap on the GPU -- two streams, two host threads, a captured
 * graph replayed concurrently with itself -- RACE; order them on one stream or with events.
 * dsmc_noalloc_setup(): the once-per-device set-up (the array's device address, SM count) for the current device;
 * dsmc_bin_noalloc does it on first use, call it beforehand where even that is unwelcome (before a graph capture). */
#define DSMC_NOALLOC_MAX_PARTICLES 1048576
#define DSMC_NOALLOC_MAX_CELLS 131072
int dsmc_noalloc_setup(void);
int dsmc_bin_noalloc(void *stream, int64_t n, int32_t n_cells, const int32_t *cell, const float *vx,
                     const float *vy, const float *vz, float *vx_s, float *vy_s, float *vz_s, int32_t *perm,
                     int32_t *cell_start, int32_t *status_dev);

/* ---- fused collision steps -------------------------------------------------------------- */
enum {
  DSMC_F_NOISE = 1,             /* feed sigma_xi * xi, xi ~ N(0,I3), to f_theta (eq. 2/9)      */
  DSMC_F_ENERGY_SHELL = 2,      /* g' = |g| h/|h| (eq. 5, guard Q4); else g' = sigma_v h */
  DSMC_F_MOMENT_MATCH = 4,      /* restore the cell's pre-collision momentum and energy (Q5)   */
  DSMC_F_ACCEPT = 8,            /* NTC acceptance test; needs the *_max array          */
  DSMC_F_BF16_TC = 16,          /* MLP layers as tcgen05 BF16 GEMMs over 128-pair tiles        */
  DSMC_F_MATCH_ENERGY_ONLY = 32, /* literal eq. 11: scale raw velocities by sqrt(E_pre/E_post)  */
  DSMC_F_PAIR_REPLACE = 128,    /* pairs drawn WITH replacement, i = mulhi(R0, N), j = mulhi(R1, N-1)
                                   + (j >= i) from Philox stream 4; every pair of a cell is evaluated on the
                                   pre-collision velocities (one batch) and the velocity changes of a
                                   particle that appears in several pairs add up.  Momentum is conserved exactly,
                                   energy is restored by DSMC_F_MOMENT_MATCH.  Both operators, on the FP32 / table
                                   paths and with DSMC_F_BF16_TC.  No key sort: the cheapest selection. */
  DSMC_F_TC_ONE_KERNEL = 256    /* with DSMC_F_BF16_TC: run the fused step as ONE kernel (chi-MLP: cell teams + a tcgen05
                                   MLP server sharing every SM; VHS-NN: chunks with a per-CTA engine) instead of the
                                   default three passes (pairing + network inputs | MLP batch on the tensor cores |
                                   rotation or eq. 5 + matching).
                                   Same pairs, same randoms; chi differs within the BF16 tolerance (the two forms add
                                   the output layer's partial sums in a different order).  Slower on large steps. */
};

typedef struct {
  float mass;        /* kg */
  float sigma_v;     /* global velocity scale */
  float T_scale;     /* K, normalises the T_cell feature */
  float noise_sigma; /* sigma_xi (BASELINE.json cfg 1: 0.1) */
  float shell_eps;   /* |h| below this skips the collision (Q4) */
  float d_ref, omega, T_ref; /* VHS sigma_T(g), used iff DSMC_F_ACCEPT */
  int32_t pairs_per_cell;    /* > 0: request per cell; -1: floor(N_k/2).  M_k = min(req, N_k/2) */
  uint32_t flags;
  int32_t cell_base;         /* RNG cell coordinate of local cell 0: a rank that owns the global cell range
                                [c0, c1) passes c0 and draws exactly the randoms of the unsharded run */
  const int32_t *pairs_count; /* NULL, or DEVICE array [n_cells]: the request of every cell, overriding
                                pairs_per_cell (e.g. the NTC candidate counts of dsmc_ntc_counts).
                                M_k = min(pairs_count[k], N_k/2); negative entries mean N_k/2 */
} dsmc_vhs_params;

typedef struct {
  float mass;
  float b_max;            /* m; b = b_max sqrt(U_b) */
  float lnE_min, lnE_max; /* normalisation of the chi-MLP energy input (Q15) */
  int32_t chi_mode;       /* 0 = table, 1 = MLP (slot 1) */
  int32_t pairs_per_cell;
  uint32_t flags;         /* NOISE / ENERGY_SHELL are ignored here */
  int32_t cell_base;      /* as in dsmc_vhs_params */
  const int32_t *pairs_count; /* as in dsmc_vhs_params */
} dsmc_abinitio_params;

/* Optional debug output (any member may be NULL).  All arrays have n entries; pair slot s of
 * cell k is written at index cell_start[k] + s (s < M_k): pair_i/pair_j = the two particle
 * slots RELATIVE to cell_start[k]; accepted = 0/1; gprime = post-collision relative velocity
 * (3 floats per index); aux = |h_hat| (VHS-NN) or chi (ab initio).  Other entries untouched. */
typedef struct {
  int32_t *pair_i;
  int32_t *pair_j;
  uint8_t *accepted;
  float *gprime;
  float *aux;
} dsmc_pair_dump;

/* Per cell k (contiguous segment [cell_start[k], cell_start[k+1]) of the sorted arrays):
 * pre-collision moments -> disjoint random pairing (Q7) -> [acceptance] -> operator ->
 * centre-of-mass update (eqs. 6-8) -> [moment matching over the whole cell] -> store.
 * Velocities are updated in place.  Cells with N_k < 2 are untouched.
 * sigma_cr_max / cr_max: [n_cells] fp32 caps for the acceptance test, or NULL (accept all). */
int dsmc_collide_vhs_nn(dsmc_ctx *ctx, int64_t n, int32_t n_cells, const int32_t *cell_start,
                        float *vx_s, float *vy_s, float *vz_s, const float *sigma_cr_max,
                        const dsmc_vhs_params *prm, uint64_t seed, uint32_t step,
                        const dsmc_pair_dump *dump);
int dsmc_collide_abinitio(dsmc_ctx *ctx, int64_t n, int32_t n_cells, const int32_t *cell_start,
                          float *vx_s, float *vy_s, float *vz_s, const float *cr_max,
                          const dsmc_abinitio_params *prm, uint64_t seed, uint32_t step,
                          const dsmc_pair_dump *dump);

/* ---- cell sums and the stand-alone correction ------------------------------------------- */
/* moments[k] = (Px, Py, Pz, E = sum |v|^2), fp64, eq. 10 */
int dsmc_cell_moments(dsmc_ctx *ctx, int64_t n, int32_t n_cells, const int32_t *cell_start,
                      const float *vx_s, const float *vy_s, const float *vz_s, double *moments);
/* v <- u_t + sqrt(Theta_t/Theta') (v - u') with (u_t, Theta_t) from target_moments[k] (Q5);
 * flags & DSMC_F_MATCH_ENERGY_ONLY: v <- v sqrt(E_t/E') (eq. 11). */
int dsmc_moment_match(dsmc_ctx *ctx, int64_t n, int32_t n_cells, const int32_t *cell_start,
                      float *vx_s, float *vy_s, float *vz_s, const double *target_moments,
                      uint32_t flags);

/* ---- a10: chi for n independent pairs (BASELINE.json cfg 4) ------------------------------
 * E_over_k [K], b [m] -> chi [rad]; chi_mode 0 = table, 1 = MLP slot 1;
 * flags & DSMC_F_BF16_TC selects the tensor-core MLP. */
int dsmc_chi_batch(dsmc_ctx *ctx, int64_t n, const float *E_over_k, const float *b, float *chi,
                   int32_t chi_mode, float b_max, float lnE_min, float lnE_max, uint32_t flags);

/* ---- "exact" chi for n independent pairs (the computation the neural operators replace) ----
 * Classical deflection integral of eq. 16 for a Lennard-Jones 12-6 potential with well depth
 * eps_over_k [K] and diameter sigma [m], per pair, in FP64: largest root r_min of eq. 21, then
 * Gauss-Legendre quadrature in the variable of P:L342 with the end-point singularity removed analytically.
 * E_over_k [K], b [m] -> chi [rad], SIGNED (negative = attractive glancing collision, Q14) unless
 * flags & DSMC_F_CHI_ABS.  b <= 0 gives pi.  Near the orbiting condition the integral is ill-conditioned (Q23). */
#define DSMC_F_CHI_ABS 64u
int dsmc_chi_exact_batch(dsmc_ctx *ctx, int64_t n, const float *E_over_k, const float *b, float *chi,
                         float eps_over_k, float sigma, uint32_t flags);

/* Generates the chi table ON THE DEVICE by that quadrature (the paper's exact 512 x 512 table takes
 * "several hours" on a CPU cluster) and installs it as the context's table exactly as dsmc_set_chi_table
 * would: nodes as documented there, abs(chi) rounded to fp32 (Q14).  chi_out: optional DEVICE array [nE][nB] that
 * receives the node values.  Synchronises the stream. */
int dsmc_build_chi_table_lj(dsmc_ctx *ctx, int32_t nE, int32_t nB, float lnE_min, float lnE_max, float b_max,
                            float eps_over_k, float sigma, float *chi_out);

/* f2 as the paper states it ("the neural network can generate a complete 512 x 512 table in less than 1.0 s"):
 * evaluates the chi-MLP of operator slot 1 (dsmc_set_mlp, readings Q13-Q15) on the nE x nB table nodes
 * ON THE DEVICE and installs the result as the context's table exactly as dsmc_set_chi_table would: node (i, j) =
 * chi(lnE_min + i (lnE_max - lnE_min) / (nE - 1), b~ = j / (nB - 1)), abs value (Q14), capped at 64 pi (Q23), fp32.
 * flags: 0 (FP32 CUDA-core MLP) or DSMC_F_BF16_TC (tensor cores; DSMC_ERR_UNSUPPORTED_SHAPE if slot 1 has no
 * tensor-core image).  chi_out: optional DEVICE array [nE][nB] that receives the node values.  Synchronises the
 * stream.  DSMC_ERR_NOT_CONFIGURED without a slot-1 network; on any error the installed table (if any) stays. */
int dsmc_build_chi_table_mlp(dsmc_ctx *ctx, int32_t nE, int32_t nB, float lnE_min, float lnE_max, uint32_t flags,
                             float *chi_out);

/* ---- end-to-end helper on HOST buffers ----------------------------------------------------
 * Copies cell/vx/vy/vz (HOST, ideally pinned) to context-owned device buffers, runs dsmc_bin and
 * one fused ab initio (vhs == NULL) or VHS-NN (abi == NULL) step, copies the sorted post-collision
 * velocities, perm and cell_start back to the HOST outputs, and synchronises. */
int dsmc_step_host(dsmc_ctx *ctx, int64_t n, int32_t n_cells, const int32_t *cell_h,
                   const float *vx_h, const float *vy_h, const float *vz_h, float *vx_out_h,
                   float *vy_out_h, float *vz_out_h, int32_t *perm_h, int32_t *cell_start_h,
                   const dsmc_vhs_params *vhs, const dsmc_abinitio_params *abi, uint64_t seed,
                   uint32_t step);

/* The same step, enqueued only: returns as soon as the copies and kernels are on the context's stream (argument
 * errors are still returned at once).  The caller's host buffers (inputs and outputs) must stay valid and untouched
 * until dsmc_sync_status(ctx) has returned, which also delivers the device-detected data errors.  One submitted step
 * per context at a time.  Two contexts on two streams, fed alternately, overlap the host->device copy of one batch
 * with the device->host copy of the previous one (the PCIe link is full duplex): that is how bench.py measures the
 * end-to-end throughput of independent batches. */
int dsmc_step_host_submit(dsmc_ctx *ctx, int64_t n, int32_t n_cells, const int32_t *cell_h,
                          const float *vx_h, const float *vy_h, const float *vz_h, float *vx_out_h,
                          float *vy_out_h, float *vz_out_h, int32_t *perm_h, int32_t *cell_start_h,
                          const dsmc_vhs_params *vhs, const dsmc_abinitio_params *abi, uint64_t seed,
                          uint32_t step);

/* ---- f1: NTC candidate count with a carried remainder (Q31) ---------------------------
 * "a number of candidate pairs is drawn proportional to N_k (N_k - 1) and a cell-wise upper bound (sigma v_r)max,k":
 * m = 1/2 N_k (N_k - 1) coef sigma_cr_max[k] + remainder[k]; counts[k] = floor(m); remainder[k] = m - counts[k],
 * evaluated in FP64 in that order, coef = F_N dt / V_c (not given by the paper: an input).  Cells with N_k < 2 get
 * 0 and keep their remainder.  sigma_cr_max [n_cells] float, remainder [n_cells] double in/out (the caller zeroes
 * it once), counts [n_cells] int32 out: pass it as pairs_count of the next fused step (with DSMC_F_ACCEPT and the
 * same sigma_cr_max this is the NTC scheme; the disjoint matching caps the count at N_k/2). */
int dsmc_ntc_counts(dsmc_ctx *ctx, int32_t n_cells, const int32_t *cell_start, const float *sigma_cr_max,
                    double coef, double *remainder, int32_t *counts);

/* ---- f4: the minimal DSMC loop around the step, 1-D Couette layout (Q30) -------
 * Walls normal to x at x = 0 (moving with y-velocity -u_wall) and x = L (+u_wall); "U_wall = +-500 m/s".
 * The paper says only "a standard DSMC simulation of Couette flow"; standard is read as (Q30): free flight for dt;
 * Maxwell wall model (a fraction `accommodation` of the wall hits is re-emitted diffusely from the wall Maxwellian
 * at rt_wall = k_B T_w / m [m^2/s^2], normal speed sqrt(-2 rt ln u), the rest reflects specularly); the flight
 * continues with the new velocity for the rest of dt (at most DSMC_MAX_BOUNCES wall hits per step, then the
 * particle is parked on the wall); cell = floor(x n_cells / L) clamped to [0, n_cells).
 * Random numbers: Philox stream 5, counter (particle index, bounce number, step, 5): word 0 decides diffuse
 * (u < accommodation), word 1 the normal speed, words 2, 3 the Box-Muller pair of the tangential components. */
#define DSMC_MAX_BOUNCES 4
typedef struct {
  float L;             /* gap [m] */
  float dt;            /* time step [s] */
  float u_wall;        /* wall speed [m/s] */
  float rt_wall;       /* k_B T_wall / m [m^2/s^2] */
  float accommodation; /* in [0, 1]: 1 = fully diffuse walls, 0 = specular */
  int32_t n_cells;
  /* used by dsmc_couette_run only: NTC rate control.  ntc_coef = F_N dt / V_c > 0 makes every step draw
   * dsmc_ntc_counts candidates per cell (remainders start at 0 and are carried through the run) against the uniform
   * bound sigma_cr_max [m^3/s]; with DSMC_F_ACCEPT the same bound caps the acceptance test (VHS-NN: sigma_T(g) g /
   * sigma_cr_max; ab initio, constant cross-section pi b_max^2: g / (sigma_cr_max / (pi b_max^2))).
   * ntc_coef = 0: the pair request of the operator's parameter struct is used as is. */
  float ntc_coef;
  float sigma_cr_max;
} dsmc_couette_params;

/* x, vx, vy, vz [n] in/out (vy, vz are written only for re-emitted particles); cell [n] out; bounces [n] out or
 * NULL (wall hits of the particle in this step). */
int dsmc_move_couette(dsmc_ctx *ctx, int64_t n, float *x, float *vx, float *vy, float *vz, int32_t *cell,
                      int32_t *bounces, const dsmc_couette_params *geo, uint64_t seed, uint32_t step);

/* dst[s] = src[perm[s]], s < n: carries a per-particle array (the position) into the order dsmc_bin produced.
 * perm values must lie in [0, n); src and dst must not overlap. */
int dsmc_gather_f32(dsmc_ctx *ctx, int64_t n, const int32_t *perm, const float *src, float *dst);

/* acc [n_cells][8] (FP64, device) += per cell (count, sum vx, vy, vz, vx^2, vy^2, vz^2, vx vy) of the sorted
 * arrays: the time-averaged sums behind U, T, rho, tau_xy.  The caller zeroes acc. */
int dsmc_sample_cells(dsmc_ctx *ctx, int64_t n, int32_t n_cells, const int32_t *cell_start, const float *vx,
                      const float *vy, const float *vz, double *acc);

/* n_steps of  move -> bin -> gather x -> fused collision step (vhs or abi, exactly one non-NULL; step index
 * step0 + k for the random numbers of both move and collide) -> sample (steps k >= sample_from, into acc if
 * non-NULL), entirely on the device in context-owned scratch.  x, vx, vy, vz [n] in/out: on return they hold the
 * state after the last step, in that step's cell-sorted order.  Synchronises and returns the sticky status. */
int dsmc_couette_run(dsmc_ctx *ctx, int64_t n, float *x, float *vx, float *vy, float *vz,
                     const dsmc_couette_params *geo, const dsmc_vhs_params *vhs, const dsmc_abinitio_params *abi,
                     uint64_t seed, uint32_t step0, int32_t n_steps, int32_t sample_from, double *acc);

#ifdef __cplusplus
}
#endif
#endif
