/*
 * dsmc_oracle.h -- CPU oracle for the neural DSMC collision step (TEST INFRASTRUCTURE).
 *
 * This is the plain, slow, single-threaded fp64 restatement of what the hot path
 * computes, written from /root/reference/PAPER.md ("P:L<line>") and the readings
 * listed in DESIGN.md ("Q<n>").  It is NOT part of the product: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code, header, table or constant generator with the CUDA
 * path under paper_2602_21244_b200/csrc/.
 *
 * All pointers are HOST pointers.  Velocities are fp64 (fp32 inputs are promoted
 * exactly by the caller).  Every function is deterministic and re-entrant.
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py
 * (-m "not gpu") except the behaviour of *trained* networks (isotropy, cos(chi)
 * PDF, viscosity, flow fields: P:L217-235), which needs the paper's
 * weights and data and is "parity unpinned".
 */
#ifndef DSMC_ORACLE_H
#define DSMC_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- flags (same numeric values as the product header; restated, not shared) ---- */
#define ORC_F_NOISE 1u              /* feed sigma_xi*xi to the network (eq. 2/9) */
#define ORC_F_ENERGY_SHELL 2u       /* eq. 5 projection */
#define ORC_F_MOMENT_MATCH 4u       /* cell-wise correction, eqs. 10-11 P:L126-131 + P:L46 */
#define ORC_F_ACCEPT 8u             /* NTC acceptance test */
#define ORC_F_MATCH_ENERGY_ONLY 32u /* literal eq. 11 (scale raw velocities) */
#define ORC_F_PAIR_REPLACE 128u     /* NTC-style selection WITH replacement, batch semantics */

#define ORC_ACT_TANH 0
#define ORC_ACT_RELU 1
#define ORC_ACT_SILU 2

#define ORC_OK 0
#define ORC_ERR_INVALID_ARG (-1)
#define ORC_ERR_BAD_CELL_INDEX (-2)

#define ORC_KB 1.380649e-23 /* CODATA k_B, J/K (Q18) */

/* h^(l) = act(W^(l) h^(l-1) + b^(l)); W[l] row-major [out][in], fp32 values */
typedef struct {
  int32_t n_layers; /* number of linear layers, 2..6 */
  int32_t dims[8];  /* dims[0] inputs ... dims[n_layers] outputs */
  int32_t act;      /* hidden activation */
  const float *W[7];
  const float *b[7];
} orc_mlp;

typedef struct {
  double mass, sigma_v, T_scale, noise_sigma, shell_eps;
  double d_ref, omega, T_ref; /* VHS cross-section, used iff ORC_F_ACCEPT */
  int32_t pairs_per_cell;     /* >0 request per cell, -1 = floor(N_k/2) */
  uint32_t flags;
  int32_t cell_base;          /* RNG cell coordinate of local cell 0 (cell-range shards) */
  const int32_t *pairs_count; /* NULL, or the request of every cell (overrides pairs_per_cell): the NTC candidate
                                 count of orc_ntc_counts, "proportional to N_k (N_k - 1) and ... (sigma v_r)max,k" */
} orc_vhs_params;

typedef struct {
  double mass, b_max;
  double lnE_min, lnE_max; /* normalisation of the chi-MLP energy input (Q15) */
  int32_t chi_mode;        /* 0 = table, 1 = MLP */
  int32_t pairs_per_cell;
  uint32_t flags;
  int32_t cell_base; /* RNG cell coordinate of local cell 0 */
  const int32_t *pairs_count; /* as in orc_vhs_params */
} orc_abinitio_params;

typedef struct { /* chi[iE*nB + iB], node (lnE_min + iE*dE, iB/(nB-1)), Q13 */
  const float *chi;
  int32_t nE, nB;
  double lnE_min, lnE_max;
} orc_chi_table;

/* potentials for the deflection integral (eq. 16) */
#define ORC_POT_LJ 0          /* 4 eps ((s/r)^12-(s/r)^6); p0 = eps [J], p1 = sigma [m]  (Q17) */
#define ORC_POT_HARD_SPHERE 1 /* +inf for r<d; p0 = d */
#define ORC_POT_INV_R 2       /* kappa / r;   p0 = kappa */
#define ORC_POT_INV_R2 3      /* kappa / r^2; p0 = kappa */
typedef struct {
  int32_t kind;
  double p0, p1;
  double r_hi; /* scan start for r_min, must exceed the largest root */
} orc_potential;

/* ---- random numbers (a4) ---- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_u01(uint32_t x); /* ((x>>9)+0.5)*2^-23 in (0,1), exact in fp32 */
/* pairing key of slot p in cell k at step t (stream 0) */
uint32_t orc_pair_key(uint64_t seed, uint32_t step, uint32_t cell, uint32_t slot);
/* with-replacement selection (stream 4): i = mulhi(R0, N), j = mulhi(R1, N-1) + (j >= i), uniform over ordered
 * pairs i != j */
void orc_pair_draw(uint64_t seed, uint32_t step, uint32_t cell, uint32_t s, int32_t N, int32_t *i, int32_t *j);
/* per-pair uniforms: U_acc (stream 3, word s&3 of block s>>2), U_b, U_eps (stream 1, words 2(s&1), 2(s&1)+1
 * of block s>>1) */
void orc_pair_uniforms(uint64_t seed, uint32_t step, uint32_t cell, uint32_t s, double u[3]);
void orc_pair_uniforms_batch(uint64_t seed, uint32_t step, int64_t n, const uint32_t *cell, const uint32_t *s, double *u);
/* per-pair latent xi ~ N(0, I3) by Box-Muller (stream 2) */
void orc_pair_normals(uint64_t seed, uint32_t step, uint32_t cell, uint32_t s, double xi[3]);

/* ---- a1: stable counting sort by cell id, P:L140 ---- */
int orc_bin(int64_t n, int32_t n_cells, const int32_t *cell, int32_t *perm, int32_t *cell_start);

/* ---- a2: cell moments, eq. 10: moments[k] = (Px,Py,Pz,E=sum|v|^2) ---- */
void orc_cell_moments(int32_t n_cells, const int32_t *cell_start, const double *vx,
                      const double *vy, const double *vz, double *moments);
/* mean velocity, centred Theta = sum|v-u|^2, T = m Theta/(3 kB N) of one segment (Q6) */
void orc_cell_state(int64_t N, const double *vx, const double *vy, const double *vz, double mass,
                    double ubar[3], double *Theta, double *T);

/* ---- a3: disjoint random matching (Q7). pi[N] = slots sorted by (key,slot). returns M ---- */
int32_t orc_pairing(uint64_t seed, uint32_t step, uint32_t cell, int32_t N, int32_t M_req,
                    int32_t *pi);
void orc_pairing_all(uint64_t seed, uint32_t step, int32_t K, const int32_t *cell_start, uint32_t cell_base,
                     int32_t M_req, int32_t *pair_i, int32_t *pair_j);

/* ---- operators ---- */
void orc_mlp_forward(const orc_mlp *net, const double *x, double *out);
double orc_vhs_sigma_g(double g, const orc_vhs_params *p); /* sigma_T(g)*g, P:L68 + BJ cfg 1 */
void orc_rotate(const double g[3], double chi, double eps, double gp[3]); /* Q16 */
double orc_chi_bilinear(const orc_chi_table *t, double lnE, double btilde);
double orc_chi_mlp(const orc_mlp *net, double lnE_min, double lnE_max, double lnE, double btilde);

/* ---- a8: moment matching against target moments, eqs. 10-11 + P:L46 (Q5) ---- */
void orc_moment_match(int32_t n_cells, const int32_t *cell_start, double *vx, double *vy,
                      double *vz, const double *target_moments, uint32_t flags);

/* ---- fused steps (a2-a9).  pair_i/pair_j/accepted (may be NULL) are indexed
 *      cell_start[k]+s for pair slot s<M_k and hold slots relative to cell_start[k].
 *      gprime_out (may be NULL): 3 doubles per dump index = post-collision relative velocity,
 *      hnorm_out (may be NULL): |h_hat| per dump index (VHS-NN only; Q21 gating). ---- */
int orc_collide_vhs_nn(int64_t n, int32_t n_cells, const int32_t *cell_start, double *vx,
                       double *vy, double *vz, const float *sigma_cr_max, const orc_mlp *net,
                       const orc_vhs_params *p, uint64_t seed, uint32_t step, int32_t *pair_i,
                       int32_t *pair_j, uint8_t *accepted, double *gprime_out, double *hnorm_out);
int orc_collide_abinitio(int64_t n, int32_t n_cells, const int32_t *cell_start, double *vx,
                         double *vy, double *vz, const float *cr_max, const orc_mlp *net,
                         const orc_chi_table *table, const orc_abinitio_params *p, uint64_t seed,
                         uint32_t step, int32_t *pair_i, int32_t *pair_j, uint8_t *accepted,
                         double *gprime_out, double *chi_out);

/* ---- a10: chi for independent (E_r/k_B [K], b [m]) pairs ---- */
void orc_chi_batch(int64_t n, const float *E_over_k, const float *b, double *chi, int32_t chi_mode,
                   const orc_mlp *net, const orc_chi_table *table, double b_max, double lnE_min,
                   double lnE_max);

/* ---- "Exact" deflection angle, eqs. 16/20/21 P:L272, P:L327, P:L338-342 ---- */
double orc_potential_eval(const orc_potential *pot, double r);
double orc_rmin(const orc_potential *pot, double E, double b);
/* signed chi by composite Gauss-Legendre (n_panels x 64 points) after u=r_min/r, u=1-s^2 */
double orc_chi_exact(const orc_potential *pot, double E, double b, int32_t n_panels);
/* fills chi[nE*nB] with |chi| rounded to fp32 (Q14) */
double orc_cap_chi(double c); /* Q23: min(c, 64 pi), NaN -> 64 pi */
void orc_build_chi_table(const orc_potential *pot, int32_t nE, int32_t nB, double lnE_min,
                         double lnE_max, double b_max, int32_t n_panels, float *chi);
/* f2: the chi-MLP evaluated on the table nodes (Q13), abs (Q14), capped (Q23), fp32 */
void orc_build_chi_table_mlp(const orc_mlp *net, int32_t nE, int32_t nB, double lnE_min, double lnE_max, float *chi);

/* ---- f1: NTC candidate count with a carried remainder (Bird 1994 eq. 11.3; Q31) ----
 * "a number of candidate pairs is drawn proportional to N_k (N_k - 1) and a cell-wise upper bound (sigma v_r)max,k":
 * m = 1/2 N_k (N_k - 1) coef (sigma v_r)max,k + R_k, count_k = floor(m), R_k <- m - count_k, with
 * coef = F_N dt / V_c (the paper does not give the constant: an input).  Evaluated in fp64 in exactly this order
 * (((0.5 * (N (N-1))) * coef) * max) + R.  Cells with N_k < 2 get 0 and keep their remainder. */
void orc_ntc_counts(int32_t n_cells, const int32_t *cell_start, const float *sigma_cr_max, double coef,
                    double *remainder, int32_t *counts);

/* ---- f4: the minimal DSMC loop around the collision step, 1-D Couette layout (Q30) ----
 * Walls at x = 0 (moving with y-velocity -u_wall) and x = L (+u_wall), "U_wall = +-500 m/s".  The paper
 * only says "a standard DSMC simulation of Couette flow"; the standard is taken to be: free flight for dt, Maxwell
 * wall model (a fraction `accommodation` of the wall hits is re-emitted diffusely from the wall Maxwellian at
 * rt_wall = k_B T_w / m, the rest reflects specularly), the flight continues for the rest of dt with the new
 * velocity (at most ORC_MAX_BOUNCES wall hits, then the position is clamped into the gap), and the cell index is
 * floor(x n_cells / L).  Random numbers: Philox stream 5, counter (particle index, bounce number, step, 5):
 * word 0 decides diffuse (u < accommodation), word 1 the wall-normal speed sqrt(-2 rt ln u) (flux-weighted),
 * words 2, 3 the Box-Muller pair for the tangential components. */
#define ORC_MAX_BOUNCES 4
typedef struct {
  double L, dt, u_wall, rt_wall, accommodation;
  int32_t n_cells;
} orc_couette_params;
/* x, vx, vy, vz in/out; cell[n], bounces[n] (may be NULL) out; margin[n] (may be NULL) out = the smallest distance
 * of any floating-point decision taken for the particle from its threshold (wall crossing and cell boundary as a
 * fraction of L, diffuse/specular draw as |u - accommodation|): a parity test compares decisions only where the
 * margin exceeds the FP32 resolution. */
void orc_move_couette(int64_t n, double *x, double *vx, double *vy, double *vz, int32_t *cell, int32_t *bounces,
                      double *margin, const orc_couette_params *p, uint64_t seed, uint32_t step);
/* acc[n_cells][8] += (count, sum vx, vy, vz, vx^2, vy^2, vz^2, vx vy) of every cell (time-averaged sampling of the
 * macroscopic fields U, T, tau_xy: P:L187) */
void orc_sample_cells(int32_t n_cells, const int32_t *cell_start, const double *vx, const double *vy,
                      const double *vz, double *acc);

#ifdef __cplusplus
}
#endif
#endif
