/*
 * dsmc_oracle.c -- CPU oracle for the neural DSMC collision step (TEST INFRASTRUCTURE,
 * see dsmc_oracle.h).  Plain C99, fp64, single-threaded, one loop per sentence of the
 * paper; no blocking, fusion or reordering.  "P:L<n>" = /root/reference/PAPER.md line n,
 * "Q<n>" = reading n in DESIGN.md.
 */
#include "dsmc_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------------------------------
 * Random numbers.  Philox4x32-10 (Salmon et al., SC'11): 10 rounds of
 *   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
 * key bumped by the Weyl constants between rounds.  The method keys it by
 * (seed, step, cell, slot) so every draw is addressable.
 * ---------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = M0 * (uint64_t)c0;
    uint64_t p1 = M1 * (uint64_t)c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* 23-bit uniform + half step: strictly inside (0,1) and (24 significant bits) exact in fp32 and fp64 */
double orc_u01(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

static void philox_at(uint64_t seed, uint32_t index, uint32_t cell, uint32_t step, uint32_t stream,
                      uint32_t out[4]) {
  uint32_t ctr[4] = {index, cell, step, stream};
  uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
  orc_philox4x32_10(ctr, key, out);
}

/* stream 0: one Philox block serves four consecutive slots; slot p takes word p&3 of block p>>2 */
uint32_t orc_pair_key(uint64_t seed, uint32_t step, uint32_t cell, uint32_t slot) {
  uint32_t r[4];
  philox_at(seed, slot >> 2, cell, step, 0u, r);
  return r[slot & 3u];
}

/* per-pair uniforms.  Stream 1: one Philox block serves two consecutive pair slots; pair s takes words
 * 2(s&1), 2(s&1)+1 of block s>>1 as (U_b, U_eps).  Stream 3: U_acc of pair s is word s&3 of block s>>2
 * (DESIGN.md "RNG addressing"). */
void orc_pair_uniforms(uint64_t seed, uint32_t step, uint32_t cell, uint32_t s, double u[3]) {
  uint32_t r[4], a[4];
  philox_at(seed, s >> 1, cell, step, 1u, r);
  philox_at(seed, s >> 2, cell, step, 3u, a);
  u[0] = orc_u01(a[s & 3u]);
  u[1] = orc_u01(r[2u * (s & 1u)]);
  u[2] = orc_u01(r[2u * (s & 1u) + 1u]);
}

/* the same for n (cell, slot) pairs: u[3 i ..] = uniforms of (cell[i], s[i]).  A loop over the function above (test
 * marshalling only: one call instead of n). */
void orc_pair_uniforms_batch(uint64_t seed, uint32_t step, int64_t n, const uint32_t *cell, const uint32_t *s, double *u) {
  for (int64_t i = 0; i < n; ++i) orc_pair_uniforms(seed, step, cell[i], s[i], u + 3 * i);
}

/* stream 4: with-replacement pair draw ("two particles i, j in C_k are selected uniformly at random") */
void orc_pair_draw(uint64_t seed, uint32_t step, uint32_t cell, uint32_t s, int32_t N, int32_t *i, int32_t *j) {
  uint32_t r[4];
  philox_at(seed, s, cell, step, 4u, r);
  int32_t ii = (int32_t)(((uint64_t)r[0] * (uint64_t)(uint32_t)N) >> 32);
  int32_t jj = (int32_t)(((uint64_t)r[1] * (uint64_t)(uint32_t)(N - 1)) >> 32);
  if (jj >= ii) jj++;
  *i = ii;
  *j = jj;
}

/* stream 2: xi ~ N(0,I3), eq. 2, by Box-Muller on four uniforms */
void orc_pair_normals(uint64_t seed, uint32_t step, uint32_t cell, uint32_t s, double xi[3]) {
  uint32_t r[4];
  philox_at(seed, s, cell, step, 2u, r);
  double rad0 = sqrt(-2.0 * log(orc_u01(r[0])));
  double ang0 = 2.0 * PI * orc_u01(r[1]);
  double rad1 = sqrt(-2.0 * log(orc_u01(r[2])));
  double ang1 = 2.0 * PI * orc_u01(r[3]);
  xi[0] = rad0 * cos(ang0);
  xi[1] = rad0 * sin(ang0);
  xi[2] = rad1 * cos(ang1);
}

/* ------------------------------------------------------------------------------------------
 * a1.  "Particles are sorted by cell index so that particles in the same cell are contiguous
 * in memory".  Stable counting sort: perm[slot] = original particle id.
 * ---------------------------------------------------------------------------------------- */
int orc_bin(int64_t n, int32_t n_cells, const int32_t *cell, int32_t *perm, int32_t *cell_start) {
  if (n < 0 || n_cells < 0) return ORC_ERR_INVALID_ARG;
  for (int32_t k = 0; k <= n_cells; ++k) cell_start[k] = 0;
  for (int64_t p = 0; p < n; ++p) {
    if (cell[p] < 0 || cell[p] >= n_cells) return ORC_ERR_BAD_CELL_INDEX;
    cell_start[cell[p] + 1] += 1;
  }
  for (int32_t k = 0; k < n_cells; ++k) cell_start[k + 1] += cell_start[k];
  int32_t *fill = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_cells > 0 ? n_cells : 1));
  for (int32_t k = 0; k < n_cells; ++k) fill[k] = cell_start[k];
  for (int64_t p = 0; p < n; ++p) perm[fill[cell[p]]++] = (int32_t)p;
  free(fill);
  return ORC_OK;
}

/* ------------------------------------------------------------------------------------------
 * a2.  Cell sums, eq. 10 P:L126 (E omits m/2, single species, Q6).
 * ---------------------------------------------------------------------------------------- */
void orc_cell_moments(int32_t n_cells, const int32_t *cell_start, const double *vx,
                      const double *vy, const double *vz, double *moments) {
  for (int32_t k = 0; k < n_cells; ++k) {
    double Px = 0, Py = 0, Pz = 0, E = 0;
    for (int32_t p = cell_start[k]; p < cell_start[k + 1]; ++p) {
      Px += vx[p];
      Py += vy[p];
      Pz += vz[p];
      E += vx[p] * vx[p] + vy[p] * vy[p] + vz[p] * vz[p];
    }
    moments[4 * k + 0] = Px;
    moments[4 * k + 1] = Py;
    moments[4 * k + 2] = Pz;
    moments[4 * k + 3] = E;
  }
}

void orc_cell_state(int64_t N, const double *vx, const double *vy, const double *vz, double mass,
                    double ubar[3], double *Theta, double *T) {
  ubar[0] = ubar[1] = ubar[2] = 0.0;
  *Theta = 0.0;
  *T = 0.0;
  if (N <= 0) return;
  for (int64_t p = 0; p < N; ++p) {
    ubar[0] += vx[p];
    ubar[1] += vy[p];
    ubar[2] += vz[p];
  }
  ubar[0] /= (double)N;
  ubar[1] /= (double)N;
  ubar[2] /= (double)N;
  double th = 0.0;
  for (int64_t p = 0; p < N; ++p) {
    double cx = vx[p] - ubar[0], cy = vy[p] - ubar[1], cz = vz[p] - ubar[2];
    th += cx * cx + cy * cy + cz * cz;
  }
  *Theta = th;
  *T = mass * th / (3.0 * ORC_KB * (double)N);
}

/* ------------------------------------------------------------------------------------------
 * a3.  Pair selection.  The paper draws (i,j) uniformly per trial and evaluates a
 * cell's pairs as one batch; the reading (Q7) is a uniformly random disjoint
 * matching: sort the slots by a random key, pair neighbours.
 * ---------------------------------------------------------------------------------------- */
static int cmp_u64(const void *a, const void *b) {
  uint64_t x = *(const uint64_t *)a, y = *(const uint64_t *)b;
  return (x > y) - (x < y);
}

int32_t orc_pairing(uint64_t seed, uint32_t step, uint32_t cell, int32_t N, int32_t M_req,
                    int32_t *pi) {
  if (N <= 0) return 0;
  uint64_t *keys = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)N);
  for (int32_t p = 0; p < N; ++p)
    keys[p] = ((uint64_t)orc_pair_key(seed, step, cell, (uint32_t)p) << 32) | (uint64_t)(uint32_t)p;
  qsort(keys, (size_t)N, sizeof(uint64_t), cmp_u64);
  for (int32_t p = 0; p < N; ++p) pi[p] = (int32_t)(keys[p] & 0xFFFFFFFFu);
  free(keys);
  int32_t M = N / 2; /* odd N: last element of pi is a spectator (Q10) */
  if (M_req >= 0 && M_req < M) M = M_req;
  return M;
}

/* orc_pairing for every cell of a population (a loop over the function above; test marshalling): pair slot s of
 * cell k at index cell_start[k] + s of pair_i / pair_j (slots relative to the cell's first slot), -1 elsewhere. */
void orc_pairing_all(uint64_t seed, uint32_t step, int32_t K, const int32_t *cell_start, uint32_t cell_base,
                     int32_t M_req, int32_t *pair_i, int32_t *pair_j) {
  for (int32_t k = 0; k < K; ++k) {
    const int32_t gs = cell_start[k], N = cell_start[k + 1] - gs;
    for (int32_t q = 0; q < N; ++q) pair_i[gs + q] = pair_j[gs + q] = -1;
    if (N < 2) continue;
    int32_t *pi = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    const int32_t M = orc_pairing(seed, step, (uint32_t)k + cell_base, N, M_req, pi);
    for (int32_t s = 0; s < M; ++s) {
      pair_i[gs + s] = pi[2 * s];
      pair_j[gs + s] = pi[2 * s + 1];
    }
    free(pi);
  }
}

/* ------------------------------------------------------------------------------------------
 * MLP, h^(l) = act(W^(l) h^(l-1) + b^(l)); last layer linear.
 * ---------------------------------------------------------------------------------------- */
static double activation(int act, double z) {
  switch (act) {
    case ORC_ACT_TANH: return tanh(z);
    case ORC_ACT_RELU: return z > 0.0 ? z : 0.0;
    default: return z / (1.0 + exp(-z)); /* SiLU */
  }
}

void orc_mlp_forward(const orc_mlp *net, const double *x, double *out) {
  double h_in[512], h_out[512];
  for (int i = 0; i < net->dims[0]; ++i) h_in[i] = x[i];
  for (int l = 0; l < net->n_layers; ++l) {
    int n_in = net->dims[l], n_out = net->dims[l + 1];
    for (int o = 0; o < n_out; ++o) {
      double z = (double)net->b[l][o];
      for (int i = 0; i < n_in; ++i) z += (double)net->W[l][o * n_in + i] * h_in[i];
      h_out[o] = (l + 1 < net->n_layers) ? activation(net->act, z) : z;
    }
    for (int o = 0; o < n_out; ++o) h_in[o] = h_out[o];
  }
  for (int o = 0; o < net->dims[net->n_layers]; ++o) out[o] = h_in[o];
}

/* ------------------------------------------------------------------------------------------
 * NTC acceptance weight sigma_T(g) g.  VHS total cross-section (Bird):
 *   sigma_T = pi d_ref^2 (2 kB T_ref / (m_r g^2))^(omega-1/2) / Gamma(5/2-omega), m_r = m/2.
 * ---------------------------------------------------------------------------------------- */
double orc_vhs_sigma_g(double g, const orc_vhs_params *p) {
  double m_r = 0.5 * p->mass;
  double ratio = 2.0 * ORC_KB * p->T_ref / (m_r * g * g);
  double sigma = PI * p->d_ref * p->d_ref * pow(ratio, p->omega - 0.5) / tgamma(2.5 - p->omega);
  return sigma * g;
}

/* ------------------------------------------------------------------------------------------
 * Rotation of the relative velocity by deflection chi and azimuth eps (Q16): |g'| = |g| and
 * g.g' = g^2 cos(chi).
 * ---------------------------------------------------------------------------------------- */
void orc_rotate(const double g[3], double chi, double eps, double gp[3]) {
  double gx = g[0], gy = g[1], gz = g[2];
  double gn = sqrt(gx * gx + gy * gy + gz * gz);
  double gperp = sqrt(gy * gy + gz * gz);
  double cc = cos(chi), sc = sin(chi), ce = cos(eps), se = sin(eps);
  if (gperp <= 1e-30 * gn) {
    gp[0] = gx * cc;
    gp[1] = fabs(gx) * sc * ce;
    gp[2] = fabs(gx) * sc * se;
    return;
  }
  gp[0] = gx * cc + gperp * sc * se;
  gp[1] = gy * cc + sc * (gn * gz * ce - gx * gy * se) / gperp;
  gp[2] = gz * cc - sc * (gn * gy * ce + gx * gz * se) / gperp;
}

/* ------------------------------------------------------------------------------------------
 * chi table: "parameterized by normalized impact parameter b~ = b/b_max and logarithmic energy
 * E~ = ln(E_r/k_B)", "bilinear interpolation".  Both coordinates clamp (Q13).
 * ---------------------------------------------------------------------------------------- */
double orc_chi_bilinear(const orc_chi_table *t, double lnE, double btilde) {
  double tE = (lnE - t->lnE_min) / (t->lnE_max - t->lnE_min) * (double)(t->nE - 1);
  double tB = btilde * (double)(t->nB - 1);
  if (!(tE > 0.0)) tE = 0.0; /* also catches -inf / NaN from g = 0 */
  if (tE > (double)(t->nE - 1)) tE = (double)(t->nE - 1);
  if (!(tB > 0.0)) tB = 0.0;
  if (tB > (double)(t->nB - 1)) tB = (double)(t->nB - 1);
  int iE = (int)floor(tE), iB = (int)floor(tB);
  if (iE > t->nE - 2) iE = t->nE - 2;
  if (iB > t->nB - 2) iB = t->nB - 2;
  double fE = tE - (double)iE, fB = tB - (double)iB;
  double c00 = (double)t->chi[(size_t)iE * t->nB + iB];
  double c01 = (double)t->chi[(size_t)iE * t->nB + iB + 1];
  double c10 = (double)t->chi[(size_t)(iE + 1) * t->nB + iB];
  double c11 = (double)t->chi[(size_t)(iE + 1) * t->nB + iB + 1];
  return (1.0 - fE) * ((1.0 - fB) * c00 + fB * c01) + fE * ((1.0 - fB) * c10 + fB * c11);
}

/* chi-MLP: SiLU hidden layers, Softplus output, target ln(1+chi) => chi = expm1(y) */
double orc_chi_mlp(const orc_mlp *net, double lnE_min, double lnE_max, double lnE, double btilde) {
  double x[2], z;
  x[0] = (lnE - lnE_min) / (lnE_max - lnE_min);
  if (!(x[0] > 0.0)) x[0] = 0.0;
  if (x[0] > 1.0) x[0] = 1.0;
  x[1] = btilde;
  if (!(x[1] > 0.0)) x[1] = 0.0;
  if (x[1] > 1.0) x[1] = 1.0;
  orc_mlp_forward(net, x, &z);
  double y = (z > 0.0 ? z : 0.0) + log1p(exp(-fabs(z))); /* softplus */
  return expm1(y);
}

/* ------------------------------------------------------------------------------------------
 * a8 standalone: restore target (P, E) of each cell.  Full version (Q5): shift to the target
 * mean and scale peculiar velocities; literal eq. 11 behind MATCH_ENERGY_ONLY.
 * ---------------------------------------------------------------------------------------- */
void orc_moment_match(int32_t n_cells, const int32_t *cell_start, double *vx, double *vy,
                      double *vz, const double *target, uint32_t flags) {
  for (int32_t k = 0; k < n_cells; ++k) {
    int32_t a = cell_start[k], N = cell_start[k + 1] - cell_start[k];
    if (N < 2) continue; /* Q11 */
    double Pt[3] = {target[4 * k], target[4 * k + 1], target[4 * k + 2]}, Et = target[4 * k + 3];
    if (flags & ORC_F_MATCH_ENERGY_ONLY) {
      double Epost = 0.0;
      for (int32_t p = a; p < a + N; ++p) Epost += vx[p] * vx[p] + vy[p] * vy[p] + vz[p] * vz[p];
      if (Epost > 0.0) { /* "If E_post > 0" */
        double alpha = sqrt(Et / Epost);
        for (int32_t p = a; p < a + N; ++p) { vx[p] *= alpha; vy[p] *= alpha; vz[p] *= alpha; }
      }
      continue;
    }
    double ut[3] = {Pt[0] / N, Pt[1] / N, Pt[2] / N};
    double Theta_t = Et - (double)N * (ut[0] * ut[0] + ut[1] * ut[1] + ut[2] * ut[2]);
    double up[3], Theta_p, Tdummy;
    orc_cell_state(N, vx + a, vy + a, vz + a, 1.0, up, &Theta_p, &Tdummy);
    double alpha = (Theta_p > 0.0 && Theta_t >= 0.0) ? sqrt(Theta_t / Theta_p) : 1.0;
    for (int32_t p = a; p < a + N; ++p) {
      vx[p] = ut[0] + alpha * (vx[p] - up[0]);
      vy[p] = ut[1] + alpha * (vy[p] - up[1]);
      vz[p] = ut[2] + alpha * (vz[p] - up[2]);
    }
  }
}

/* in-step version: match post-collision cell to its own pre-collision (ubar, Theta) */
static void match_cell(int32_t N, double *vx, double *vy, double *vz, const double ubar[3],
                       double Theta, double E_pre, uint32_t flags) {
  if (flags & ORC_F_MATCH_ENERGY_ONLY) {
    double Epost = 0.0;
    for (int32_t p = 0; p < N; ++p) Epost += vx[p] * vx[p] + vy[p] * vy[p] + vz[p] * vz[p];
    if (Epost > 0.0) {
      double alpha = sqrt(E_pre / Epost);
      for (int32_t p = 0; p < N; ++p) { vx[p] *= alpha; vy[p] *= alpha; vz[p] *= alpha; }
    }
    return;
  }
  double up[3], Theta_p, Tdummy;
  orc_cell_state(N, vx, vy, vz, 1.0, up, &Theta_p, &Tdummy);
  double alpha = (Theta_p > 0.0) ? sqrt(Theta / Theta_p) : 1.0;
  for (int32_t p = 0; p < N; ++p) {
    vx[p] = ubar[0] + alpha * (vx[p] - up[0]);
    vy[p] = ubar[1] + alpha * (vy[p] - up[1]);
    vz[p] = ubar[2] + alpha * (vz[p] - up[2]);
  }
}

/* ------------------------------------------------------------------------------------------
 * Fused VHS-NN step, cell by cell, in the paper's order: pre-moments -> pair
 * selection/acceptance -> f_theta (eqs. 1-4) -> energy shell (eq. 5) -> CM update
 * (eqs. 6-8) -> cell-wise correction (eqs. 10-11).
 * ---------------------------------------------------------------------------------------- */
int orc_collide_vhs_nn(int64_t n, int32_t n_cells, const int32_t *cell_start, double *vx,
                       double *vy, double *vz, const float *sigma_cr_max, const orc_mlp *net,
                       const orc_vhs_params *prm, uint64_t seed, uint32_t step, int32_t *pair_i,
                       int32_t *pair_j, uint8_t *accepted, double *gprime_out, double *hnorm_out) {
  (void)n;
  int n_in = net->dims[0];
  if (!(n_in == 8 || n_in == 6) || net->dims[net->n_layers] != 3) return ORC_ERR_INVALID_ARG;
  for (int32_t k = 0; k < n_cells; ++k) {
    int32_t a = cell_start[k], N = cell_start[k + 1] - cell_start[k];
    if (N < 2) continue;
    double *cx = vx + a, *cy = vy + a, *cz = vz + a;
    double ubar[3], Theta, Tk, E_pre = 0.0;
    orc_cell_state(N, cx, cy, cz, prm->mass, ubar, &Theta, &Tk);
    for (int32_t p = 0; p < N; ++p) E_pre += cx[p] * cx[p] + cy[p] * cy[p] + cz[p] * cz[p];
    /* with replacement (the paper's literal NTC text), batch semantics as in
     * orc_collide_abinitio below: every pair sees the PRE-collision velocities, changes add up (Q29) */
    const int replace = (prm->flags & ORC_F_PAIR_REPLACE) != 0;
    const int32_t M_req = prm->pairs_count ? prm->pairs_count[k] : prm->pairs_per_cell;
    int32_t *pi = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    double *dv = replace ? (double *)calloc((size_t)(3 * N), sizeof(double)) : NULL;
    int32_t M;
    if (replace) {
      M = N / 2;
      if (M_req >= 0 && M_req < M) M = M_req;
    } else {
      M = orc_pairing(seed, step, (uint32_t)(k + prm->cell_base), N, M_req, pi);
    }
    int32_t n_collided = 0;
    for (int32_t s = 0; s < M; ++s) {
      int32_t i, j;
      if (replace) orc_pair_draw(seed, step, (uint32_t)(k + prm->cell_base), (uint32_t)s, N, &i, &j);
      else { i = pi[2 * s]; j = pi[2 * s + 1]; }
      double g[3] = {cx[i] - cx[j], cy[i] - cy[j], cz[i] - cz[j]}; /* eq. 1 */
      double gn = sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
      double U[3], xi[3];
      orc_pair_uniforms(seed, step, (uint32_t)(k + prm->cell_base), (uint32_t)s, U);
      orc_pair_normals(seed, step, (uint32_t)(k + prm->cell_base), (uint32_t)s, xi);
      int acc = 1;
      if ((prm->flags & ORC_F_ACCEPT) && sigma_cr_max != NULL)
        acc = (U[0] * (double)sigma_cr_max[k] < orc_vhs_sigma_g(gn, prm)) ? 1 : 0;
      if (pair_i) pair_i[a + s] = i;
      if (pair_j) pair_j[a + s] = j;
      if (accepted) accepted[a + s] = (uint8_t)acc;
      double gp[3] = {g[0], g[1], g[2]}, hn = 0.0;
      if (acc) {
        double x[8], h[3];
        double nz = (prm->flags & ORC_F_NOISE) ? prm->noise_sigma : 0.0;
        if (n_in == 8) { /* BJ form: g/sigma_v, |g|/sigma_v, T_cell/T_scale, noise (Q2, Q3) */
          x[0] = g[0] / prm->sigma_v; x[1] = g[1] / prm->sigma_v; x[2] = g[2] / prm->sigma_v;
          x[3] = gn / prm->sigma_v;   x[4] = Tk / prm->T_scale;
          x[5] = nz * xi[0]; x[6] = nz * xi[1]; x[7] = nz * xi[2];
        } else { /* paper form, eq. 3 as read in Q1: (v_r/sigma_v) (+) xi */
          x[0] = g[0] / prm->sigma_v; x[1] = g[1] / prm->sigma_v; x[2] = g[2] / prm->sigma_v;
          x[3] = nz * xi[0]; x[4] = nz * xi[1]; x[5] = nz * xi[2];
        }
        orc_mlp_forward(net, x, h); /* eq. 4 */
        hn = sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
        if (prm->flags & ORC_F_ENERGY_SHELL) {
          if (hn >= prm->shell_eps) { /* eq. 5 with the guard of Q4 */
            gp[0] = gn * h[0] / hn; gp[1] = gn * h[1] / hn; gp[2] = gn * h[2] / hn;
          }
        } else {
          gp[0] = prm->sigma_v * h[0]; gp[1] = prm->sigma_v * h[1]; gp[2] = prm->sigma_v * h[2];
        }
        if (replace) { /* v_i' - v_i = (g' - g) / 2 = -(v_j' - v_j), eqs. 6-8 */
          for (int d = 0; d < 3; ++d) {
            dv[3 * i + d] += 0.5 * (gp[d] - g[d]);
            dv[3 * j + d] -= 0.5 * (gp[d] - g[d]);
          }
        } else {
          double cm[3] = {0.5 * (cx[i] + cx[j]), 0.5 * (cy[i] + cy[j]), 0.5 * (cz[i] + cz[j])};
          cx[i] = cm[0] + 0.5 * gp[0]; cy[i] = cm[1] + 0.5 * gp[1]; cz[i] = cm[2] + 0.5 * gp[2];
          cx[j] = cm[0] - 0.5 * gp[0]; cy[j] = cm[1] - 0.5 * gp[1]; cz[j] = cm[2] - 0.5 * gp[2];
        }
        n_collided++;
      }
      if (gprime_out) { gprime_out[3 * (a + s)] = gp[0]; gprime_out[3 * (a + s) + 1] = gp[1]; gprime_out[3 * (a + s) + 2] = gp[2]; }
      if (hnorm_out) hnorm_out[a + s] = hn;
    }
    free(pi);
    if (replace) {
      for (int32_t p = 0; p < N; ++p) { cx[p] += dv[3 * p]; cy[p] += dv[3 * p + 1]; cz[p] += dv[3 * p + 2]; }
      free(dv);
    }
    if ((prm->flags & ORC_F_MOMENT_MATCH) && n_collided > 0)
      match_cell(N, cx, cy, cz, ubar, Theta, E_pre, prm->flags);
  }
  return ORC_OK;
}

/* ------------------------------------------------------------------------------------------
 * Fused ab initio step: E_r = 1/2 mu v_r^2 (mu = m/2, Q12) -> (E~, b~) -> chi by table
 * or MLP -> rotation -> CM update -> cell-wise correction.
 * ---------------------------------------------------------------------------------------- */
int orc_collide_abinitio(int64_t n, int32_t n_cells, const int32_t *cell_start, double *vx,
                         double *vy, double *vz, const float *cr_max, const orc_mlp *net,
                         const orc_chi_table *table, const orc_abinitio_params *prm, uint64_t seed,
                         uint32_t step, int32_t *pair_i, int32_t *pair_j, uint8_t *accepted,
                         double *gprime_out, double *chi_out) {
  (void)n;
  if (prm->chi_mode == 0 && table == NULL) return ORC_ERR_INVALID_ARG;
  if (prm->chi_mode == 1 && (net == NULL || net->dims[0] != 2 || net->dims[net->n_layers] != 1))
    return ORC_ERR_INVALID_ARG;
  for (int32_t k = 0; k < n_cells; ++k) {
    int32_t a = cell_start[k], N = cell_start[k + 1] - cell_start[k];
    if (N < 2) continue;
    double *cx = vx + a, *cy = vy + a, *cz = vz + a;
    double ubar[3], Theta, Tk, E_pre = 0.0;
    orc_cell_state(N, cx, cy, cz, prm->mass, ubar, &Theta, &Tk);
    for (int32_t p = 0; p < N; ++p) E_pre += cx[p] * cx[p] + cy[p] * cy[p] + cz[p] * cz[p];
    /* with replacement, every pair of the cell is evaluated on the PRE-collision velocities
     * ("all collision pairs in a cell are evaluated in a single forward pass") and the velocity changes
     * of a particle that appears in several pairs add up; momentum is conserved exactly, energy is restored by
     * the cell-wise correction. */
    const int replace = (prm->flags & ORC_F_PAIR_REPLACE) != 0;
    int32_t *pi = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    double *dv = replace ? (double *)calloc((size_t)(3 * N), sizeof(double)) : NULL;
    int32_t M;
    const int32_t M_req = prm->pairs_count ? prm->pairs_count[k] : prm->pairs_per_cell;
    if (replace) {
      M = N / 2;
      if (M_req >= 0 && M_req < M) M = M_req;
    } else {
      M = orc_pairing(seed, step, (uint32_t)(k + prm->cell_base), N, M_req, pi);
    }
    int32_t n_collided = 0;
    for (int32_t s = 0; s < M; ++s) {
      int32_t i, j;
      if (replace) orc_pair_draw(seed, step, (uint32_t)(k + prm->cell_base), (uint32_t)s, N, &i, &j);
      else { i = pi[2 * s]; j = pi[2 * s + 1]; }
      double g[3] = {cx[i] - cx[j], cy[i] - cy[j], cz[i] - cz[j]};
      double g2 = g[0] * g[0] + g[1] * g[1] + g[2] * g[2];
      double gn = sqrt(g2);
      double U[3];
      orc_pair_uniforms(seed, step, (uint32_t)(k + prm->cell_base), (uint32_t)s, U);
      int acc = 1; /* constant sigma = pi b_max^2 => accept iff U g_max < g (Q9) */
      if ((prm->flags & ORC_F_ACCEPT) && cr_max != NULL) acc = (U[0] * (double)cr_max[k] < gn) ? 1 : 0;
      if (pair_i) pair_i[a + s] = i;
      if (pair_j) pair_j[a + s] = j;
      if (accepted) accepted[a + s] = (uint8_t)acc;
      double gp[3] = {g[0], g[1], g[2]}, chi = 0.0;
      if (acc) {
        double E_over_k = prm->mass * g2 / (4.0 * ORC_KB);
        double lnE = log(E_over_k);
        double btilde = sqrt(U[1]); /* b = b_max sqrt(U) */
        chi = (prm->chi_mode == 0) ? orc_chi_bilinear(table, lnE, btilde)
                                   : orc_chi_mlp(net, prm->lnE_min, prm->lnE_max, lnE, btilde);
        double eps = 2.0 * PI * U[2];
        if (gn > 0.0) orc_rotate(g, chi, eps, gp);
        if (replace) { /* v_i' - v_i = (g' - g) / 2 = -(v_j' - v_j), eqs. 6-8 */
          for (int d = 0; d < 3; ++d) {
            dv[3 * i + d] += 0.5 * (gp[d] - g[d]);
            dv[3 * j + d] -= 0.5 * (gp[d] - g[d]);
          }
        } else {
          double cm[3] = {0.5 * (cx[i] + cx[j]), 0.5 * (cy[i] + cy[j]), 0.5 * (cz[i] + cz[j])};
          cx[i] = cm[0] + 0.5 * gp[0]; cy[i] = cm[1] + 0.5 * gp[1]; cz[i] = cm[2] + 0.5 * gp[2];
          cx[j] = cm[0] - 0.5 * gp[0]; cy[j] = cm[1] - 0.5 * gp[1]; cz[j] = cm[2] - 0.5 * gp[2];
        }
        n_collided++;
      }
      if (gprime_out) { gprime_out[3 * (a + s)] = gp[0]; gprime_out[3 * (a + s) + 1] = gp[1]; gprime_out[3 * (a + s) + 2] = gp[2]; }
      if (chi_out) chi_out[a + s] = chi;
    }
    free(pi);
    if (replace) {
      for (int32_t p = 0; p < N; ++p) { cx[p] += dv[3 * p]; cy[p] += dv[3 * p + 1]; cz[p] += dv[3 * p + 2]; }
      free(dv);
    }
    if ((prm->flags & ORC_F_MOMENT_MATCH) && n_collided > 0)
      match_cell(N, cx, cy, cz, ubar, Theta, E_pre, prm->flags);
  }
  return ORC_OK;
}

/* a10 */
void orc_chi_batch(int64_t n, const float *E_over_k, const float *b, double *chi, int32_t chi_mode,
                   const orc_mlp *net, const orc_chi_table *table, double b_max, double lnE_min,
                   double lnE_max) {
  for (int64_t p = 0; p < n; ++p) {
    double lnE = log((double)E_over_k[p]);
    double btilde = (double)b[p] / b_max;
    chi[p] = (chi_mode == 0) ? orc_chi_bilinear(table, lnE, btilde)
                             : orc_chi_mlp(net, lnE_min, lnE_max, lnE, btilde);
  }
}

/* ------------------------------------------------------------------------------------------
 * "Exact" deflection angle (eqs. 16/20 P:L272).
 * ---------------------------------------------------------------------------------------- */
double orc_potential_eval(const orc_potential *pot, double r) {
  switch (pot->kind) {
    case ORC_POT_LJ: {
      double s = pot->p1 / r, s2 = s * s, s6 = s2 * s2 * s2;
      return 4.0 * pot->p0 * (s6 * s6 - s6);
    }
    case ORC_POT_HARD_SPHERE: return r < pot->p0 ? 1e300 : 0.0;
    case ORC_POT_INV_R: return pot->p0 / r;
    default: return pot->p0 / (r * r);
  }
}

static double F_of_r(const orc_potential *pot, double E, double b, double r) {
  return 1.0 - (b * b) / (r * r) - orc_potential_eval(pot, r) / E; /* eq. 21 */
}

/* r_min = LARGEST root of eq. 21: walk inward from r_hi on a geometric grid to the first sign
 * change, then bisect to the last bit (the paper uses Brent to 1e-14). */
double orc_rmin(const orc_potential *pot, double E, double b) {
  double hi = pot->r_hi > 2.0 * b ? pot->r_hi : 2.0 * b;
  double lo = hi;
  for (int it = 0; it < 100000; ++it) {
    lo = hi * 0.99;
    if (F_of_r(pot, E, b, lo) < 0.0) break;
    hi = lo;
    if (lo < 1e-300) return 0.0; /* no turning point (cannot happen for repulsive cores) */
  }
  for (int it = 0; it < 200; ++it) {
    double mid = 0.5 * (lo + hi);
    if (mid <= lo || mid >= hi) break;
    if (F_of_r(pot, E, b, mid) < 0.0) lo = mid; else hi = mid;
  }
  return hi; /* F(hi) >= 0 */
}

/* Gauss-Legendre nodes/weights on [-1,1], Newton on P_n (computed, not tabulated) */
#define GLN 64
static double gl_x[GLN], gl_w[GLN];
static int gl_ready = 0;
static void gl_init(void) {
  for (int i = 0; i < GLN; ++i) {
    double x = cos(PI * (i + 0.75) / (GLN + 0.5)), dp = 1.0;
    for (int it = 0; it < 100; ++it) {
      double p0 = 1.0, p1 = x;
      for (int k = 2; k <= GLN; ++k) {
        double p2 = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
        p0 = p1; p1 = p2;
      }
      dp = GLN * (x * p1 - p0) / (x * x - 1.0);
      double dx = p1 / dp;
      x -= dx;
      if (fabs(dx) < 1e-16) break;
    }
    { /* recompute derivative at the converged node */
      double p0 = 1.0, p1 = x;
      for (int k = 2; k <= GLN; ++k) {
        double p2 = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
        p0 = p1; p1 = p2;
      }
      dp = GLN * (x * p1 - p0) / (x * x - 1.0);
    }
    gl_x[i] = x;
    gl_w[i] = 2.0 / ((1.0 - x * x) * dp * dp);
  }
  gl_ready = 1;
}

/* chi = pi - 2b int_{rmin}^inf dr / (r^2 sqrt(F(r))).  With u = r_min/r, beta = b/r_min:
 *   chi = pi - 2 beta int_0^1 du / sqrt(Ft(u)),  Ft(u) = 1 - beta^2 u^2 - V(r_min/u)/E,
 * and u = 1 - s^2 removes the inverse-square-root end point at u = 1:
 *   chi = pi - 4 beta int_0^1 s ds / sqrt(Ft(1 - s^2)). */
double orc_chi_exact(const orc_potential *pot, double E, double b, int32_t n_panels) {
  if (b <= 0.0) return PI; /* head-on */
  if (!gl_ready) gl_init();
  double rmin = orc_rmin(pot, E, b);
  if (rmin <= 0.0) return 0.0;
  double beta = b / rmin;
  double sum = 0.0;
  for (int32_t pnl = 0; pnl < n_panels; ++pnl) {
    double a0 = (double)pnl / n_panels, a1 = (double)(pnl + 1) / n_panels;
    double half = 0.5 * (a1 - a0), mid = 0.5 * (a1 + a0);
    for (int i = 0; i < GLN; ++i) {
      double s = mid + half * gl_x[i];
      double u = 1.0 - s * s;
      double Ft = 1.0 - beta * beta * u * u - (u > 0.0 ? orc_potential_eval(pot, rmin / u) / E : 0.0);
      if (Ft > 0.0) sum += half * gl_w[i] * s / sqrt(Ft);
    }
  }
  return PI - 4.0 * beta * sum;
}

/* Q23: a node that falls on the orbiting singularity (chi -> infinity: the pair spirals) is capped at 32 revolutions so
 * that the fp32 table stays finite; any such angle is as good as another.  Written so that NaN is capped too. */
double orc_cap_chi(double c) { return (c <= 64.0 * PI) ? c : 64.0 * PI; }

void orc_build_chi_table(const orc_potential *pot, int32_t nE, int32_t nB, double lnE_min,
                         double lnE_max, double b_max, int32_t n_panels, float *chi) {
  for (int32_t iE = 0; iE < nE; ++iE) {
    double lnE = lnE_min + (lnE_max - lnE_min) * (double)iE / (double)(nE - 1);
    double E = ORC_KB * exp(lnE);
    for (int32_t iB = 0; iB < nB; ++iB) {
      double b = b_max * (double)iB / (double)(nB - 1);
      double c = orc_cap_chi(fabs(orc_chi_exact(pot, E, b, n_panels))); /* Q14, Q23 */
      chi[(size_t)iE * nB + iB] = (float)c;
    }
  }
}


/* f2, the paper's neural table generation ("the neural network can generate a complete 512 x 512 table in less
 * than 1.0 s"): the chi-MLP of P:L277-283 evaluated on the table nodes of Q13 (lnE uniform in [lnE_min, lnE_max],
 * b~ = j / (nB - 1)), abs value (Q14), capped (Q23), rounded to fp32 like the quadrature table. */
void orc_build_chi_table_mlp(const orc_mlp *net, int32_t nE, int32_t nB, double lnE_min, double lnE_max, float *chi) {
  for (int32_t iE = 0; iE < nE; ++iE) {
    double lnE = lnE_min + (lnE_max - lnE_min) * (double)iE / (double)(nE - 1);
    for (int32_t iB = 0; iB < nB; ++iB) {
      double bt = (double)iB / (double)(nB - 1);
      chi[(size_t)iE * nB + iB] = (float)orc_cap_chi(fabs(orc_chi_mlp(net, lnE_min, lnE_max, lnE, bt)));
    }
  }
}


/* ------------------------------------------------------------------------------------------
 * f4.  Free flight + Maxwell walls for the 1-D Couette layout (Q30), and the
 * per-cell sampling sums.
 * ---------------------------------------------------------------------------------------- */
void orc_move_couette(int64_t n, double *x, double *vx, double *vy, double *vz, int32_t *cell, int32_t *bounces,
                      double *margin, const orc_couette_params *p, uint64_t seed, uint32_t step) {
  const double L = p->L, srt = sqrt(p->rt_wall);
  for (int64_t q = 0; q < n; ++q) {
    double xx = x[q], t_left = p->dt, mg = 1e300;
    int nb = 0;
    for (;;) {
      double xn = xx + vx[q] * t_left;
      if (xn >= 0.0 && xn <= L) { /* no (further) wall hit */
        double d0 = fabs(xn) / L, d1 = fabs(L - xn) / L;
        if (d0 < mg) mg = d0;
        if (d1 < mg) mg = d1;
        xx = xn;
        break;
      }
      {
        double d = (xn < 0.0 ? -xn : xn - L) / L;
        if (d < mg) mg = d;
      }
      if (nb == ORC_MAX_BOUNCES) { /* give up: clamp into the gap */
        xx = xn < 0.0 ? 0.0 : L;
        break;
      }
      {
        const int upper = xn > L;
        const double wall = upper ? L : 0.0;
        uint32_t r[4];
        t_left -= (wall - xx) / vx[q]; /* time of the hit */
        xx = wall;
        philox_at(seed, (uint32_t)q, (uint32_t)nb, step, 5u, r);
        {
          double u0 = orc_u01(r[0]), da = fabs(u0 - p->accommodation);
          if (da < mg) mg = da;
          if (u0 < p->accommodation) { /* diffuse re-emission from the wall Maxwellian */
            double vn = sqrt(-2.0 * p->rt_wall * log(orc_u01(r[1])));
            double rad = sqrt(-2.0 * log(orc_u01(r[2]))), ang = 2.0 * PI * orc_u01(r[3]);
            vx[q] = upper ? -vn : vn;
            vy[q] = srt * rad * cos(ang) + (upper ? p->u_wall : -p->u_wall);
            vz[q] = srt * rad * sin(ang);
          } else { /* specular */
            vx[q] = -vx[q];
          }
        }
        nb++;
      }
    }
    x[q] = xx;
    {
      double s = xx * (double)p->n_cells / L;
      int32_t k = (int32_t)floor(s);
      double f = fabs(s - floor(s + 0.5)) / (double)p->n_cells; /* distance to the nearest cell boundary / L */
      if (k > p->n_cells - 1) k = p->n_cells - 1;
      if (k < 0) k = 0;
      if (f < mg) mg = f;
      cell[q] = k;
    }
    if (bounces) bounces[q] = nb;
    if (margin) margin[q] = mg;
  }
}

void orc_sample_cells(int32_t n_cells, const int32_t *cell_start, const double *vx, const double *vy,
                      const double *vz, double *acc) {
  for (int32_t k = 0; k < n_cells; ++k) {
    double *a = acc + 8 * (size_t)k;
    for (int32_t s = cell_start[k]; s < cell_start[k + 1]; ++s) {
      a[0] += 1.0;
      a[1] += vx[s];
      a[2] += vy[s];
      a[3] += vz[s];
      a[4] += vx[s] * vx[s];
      a[5] += vy[s] * vy[s];
      a[6] += vz[s] * vz[s];
      a[7] += vx[s] * vy[s];
    }
  }
}


/* f1: NTC candidate count with carried remainder (Q31) */
void orc_ntc_counts(int32_t n_cells, const int32_t *cell_start, const float *sigma_cr_max, double coef,
                    double *remainder, int32_t *counts) {
  for (int32_t k = 0; k < n_cells; ++k) {
    int32_t N = cell_start[k + 1] - cell_start[k];
    if (N < 2) {
      counts[k] = 0;
      continue;
    }
    {
      double pairs = (double)N * (double)(N - 1);
      double m = 0.5 * pairs;
      m = m * coef;
      m = m * (double)sigma_cr_max[k];
      m = m + remainder[k];
      {
        double f = floor(m);
        counts[k] = (int32_t)f;
        remainder[k] = m - f;
      }
    }
  }
}
