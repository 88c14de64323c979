// "Exact" ab initio deflection angle on the GPU: the classical deflection integral
// of eq. 16 for a Lennard-Jones 12-6 potential, per pair, in FP64 -- the computation the paper's
// neural / tabulated operators replace, so that the exact-vs-neural KERNEL ratio the paper
// leaves unquantified can be measured on one box.  Written from the paper's equations, independent of
// oracle/.
//
// Reduced units E* = E / eps, b* = b / sigma, V*(r) = 4 (r^-12 - r^-6).
//   1. r_min = largest root of F(r) = 1 - b^2/r^2 - V(r)/E (eq. 21): scan inward from r_hi = max(50, 2 b*)
//      on a geometric grid to the first sign change, then bisection to machine precision;
//   2. with beta = b / r_min and u = r_min / r, and u = 1 - s^2 to remove the inverse-square-root end
//      point:  chi = pi - 4 beta int_0^1 s ds / sqrt(F~(1 - s^2)),  F~(u) = 1 - beta^2 u^2 - V(r_min/u)/E;
//      since F~(1) = 0 the factor s^2 is divided out of F~ analytically (see the kernel), leaving a smooth
//      integrand for composite Gauss-Legendre (kPanels panels x 32 nodes; nodes by Newton on P_32 at first use).
// b = 0 gives chi = pi.  The result is the SIGNED angle (negative for attractive glancing collisions, Q14).
#include <algorithm>
#include <cmath>
#include <mutex>

#include "dsmc_internal.h"

namespace dsmc {

constexpr int kGl = 32;      // Gauss-Legendre nodes per panel
constexpr int kPanels = 8;   // panels on s in [0, 1], graded towards s = 0

__constant__ double c_gl_x[kGl];  // nodes on [0, 1]
__constant__ double c_gl_w[kGl];  // weights on [0, 1]

__device__ __forceinline__ double lj_over_E(double r, double inv_E) {  // V*(r) / E*
  const double i2 = 1.0 / (r * r), i6 = i2 * i2 * i2;
  return 4.0 * (i6 * i6 - i6) * inv_E;
}

// signed chi for reduced energy Es = E / eps and reduced impact parameter bs = b / sigma
__device__ double chi_exact_lj(double Es, double bs) {
  double out;
  if (!(bs > 0.0) || !(Es > 0.0)) {
    out = 3.141592653589793;
  } else {
    const double inv_E = 1.0 / Es, b2 = bs * bs;
    // 1. largest root of F
    double hi = fmax(50.0, 2.0 * bs), lo = hi;
    {
      const double q = 0.97;
      for (int it = 0; it < 400; ++it) {
        lo = hi * q;
        const double F = 1.0 - b2 / (lo * lo) - lj_over_E(lo, inv_E);
        if (F < 0.0) break;
        hi = lo;
      }
    }
    for (int it = 0; it < 64; ++it) {  // F(lo) < 0 <= F(hi)
      const double mid = 0.5 * (lo + hi);
      const double F = 1.0 - b2 / (mid * mid) - lj_over_E(mid, inv_E);
      if (F < 0.0) lo = mid; else hi = mid;
    }
    const double rmin = hi, beta = bs / rmin, beta2 = beta * beta;
    // 2. quadrature in s.  F~(1) = 0 at the root, so F~(u) = F~(u) - F~(1) = s^2 G(s) with
    //    G = beta^2 (1 + u) + (4 / E) [a^12 P12(u) - a^6 P6(u)],  a = 1 / r_min,  Pn(u) = 1 + u + ... + u^(n-1)
    //    (1 - u^n = (1 - u) Pn(u), 1 - u = s^2): the integrand s / sqrt(F~) = 1 / sqrt(G) is smooth and free of
    //    cancellation.  Panel edges graded as (k / kPanels)^2 (G(0) is small near orbiting).
    const double a2 = 1.0 / (rmin * rmin), a6 = a2 * a2 * a2, a12 = a6 * a6;
    const double c12 = 4.0 * inv_E * a12, c6 = 4.0 * inv_E * a6;
    double acc = 0.0;
    for (int k = 0; k < kPanels; ++k) {
      const double e0 = (double)(k * k) / (kPanels * kPanels), e1 = (double)((k + 1) * (k + 1)) / (kPanels * kPanels);
      const double h = e1 - e0;
      double part = 0.0;
#pragma unroll 4
      for (int j = 0; j < kGl; ++j) {
        const double sx = e0 + h * c_gl_x[j];
        const double u = 1.0 - sx * sx;
        const double u2 = u * u, u3 = u2 * u;
        const double p6 = (1.0 + u + u2) * (1.0 + u3);  // 1 + u + ... + u^5
        const double p12 = p6 * (1.0 + u3 * u3);        // 1 + u + ... + u^11
        const double G = beta2 * (1.0 + u) + c12 * p12 - c6 * p6;
        part += c_gl_w[j] * rsqrt(fmax(G, 1e-300));
      }
      acc += h * part;
    }
    out = 3.141592653589793 - 4.0 * beta * acc;
  }
  return out;
}

__global__ void __launch_bounds__(128) k_chi_exact(int64_t n, const float *__restrict__ E_over_k,
                                                  const float *__restrict__ b, float *__restrict__ chi,
                                                  double inv_eps_k, double inv_sigma, int take_abs) {
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
    const double out = chi_exact_lj((double)__ldg(E_over_k + p) * inv_eps_k, (double)__ldg(b + p) * inv_sigma);
    chi[p] = (float)(take_abs ? fabs(out) : out);
  }
}

// chi table nodes (Q13): node (iE, iB) at E~ = lnE_min + iE dlnE (E~ = ln(E_r / k_B [K])), b~ = iB / (nB - 1);
// stores abs(chi) (Q14) rounded to fp32, chi[iE * nB + iB]
__global__ void __launch_bounds__(128) k_chi_table_lj(int nE, int nB, double lnE_min, double dlnE, double bmax_star,
                                                     double inv_eps_k, float *__restrict__ table) {
  const int64_t total = (int64_t)nE * nB;
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < total; p += (int64_t)gridDim.x * blockDim.x) {
    const int iE = (int)(p / nB), iB = (int)(p % nB);
    const double Es = exp(lnE_min + iE * dlnE) * inv_eps_k;
    const double bs = bmax_star * ((double)iB / (double)(nB - 1));
    // Q23: a node on the orbiting singularity (chi -> infinity) is capped at 32 revolutions: the table stays finite
    table[p] = (float)fmin(fabs(chi_exact_lj(Es, bs)), 64.0 * 3.141592653589793);
  }
}

// quad[iE (nB-1) + iB] = the four nodes around grid cell (iE, iB): one 16-byte load per lookup
__global__ void k_quad_from_table(int nE, int nB, const float *__restrict__ table, float4 *__restrict__ quad) {
  const int64_t total = (int64_t)(nE - 1) * (nB - 1);
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < total; p += (int64_t)gridDim.x * blockDim.x) {
    const int iE = (int)(p / (nB - 1)), iB = (int)(p % (nB - 1));
    const float *t = table + (size_t)iE * nB + iB;
    quad[p] = make_float4(t[0], t[1], t[nB], t[nB + 1]);
  }
}

// f2, neural table generation: the node coordinates of the table as a pair batch (E_r / k_B, b / b_max) ...
__global__ void k_table_node_coords(int nE, int nB, double lnE_min, double dlnE, float *__restrict__ E,
                                    float *__restrict__ b) {
  const int64_t total = (int64_t)nE * nB;
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < total; p += (int64_t)gridDim.x * blockDim.x) {
    const int iE = (int)(p / nB), iB = (int)(p % nB);
    E[p] = (float)exp(lnE_min + dlnE * iE);
    b[p] = (float)((double)iB / (double)(nB - 1));
  }
}

// ... and, after the network: abs (Q14), cap at 64 pi (Q23, written so that NaN is capped too), quad layout
__global__ void k_cap_nodes(int64_t total, float *__restrict__ table) {
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < total; p += (int64_t)gridDim.x * blockDim.x) {
    const float cap = (float)(64.0 * 3.141592653589793);
    const float c = fabsf(table[p]);
    table[p] = (c <= cap) ? c : cap;
  }
}

int launch_table_node_coords(dsmc_ctx *c, int nE, int nB, double lnE_min, double lnE_max, float *E, float *b) {
  const int64_t total = (int64_t)nE * nB;
  const int grid = (int)std::min<int64_t>((total + 255) / 256, (int64_t)c->num_sms * 8);
  k_table_node_coords<<<grid, 256, 0, c->stream>>>(nE, nB, lnE_min, (lnE_max - lnE_min) / (nE - 1), E, b);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_cap_and_quad(dsmc_ctx *c, int nE, int nB, float *table_dev, float4 *quad_dev) {
  const int64_t total = (int64_t)nE * nB;
  const int grid = (int)std::min<int64_t>((total + 255) / 256, (int64_t)c->num_sms * 8);
  k_cap_nodes<<<grid, 256, 0, c->stream>>>(total, table_dev);
  k_quad_from_table<<<grid, 256, 0, c->stream>>>(nE, nB, table_dev, quad_dev);
  c->launches += 2;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

// Gauss-Legendre nodes / weights on [0, 1] by Newton iteration on the Legendre polynomial P_n (host, once)
static void gauss_legendre_01(int n, double *x, double *w) {
  for (int i = 0; i < n; ++i) {
    double z = std::cos(3.141592653589793 * (i + 0.75) / (n + 0.5));
    double pp = 1.0;
    for (int it = 0; it < 100; ++it) {
      double p1 = 1.0, p2 = 0.0;
      for (int j = 0; j < n; ++j) {
        const double p3 = p2;
        p2 = p1;
        p1 = ((2.0 * j + 1.0) * z * p2 - j * p3) / (j + 1.0);
      }
      pp = n * (z * p1 - p2) / (z * z - 1.0);
      const double dz = p1 / pp;
      z -= dz;
      if (std::fabs(dz) < 1e-16) break;
    }
    x[i] = 0.5 * (1.0 - z);  // descending z -> ascending x
    w[i] = 1.0 / ((1.0 - z * z) * pp * pp);
  }
}

static int upload_gl_nodes(dsmc_ctx *c);

// generates the table on the device and installs it as the context's chi table (device copy in `table_dev`,
// nE * nB floats, owned by the caller / context)
int launch_chi_table_lj(dsmc_ctx *c, int nE, int nB, double lnE_min, double lnE_max, double b_max, double eps_over_k,
                        double sigma, float *table_dev, float4 *quad_dev) {
  int rc = upload_gl_nodes(c);
  if (rc != DSMC_OK) return rc;
  const int64_t total = (int64_t)nE * nB;
  const int grid = (int)std::min<int64_t>((total + 127) / 128, (int64_t)c->num_sms * 16);
  k_chi_table_lj<<<grid, 128, 0, c->stream>>>(nE, nB, lnE_min, (lnE_max - lnE_min) / (nE - 1), b_max / sigma,
                                              1.0 / eps_over_k, table_dev);
  k_quad_from_table<<<grid, 128, 0, c->stream>>>(nE, nB, table_dev, quad_dev);
  c->launches += 2;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

static int upload_gl_nodes(dsmc_ctx *c) {
  static std::once_flag once[64];
  static cudaError_t upload_rc[64];
  const int dev = c->device < 64 ? c->device : 63;
  std::call_once(once[dev], [&] {
    double x[kGl], w[kGl];
    gauss_legendre_01(kGl, x, w);
    upload_rc[dev] = cudaMemcpyToSymbol(c_gl_x, x, sizeof(x));
    if (upload_rc[dev] == cudaSuccess) upload_rc[dev] = cudaMemcpyToSymbol(c_gl_w, w, sizeof(w));
  });
  return upload_rc[dev] == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_chi_exact(dsmc_ctx *c, int64_t n, const float *E_over_k, const float *b, float *chi, double eps_over_k,
                     double sigma, int take_abs) {
  const int rc = upload_gl_nodes(c);
  if (rc != DSMC_OK) return rc;
  const int grid = (int)std::min<int64_t>((n + 127) / 128, (int64_t)c->num_sms * 16);
  k_chi_exact<<<grid, 128, 0, c->stream>>>(n, E_over_k, b, chi, 1.0 / eps_over_k, 1.0 / sigma, take_abs);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

}  // namespace dsmc
