// common.cuh -- device-side context and small helpers of the PTEFIT hot path (sm_100a).
// Product code: shares nothing with oracle/.  See include/ptefit.h for the ABI and DESIGN.md
// for the data layout.  Citations are PAPER.md lines (arxiv 2601.12378).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define PTEFIT_MAX_TERMS 16
#define PTEFIT_MAX_KNOTS 16
#define PTEFIT_MAX_CAND 32
#define PTEFIT_MAX_LIM 256
#define PTEFIT_MAX_NR 257
#define PTEFIT_MAX_DEG 8      /* largest exponent N of a polynomial term */

namespace ptefit {

constexpr double kMu0 = 1.25663706143591729e-6;  // 4 pi 1e-7 (reading O0)

struct TermDev { int kind, family, i, N; };

// Tension-spline tables (family 1 terms; reading O4c), FP64, in global memory.
// On [knot_r, knot_r+1], t = (x - knot_r)/h_r:
//   phi_q = d_qr (1-t) + d_q,r+1 t + m[r][q] (sinh(tau h (1-t))/sinh(tau h) - (1-t))/tau^2 + m[r+1][q] (sinh(tau h t)/sinh(tau h) - t)/tau^2
struct SplineDev {
  int nk;
  double tau, inv_tau2;
  double knot[PTEFIT_MAX_KNOTS], inv_h[PTEFIT_MAX_KNOTS], tau_h[PTEFIT_MAX_KNOTS], inv_sinh[PTEFIT_MAX_KNOTS];
  double m[PTEFIT_MAX_KNOTS][PTEFIT_MAX_KNOTS];      // m[r][q] = second derivative of phi_q at knot r
};

// Caller-owned device pointers of one ptefit_reconstruct call.  The block lives in device memory at a
// fixed address and is rewritten by k_set_args before every call, so that the captured CUDA graph
// does not depend on the pointers a caller passes.
struct CallArgs {
  const void *b, *ic;
  void *psi, *coeffs;
  int *axis_ij; void *axis_rzpsi;
  int *xpt_ij; void *xpt_rzpsi;
  void *psi_bnd; int *limited; void *chi2; int *status;
};

// Per-slice result of the search, kept in double on the device.
struct SearchOut {
  double axis_r, axis_z, axis_psi;
  double xpt_r, xpt_z, xpt_psi;
  double psi_b;
  int axis_i, axis_j, xpt_i, xpt_j;
  int limited, n_cand;
};

// Everything the kernels need, passed by value (fits the 4 KB kernel-parameter space).
template <typename T>
struct Dev {
  int nr, nz, N, nri, nzi, nbnd, M, nc, nt, npoly, has_delz, nlim, ip_sign;
  int nspl, maxdeg;               // spline terms among the npoly basis terms; largest polynomial exponent
  int lsq_method;                 // 0 normal equations + Cholesky, 1 modified Gram-Schmidt
  int fit_coils;                  // 1 = joint fit of the coil currents, Eq. 7 (joint_fit.cuh)
  const double *gcw, *c22s, *tcoil, *inv_sic2;   // W G_C [M][nc]; scaled G_C^T W^2 G_C + diag(1/sigma_ic^2) [nc][nc]; column scales; 1/sigma_ic^2
  double *icf, *icm;              // [B][nc] fitted / measured coil currents
  const SplineDev *spl;           // nullptr unless nspl > 0
  const CallArgs *ca;             // device copy of the caller's pointers (k_set_args)
  double rmin, zmin, dr, dz, dA, lambda_reg, relax;
  double cold_rc, cold_zc, cold_a, cold_b;
  TermDev terms[PTEFIT_MAX_TERMS];
  // tables (device)
  const T *gp, *gc, *gb, *ggc;
  const T *ggc_t;                 // ggc transposed: [n_c][N]
  const double *inv_sigma;        // [M]
  const uint8_t *lim_mask, *xpt_mask;
  const unsigned *lim_bits, *xpt_bits;   // the same masks bit-packed: bit (n & 31) of word n >> 5
  const unsigned *edge_bits;             // bit set for the nodes of the grid edge
  const unsigned *dil_bits;              // lim_mask dilated by one row up and down, edge nodes excluded (compact node list)
  const unsigned *dil2_bits;             // lim_mask dilated by two rows up and down (all nodes)
  const double *lim_r, *lim_z;    // [nlim]
  const int *lim_n0;              // [nlim] flat index of the lower-left node of each vertex's bilinear cell
  const double *lim_tx, *lim_ty;  // [nlim] bilinear weights inside that cell
  // Delta* solve factors: [nri][nzi] (i-major so that threads over m coalesce)
  const double *tri_w, *tri_invb; // Thomas multipliers and inverse pivots
  const double *tri_ce;           // [nri] super-diagonal
  const double *tw2, *tib2;       // [nri][nzi] twisted factorisation (two threads per mode), see ptefit.cu
  const double *tw2k, *tod2;      // [nzi] right multiplier of the middle row; [nri] off-diagonals
  const T *sintab;                // [2*(nz-1)] sin(pi k/(nz-1))
  const T *dst_tab;               // folded DST matrices So[n2][n2], Se[n2][n2] (fused_solve.cuh)
  // workspaces [max_batch][...]
  T *xn, *psi_coil, *dred, *resp, *cur, *dzc, *psi_bdry, *fhat;
  double *ytmp;                   // [B][nri][nzi]
  double *X, *Xprev;              // [B][nt]
  float *pco;                     // [B][PCO_STRIDE] polynomial form of I'(x) = R dA P(x) + (mu0 dA / R) Q(x) of the last fit: P[0..MAX_DEG], Q[0..MAX_DEG], X_delz
  double *chi2;                   // [B]
  SearchOut *so;                  // [B]
  int *status;                    // [B]
};

constexpr int PCO_STRIDE = 2 * (PTEFIT_MAX_DEG + 1) + 2;

// After a fit kernel has stored X of slice s (same warp): the P' and FF' sums of I' = J_b(x) X are polynomials in x;
// their coefficients (FP64 sums, rounded to float) are written once here instead of being rebuilt by every consumer
// (k_current_split, k_solve_tc).  Entry 2 (MAX_DEG + 1) = the coefficient of the vertical-shift column.
template <typename T>
__device__ __forceinline__ void emit_pco(const Dev<T> &D, int s, int lane) {
  __syncwarp();
  const double *X = D.X + (size_t)s * D.nt;
  if (lane < 2 * (PTEFIT_MAX_DEG + 1)) {
    const int kind = lane / (PTEFIT_MAX_DEG + 1), k = lane - kind * (PTEFIT_MAX_DEG + 1);
    double c = 0.0;
    for (int l = 0; l < D.npoly; ++l)
      if (D.terms[l].kind == kind && D.terms[l].family == 0) c += X[l] * ((D.terms[l].i == k ? 1.0 : 0.0) - (D.terms[l].N == k ? 1.0 : 0.0));
    D.pco[(size_t)s * PCO_STRIDE + lane] = float(c);
  }
  if (lane == 2 * (PTEFIT_MAX_DEG + 1)) D.pco[(size_t)s * PCO_STRIDE + lane] = D.has_delz ? float(X[D.nt - 1]) : 0.f;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Polynomial basis value of one node: fac_l * (x^i_l - x^N_l), l < npoly, where
// fac = R dA (P' terms) or mu0 dA / R (FF' terms) -- Eq. 10.  x < 0 = outside.
template <typename T>
__device__ __forceinline__ T ipow(T x, int e) {
  T p = T(1);
  for (int k = 0; k < e; ++k) p *= x;   // repeated multiply, exponents are <= 8
  return p;
}

// Cardinal tension spline phi_q(x) (family 1).  Evaluated in FP64 (sinh), x in [0, 1].
__device__ __forceinline__ double spline_phi(const SplineDev &sp, int q, double x) {
  if (!(x >= sp.knot[0]) || !(x <= sp.knot[sp.nk - 1])) return 0.0;
  int r = 0;
  while (r < sp.nk - 2 && x >= sp.knot[r + 1]) ++r;
  const double t = fmin(fmax((x - sp.knot[r]) * sp.inv_h[r], 0.0), 1.0), th = sp.tau_h[r];
  const double A = sinh(th * (1.0 - t)) * sp.inv_sinh[r] - (1.0 - t), Bc = sinh(th * t) * sp.inv_sinh[r] - t;
  double v = (sp.m[r][q] * A + sp.m[r + 1][q] * Bc) * sp.inv_tau2;
  if (q == r) v += 1.0 - t;
  if (q == r + 1) v += t;
  return v;
}

// The pieces of spline_phi that do not depend on q: interval r, t, and the two sinh brackets (one pair of
// sinh per node instead of one per spline term).
struct SplinePt { int r; double t, A, Bc; bool in; };
__device__ __forceinline__ SplinePt spline_point(const SplineDev &sp, double x) {
  SplinePt p;
  p.in = (x >= sp.knot[0]) && (x <= sp.knot[sp.nk - 1]);
  int r = 0;
  while (r < sp.nk - 2 && x >= sp.knot[r + 1]) ++r;
  p.r = r;
  p.t = fmin(fmax((x - sp.knot[r]) * sp.inv_h[r], 0.0), 1.0);
  const double th = sp.tau_h[r];
  p.A = sinh(th * (1.0 - p.t)) * sp.inv_sinh[r] - (1.0 - p.t);
  p.Bc = sinh(th * p.t) * sp.inv_sinh[r] - p.t;
  return p;
}
__device__ __forceinline__ double spline_phi_at(const SplineDev &sp, const SplinePt &p, int q) {
  if (!p.in) return 0.0;
  double v = (sp.m[p.r][q] * p.A + sp.m[p.r + 1][q] * p.Bc) * sp.inv_tau2;
  if (q == p.r) v += 1.0 - p.t;
  if (q == p.r + 1) v += p.t;
  return v;
}

template <typename T>
__device__ __forceinline__ T basis_term(const Dev<T> &D, int l, T x, T rdA, T mu0dA_over_r) {
  const TermDev t = D.terms[l];
  if (x < T(0)) return T(0);
  T v;
  if (t.family == 1) v = T(spline_phi(*D.spl, t.i, (double)x));
  else v = ipow(x, t.i) - ipow(x, t.N);
  return v * (t.kind == 0 ? rdA : mu0dA_over_r);
}

// Contribution of the spline terms (family 1) to I' = J_b(x) X; the polynomial terms are summed by
// Horner where this is used.
template <typename T>
__device__ __forceinline__ T spline_current(const Dev<T> &D, const double *__restrict__ X, T x, T rdA, T fdA) {
  T acc = T(0);
  for (int l = 0; l < D.npoly; ++l)
    if (D.terms[l].family == 1) acc = fma(basis_term(D, l, x, rdA, fdA), T(X[l]), acc);
  return acc;
}

}  // namespace ptefit
