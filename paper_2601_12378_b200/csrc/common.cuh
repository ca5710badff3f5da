// common.cuh -- device-side context and small helpers of the PTEFIT hot path (sm_100a).
// Product code: shares nothing with oracle/.  See include/ptefit.h for the ABI and DESIGN.md
// for the data layout.  Citations are PAPER.md lines (arxiv 2601.12378).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define PTEFIT_MAX_TERMS 12
#define PTEFIT_MAX_CAND 32
#define PTEFIT_MAX_LIM 256
#define PTEFIT_MAX_NR 257
#define PTEFIT_MAX_DEG 8      /* largest exponent N of a polynomial term */

namespace ptefit {

constexpr double kMu0 = 1.25663706143591729e-6;  // 4 pi 1e-7 (reading O0)

struct TermDev { int kind, i, N; };

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
  const double *lim_r, *lim_z;    // [nlim]
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
  double *chi2;                   // [B]
  SearchOut *so;                  // [B]
  int *status;                    // [B]
  long long *phase_clk;           // [8] optional in-kernel phase timers (ptefit_debug_phase_clocks), else nullptr
};

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

template <typename T>
__device__ __forceinline__ T basis_term(const Dev<T> &D, int l, T x, T rdA, T mu0dA_over_r) {
  const TermDev t = D.terms[l];
  T v = ipow(x, t.i) - ipow(x, t.N);
  return (x < T(0)) ? T(0) : v * (t.kind == 0 ? rdA : mu0dA_over_r);
}

}  // namespace ptefit
