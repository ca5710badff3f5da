// solve_kernels.cuh -- A7/A8: Delta* psi = -mu0 R J_phi (Eq. 1) on the 5-point
// stencil with Dirichlet data, as N_Z-2 independent tridiagonal systems:
// DST-I in Z, Thomas sweeps in R with precomputed FP64 factors, inverse DST-I, then
// psi = psi_pl + psi_coil with relaxation.  v1: three kernels, intermediates in global memory.
#pragma once
#include "common.cuh"

namespace ptefit {

constexpr int DST_COLS = 32;      // R-columns per block
constexpr int DST_THREADS = 256;

// Right-hand side + forward DST-I along Z.  grid (ceil(nri/DST_COLS), B), dyn smem nzi*DST_COLS*T.
// Output fhat[s][i-1][m-1]  (i-major so the tridiagonal kernel coalesces over m).
template <typename T>
__global__ void __launch_bounds__(DST_THREADS) k_rhs_dst(Dev<T> D, const T *__restrict__ cur,
                                                          const T *__restrict__ pbd) {
  extern __shared__ unsigned char smem_raw[];
  T *f = reinterpret_cast<T *>(smem_raw);          // [nzi][DST_COLS]
  const int s = blockIdx.y, i0 = 1 + blockIdx.x * DST_COLS;
  const int nr = D.nr, nz = D.nz, nri = D.nri, nzi = D.nzi;
  const T *I = cur + (size_t)s * D.N;
  const T *pb = pbd + (size_t)s * D.nbnd;          // bottom[nr], top[nr], left[nzi], right[nzi]
  const T cz = T(1.0 / (D.dz * D.dz));
  for (int e = threadIdx.x; e < nzi * DST_COLS; e += DST_THREADS) {
    const int jj = e / DST_COLS, c = e - jj * DST_COLS;
    const int i = i0 + c, j = jj + 1;
    T v = T(0);
    if (i <= nri) {
      const double R = D.rmin + i * D.dr;
      v = T(-kMu0 * R / D.dA) * I[j * nr + i];
      if (i == 1) v -= T((1.0 + D.dr / (2.0 * R)) / (D.dr * D.dr)) * pb[2 * nr + jj];
      if (i == nri) v -= T((1.0 - D.dr / (2.0 * R)) / (D.dr * D.dr)) * pb[2 * nr + nzi + jj];
      if (j == 1) v -= cz * pb[i];
      if (j == nzi) v -= cz * pb[nr + i];
    }
    f[e] = v;
  }
  __syncthreads();
  const int period = 2 * (nz - 1);
  T *out = D.fhat + (size_t)s * nri * nzi;
  for (int e = threadIdx.x; e < nzi * DST_COLS; e += DST_THREADS) {
    const int c = e / nzi, mm = e - c * nzi;        // consecutive threads -> consecutive m
    const int i = i0 + c, m = mm + 1;
    if (i > nri) continue;
    T acc = T(0);
    int k = m;                                      // (j*m) mod period
    for (int jj = 0; jj < nzi; ++jj) {
      acc = fma(f[jj * DST_COLS + c], D.sintab[k], acc);
      k += m; if (k >= period) k -= period;
    }
    out[(size_t)(i - 1) * nzi + mm] = acc;
  }
}

// Thomas sweeps along R in FP64, one thread per (slice, mode m).  grid (ceil(nzi/128), B).
// In place on ytmp (double) -> result written back to fhat as T.
template <typename T>
__global__ void k_tridiag(Dev<T> D) {
  const int s = blockIdx.y, mm = blockIdx.x * blockDim.x + threadIdx.x;
  if (mm >= D.nzi) return;
  const int nri = D.nri, nzi = D.nzi;
  T *fh = D.fhat + (size_t)s * nri * nzi;
  double *y = D.ytmp + (size_t)s * nri * nzi;
  double prev = 0.0;
  for (int i = 0; i < nri; ++i) {
    const size_t o = (size_t)i * nzi + mm;
    const double v = (double)fh[o] - D.tri_w[o] * prev;   // tri_w[0][m] = 0
    y[o] = v;
    prev = v;
  }
  double x = 0.0;
  for (int i = nri - 1; i >= 0; --i) {
    const size_t o = (size_t)i * nzi + mm;
    x = (y[o] - D.tri_ce[i] * x) * D.tri_invb[o];         // ce[nri-1] multiplies x = 0
    fh[o] = T(x);
  }
}

// Inverse DST-I along Z + total flux + relaxation.  grid (ceil(nri/DST_COLS), B).
// psi_out[s][j][i] = old + relax * (psi_pl + psi_coil - old)  (relax applied iff use_relax).
template <typename T>
__global__ void __launch_bounds__(DST_THREADS) k_idst_total(Dev<T> D, T *__restrict__ psi, int use_relax,
                                                             int add_coil) {
  extern __shared__ unsigned char smem_raw[];
  if (!psi) psi = reinterpret_cast<T *>(D.ca->psi);
  T *f = reinterpret_cast<T *>(smem_raw);          // [DST_COLS][nzi+1]
  const int s = blockIdx.y, i0 = 1 + blockIdx.x * DST_COLS;
  const int nr = D.nr, nz = D.nz, nri = D.nri, nzi = D.nzi, ld = nzi + 1;
  const T *fh = D.fhat + (size_t)s * nri * nzi;
  for (int e = threadIdx.x; e < nzi * DST_COLS; e += DST_THREADS) {
    const int c = e / nzi, mm = e - c * nzi;
    const int i = i0 + c;
    f[c * ld + mm] = (i <= nri) ? fh[(size_t)(i - 1) * nzi + mm] : T(0);
  }
  __syncthreads();
  const int period = 2 * (nz - 1);
  const T scale = T(2.0 / (nz - 1));
  const T om = T(D.relax);
  T *p = psi + (size_t)s * D.N;
  const T *pc = D.psi_coil + (size_t)s * D.N;
  for (int e = threadIdx.x; e < nzi * DST_COLS; e += DST_THREADS) {
    const int jj = e / DST_COLS, c = e - jj * DST_COLS;   // consecutive threads -> consecutive i
    const int i = i0 + c, j = jj + 1;
    if (i > nri) continue;
    T acc = T(0);
    int k = j;
    for (int mm = 0; mm < nzi; ++mm) {
      acc = fma(f[c * ld + mm], D.sintab[k], acc);
      k += j; if (k >= period) k -= period;
    }
    T v = acc * scale;
    if (add_coil) v += pc[j * nr + i];
    if (use_relax) { const T old = p[j * nr + i]; v = old + om * (v - old); }
    p[j * nr + i] = v;
  }
}

// Edge nodes: psi = psi_bdry + psi_coil (same relaxation).  grid (ceil(nbnd/256), B).
template <typename T>
__global__ void k_edge_total(Dev<T> D, T *__restrict__ psi, const T *__restrict__ pbd, int use_relax,
                             int add_coil) {
  const int s = blockIdx.y, k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= D.nbnd) return;
  if (!psi) psi = reinterpret_cast<T *>(D.ca->psi);
  const int nr = D.nr, nz = D.nz, nzi = D.nzi;
  int n;
  if (k < nr) n = k;
  else if (k < 2 * nr) n = (nz - 1) * nr + (k - nr);
  else if (k < 2 * nr + nzi) n = (k - 2 * nr + 1) * nr;
  else n = (k - 2 * nr - nzi + 1) * nr + nr - 1;
  T v = pbd[(size_t)s * D.nbnd + k];
  if (add_coil) v += D.psi_coil[(size_t)s * D.N + n];
  T *p = psi + (size_t)s * D.N;
  if (use_relax) { const T old = p[n]; v = old + T(D.relax) * (v - old); }
  p[n] = v;
}

}  // namespace ptefit
