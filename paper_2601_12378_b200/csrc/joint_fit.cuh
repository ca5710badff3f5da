// joint_fit.cuh -- NEXT-1: joint fit of the basis coefficients and the coil currents,
// Eq. 7.  Unknowns [X; I_C'], block system [[R, G_C], [0, I]] [X; I_C'] = [b; I_C] with
// measurement rows weighted 1/sigma and coil rows 1/sigma_ic (reading O5b); the Tikhonov term
// acts on X only.  Normal equations + Cholesky in FP64, one CTA per slice, matrix in shared memory.
// The coil -> grid flux psi_coil = G_GC I_C' is then recomputed every iteration (k_coil_flux).
#pragma once
#include "common.cuh"

namespace ptefit {

constexpr int JOINT_THREADS = 128;
constexpr int JOINT_MAX_N = 96;          // n_terms + n_coil

__host__ __device__ inline size_t joint_smem_bytes(int M, int nt, int nc) {
  const size_t n = (size_t)nt + nc;
  return (n * n + 2 * n + (size_t)M * nt + M + 64) * sizeof(double);
}

// grid B, block JOINT_THREADS, dyn smem joint_smem_bytes.  dred holds b (k_setup in joint mode).
template <typename T>
__global__ void __launch_bounds__(JOINT_THREADS) k_lsq_joint(Dev<T> D, int B) {
  extern __shared__ __align__(16) unsigned char jf_raw[];
  const int s = blockIdx.x, tid = threadIdx.x, nth = blockDim.x, lane = tid & 31, warp = tid >> 5;
  const int M = D.M, nt = D.nt, nc = D.nc, n = nt + nc;
  double *A = reinterpret_cast<double *>(jf_raw);        // [n][n] normal matrix, lower triangle used
  double *g = A + (size_t)n * n;                          // [n] right-hand side -> solution
  double *sc = g + n;                                     // [n] column scales
  double *WR = sc + n;                                    // [M][nt] weighted response
  double *Wb = WR + (size_t)M * nt;                       // [M] weighted measurements
  double *red = Wb + M;                                   // [64] reductions / flags
  const T *resp = D.resp + (size_t)s * M * nt;
  const T *b = D.dred + (size_t)s * M;
  const double *icm = D.icm + (size_t)s * nc;
  if (tid == 0) { red[32] = 0.0; red[33] = 0.0; }
  __syncthreads();
  bool finite = true;
  for (int e = tid; e < M * nt; e += nth) {
    const int m = e / nt;
    const double v = (double)resp[e] * D.inv_sigma[m];
    WR[e] = v;
    finite &= isfinite(v);
  }
  for (int m = tid; m < M; m += nth) { const double v = (double)b[m] * D.inv_sigma[m]; Wb[m] = v; finite &= isfinite(v); }
  for (int c = tid; c < nc; c += nth) finite &= isfinite(icm[c]);
  if (!finite) red[32] = 1.0;
  __syncthreads();
  // rows of X: N11 (lower), N12^T into A[nt + c][l], right-hand side
  for (int e = tid; e < nt * (n + 1); e += nth) {
    const int l = e / (n + 1), j = e - l * (n + 1);
    double acc = 0.0;
    if (j < nt) { if (j <= l) for (int m = 0; m < M; ++m) acc = fma(WR[m * nt + l], WR[m * nt + j], acc); }
    else if (j < n) { const double *gw = D.gcw + (j - nt); for (int m = 0; m < M; ++m) acc = fma(WR[m * nt + l], gw[(size_t)m * nc], acc); }
    else for (int m = 0; m < M; ++m) acc = fma(WR[m * nt + l], Wb[m], acc);
    if (j < nt) { if (j <= l) A[l * n + j] = acc; }
    else if (j < n) A[j * n + l] = acc;
    else g[l] = acc;
  }
  for (int c = tid; c < nc; c += nth) {
    const double *gw = D.gcw + c;
    double acc = 0.0;
    for (int m = 0; m < M; ++m) acc = fma(gw[(size_t)m * nc], Wb[m], acc);
    g[nt + c] = (acc + icm[c] * D.inv_sic2[c]) / D.tcoil[c];
    sc[nt + c] = D.tcoil[c];
  }
  __syncthreads();
  if (tid < nt) sc[tid] = sqrt(A[tid * n + tid]);
  __syncthreads();
  bool any = false;
  for (int l = 0; l < nt; ++l) any |= sc[l] > 0.0;
  int st = red[32] != 0.0 ? 2 : (!any ? 3 : 0);
  const double reg = D.lambda_reg * D.lambda_reg * (double)M;
  for (int e = tid; e < n * n; e += nth) {
    const int i = e / n, j = e - i * n;
    if (j > i) continue;
    double v;
    if (i < nt) {                                          // N11
      v = (sc[i] > 0.0 && sc[j] > 0.0) ? A[e] / (sc[i] * sc[j]) + (i == j ? reg : 0.0) : (i == j ? 1.0 : 0.0);
    } else if (j < nt) {                                   // N12^T
      v = sc[j] > 0.0 ? A[e] / (sc[j] * sc[i]) : 0.0;
    } else {                                               // N22: constant, scaled at create
      v = D.c22s[(size_t)(i - nt) * nc + (j - nt)];
    }
    A[e] = v;
  }
  if (tid < nt) g[tid] = sc[tid] > 0.0 ? g[tid] / sc[tid] : 0.0;
  __syncthreads();
  // Cholesky A = L L^T in place (lower triangle), right-looking
  for (int j = 0; j < n && st == 0; ++j) {
    if (tid == 0) {
      const double v = A[j * n + j];
      if (j == 0) red[34] = v;
      if (!(v > 1e-13 * red[34]) || !(v > 0.0)) red[33] = 1.0; else A[j * n + j] = sqrt(v);
    }
    __syncthreads();
    if (red[33] != 0.0) { st = 3; break; }
    const double piv = A[j * n + j];
    for (int i = j + 1 + tid; i < n; i += nth) A[i * n + j] /= piv;
    __syncthreads();
    const int rem = n - j - 1;
    for (int e = tid; e < rem * rem; e += nth) {
      const int i = j + 1 + e / rem, k = j + 1 + e % rem;
      if (k <= i) A[i * n + k] = fma(-A[i * n + j], A[k * n + j], A[i * n + k]);
    }
    __syncthreads();
  }
  // L z = g, L^T x = z by warp 0 (dot products across lanes)
  if (warp == 0 && st == 0) {
    for (int i = 0; i < n; ++i) {
      double acc = 0.0;
      for (int k = lane; k < i; k += 32) acc = fma(A[i * n + k], g[k], acc);
      acc = warp_sum(acc);
      if (lane == 0) g[i] = (g[i] - acc) / A[i * n + i];
      __syncwarp();
    }
    for (int i = n - 1; i >= 0; --i) {
      double acc = 0.0;
      for (int k = i + 1 + lane; k < n; k += 32) acc = fma(A[k * n + i], g[k], acc);
      acc = warp_sum(acc);
      if (lane == 0) g[i] = (g[i] - acc) / A[i * n + i];
      __syncwarp();
    }
  }
  __syncthreads();
  if (st == 0) for (int i = tid; i < n; i += nth) g[i] = sc[i] > 0.0 ? g[i] / sc[i] : 0.0;
  else for (int i = tid; i < n; i += nth) g[i] = i < nt ? 0.0 : icm[i - nt];
  __syncthreads();
  // chi^2 over the measurement rows
  double c2 = 0.0;
  for (int m = tid; m < M; m += nth) {
    double r = -Wb[m];
    for (int l = 0; l < nt; ++l) r = fma(WR[m * nt + l], g[l], r);
    const double *gw = D.gcw + (size_t)m * nc;
    for (int c = 0; c < nc; ++c) r = fma(gw[c], g[nt + c], r);
    c2 = fma(r, r, c2);
  }
  c2 = warp_sum(c2);
  if (lane == 0) red[warp] = c2;
  __syncthreads();
  if (tid == 0 && D.status[s] == 0) {
    double tot = 0.0;
    for (int w = 0; w < (nth >> 5); ++w) tot += red[w];
    for (int l = 0; l < nt; ++l) { D.Xprev[(size_t)s * nt + l] = D.X[(size_t)s * nt + l]; D.X[(size_t)s * nt + l] = g[l]; }
    for (int c = 0; c < nc; ++c) D.icf[(size_t)s * nc + c] = g[nt + c];
    D.chi2[s] = tot;
    if (st != 0) D.status[s] = st;
  }
  __syncthreads();
  if (tid < 32) emit_pco(D, s, tid);
}

// psi_coil = G_GC I_C' with the fitted currents (Eq. 7: the coil flux follows the fit).  grid (ceil(N/256), B).
template <typename T>
__global__ void k_coil_flux(Dev<T> D) {
  extern __shared__ unsigned char cf_raw[];
  T *sic = reinterpret_cast<T *>(cf_raw);
  const int s = blockIdx.y;
  for (int c = threadIdx.x; c < D.nc; c += blockDim.x) sic[c] = T(D.icf[(size_t)s * D.nc + c]);
  __syncthreads();
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= D.N) return;
  const T *g = D.ggc_t + n;
  T acc = T(0);
#pragma unroll 4
  for (int c = 0; c < D.nc; ++c) acc = fma(g[(size_t)c * D.N], sic[c], acc);
  D.psi_coil[(size_t)s * D.N + n] = acc;
}

// fitted coil currents -> caller buffer [B][n_coil] real.  grid ceil(B nc / 256).
template <typename T>
__global__ void k_export_ic(Dev<T> D, int B, T *out) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e < B * D.nc) out[e] = T(D.icf[e]);
}

}  // namespace ptefit
