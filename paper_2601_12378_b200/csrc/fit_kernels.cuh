// fit_kernels.cuh -- once-per-call setup, basis/response contraction, least squares, current.
// v1: plain FMA kernels (correctness first); the tensor-core contractions replace
// k_response / k_boundary.
#pragma once
#include "common.cuh"

namespace ptefit {

// A0 / A0': d = b - G_C I_C (Eq. 2/6) and psi_coil = G_GC I_C; resets state (keep_x: not the coefficients).
// Each block handles SETUP_S slices of 256 nodes, so that a table value read once feeds SETUP_S products
// (the coil -> grid table is re-read from L2 for every slice otherwise).
// grid (ceil(N/256), ceil(B/SETUP_S)), block 256, dyn smem SETUP_S * nc * sizeof(T).
constexpr int SETUP_S = 8;
template <typename T>
__global__ void __launch_bounds__(256) k_setup(Dev<T> D, const T *__restrict__ b, const T *__restrict__ ic, int B, int keep_x) {
  extern __shared__ unsigned char smem_raw[];
  T *sic = reinterpret_cast<T *>(smem_raw);                 // [SETUP_S][nc]
  const int s0 = blockIdx.y * SETUP_S, ns = min(SETUP_S, B - s0);
  if (!b) { b = reinterpret_cast<const T *>(D.ca->b); ic = reinterpret_cast<const T *>(D.ca->ic); }   // graph replay: caller pointers from the argument block
  for (int e = threadIdx.x; e < SETUP_S * D.nc; e += blockDim.x) {
    const int q = e / D.nc, c = e - q * D.nc;
    sic[e] = q < ns ? ic[(size_t)(s0 + q) * D.nc + c] : T(0);
  }
  __syncthreads();
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n < D.N) {
    const T *g = D.ggc_t + n;                       // transposed table [n_c][N]: coalesced over nodes
    T acc[SETUP_S];
#pragma unroll
    for (int q = 0; q < SETUP_S; ++q) acc[q] = T(0);
#pragma unroll 2
    for (int c = 0; c < D.nc; ++c) {
      const T gv = g[(size_t)c * D.N];
#pragma unroll
      for (int q = 0; q < SETUP_S; ++q) acc[q] = fma(gv, sic[q * D.nc + c], acc[q]);
    }
#pragma unroll
    for (int q = 0; q < SETUP_S; ++q)
      if (q < ns) D.psi_coil[(size_t)(s0 + q) * D.N + n] = acc[q];
  }
  for (int q = 0; q < ns; ++q) {
    const int s = s0 + q;
    const T *sq = sic + q * D.nc;
    for (int m = n; m < D.M; m += gridDim.x * blockDim.x) {       // M may exceed the node count of a small grid
      // FP64 accumulation: b and G_C I_C nearly cancel when the coil signal dominates the plasma signal, and an
      // FP32 sum of n_c terms would leave d with a relative error of ~1e-6 |G_C I_C| / |d|
      const T *g = D.gc + (size_t)m * D.nc;
      double acc = 0.0;
      for (int c = 0; c < D.nc; ++c) acc = fma((double)g[c], (double)sq[c], acc);
      D.dred[(size_t)s * D.M + m] = D.fit_coils ? b[(size_t)s * D.M + m] : T((double)b[(size_t)s * D.M + m] - acc);   // Eq. 7 fits b itself
    }
    if (D.fit_coils)
      for (int c = n; c < D.nc; c += gridDim.x * blockDim.x) {
        const double v = (double)ic[(size_t)s * D.nc + c];
        D.icm[(size_t)s * D.nc + c] = v; D.icf[(size_t)s * D.nc + c] = v;
      }
    // a warm start keeps the coefficients of the handle's previous call: they seed the vertical-shift column
    if (n < D.nt && !keep_x) { D.X[(size_t)s * D.nt + n] = 0.0; D.Xprev[(size_t)s * D.nt + n] = 0.0; }
    if (n == 0) { D.status[s] = 0; D.chi2[s] = 0.0; }
  }
}

// O2 cold start (paper silent): xn = ((R-Rc)/a)^2 + ((Z-Zc)/b)^2 where < 1 and
// inside the limiter mask, else -1.  grid (ceil(N/256), B).
template <typename T>
__global__ void k_cold_start(Dev<T> D) {
  const int s = blockIdx.y;
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= D.N) return;
  const int j = n / D.nr, i = n - j * D.nr;
  const double R = D.rmin + i * D.dr, Z = D.zmin + j * D.dz;
  const double u = (R - D.cold_rc) / D.cold_a, v = (Z - D.cold_zc) / D.cold_b;
  const double x = u * u + v * v;
  D.xn[(size_t)s * D.N + n] = (x < 1.0 && D.lim_mask[n]) ? T(x) : T(-1);
}

// Vertical-shift column (O4b): dzc[n] = -(I'[n+nr] - I'[n-nr]) / (2 dZ) with
// I' = J_b(xn) X over the polynomial terms, X = the coefficients of the previous fit (D.X is
// only overwritten by k_lsq, which runs after this kernel).  grid (ceil(N/256), B).
template <typename T>
__global__ void k_delz_column(Dev<T> D) {
  const int s = blockIdx.y;
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= D.N) return;
  const int j = n / D.nr, i = n - j * D.nr;
  T out = T(0);
  if (j >= 1 && j <= D.nz - 2 && i >= 1 && i <= D.nr - 2) {
    const T R = T(D.rmin + i * D.dr);
    const T rdA = R * T(D.dA), fdA = T(kMu0 * D.dA) / R;
    const T *x = D.xn + (size_t)s * D.N;
    const double *Xp = D.X + (size_t)s * D.nt;
    T up = T(0), dn = T(0);
    for (int l = 0; l < D.npoly; ++l) {
      const T c = T(Xp[l]);
      up = fma(basis_term(D, l, x[n + D.nr], rdA, fdA), c, up);
      dn = fma(basis_term(D, l, x[n - D.nr], rdA, fdA), c, dn);
    }
    out = -(up - dn) * T(0.5 / D.dz);
  }
  D.dzc[(size_t)s * D.N + n] = out;
}

// A2+A3: resp[s][m][l] = sum_n G_P[m][n] J_b[s][n][l]  (Eq. 6), J_b evaluated on
// the fly from xn (Eq. 10).  grid (ceil(M/MT), B), block RESP_THREADS; each block: MT rows.
constexpr int RESP_THREADS = 256;
constexpr int RESP_MT = 4;
template <typename T, int NT>
__global__ void __launch_bounds__(RESP_THREADS) k_response(Dev<T> D) {
  const int s = blockIdx.y;
  const int m0 = blockIdx.x * RESP_MT;
  const T *x = D.xn + (size_t)s * D.N;
  const T *dzc = D.dzc + (size_t)s * D.N;
  T acc[RESP_MT][NT];
#pragma unroll
  for (int a = 0; a < RESP_MT; ++a)
#pragma unroll
    for (int l = 0; l < NT; ++l) acc[a][l] = T(0);
  for (int n = threadIdx.x; n < D.N; n += RESP_THREADS) {
    const T xv = x[n];
    const T dz = D.has_delz ? dzc[n] : T(0);
    if (xv < T(0) && dz == T(0)) continue;
    const int i = n % D.nr;
    const T R = T(D.rmin + i * D.dr);
    const T rdA = R * T(D.dA), fdA = T(kMu0 * D.dA) / R;
    T bv[NT];
#pragma unroll
    for (int l = 0; l < NT; ++l) bv[l] = (l < D.npoly) ? basis_term(D, l, xv, rdA, fdA) : dz;
#pragma unroll
    for (int a = 0; a < RESP_MT; ++a) {
      const int m = min(m0 + a, D.M - 1);
      const T g = D.gp[(size_t)m * D.N + n];
#pragma unroll
      for (int l = 0; l < NT; ++l) acc[a][l] = fma(g, bv[l], acc[a][l]);
    }
  }
  __shared__ T red[RESP_THREADS / 32][RESP_MT * NT];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int a = 0; a < RESP_MT; ++a)
#pragma unroll
    for (int l = 0; l < NT; ++l) {
      T v = warp_sum(acc[a][l]);
      if (lane == 0) red[w][a * NT + l] = v;
    }
  __syncthreads();
  if (threadIdx.x < RESP_MT * NT) {
    T v = T(0);
    for (int k = 0; k < RESP_THREADS / 32; ++k) v += red[k][threadIdx.x];
    const int a = threadIdx.x / NT, l = threadIdx.x - a * NT;
    if (m0 + a < D.M && l < D.nt) D.resp[((size_t)s * D.M + m0 + a) * D.nt + l] = v;
  }
}

// A4: least squares by normal equations + Cholesky in FP64 registers, column
// equilibration and Tikhonov term per DESIGN.md reading O5.  One warp per slice.
// grid ceil(B/4), block 128.
template <typename T, int NT>
__global__ void __launch_bounds__(128) k_lsq(Dev<T> D, int B) {
  const int s = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (s >= B) return;
  constexpr int nt = NT;                       // compile-time so that A, g, X stay in registers
  const T *resp = D.resp + (size_t)s * D.M * nt;
  const T *d = D.dred + (size_t)s * D.M;
  constexpr int NA = NT * (NT + 1) / 2;
  // the sticky status and the previous coefficients are only needed at the very end: load them now
  const int status_in = D.status[s];
  double xold = 0.0;
  if (lane < nt) xold = D.X[(size_t)s * nt + lane];
  double A[NA], g[NT];
#pragma unroll
  for (int k = 0; k < NA; ++k) A[k] = 0.0;
#pragma unroll
  for (int k = 0; k < NT; ++k) g[k] = 0.0;
  bool finite = true;
  for (int m = lane; m < D.M; m += 32) {
    const double w = D.inv_sigma[m];
    const double y = (double)d[m] * w;
    double r[NT];
    #pragma unroll
    for (int l = 0; l < nt; ++l) { r[l] = (double)resp[m * nt + l] * w; finite &= isfinite(r[l]); }
    finite &= isfinite(y);
    int k = 0;
    #pragma unroll
    for (int l = 0; l < nt; ++l) {
      g[l] = fma(r[l], y, g[l]);
      #pragma unroll
      for (int q = 0; q <= l; ++q, ++k) A[k] = fma(r[l], r[q], A[k]);
    }
  }
  const int na = nt * (nt + 1) / 2;
  #pragma unroll
  for (int k = 0; k < na; ++k) A[k] = warp_sum(A[k]);
  #pragma unroll
  for (int l = 0; l < nt; ++l) g[l] = warp_sum(g[l]);
  finite = __all_sync(0xffffffffu, finite);
  double X[NT];
  int st = 0;
  // every lane runs the tiny factorisation redundantly (no divergence, no broadcast needed)
  double sc[NT];
  bool any = false;
  #pragma unroll
  for (int l = 0; l < nt; ++l) { sc[l] = sqrt(A[l * (l + 1) / 2 + l]); any |= sc[l] > 0.0; }
  double isc[NT];                              // reciprocal scales: one division per column instead of one per entry
  #pragma unroll
  for (int l = 0; l < nt; ++l) isc[l] = sc[l] > 0.0 ? 1.0 / sc[l] : 0.0;
  if (!finite) st = 2; else if (!any) st = 3;
  const double reg = D.lambda_reg * D.lambda_reg * (double)D.M;
  // scaled matrix (unit diagonal + reg); dropped columns (sc = 0) become identity rows
  {
    int k = 0;
    #pragma unroll
    for (int l = 0; l < nt; ++l)
      #pragma unroll
      for (int q = 0; q <= l; ++q, ++k) {
        if (sc[l] > 0.0 && sc[q] > 0.0) A[k] = A[k] * (isc[l] * isc[q]) + (l == q ? reg : 0.0);
        else A[k] = (l == q) ? 1.0 : 0.0;
      }
    #pragma unroll
    for (int l = 0; l < nt; ++l) g[l] = g[l] * isc[l];
  }
  // Cholesky A = L L^T in place (row-packed lower triangle)
  double first_piv = 0.0;
  double idg[NT];                              // 1 / L_ll
  #pragma unroll
  for (int l = 0; l < nt; ++l) idg[l] = 0.0;
  #pragma unroll
  for (int l = 0; l < nt; ++l) {
    if (st != 0) break;
    #pragma unroll
    for (int q = 0; q <= l; ++q) {
      double v = A[l * (l + 1) / 2 + q];
      #pragma unroll
      for (int p = 0; p < q; ++p) v -= A[l * (l + 1) / 2 + p] * A[q * (q + 1) / 2 + p];
      if (q == l) {
        if (l == 0) first_piv = v;
        if (!(v > 1e-13 * first_piv) || !(v > 0.0)) { st = 3; break; }
        idg[l] = rsqrt(v);
        A[l * (l + 1) / 2 + l] = v * idg[l];
      } else {
        A[l * (l + 1) / 2 + q] = v * idg[q];
      }
    }
  }
  #pragma unroll
  for (int l = 0; l < nt; ++l) X[l] = 0.0;
  if (st == 0) {
    #pragma unroll
    for (int l = 0; l < nt; ++l) {           // L z = g
      double v = g[l];
      #pragma unroll
      for (int p = 0; p < l; ++p) v -= A[l * (l + 1) / 2 + p] * X[p];
      X[l] = v * idg[l];
    }
    #pragma unroll
    for (int l = nt - 1; l >= 0; --l) {      // L^T x = z
      double v = X[l];
      #pragma unroll
      for (int p = l + 1; p < nt; ++p) v -= A[p * (p + 1) / 2 + l] * X[p];
      X[l] = v * idg[l];
    }
    #pragma unroll
    for (int l = 0; l < nt; ++l) X[l] = X[l] * isc[l];
  }
  // chi^2 over the measurement rows
  double c2 = 0.0;
  for (int m = lane; m < D.M; m += 32) {
    double rsum = -(double)d[m];
    #pragma unroll
    for (int l = 0; l < nt; ++l) rsum = fma((double)resp[m * nt + l], X[l], rsum);
    rsum *= D.inv_sigma[m];
    c2 = fma(rsum, rsum, c2);
  }
  c2 = warp_sum(c2);
  if (status_in == 0) {                        // status is sticky: a failed slice keeps its outputs
    if (lane < nt) D.Xprev[(size_t)s * nt + lane] = xold;
    if (lane == 0) {
      #pragma unroll
      for (int l = 0; l < nt; ++l) D.X[(size_t)s * nt + l] = X[l];
      D.chi2[s] = c2;
      if (st != 0) D.status[s] = st;
    }
  }
  emit_pco(D, s, lane);
}

// A4, second driver: modified Gram-Schmidt QR ("Gram-Schmidt QR ... stable, slower") of the
// stacked, column-equilibrated, Tikhonov-augmented matrix [W R S^-1 ; lambda sqrt(M) I] in FP64, one warp
// per slice, matrix in shared memory: (M + nt) rows x (nt + 1) columns (last column = right-hand side).
// Same scaling, regularisation, chi^2 and status rules as k_lsq.  grid B, block 32,
// dyn smem ((M + nt) (nt + 1) + nt (nt + 1) + nt) doubles.
template <typename T>
__global__ void __launch_bounds__(32) k_lsq_mgs(Dev<T> D, int B) {
  extern __shared__ __align__(16) unsigned char mgs_raw[];
  const int s = blockIdx.x, lane = threadIdx.x;
  if (s >= B) return;
  const int M = D.M, nt = D.nt, rows = M + nt, ld = nt + 1;
  double *A = reinterpret_cast<double *>(mgs_raw);     // [rows][ld]
  double *Rm = A + (size_t)rows * ld;                    // [nt][ld] upper triangle + transformed rhs
  double *sc = Rm + nt * ld;                             // [nt] column scales
  const T *resp = D.resp + (size_t)s * M * nt;
  const T *d = D.dred + (size_t)s * M;
  bool finite = true;
  for (int m = lane; m < M; m += 32) {
    const double w = D.inv_sigma[m];
    for (int l = 0; l < nt; ++l) { const double v = (double)resp[m * nt + l] * w; A[m * ld + l] = v; finite &= isfinite(v); }
    const double y = (double)d[m] * w;
    A[m * ld + nt] = y;
    finite &= isfinite(y);
  }
  finite = __all_sync(0xffffffffu, finite);
  __syncwarp();
  bool any = false;
  for (int l = 0; l < nt; ++l) {
    double q = 0.0;
    for (int m = lane; m < M; m += 32) q = fma(A[m * ld + l], A[m * ld + l], q);
    q = sqrt(warp_sum(q));
    if (lane == 0) sc[l] = q;
    any |= q > 0.0;
  }
  __syncwarp();
  int st = !finite ? 2 : (!any ? 3 : 0);
  const double reg = D.lambda_reg * sqrt((double)M);
  for (int m = lane; m < M; m += 32)
    for (int l = 0; l < nt; ++l) A[m * ld + l] = sc[l] > 0.0 ? A[m * ld + l] / sc[l] : 0.0;
  for (int e = lane; e < nt * ld; e += 32) {             // regularisation rows; a dropped column gets a unit pivot
    const int r = e / ld, l = e - r * ld;
    A[(M + r) * ld + l] = (l == r) ? (sc[r] > 0.0 ? reg : 1.0) : 0.0;
  }
  __syncwarp();
  double r11 = 0.0;
  for (int l = 0; l < nt && st == 0; ++l) {
    double q = 0.0;
    for (int r = lane; r < rows; r += 32) q = fma(A[r * ld + l], A[r * ld + l], q);
    const double rll = sqrt(warp_sum(q));
    if (l == 0) r11 = rll;
    if (!(rll > 1e-13 * r11) || !(rll > 0.0)) { st = 3; break; }
    const double inv = 1.0 / rll;
    for (int r = lane; r < rows; r += 32) A[r * ld + l] *= inv;
    if (lane == 0) Rm[l * ld + l] = rll;
    __syncwarp();
    for (int p = l + 1; p <= nt; ++p) {
      double dot = 0.0;
      for (int r = lane; r < rows; r += 32) dot = fma(A[r * ld + l], A[r * ld + p], dot);
      dot = warp_sum(dot);
      for (int r = lane; r < rows; r += 32) A[r * ld + p] = fma(-dot, A[r * ld + l], A[r * ld + p]);
      if (lane == 0) Rm[l * ld + p] = dot;
    }
    __syncwarp();
  }
  // back substitution R x = Q^T y (every lane redundantly, nt <= 16), then undo the column scaling
  double X[PTEFIT_MAX_TERMS];
  for (int l = 0; l < PTEFIT_MAX_TERMS; ++l) X[l] = 0.0;
  if (st == 0) {
    for (int l = nt - 1; l >= 0; --l) {
      double v = Rm[l * ld + nt];
      for (int p = l + 1; p < nt; ++p) v -= Rm[l * ld + p] * X[p];
      X[l] = v / Rm[l * ld + l];
    }
    for (int l = 0; l < nt; ++l) X[l] = sc[l] > 0.0 ? X[l] / sc[l] : 0.0;
  }
  double c2 = 0.0;
  for (int m = lane; m < M; m += 32) {
    double rsum = -(double)d[m];
    for (int l = 0; l < nt; ++l) rsum = fma((double)resp[m * nt + l], X[l], rsum);
    rsum *= D.inv_sigma[m];
    c2 = fma(rsum, rsum, c2);
  }
  c2 = warp_sum(c2);
  if (lane == 0 && D.status[s] == 0) {
    for (int l = 0; l < nt; ++l) { D.Xprev[(size_t)s * nt + l] = D.X[(size_t)s * nt + l]; D.X[(size_t)s * nt + l] = X[l]; }
    D.chi2[s] = c2;
    if (st != 0) D.status[s] = st;
  }
  emit_pco(D, s, lane);
}

// A5: node currents I = J_b X in amperes.  grid (ceil(N/256), B).
template <typename T>
__global__ void k_current(Dev<T> D) {
  const int s = blockIdx.y;
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= D.N) return;
  const T xv = D.xn[(size_t)s * D.N + n];
  const int i = n % D.nr;
  const T R = T(D.rmin + i * D.dr);
  const T rdA = R * T(D.dA), fdA = T(kMu0 * D.dA) / R;
  const double *X = D.X + (size_t)s * D.nt;
  T acc = T(0);
  for (int l = 0; l < D.npoly; ++l) acc = fma(basis_term(D, l, xv, rdA, fdA), T(X[l]), acc);
  if (D.has_delz) acc = fma(D.dzc[(size_t)s * D.N + n], T(X[D.nt - 1]), acc);
  D.cur[(size_t)s * D.N + n] = acc;
}

// A6: psi_bdry[s][k] = sum_n G_B[k][n] I[s][n] (Dirichlet data of the Delta* solve; named by
// north_star, PAPER.md:120 says only "Dirichlet").  grid (ceil(nbnd/KT), ceil(B/ST)).
constexpr int BND_THREADS = 256;
constexpr int BND_KT = 8;
constexpr int BND_ST = 4;
template <typename T>
__global__ void __launch_bounds__(BND_THREADS) k_boundary(Dev<T> D, int B) {
  const int k0 = blockIdx.x * BND_KT, s0 = blockIdx.y * BND_ST;
  T acc[BND_KT][BND_ST];
#pragma unroll
  for (int a = 0; a < BND_KT; ++a)
#pragma unroll
    for (int c = 0; c < BND_ST; ++c) acc[a][c] = T(0);
  for (int n = threadIdx.x; n < D.N; n += BND_THREADS) {
    T cv[BND_ST];
    bool any = false;
#pragma unroll
    for (int c = 0; c < BND_ST; ++c) {
      const int s = min(s0 + c, B - 1);
      cv[c] = D.cur[(size_t)s * D.N + n];
      any |= cv[c] != T(0);
    }
    if (!any) continue;
#pragma unroll
    for (int a = 0; a < BND_KT; ++a) {
      const int k = min(k0 + a, D.nbnd - 1);
      const T g = D.gb[(size_t)k * D.N + n];
#pragma unroll
      for (int c = 0; c < BND_ST; ++c) acc[a][c] = fma(g, cv[c], acc[a][c]);
    }
  }
  __shared__ T red[BND_THREADS / 32][BND_KT * BND_ST];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int a = 0; a < BND_KT; ++a)
#pragma unroll
    for (int c = 0; c < BND_ST; ++c) {
      T v = warp_sum(acc[a][c]);
      if (lane == 0) red[w][a * BND_ST + c] = v;
    }
  __syncthreads();
  if (threadIdx.x < BND_KT * BND_ST) {
    T v = T(0);
    for (int q = 0; q < BND_THREADS / 32; ++q) v += red[q][threadIdx.x];
    const int a = threadIdx.x / BND_ST, c = threadIdx.x - a * BND_ST;
    if (k0 + a < D.nbnd && s0 + c < B) D.psi_bdry[(size_t)(s0 + c) * D.nbnd + k0 + a] = v;
  }
}

}  // namespace ptefit
