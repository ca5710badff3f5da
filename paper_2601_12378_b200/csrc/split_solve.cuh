// split_solve.cuh -- the Delta* solve (A7) of a whole batch as two batched DST products on the
// tensor cores (k_gemm_3xtf32) around a massively parallel FP64 tridiagonal kernel, instead of one
// CTA per slice:
//   k_rhs_t     rhs of Eq. 1 with the Dirichlet data moved over, written
//               transposed [(s, i)][j] and split hi / lo for 3xTF32
//   GEMM 1      Y[(s, i)][m] = sum_j rhs[(s, i)][j] sin(pi j m / Nz)          (DST-I in Z)
//   k_thomas_t  one thread per (slice, mode): FP64 Thomas sweeps along R
//   GEMM 2      psi_pl[s][j][i] = 2/Nz sum_m X[(s, i)][m] sin(pi j m / Nz)     (transposed store)
// FP32 only; grids with N_Z - 2 padded to P = 128 or 256.
#pragma once
#include "common.cuh"
#include "tc_kernels.cuh"

namespace ptefit {

struct SplitDev {
  int RS, P, rows;          // rows per slice (N_R-2 padded to 32), padded transform length, total rows (multiple of 128)
  float *a_hi, *a_lo;       // [rows][P]  transposed right-hand side
  float *y1;                // [rows][P]  after the forward DST
  float *x_hi, *x_lo;       // [rows][P]  after the tridiagonal solves
  float *psi_pl;            // [B][N]     plasma flux on the grid (interior nodes)
};

// grid (RS/32, P/32, B), block (32, 8).
__global__ void __launch_bounds__(256) k_rhs_t(Dev<float> D, SplitDev S, const float *__restrict__ cur_all,
                                               const float *__restrict__ pbd_all) {
  __shared__ float tile[32][33];
  const int s = blockIdx.z, it = blockIdx.x * 32, jt = blockIdx.y * 32;
  const int nr = D.nr, nri = D.nri, nzi = D.nzi;
  const float *I = cur_all + (size_t)s * D.N;
  const float *pb = pbd_all + (size_t)s * D.nbnd;          // bottom[nr], top[nr], left[nzi], right[nzi]
  const float cz = float(1.0 / (D.dz * D.dz));
  const int ii = it + threadIdx.x, i = ii + 1;              // grid column of this thread while reading
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int jj = jt + threadIdx.y + 8 * k, j = jj + 1;
    float v = 0.f;
    if (ii < nri && jj < nzi) {
      const double R = D.rmin + i * D.dr;
      v = float(-kMu0 * R / D.dA) * I[j * nr + i];
      if (i == 1) v -= float((1.0 + D.dr / (2.0 * R)) / (D.dr * D.dr)) * pb[2 * nr + jj];
      if (i == nri) v -= float((1.0 - D.dr / (2.0 * R)) / (D.dr * D.dr)) * pb[2 * nr + nzi + jj];
      if (j == 1) v -= cz * pb[i];
      if (j == nzi) v -= cz * pb[nr + i];
    }
    tile[threadIdx.y + 8 * k][threadIdx.x] = v;            // tile[jj local][ii local]
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int il = threadIdx.y + 8 * k;                     // local row index i of the output
    const float v = tile[threadIdx.x][il];                  // [jj local = tx][ii local]
    const size_t o = ((size_t)s * S.RS + it + il) * S.P + jt + threadIdx.x;
    const float hi = tf32_rna(v);
    S.a_hi[o] = hi;
    S.a_lo[o] = tf32_rna(v - hi);
  }
}

// grid (ceil(nzi/128), B), block 128: thread = one (slice, mode) system of size nri.
__global__ void __launch_bounds__(128) k_thomas_t(Dev<float> D, SplitDev S) {
  const int s = blockIdx.y, mm = blockIdx.x * blockDim.x + threadIdx.x;
  if (mm >= D.nzi) return;
  const int nri = D.nri, nzi = D.nzi;
  const float *__restrict__ f = S.y1 + (size_t)s * S.RS * S.P + mm;
  double *__restrict__ y = D.ytmp + (size_t)s * nri * nzi + mm;
  const double *__restrict__ tw = D.tri_w + mm;
  const double *__restrict__ tb = D.tri_invb + mm;
  const double *__restrict__ tce = D.tri_ce;
  constexpr int U = 8;
  double prev = 0.0;
  for (int i0 = 0; i0 < nri; i0 += U) {
    double w[U];
    float g[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int i = min(i0 + u, nri - 1);
      w[u] = __ldg(tw + (size_t)i * nzi);
      g[u] = f[(size_t)i * S.P];
    }
#pragma unroll
    for (int u = 0; u < U; ++u)
      if (i0 + u < nri) {
        const double v = fma(-w[u], prev, (double)g[u]);
        y[(size_t)(i0 + u) * nzi] = v;
        prev = v;
      }
  }
  float *__restrict__ xh = S.x_hi + (size_t)s * S.RS * S.P + mm;
  float *__restrict__ xl = S.x_lo + (size_t)s * S.RS * S.P + mm;
  double x = 0.0;
  for (int i0 = nri - 1; i0 >= 0; i0 -= U) {
    double a[U], b[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int i = max(i0 - u, 0);
      const double ib = __ldg(tb + (size_t)i * nzi);
      a[u] = y[(size_t)i * nzi] * ib;
      b[u] = __ldg(tce + i) * ib;
    }
#pragma unroll
    for (int u = 0; u < U; ++u)
      if (i0 - u >= 0) {
        x = fma(-b[u], x, a[u]);
        const float xf = (float)x, hi = tf32_rna(xf);
        xh[(size_t)(i0 - u) * S.P] = hi;
        xl[(size_t)(i0 - u) * S.P] = tf32_rna(xf - hi);
      }
  }
}

}  // namespace ptefit
