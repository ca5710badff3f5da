// dmma_kernels.cuh -- operand producers and consumers around k_gemm_dmma (dmma_gemm.cuh) for the FP64
// path: basis columns and node currents on the compact node list, fixed-order split-K sums, and the
// transposing kernels that turn the two DSTs of the Delta* solve into plain K-major products.
#pragma once
#include "common.cuh"

namespace ptefit {

struct DmDev {
  int Kc;                    // compact node count padded to a multiple of 16
  int ld_resp, ld_pbd;       // leading dimensions of the partial buffers (even)
  int split_resp, split_pbd;
  int ldS;                   // row length of the DST operands (nzi rounded up to even)
  const int *cnode;          // [Kc] grid index of compact node kc (padding entries: node 0, zero table columns)
  double *jb;                // [B * nt][Kc] basis columns (Eq. 10) of the current flux map
  double *curc;              // [B][Kc] node currents on the compact list
  const double *gp_c;        // [M][Kc]
  const double *gb_c;        // [nbnd][Kc]
  double *resp_part;         // [split_resp][B * nt][ld_resp]
  double *pbd_part;          // [split_pbd][B][ld_pbd]
  const double *S;           // [nzi][ldS] DST-I matrix sin(pi (m+1)(j+1)/(nz-1))
  double *ft, *fh, *gt;      // [B * nri][ldS] transposed right-hand side, mode coefficients, transposed flux
};

// A2: J_b[(s, l)][kc] for all terms l (Eq. 10; the vertical-shift column from dzc).
// grid (Kc/128, B), block 128.
__global__ void __launch_bounds__(128) k_basis_c(Dev<double> D, DmDev Dm) {
  const int s = blockIdx.y, kc = blockIdx.x * 128 + threadIdx.x;
  if (kc >= Dm.Kc) return;
  const int n = Dm.cnode[kc];
  const double x = D.xn[(size_t)s * D.N + n];
  const int i = n % D.nr;
  const double R = D.rmin + i * D.dr;
  const double rdA = R * D.dA, fdA = kMu0 * D.dA / R;
  SplinePt sp{};
  if (D.nspl && x >= 0.0) sp = spline_point(*D.spl, x);
  for (int l = 0; l < D.nt; ++l) {
    double v;
    if (l >= D.npoly) v = D.dzc[(size_t)s * D.N + n];
    else if (D.terms[l].family == 1) v = x < 0.0 ? 0.0 : spline_phi_at(*D.spl, sp, D.terms[l].i) * (D.terms[l].kind == 0 ? rdA : fdA);
    else v = basis_term(D, l, x, rdA, fdA);
    Dm.jb[((size_t)s * D.nt + l) * Dm.Kc + kc] = v;
  }
}

// resp[s][m][l] = sum_z resp_part[z][s nt + l][m] (fixed order).  grid (ceil(M nt/256), B).
__global__ void k_resp_reduce_d(Dev<double> D, DmDev Dm, int B) {
  const int s = blockIdx.y, e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= D.M * D.nt) return;
  const int l = e / D.M, m = e - l * D.M;
  const size_t zs = (size_t)B * D.nt * Dm.ld_resp;
  const double *p = Dm.resp_part + ((size_t)s * D.nt + l) * Dm.ld_resp + m;
  double acc = 0.0;
  for (int z = 0; z < Dm.split_resp; ++z) acc += p[z * zs];
  D.resp[((size_t)s * D.M + m) * D.nt + l] = acc;
}

// A5: I = J_b X from the basis columns already in jb.  Writes cur[s][n] (Delta* solve) and
// curc[s][kc] (boundary product).  grid (Kc/128, B), block 128.
__global__ void __launch_bounds__(128) k_current_c(Dev<double> D, DmDev Dm) {
  const int s = blockIdx.y, kc = blockIdx.x * 128 + threadIdx.x;
  if (kc >= Dm.Kc) return;
  const double *X = D.X + (size_t)s * D.nt;
  double acc = 0.0;
  for (int l = 0; l < D.nt; ++l) acc = fma(Dm.jb[((size_t)s * D.nt + l) * Dm.Kc + kc], X[l], acc);
  const int n = Dm.cnode[kc];
  if (n != 0) D.cur[(size_t)s * D.N + n] = acc;
  Dm.curc[(size_t)s * Dm.Kc + kc] = n != 0 ? acc : 0.0;
}

// psi_bdry[s][k] = sum_z pbd_part[z][s][k].  grid (ceil(nbnd/256), B).
__global__ void k_pbd_reduce_d(Dev<double> D, DmDev Dm, int B) {
  const int s = blockIdx.y, k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= D.nbnd) return;
  const size_t zs = (size_t)B * Dm.ld_pbd;
  const double *p = Dm.pbd_part + (size_t)s * Dm.ld_pbd + k;
  double acc = 0.0;
  for (int z = 0; z < Dm.split_pbd; ++z) acc += p[z * zs];
  D.psi_bdry[(size_t)s * D.nbnd + k] = acc;
}

// Right-hand side -mu0 R I / dA with the Dirichlet data moved over, written
// transposed: ft[(s, i-1)][j-1], so that the DST along Z is a K-major product.
// grid (ceil(nri/32), ceil(nzi/32), B), block (32, 8).
__global__ void __launch_bounds__(256) k_rhs_t(Dev<double> D, DmDev Dm, const double *__restrict__ cur, const double *__restrict__ pbd) {
  __shared__ double tile[32][33];
  const int s = blockIdx.z, i0 = 1 + blockIdx.x * 32, j0 = 1 + blockIdx.y * 32;
  const int nr = D.nr, nri = D.nri, nzi = D.nzi;
  const double *I = cur + (size_t)s * D.N;
  const double *pb = pbd + (size_t)s * D.nbnd;      // bottom[nr], top[nr], left[nzi], right[nzi]
  const double cz = 1.0 / (D.dz * D.dz);
  for (int r = threadIdx.y; r < 32; r += 8) {
    const int j = j0 + r, i = i0 + threadIdx.x;
    double v = 0.0;
    if (j <= nzi && i <= nri) {
      const double R = D.rmin + i * D.dr;
      v = (-kMu0 * R / D.dA) * I[j * nr + i];
      if (i == 1) v -= ((1.0 + D.dr / (2.0 * R)) / (D.dr * D.dr)) * pb[2 * nr + j - 1];
      if (i == nri) v -= ((1.0 - D.dr / (2.0 * R)) / (D.dr * D.dr)) * pb[2 * nr + nzi + j - 1];
      if (j == 1) v -= cz * pb[i];
      if (j == nzi) v -= cz * pb[nr + i];
    }
    tile[r][threadIdx.x] = v;
  }
  __syncthreads();
  for (int r = threadIdx.y; r < 32; r += 8) {
    const int i = i0 + r, j = j0 + threadIdx.x;
    if (i <= nri && j <= nzi) Dm.ft[((size_t)s * nri + i - 1) * Dm.ldS + j - 1] = tile[threadIdx.x][r];
  }
}

// Thomas sweeps along R in FP64, one thread per (slice, mode), in place on fh[(s, i)][m] (row length ldS);
// the forward-sweep values are kept in ytmp.  grid (ceil(nzi/128), B), block 128.
__global__ void k_tridiag_ld(Dev<double> D, DmDev Dm) {
  const int s = blockIdx.y, mm = blockIdx.x * blockDim.x + threadIdx.x;
  if (mm >= D.nzi) return;
  const int nri = D.nri, nzi = D.nzi, ld = Dm.ldS;
  double *fh = Dm.fh + (size_t)s * nri * ld;
  double *y = D.ytmp + (size_t)s * nri * nzi;
  double prev = 0.0;
  for (int i = 0; i < nri; ++i) {
    const double v = fh[(size_t)i * ld + mm] - D.tri_w[(size_t)i * nzi + mm] * prev;
    y[(size_t)i * nzi + mm] = v;
    prev = v;
  }
  double x = 0.0;
  for (int i = nri - 1; i >= 0; --i) {
    x = (y[(size_t)i * nzi + mm] - D.tri_ce[i] * x) * D.tri_invb[(size_t)i * nzi + mm];
    fh[(size_t)i * ld + mm] = x;
  }
}

// Interior nodes: psi[s][j][i] = old + relax (gt[(s, i-1)][j-1] + psi_coil - old); gt already carries the
// 2/(nz-1) normalisation of the inverse DST.  grid (ceil(nri/32), ceil(nzi/32), B), block (32, 8).
__global__ void __launch_bounds__(256) k_total_t(Dev<double> D, DmDev Dm, double *__restrict__ psi, int use_relax, int add_coil) {
  __shared__ double tile[32][33];
  if (!psi) psi = reinterpret_cast<double *>(D.ca->psi);
  const int s = blockIdx.z, i0 = 1 + blockIdx.x * 32, j0 = 1 + blockIdx.y * 32;
  const int nr = D.nr, nri = D.nri, nzi = D.nzi;
  for (int r = threadIdx.y; r < 32; r += 8) {
    const int i = i0 + r, j = j0 + threadIdx.x;
    tile[r][threadIdx.x] = (i <= nri && j <= nzi) ? Dm.gt[((size_t)s * nri + i - 1) * Dm.ldS + j - 1] : 0.0;
  }
  __syncthreads();
  double *p = psi + (size_t)s * D.N;
  const double *pc = D.psi_coil + (size_t)s * D.N;
  for (int r = threadIdx.y; r < 32; r += 8) {
    const int j = j0 + r, i = i0 + threadIdx.x;
    if (j <= nzi && i <= nri) {
      double v = tile[threadIdx.x][r];
      if (add_coil) v += pc[j * nr + i];
      if (use_relax) { const double old = p[j * nr + i]; v = old + D.relax * (v - old); }
      p[j * nr + i] = v;
    }
  }
}

}  // namespace ptefit
