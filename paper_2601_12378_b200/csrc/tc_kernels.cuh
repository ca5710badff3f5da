// tc_kernels.cuh -- operand producers and partial-sum reducers around k_gemm_3xtf32 (tc_gemm.cuh).
// Compact node list: cnode[kc] = grid index of the kc-th node with lim_mask = 1 (padded to a
// multiple of 32 with node 0, whose table columns are zero).  All FP32 (the FP64 path and the
// FFMA mode use fit_kernels.cuh).
#pragma once
#include "common.cuh"

namespace ptefit {

struct TcDev {
  int Kc;                 // padded compact node count (multiple of 32)
  int ntp;                // rows per slice in the response GEMM (8 or 16 >= n_terms)
  int bn_resp;            // N tile of the response GEMM (144 or 256)
  int ld_resp, ld_pbd;    // leading dimensions of the partial buffers
  int rows_resp, rows_pbd;  // padded row counts (multiples of 128)
  int split_resp, split_pbd;
  const int *cnode;       // [Kc]
  const float *rdA, *fdA; // [Kc] R dA and mu0 dA / R of the compact nodes (Eq. 10 factors)
  float *jb_hi, *jb_lo;   // [rows_resp][Kc]
  float *cur_hi, *cur_lo; // [rows_pbd][Kc]
  float *resp_part;       // [split_resp][rows_resp][ld_resp]
  float *pbd_part;        // [split_pbd][rows_pbd][ld_pbd]
};

__device__ __forceinline__ float tf32_rna(float a) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;\n" : "=r"(r) : "f"(a));
  return __uint_as_float(r);
}

// A2: basis columns of Eq. 10 on the compact node list, split for 3xTF32.
// Row s*ntp + l of jb = term l of slice s.  grid (Kc/128, B), block 128.
__global__ void __launch_bounds__(128) k_basis_split(Dev<float> D, TcDev Tc) {
  const int s = blockIdx.y, kc = blockIdx.x * 128 + threadIdx.x;
  if (kc >= Tc.Kc) return;
  const int n = Tc.cnode[kc];
  const float x = D.xn[(size_t)s * D.N + n];
  const int i = n % D.nr;
  const float R = float(D.rmin + i * D.dr);
  const float rdA = R * float(D.dA), fdA = float(kMu0 * D.dA) / R;
  float pw[PTEFIT_MAX_DEG + 1];
  pw[0] = 1.f;
#pragma unroll
  for (int k = 1; k <= PTEFIT_MAX_DEG; ++k) pw[k] = pw[k - 1] * x;
  const size_t row0 = (size_t)s * Tc.ntp;
  for (int l = 0; l < D.nt; ++l) {
    float v;
    if (l < D.npoly) {
      const TermDev t = D.terms[l];
      float a = 0.f, b = 0.f;
#pragma unroll
      for (int k = 0; k <= PTEFIT_MAX_DEG; ++k) { a = (k == t.i) ? pw[k] : a; b = (k == t.N) ? pw[k] : b; }
      v = (x < 0.f) ? 0.f : (a - b) * (t.kind == 0 ? rdA : fdA);
      if (t.family == 1) v = basis_term(D, l, x, rdA, fdA);
    } else {
      v = D.dzc[(size_t)s * D.N + n];
    }
    const float hi = tf32_rna(v);
    Tc.jb_hi[(row0 + l) * Tc.Kc + kc] = hi;
    Tc.jb_lo[(row0 + l) * Tc.Kc + kc] = tf32_rna(v - hi);
  }
}

// resp[s][m][l] = sum_z resp_part[z][s*ntp + l][m]  (fixed order).  grid (ceil(M*nt/256), B).
__global__ void k_resp_reduce(Dev<float> D, TcDev Tc) {
  const int s = blockIdx.y, e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= D.M * D.nt) return;
  const int l = e / D.M, m = e - l * D.M;           // consecutive threads -> consecutive m (coalesced reads)
  const size_t zs = (size_t)Tc.rows_resp * Tc.ld_resp;
  const float *p = Tc.resp_part + ((size_t)s * Tc.ntp + l) * Tc.ld_resp + m;
  float acc = 0.f;
  for (int z = 0; z < Tc.split_resp; ++z) acc += p[z * zs];
  D.resp[((size_t)s * D.M + m) * D.nt + l] = acc;
}

// A5 on the compact node list: I = J_b X by Horner evaluation of the per-slice
// polynomials rdA P(x) + fdA Q(x) (+ delz column), written to cur[s][n] (for the Delta* solve; nodes
// outside the list stay zero) and, split for 3xTF32, to cur_hi/lo[s][kc].  grid (Kc/1024, B), block 256.
__global__ void __launch_bounds__(256) k_current_split(Dev<float> D, TcDev Tc) {
  __shared__ float pco[2 * (PTEFIT_MAX_DEG + 1)];
  __shared__ float xdz;
  const int s = blockIdx.y;
  const double *X = D.X + (size_t)s * D.nt;
  if (threadIdx.x < 2 * (PTEFIT_MAX_DEG + 1)) {
    const int kind = threadIdx.x / (PTEFIT_MAX_DEG + 1), k = threadIdx.x - kind * (PTEFIT_MAX_DEG + 1);
    double c = 0.0;
    for (int l = 0; l < D.npoly; ++l)
      if (D.terms[l].kind == kind && D.terms[l].family == 0) c += X[l] * ((D.terms[l].i == k ? 1.0 : 0.0) - (D.terms[l].N == k ? 1.0 : 0.0));
    pco[threadIdx.x] = float(c);
  }
  if (threadIdx.x == 32) xdz = D.has_delz ? float(X[D.nt - 1]) : 0.f;
  __syncthreads();
  float cp[2 * (PTEFIT_MAX_DEG + 1)];
#pragma unroll
  for (int k = 0; k < 2 * (PTEFIT_MAX_DEG + 1); ++k) cp[k] = pco[k];
  const float xd = xdz;
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const int kq = (blockIdx.x * 4 + u) * blockDim.x + threadIdx.x;
    if (kq >= Tc.Kc) continue;
    const int n = Tc.cnode[kq];
    const float x = D.xn[(size_t)s * D.N + n];
    const float rdA = Tc.rdA[kq], fdA = Tc.fdA[kq];
    float hp = cp[PTEFIT_MAX_DEG], hq = cp[2 * PTEFIT_MAX_DEG + 1];
#pragma unroll
    for (int k = PTEFIT_MAX_DEG - 1; k >= 0; --k) { hp = fmaf(hp, x, cp[k]); hq = fmaf(hq, x, cp[PTEFIT_MAX_DEG + 1 + k]); }
    float v = (x < 0.f) ? 0.f : fmaf(rdA, hp, fdA * hq);
    if (D.nspl) v += spline_current(D, X, x, rdA, fdA);
    if (D.has_delz) v = fmaf(D.dzc[(size_t)s * D.N + n], xd, v);
    if (n != 0) D.cur[(size_t)s * D.N + n] = v;        // padding entries point at node 0
    const float hi = tf32_rna(v);
    Tc.cur_hi[(size_t)s * Tc.Kc + kq] = hi;
    Tc.cur_lo[(size_t)s * Tc.Kc + kq] = tf32_rna(v - hi);
  }
}

// psi_bdry[s][k] = sum_z pbd_part[z][s][k].  grid (ceil(nbnd/256), B).
__global__ void k_pbd_reduce(Dev<float> D, TcDev Tc) {
  const int s = blockIdx.y, k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= D.nbnd) return;
  const size_t zs = (size_t)Tc.rows_pbd * Tc.ld_pbd;
  const float *p = Tc.pbd_part + (size_t)s * Tc.ld_pbd + k;
  float acc = 0.f;
  for (int z = 0; z < Tc.split_pbd; ++z) acc += p[z * zs];
  D.psi_bdry[(size_t)s * D.nbnd + k] = acc;
}

}  // namespace ptefit
