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

// resp[s][m][l] = sum_z resp_part[z][s*ntp + l][m]  (fixed order; few splits).  grid (ceil(M*nt/256), B).
__global__ void k_resp_reduce1(Dev<float> D, TcDev Tc) {
  const int s = blockIdx.y, e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= D.M * D.nt) return;
  const int l = e / D.M, m = e - l * D.M;           // consecutive threads -> consecutive m (coalesced reads)
  const size_t zs = (size_t)Tc.rows_resp * Tc.ld_resp;
  const float *p = Tc.resp_part + ((size_t)s * Tc.ntp + l) * Tc.ld_resp + m;
  float acc = 0.f;
  for (int z = 0; z < Tc.split_resp; ++z) acc += p[z * zs];
  D.resp[((size_t)s * D.M + m) * D.nt + l] = acc;
}

// Many splits (small batches): four threads share one output (z = g, g + 4, ...) and
// are combined in a fixed order, so the sum is bit-reproducible.  grid (ceil(M*nt/64), B), block 256.
__global__ void __launch_bounds__(256) k_resp_reduce(Dev<float> D, TcDev Tc) {
  __shared__ float part[4][64];
  const int s = blockIdx.y, o = threadIdx.x & 63, g = threadIdx.x >> 6, e = blockIdx.x * 64 + o;
  const bool live = e < D.M * D.nt;
  const int l = live ? e / D.M : 0, m = live ? e - l * D.M : 0;       // consecutive threads -> consecutive m (coalesced reads)
  const size_t zs = (size_t)Tc.rows_resp * Tc.ld_resp;
  const float *p = Tc.resp_part + ((size_t)s * Tc.ntp + l) * Tc.ld_resp + m;
  float acc = 0.f;
  if (live) {
#pragma unroll 4
    for (int z = g; z < Tc.split_resp; z += 4) acc += p[z * zs];
  }
  part[g][o] = acc;
  __syncthreads();
  if (g == 0 && live) D.resp[((size_t)s * D.M + m) * D.nt + l] = (part[0][o] + part[1][o]) + (part[2][o] + part[3][o]);
}

// A5 on the compact node list: I = J_b X by Horner evaluation of the per-slice
// polynomials rdA P(x) + fdA Q(x) (+ delz column), written to cur[s][n] (for the Delta* solve; nodes
// outside the list stay zero) and, split for 3xTF32, to cur_hi/lo[s][kc].  Four consecutive compact nodes
// per thread (16-byte loads of the node list and factors, 16-byte stores of the split currents).
// grid (ceil(Kc/2048), B), block 256.
__global__ void __launch_bounds__(256) k_current_split(Dev<float> D, TcDev Tc) {
  __shared__ float pco[2 * (PTEFIT_MAX_DEG + 1)];
  const int s = blockIdx.y;
  const double *X = D.X + (size_t)s * D.nt;
  const float *pg = D.pco + (size_t)s * PCO_STRIDE;     // polynomial form of the fitted current profile, written by the fit kernel
  constexpr int MD = PTEFIT_MAX_DEG;
  const bool lowdeg = D.maxdeg <= 4;
  float pp[5], pq[5];
#pragma unroll
  for (int k = 0; k < 5; ++k) { pp[k] = __ldg(pg + k); pq[k] = __ldg(pg + MD + 1 + k); }
  const float xd = __ldg(pg + 2 * (MD + 1));
  if (!lowdeg) {                                        // uniform: high-degree terms read the coefficients from shared memory
    if (threadIdx.x < 2 * (MD + 1)) pco[threadIdx.x] = pg[threadIdx.x];
    __syncthreads();
  }
  const float *xs = D.xn + (size_t)s * D.N, *ds = D.dzc + (size_t)s * D.N;
  float *cs = D.cur + (size_t)s * D.N;
#pragma unroll
  for (int u = 0; u < 2; ++u) {
    const int kq = 4 * ((blockIdx.x * 2 + u) * blockDim.x + threadIdx.x);
    if (kq >= Tc.Kc) continue;
    const int4 n4 = *reinterpret_cast<const int4 *>(Tc.cnode + kq);
    const float4 r4 = *reinterpret_cast<const float4 *>(Tc.rdA + kq), f4 = *reinterpret_cast<const float4 *>(Tc.fdA + kq);
    const int n[4] = {n4.x, n4.y, n4.z, n4.w};
    const float r[4] = {r4.x, r4.y, r4.z, r4.w}, f[4] = {f4.x, f4.y, f4.z, f4.w};
    float x[4], d[4], v[4];
#pragma unroll
    for (int t = 0; t < 4; ++t) { x[t] = xs[n[t]]; d[t] = D.has_delz ? ds[n[t]] : 0.f; }
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      float hp, hq;
      if (lowdeg) {
        hp = pp[4]; hq = pq[4];
#pragma unroll
        for (int k = 3; k >= 0; --k) { hp = fmaf(hp, x[t], pp[k]); hq = fmaf(hq, x[t], pq[k]); }
      } else {
        hp = pco[MD]; hq = pco[2 * MD + 1];
#pragma unroll
        for (int k = MD - 1; k >= 0; --k) { hp = fmaf(hp, x[t], pco[k]); hq = fmaf(hq, x[t], pco[MD + 1 + k]); }
      }
      v[t] = (x[t] < 0.f) ? 0.f : fmaf(r[t], hp, f[t] * hq);
      if (D.nspl) v[t] += spline_current(D, X, x[t], r[t], f[t]);
      v[t] = fmaf(d[t], xd, v[t]);
      if (n[t] != 0) cs[n[t]] = v[t];                  // padding entries point at node 0
      else v[t] = 0.f;
      hi[t] = __float_as_uint(tf32_rna(v[t]));
      lo[t] = __float_as_uint(tf32_rna(v[t] - __uint_as_float(hi[t])));
    }
    *reinterpret_cast<uint4 *>(Tc.cur_hi + (size_t)s * Tc.Kc + kq) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4 *>(Tc.cur_lo + (size_t)s * Tc.Kc + kq) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
  }
}

// psi_bdry[s][k] = sum_z pbd_part[z][s][k], four threads per output as in k_resp_reduce.
// grid (ceil(nbnd/64), B), block 256.
__global__ void __launch_bounds__(256) k_pbd_reduce(Dev<float> D, TcDev Tc) {
  __shared__ float part[4][64];
  const int s = blockIdx.y, o = threadIdx.x & 63, g = threadIdx.x >> 6, k = blockIdx.x * 64 + o;
  const bool live = k < D.nbnd;
  const size_t zs = (size_t)Tc.rows_pbd * Tc.ld_pbd;
  const float *p = Tc.pbd_part + (size_t)s * Tc.ld_pbd + (live ? k : 0);
  float acc = 0.f;
  if (live) {
#pragma unroll 4
    for (int z = g; z < Tc.split_pbd; z += 4) acc += p[z * zs];
  }
  part[g][o] = acc;
  __syncthreads();
  if (g == 0 && live) D.psi_bdry[(size_t)s * D.nbnd + k] = (part[0][o] + part[1][o]) + (part[2][o] + part[3][o]);
}

}  // namespace ptefit
