// search_kernels.cuh -- A1/A9: magnetic axis, X-point candidates, limiter fluxes, boundary flux,
// plasma mask and normalised flux (Sec. II.D; rules per DESIGN.md reading O3).
// One CTA per slice; all fit arithmetic in FP64 on the T-typed flux so that classification
// decisions (det < 0, |x*| <= 1/2) are taken in the same precision on both code paths.
#pragma once
#include "common.cuh"

namespace ptefit {

constexpr int SEARCH_THREADS = 512;

struct Fit { double det, xs, ys, ps; };

// 3x3 least-squares quadratic with the pre-inverted normal equations: integer
// weight table, index units.  p points at the centre node, ld = nr.
struct Quad { double cx, cy, cxx, cyy, cxy, c0, det; };
template <typename T>
__device__ __forceinline__ Quad quad_coef(const T *__restrict__ p, int ld) {
  const double a = p[-ld - 1], b = p[-ld], c = p[-ld + 1];
  const double d = p[-1], e = p[0], f = p[1];
  const double g = p[ld - 1], h = p[ld], k = p[ld + 1];
  Quad q;
  q.cx = ((c + f + k) - (a + d + g)) * (1.0 / 6.0);
  q.cy = ((g + h + k) - (a + b + c)) * (1.0 / 6.0);
  q.cxx = ((a + d + g) - 2.0 * (b + e + h) + (c + f + k)) * (1.0 / 6.0);
  q.cyy = ((a + b + c) - 2.0 * (d + e + f) + (g + h + k)) * (1.0 / 6.0);
  q.cxy = (k + a - g - c) * 0.25;
  q.c0 = (5.0 * e + 2.0 * (b + d + f + h) - (a + c + g + k)) * (1.0 / 9.0);
  q.det = 4.0 * q.cxx * q.cyy - q.cxy * q.cxy;
  return q;
}
__device__ __forceinline__ Fit quad_finish(const Quad &q) {
  Fit o;
  o.det = q.det;
  o.xs = -(2.0 * q.cyy * q.cx - q.cxy * q.cy) / q.det;
  o.ys = -(2.0 * q.cxx * q.cy - q.cxy * q.cx) / q.det;
  o.ps = q.c0 + 0.5 * (q.cx * o.xs + q.cy * o.ys);
  return o;
}
template <typename T>
__device__ __forceinline__ Fit quad_fit(const T *__restrict__ p, int ld) {
  return quad_finish(quad_coef<T>(p, ld));
}

struct ArgMax { double v; int n; };
__device__ __forceinline__ ArgMax better(ArgMax a, ArgMax b) {   // larger v, tie -> smaller n
  return (b.v > a.v || (b.v == a.v && b.n < a.n)) ? b : a;
}
__device__ __forceinline__ ArgMax block_argmax(ArgMax a, ArgMax *sh) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    ArgMax b;
    b.v = __shfl_xor_sync(0xffffffffu, a.v, o);
    b.n = __shfl_xor_sync(0xffffffffu, a.n, o);
    a = better(a, b);
  }
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  __syncthreads();
  if (lane == 0) sh[w] = a;
  __syncthreads();
  ArgMax r = sh[0];
  const int nw = (blockDim.x + 31) >> 5;
  for (int k = 1; k < nw; ++k) r = better(r, sh[k]);
  return r;
}

// Optional shared-memory helpers of search_body (all nullptr / default = plain global-memory path).
template <typename T>
struct SearchOpt {
  const unsigned *lbits = nullptr;   // bit-packed lim_mask in shared memory (bit n&31 of word n>>5)
  const unsigned *xbits = nullptr;   // bit-packed xpt_mask
  bool have_am = false;              // pass 0 done by the caller: this thread's partial arg-max + finiteness
  ArgMax am;
  bool bad = false;
  T *local = nullptr;                // per-node output in shared memory (may alias psi)
  const T *pc = nullptr;             // if set: local gets I'(xn) = rdA P(xn) + fdA Q(xn) instead of xn
  const T *rdA = nullptr, *fdA = nullptr;
  const double *Xs = nullptr;        // coefficients of this slice (spline terms of I', if any)
};

// Search of one slice by one CTA (any block size that is a multiple of 32, <= 1024).  Reads
// psi[nz][nr] (global or shared memory), writes xn (normalised flux in the mask, -1 outside) to
// global memory and, if o.local != nullptr, a per-node value to o.local (may alias psi: every
// thread overwrites only nodes it alone reads after the last barrier).  Updates D.so[s],
// D.status[s] (sticky).  All threads of the CTA must call it.

template <typename T>
__device__ void search_body(const Dev<T> &D, int s, const T *psi, T *__restrict__ xn, const SearchOpt<T> &o) {
  const int nth = blockDim.x, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nwarp = nth >> 5;
  const int nr = D.nr, nz = D.nz, N = D.N;
  const double sg = (double)D.ip_sign;
  __shared__ ArgMax sh_am[32];
  __shared__ int sh_flag, sh_ncand, sh_count;
  __shared__ double cR[PTEFIT_MAX_CAND], cZ[PTEFIT_MAX_CAND], cP[PTEFIT_MAX_CAND];
  __shared__ int cN[PTEFIT_MAX_CAND];
  __shared__ SearchOut so;
  if (tid == 0) { sh_flag = 0; sh_ncand = 0; sh_count = 0; }
  __syncthreads();
  // 0. finiteness + 1. axis node: arg-max of s*psi over lim_mask, tie -> smallest n
  ArgMax am; am.v = -INFINITY; am.n = 0x7fffffff;
  bool bad = false;
  if (o.have_am) { am = o.am; bad = o.bad; }
  else {
    for (int j = warp; j < nz; j += nwarp)
      for (int i = lane; i < nr; i += 32) {
        const int n = j * nr + i;
        const double v = (double)psi[n];
        bad |= !isfinite(v);
        const bool lm = o.lbits ? ((o.lbits[n >> 5] >> (n & 31)) & 1u) : D.lim_mask[n];
        if (lm) { ArgMax c; c.v = sg * v; c.n = n; am = better(am, c); }
      }
  }
  if (bad) atomicOr(&sh_flag, 1);
  am = block_argmax(am, sh_am);
  int status = 0;
  if (sh_flag) status = 2;
  double Ra = 0, Za = 0, Pa = 0;
  int ia = -1, ja = -1;
  if (status == 0) {
    ja = am.n / nr; ia = am.n - ja * nr;
    const Fit f = quad_fit(psi + am.n, nr);
    if (!(f.det > 0.0) || fmax(fabs(f.xs), fabs(f.ys)) > 1.0) status = 1;
    Ra = D.rmin + (ia + f.xs) * D.dr; Za = D.zmin + (ja + f.ys) * D.dz; Pa = f.ps;
  }
  // 2. X-point candidates (det H < 0, stationary point inside the half cell, below the axis flux)
  if (status == 0) {
    for (int j = warp + 1; j < nz - 1; j += nwarp)
     for (int i = lane; i < nr - 1; i += 32) {
      if (i == 0) continue;
      const int n = j * nr + i;
      const bool xm = o.xbits ? ((o.xbits[n >> 5] >> (n & 31)) & 1u) : D.xpt_mask[n];
      if (!xm) continue;
      if (sizeof(T) == 4) {
        // FP32 pre-filter with wide margins (the coefficients carry ~1e-4 relative error in FP32):
        // skip nodes whose Hessian determinant is certainly positive or whose stationary point is
        // certainly outside the half cell; everything else is decided below in FP64.
        const T *p = psi + n;
        const float a = p[-nr - 1], b = p[-nr], c = p[-nr + 1], d = p[-1], e = p[0], f = p[1], g = p[nr - 1], hh = p[nr], k = p[nr + 1];
        const float l3 = a + d + g, r3 = c + f + k, m3 = b + e + hh, t3 = a + b + c, u3 = g + hh + k, w3 = d + e + f;
        const float fcx = (r3 - l3) * (1.f / 6.f), fcy = (u3 - t3) * (1.f / 6.f);
        const float fcxx = (l3 - 2.f * m3 + r3) * (1.f / 6.f), fcyy = (t3 - 2.f * w3 + u3) * (1.f / 6.f);
        const float fcxy = (k + a - g - c) * 0.25f;
        const float p1 = 4.f * fcxx * fcyy, p2 = fcxy * fcxy, fdet = p1 - p2, mag = fabsf(p1) + p2;
        if (fdet > 0.02f * mag) continue;
        if (fdet < -0.02f * mag) {
          const float lim = 0.6f * fabsf(fdet);
          const float sx = fabsf(fcyy * fcx) + fabsf(fcxy * fcy), sy = fabsf(fcxx * fcy) + fabsf(fcxy * fcx);
          const float nx = fabsf(2.f * fcyy * fcx - fcxy * fcy), ny = fabsf(2.f * fcxx * fcy - fcxy * fcx);
          if (nx > lim + 0.02f * sx || ny > lim + 0.02f * sy) continue;
        }
      }
      const Quad qc = quad_coef(psi + n, nr);
      if (!(qc.det < 0.0)) continue;
      // division-free pre-test with a margin; the decision itself is taken below on x*, y*
      const double lim = 0.5000001 * fabs(qc.det);
      if (fabs(2.0 * qc.cyy * qc.cx - qc.cxy * qc.cy) > lim || fabs(2.0 * qc.cxx * qc.cy - qc.cxy * qc.cx) > lim) continue;
      const Fit f = quad_finish(qc);
      if (f.det < 0.0 && fabs(f.xs) <= 0.5 && fabs(f.ys) <= 0.5 && sg * f.ps < sg * Pa) {
        const int q = atomicAdd(&sh_ncand, 1);
        if (q < PTEFIT_MAX_CAND) {
          cR[q] = D.rmin + (i + f.xs) * D.dr; cZ[q] = D.zmin + (j + f.ys) * D.dz; cP[q] = f.ps; cN[q] = n;
        }
      }
    }
  }
  __syncthreads();
  const int ncand = sh_ncand;
  if (status == 0 && ncand > PTEFIT_MAX_CAND) status = 4;
  // 3. limiter vertices: bilinear flux, valid iff not behind any candidate as seen from the axis
  ArgMax lm; lm.v = -INFINITY; lm.n = 0x7fffffff;
  if (status == 0) {
    for (int v = tid; v < D.nlim; v += nth) {
      const double lr = D.lim_r[v], lz = D.lim_z[v];
      const double fi = (lr - D.rmin) / D.dr, fj = (lz - D.zmin) / D.dz;
      int i0 = (int)floor(fi), j0 = (int)floor(fj);
      i0 = max(0, min(i0, nr - 2)); j0 = max(0, min(j0, D.nz - 2));
      const double tx = fi - i0, ty = fj - j0;
      const T *p = psi + j0 * nr + i0;
      const double pv = (1.0 - ty) * ((1.0 - tx) * (double)p[0] + tx * (double)p[1]) +
                        ty * ((1.0 - tx) * (double)p[nr] + tx * (double)p[nr + 1]);
      bool valid = true;
      for (int c = 0; c < ncand; ++c)
        valid &= ((lr - cR[c]) * (Ra - cR[c]) + (lz - cZ[c]) * (Za - cZ[c])) >= 0.0;
      if (valid) { ArgMax c; c.v = sg * pv; c.n = v; lm = better(lm, c); }
    }
  }
  lm = block_argmax(lm, sh_am);
  // 4. boundary flux
  double Pb = 0.0;
  if (status == 0) {
    ArgMax bx; bx.v = -INFINITY; bx.n = 0x7fffffff;
    int qbest = -1;
    for (int c = 0; c < ncand; ++c) {
      ArgMax t; t.v = sg * cP[c]; t.n = cN[c];
      if (t.v > bx.v || (t.v == bx.v && t.n < bx.n)) { bx = t; qbest = c; }
    }
    const bool xwins = bx.v > lm.v;
    const double spb = xwins ? bx.v : lm.v;
    if (!isfinite(spb)) status = 1;
    Pb = sg * spb;
    if (tid == 0) {
      so.axis_i = ia; so.axis_j = ja; so.axis_r = Ra; so.axis_z = Za; so.axis_psi = Pa;
      so.n_cand = ncand; so.limited = xwins ? 0 : 1; so.psi_b = Pb;
      if (qbest >= 0) {
        so.xpt_j = cN[qbest] / nr; so.xpt_i = cN[qbest] - so.xpt_j * nr;
        so.xpt_r = cR[qbest]; so.xpt_z = cZ[qbest]; so.xpt_psi = cP[qbest];
      } else {
        so.xpt_i = so.xpt_j = -1; so.xpt_r = so.xpt_z = so.xpt_psi = nan("");
      }
    }
    if (Pb == Pa) status = 1;
  }
  // 5./6. plasma region and normalised flux
  int cnt = 0;
  if (status == 0) {
    const double inv = 1.0 / (Pb - Pa);
    T pco[2 * (PTEFIT_MAX_DEG + 1)];                   // registers: the stores below may alias o.pc for the compiler
#pragma unroll
    for (int k = 0; k < 2 * (PTEFIT_MAX_DEG + 1); ++k) pco[k] = o.pc ? o.pc[k] : T(0);
    for (int j = warp; j < nz; j += nwarp)
     for (int i = lane; i < nr; i += 32) {
      const int n = j * nr + i;
      T out = T(-1);
      const bool lmk = o.lbits ? ((o.lbits[n >> 5] >> (n & 31)) & 1u) : D.lim_mask[n];
      if (lmk) {
        const double v = (double)psi[n];
        if (sg * (v - Pb) > 0.0) {
          bool in = true;
          if (ncand) {
            const double R = D.rmin + i * D.dr, Z = D.zmin + j * D.dz;
            for (int c = 0; c < ncand; ++c)
              in &= ((R - cR[c]) * (Ra - cR[c]) + (Z - cZ[c]) * (Za - cZ[c])) > 0.0;
          }
          if (in) { out = T(fmin(fmax((v - Pa) * inv, 0.0), 1.0)); ++cnt; }
        }
      }
      xn[n] = out;
      if (o.local) {
        T lv = out;
        if (o.pc) {                                   // I'(x) by Horner (fused_solve.cuh, delz column)
          T hp = pco[PTEFIT_MAX_DEG], hq = pco[2 * PTEFIT_MAX_DEG + 1];
#pragma unroll
          for (int k = PTEFIT_MAX_DEG - 1; k >= 0; --k) {
            hp = fma(hp, out, pco[k]);
            hq = fma(hq, out, pco[PTEFIT_MAX_DEG + 1 + k]);
          }
          lv = (out < T(0)) ? T(0) : fma(o.rdA[i], hp, o.fdA[i] * hq);
          if (D.nspl && o.Xs) lv += spline_current(D, o.Xs, out, o.rdA[i], o.fdA[i]);
        }
        o.local[n] = lv;
      }
    }
  } else {
    for (int n = tid; n < N; n += nth) {
      xn[n] = T(-1);
      if (o.local) o.local[n] = o.pc ? T(0) : T(-1);
    }
  }
  if (cnt) atomicAdd(&sh_count, cnt);
  __syncthreads();
  if (status == 0 && sh_count == 0) status = 1;
  if (tid == 0) {
    if (D.status[s] == 0) {
      if (status == 0 || status == 4) D.so[s] = so;
      if (status == 1 || status == 2) { SearchOut z = {}; z.axis_i = ia; z.axis_j = ja; z.xpt_i = z.xpt_j = -1; D.so[s] = z; }
      D.status[s] = status;
    }
  }
}

// grid B, block SEARCH_THREADS.
template <typename T>
__global__ void __launch_bounds__(SEARCH_THREADS) k_search(Dev<T> D, const T *__restrict__ psi_all,
                                                            T *__restrict__ xn_all) {
  const int s = blockIdx.x;
  if (!psi_all) psi_all = reinterpret_cast<const T *>(D.ca->psi);
  SearchOpt<T> o;
  search_body<T>(D, s, psi_all + (size_t)s * D.N, xn_all + (size_t)s * D.N, o);
}

// Copy the per-slice search results and fit outputs to the caller's arrays.  grid ceil(B/128).
template <typename T>
__global__ void k_export(Dev<T> D, int B, T *coeffs, int *axis_ij, T *axis_rzpsi, int *xpt_ij,
                         T *xpt_rzpsi, T *psi_bnd, int *limited, T *chi2, int *status) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= B) return;
  if (!coeffs && !axis_ij && !status && !chi2 && !psi_bnd) {     // graph replay: caller pointers from the argument block
    const CallArgs a = *D.ca;
    coeffs = reinterpret_cast<T *>(a.coeffs); axis_ij = a.axis_ij; axis_rzpsi = reinterpret_cast<T *>(a.axis_rzpsi);
    xpt_ij = a.xpt_ij; xpt_rzpsi = reinterpret_cast<T *>(a.xpt_rzpsi); psi_bnd = reinterpret_cast<T *>(a.psi_bnd);
    limited = a.limited; chi2 = reinterpret_cast<T *>(a.chi2); status = a.status;
  }
  const SearchOut o = D.so[s];
  if (coeffs) for (int l = 0; l < D.nt; ++l) coeffs[(size_t)s * D.nt + l] = T(D.X[(size_t)s * D.nt + l]);
  if (axis_ij) { axis_ij[2 * s] = o.axis_i; axis_ij[2 * s + 1] = o.axis_j; }
  if (axis_rzpsi) { axis_rzpsi[3 * s] = T(o.axis_r); axis_rzpsi[3 * s + 1] = T(o.axis_z); axis_rzpsi[3 * s + 2] = T(o.axis_psi); }
  if (xpt_ij) { xpt_ij[2 * s] = o.xpt_i; xpt_ij[2 * s + 1] = o.xpt_j; }
  if (xpt_rzpsi) { xpt_rzpsi[3 * s] = T(o.xpt_r); xpt_rzpsi[3 * s + 1] = T(o.xpt_z); xpt_rzpsi[3 * s + 2] = T(o.xpt_psi); }
  if (psi_bnd) psi_bnd[s] = T(o.psi_b);
  if (limited) limited[s] = o.limited;
  if (chi2) chi2[s] = T(D.chi2[s]);
  if (status) status[s] = D.status[s];
}

}  // namespace ptefit
