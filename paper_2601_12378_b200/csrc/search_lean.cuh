// search_lean.cuh -- A1/A9 for the FP32 tensor-core solve kernel (k_solve_tc): the same rules as
// search_body (search_kernels.cuh, reading O3), organised for a low
// instruction count (the kernel is issue-bound, not bandwidth-bound):
//   * flat node order: warp w of pass k owns nodes 32 (k nwarp + w) .. +31 = exactly one word of the
//     bit-packed masks; words that are zero are skipped by the whole warp;
//   * scalar work (final arg-max, FP64 axis fit, boundary flux, thresholds) is done once by warp 0 and
//     published through shared memory instead of redundantly by every thread;
//   * X-point candidates: FP32 pre-filter (wide margins) -> survivors compacted into a shared list ->
//     the FP64 fit of quad_coef / quad_finish on the list only (no divergent FP64 in the scan);
//   * plasma region: s psi > s psi_b is decided in FP32 against the largest float <= s psi_b (exact for
//     float flux); the half-plane test of every candidate is a*i + b*j + c in FP32 and falls back to
//     the FP64 expression of search_body when |value| is within the FP32 error margin;
//   * normalised flux in FP32 with two-float psi_axis and 1/(psi_b - psi_axis) (error ~1 ulp);
//   * limiter vertices use the bilinear cells and weights precomputed by ptefit_create.
// Nodes outside lim_mask are not touched: xn there keeps the -1 that k_cold_start / k_search wrote.
#pragma once
#include "common.cuh"
#include "search_kernels.cuh"

namespace ptefit {

constexpr int LEAN_LIST = 1024;      // survivors of the FP32 pre-filter kept for the FP64 pass

struct LeanShared {
  float wv[32]; int wn[32];          // per-warp arg-max (key, node)
  double lv[32]; int ln[32];         // per-warp best limiter vertex
  int flag, ncand, count, nlist, status, ia, ja;
  double Ra, Za, Pa, Pb;
  float thr, pa_hi, pa_lo, inv_hi, inv_lo;
  double cR[PTEFIT_MAX_CAND], cZ[PTEFIT_MAX_CAND], cP[PTEFIT_MAX_CAND];
  int cN[PTEFIT_MAX_CAND];
  float hR[PTEFIT_MAX_CAND], hZ[PTEFIT_MAX_CAND], h0[PTEFIT_MAX_CAND], hm[PTEFIT_MAX_CAND];
  SearchOut so;
  int list[LEAN_LIST];
#ifdef PTEFIT_TUNING
  long long clk[8], t0;
#endif
};
#ifdef PTEFIT_TUNING
#define LS_T(k) do { if (threadIdx.x == 0) { const long long t_ = clock64(); S.clk[k] += t_ - S.t0; S.t0 = t_; } } while (0)
#else
#define LS_T(k) do { } while (0)
#endif

// Indices of the non-zero words of the static masks (host-built, copied to shared memory): the loops of the
// search run over these lists, so every warp iteration does useful work and the words are dealt round-robin.
struct WordLists {
  const unsigned short *lim, *xpt, *dil, *zero;      // lim_mask words, xpt_mask words, dilated-by-one words, words with dil2 bits but no lim bit
  int n_lim, n_xpt, n_dil, n_zero;
};

// FP32 pre-filter of one node: false = certainly not a candidate.  A candidate has its stationary
// point (x*, y*) inside the half cell, and the fitted gradient at the node is -H (x*, y*), hence
// |cx| <= |cxx| + |cxy|/2 and |cy| <= |cyy| + |cxy|/2.  Tested in FP32 with a 2 % margin plus an absolute
// slack of 2e-6 |psi| (the FP32 coefficients carry at most ~5e-7 |psi| of rounding error); the
// classification itself (det H < 0, |x*|, |y*| <= 1/2, flux below the axis) is taken in FP64 on the survivors.
__device__ __forceinline__ bool xpt_prefilter(const float *__restrict__ p, int nr) {
  const float a = p[-nr - 1], b = p[-nr], c = p[-nr + 1], d = p[-1], e = p[0], f = p[1], g = p[nr - 1], hh = p[nr], k = p[nr + 1];
  const float l3 = a + d + g, r3 = c + f + k, m3 = b + e + hh, t3 = a + b + c, u3 = g + hh + k, w3 = d + e + f;
  const float fcx = r3 - l3, fcy = u3 - t3;                                    // 6 cx, 6 cy
  const float fcxx = (l3 + r3) - 2.f * m3, fcyy = (t3 + u3) - 2.f * w3;        // 6 cxx, 6 cyy
  const float hxy = 0.75f * fabsf((k + a) - (g + c));                          // 6 |cxy| / 2
  const float slack = 1.2e-5f * fabsf(e);                                      // 6 x 2e-6 |psi|
  return fabsf(fcx) <= 1.02f * (fabsf(fcxx) + hxy) + slack && fabsf(fcy) <= 1.02f * (fabsf(fcyy) + hxy) + slack;
}

// FP64 decision on one node (identical arithmetic to search_body); appends to the candidate arrays.
__device__ __noinline__ void xpt_decide(double rmin, double zmin, double dr, double dz, int nr, LeanShared *S, const float *psi, int n,
                                        double sg, double Pa) {
  const Quad qc = quad_coef(psi + n, nr);
  if (!(qc.det < 0.0)) return;
  const double lim = 0.5000001 * fabs(qc.det);
  if (fabs(2.0 * qc.cyy * qc.cx - qc.cxy * qc.cy) > lim || fabs(2.0 * qc.cxx * qc.cy - qc.cxy * qc.cx) > lim) return;
  const Fit f = quad_finish(qc);
  if (f.det < 0.0 && fabs(f.xs) <= 0.5 && fabs(f.ys) <= 0.5 && sg * f.ps < sg * Pa) {
    const int q = atomicAdd(&S->ncand, 1);
    if (q < PTEFIT_MAX_CAND) {
      const int j = n / nr, i = n - j * nr;
      S->cR[q] = rmin + (i + f.xs) * dr; S->cZ[q] = zmin + (j + f.ys) * dz; S->cP[q] = f.ps; S->cN[q] = n;
    }
  }
}

// All threads of the CTA call it (block size a multiple of 32, <= 1024).  psi: flux map in shared
// memory, overwritten per lim_mask word with I'(xn) (pc != nullptr) or xn; xn: global, lim_mask words
// only.  (am_v, am_n) / bad: this thread's partial arg-max of s psi over lim_mask and finiteness flag.
__device__ __forceinline__ void search_lean(const Dev<float> &D, LeanShared &S, int s, float *psi, float *__restrict__ xn,
                                            const unsigned *__restrict__ lbits, const unsigned *__restrict__ xbits, const unsigned *__restrict__ d2bits,
                                            const WordLists &WL, float am_v, int am_n, bool bad, const float *pc, const float *rdA, const float *fdA, const double *Xs) {
  const int nth = blockDim.x, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nwarp = nth >> 5;
  const int nr = D.nr, N = D.N;
  const double sg = (double)D.ip_sign;
  if (tid == 0) { S.flag = 0; S.ncand = 0; S.count = 0; S.nlist = 0; }
#ifdef PTEFIT_TUNING
  if (tid == 0) S.t0 = clock64();
#endif
  // 1. axis node: arg-max of s psi over lim_mask, tie -> smallest n.  Warp level, then warp 0.
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float bv = __shfl_xor_sync(0xffffffffu, am_v, o);
    const int bn = __shfl_xor_sync(0xffffffffu, am_n, o);
    if (bv > am_v || (bv == am_v && bn < am_n)) { am_v = bv; am_n = bn; }
  }
  bad = __any_sync(0xffffffffu, bad);
  __syncthreads();                               // S.flag reset above is ordered before the writes below
  if (lane == 0) { S.wv[warp] = am_v; S.wn[warp] = am_n; if (bad) S.flag = 1; }
  __syncthreads();
  if (warp == 0) {
    float v = lane < nwarp ? S.wv[lane] : -INFINITY;
    int n = lane < nwarp ? S.wn[lane] : 0x7fffffff;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float bv = __shfl_xor_sync(0xffffffffu, v, o);
      const int bn = __shfl_xor_sync(0xffffffffu, n, o);
      if (bv > v || (bv == v && bn < n)) { v = bv; n = bn; }
    }
    if (lane == 0) {
      int st = S.flag ? 2 : 0;
      int ia = -1, ja = -1;
      double Ra = 0, Za = 0, Pa = 0;
      if (st == 0) {
        ja = n / nr; ia = n - ja * nr;
        const Fit f = quad_fit(psi + n, nr);
        if (!(f.det > 0.0) || fmax(fabs(f.xs), fabs(f.ys)) > 1.0) st = 1;
        Ra = D.rmin + (ia + f.xs) * D.dr; Za = D.zmin + (ja + f.ys) * D.dz; Pa = f.ps;
      }
      S.status = st; S.ia = ia; S.ja = ja; S.Ra = Ra; S.Za = Za; S.Pa = Pa;
    }
  }
  LS_T(0);
  // 2. X-point candidates: FP32 scan of the xpt_mask words -> compact list (the scan does not need the axis)
  {                                              // word index and mask word of the next iteration are fetched one iteration ahead
    int k = warp;
    int w = k < WL.n_xpt ? WL.xpt[k] : 0;
    unsigned xb = xbits[w];
    while (k < WL.n_xpt) {
      const int kn = k + nwarp;
      const int wn = kn < WL.n_xpt ? WL.xpt[kn] : 0;
      const unsigned xbn = xbits[wn];
      const int n = (w << 5) + lane;
      const bool bit = (xb >> lane) & 1u;
      if (xpt_prefilter(psi + (bit ? n : nr + 1), nr) && bit) {         // masked-off lanes read a harmless interior node
        const int q = atomicAdd(&S.nlist, 1);
        if (q < LEAN_LIST) S.list[q] = n;
      }
      k = kn; w = wn; xb = xbn;
    }
  }
  __syncthreads();
  LS_T(1);
  int status = S.status;
  const double Ra = S.Ra, Za = S.Za, Pa = S.Pa;
  if (status == 0) {                             // FP64 decision on the survivors
    const int nl = S.nlist;
    if (nl <= LEAN_LIST) {
      for (int q = tid; q < nl; q += nth) xpt_decide(D.rmin, D.zmin, D.dr, D.dz, nr, &S, psi, S.list[q], sg, Pa);
    } else {                                     // list overflow (not seen on smooth flux): decide in place
      for (int k = warp; k < WL.n_xpt; k += nwarp) {
        const int w = WL.xpt[k];
        const int n = (w << 5) + lane;
        if (((xbits[w] >> lane) & 1u) && xpt_prefilter(psi + n, nr)) xpt_decide(D.rmin, D.zmin, D.dr, D.dz, nr, &S, psi, n, sg, Pa);
      }
    }
  }
  __syncthreads();
  LS_T(2);
  const int ncand = S.ncand;
  if (status == 0 && ncand > PTEFIT_MAX_CAND) status = 4;
  // 3. limiter vertices: bilinear flux (precomputed cells and weights), valid iff not behind any
  // candidate as seen from the axis
  const int lim_warps = (D.nlim + 31) >> 5;
  if (warp < lim_warps) {
    double bv = -INFINITY;
    int bn = 0x7fffffff;
    if (status == 0) {
      for (int v = tid; v < D.nlim; v += 32 * lim_warps) {
        const double tx = D.lim_tx[v], ty = D.lim_ty[v];
        const float *p = psi + D.lim_n0[v];
        const double pv = (1.0 - ty) * ((1.0 - tx) * (double)p[0] + tx * (double)p[1]) +
                          ty * ((1.0 - tx) * (double)p[nr] + tx * (double)p[nr + 1]);
        bool valid = true;
        if (ncand) {
          const double lr = D.lim_r[v], lz = D.lim_z[v];
          for (int c = 0; c < ncand; ++c)
            valid &= ((lr - S.cR[c]) * (Ra - S.cR[c]) + (lz - S.cZ[c]) * (Za - S.cZ[c])) >= 0.0;
        }
        const double key = sg * pv;
        if (valid && (key > bv || (key == bv && v < bn))) { bv = key; bn = v; }
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
      const int on = __shfl_xor_sync(0xffffffffu, bn, o);
      if (ov > bv || (ov == bv && on < bn)) { bv = ov; bn = on; }
    }
    if (lane == 0) { S.lv[warp] = bv; S.ln[warp] = bn; }
  }
  __syncthreads();
  LS_T(3);
  // 4. boundary flux, thresholds of the mask pass: one thread, published through shared memory
  if (tid == 0) {
    int st = status;
    if (st == 0) {
      double lmv = -INFINITY;
      int lmn = 0x7fffffff;
      for (int k = 0; k < lim_warps; ++k)
        if (S.lv[k] > lmv || (S.lv[k] == lmv && S.ln[k] < lmn)) { lmv = S.lv[k]; lmn = S.ln[k]; }
      double bxv = -INFINITY;
      int bxn = 0x7fffffff, qbest = -1;
      for (int c = 0; c < ncand; ++c) {
        const double tv = sg * S.cP[c];
        if (tv > bxv || (tv == bxv && S.cN[c] < bxn)) { bxv = tv; bxn = S.cN[c]; qbest = c; }
      }
      const bool xwins = bxv > lmv;
      const double spb = xwins ? bxv : lmv;
      if (!isfinite(spb)) st = 1;
      const double Pb = sg * spb;
      SearchOut &so = S.so;
      so.axis_i = S.ia; so.axis_j = S.ja; so.axis_r = Ra; so.axis_z = Za; so.axis_psi = Pa;
      so.n_cand = ncand; so.limited = xwins ? 0 : 1; so.psi_b = Pb;
      if (qbest >= 0) {
        so.xpt_j = S.cN[qbest] / nr; so.xpt_i = S.cN[qbest] - so.xpt_j * nr;
        so.xpt_r = S.cR[qbest]; so.xpt_z = S.cZ[qbest]; so.xpt_psi = S.cP[qbest];
      } else {
        so.xpt_i = so.xpt_j = -1; so.xpt_r = so.xpt_z = so.xpt_psi = nan("");
      }
      if (st == 0 && Pb == Pa) st = 1;
      S.Pb = Pb;
      S.thr = __double2float_rd(sg * Pb);              // float key > thr  <=>  (double) key > s psi_b
      S.pa_hi = (float)Pa; S.pa_lo = (float)(Pa - (double)S.pa_hi);
      const double invd = 1.0 / (Pb - Pa);
      S.inv_hi = (float)invd; S.inv_lo = (float)(invd - (double)S.inv_hi);
    }
    S.status = st;
  }
  // FP32 form of the half-plane test of candidate c: hR i + hZ j + h0, decided in FP64 inside +-hm
  if (status == 0 && tid >= 32 && tid - 32 < ncand) {
    const int c = tid - 32;
    const double aR = Ra - S.cR[c], aZ = Za - S.cZ[c];
    const double c0 = aR * (D.rmin - S.cR[c]) + aZ * (D.zmin - S.cZ[c]);
    S.hR[c] = (float)(aR * D.dr); S.hZ[c] = (float)(aZ * D.dz); S.h0[c] = (float)c0;
    S.hm[c] = 4e-6f * (float)(fabs(aR * D.dr) * nr + fabs(aZ * D.dz) * D.nz + fabs(c0));
  }
  __syncthreads();
  LS_T(4);
  // 5./6. plasma region and normalised flux, lim_mask words only
  status = S.status;
  int cnt = 0;
  if (status == 0) {
    const float sgf = (float)D.ip_sign;
    const float thr = S.thr, pa_hi = S.pa_hi, pa_lo = S.pa_lo, inv_hi = S.inv_hi, inv_lo = S.inv_lo;
    const float inv_nr = 1.0f / (float)nr;
    constexpr int MD = PTEFIT_MAX_DEG;
    const bool lowdeg = D.maxdeg <= 4;
    float pp[5], pq[5];                               // low-degree fast path: coefficients in registers
#pragma unroll
    for (int k = 0; k < 5; ++k) { pp[k] = pc ? pc[k] : 0.f; pq[k] = pc ? pc[MD + 1 + k] : 0.f; }
    const bool spl = D.nspl && Xs;
    // half-plane tests of candidates 0 and 1 from registers; an absent candidate reads as "always in front,
    // never near the margin" (value 1, margin 0).  More than two candidates (rare) take the loop below.
    const float a0R = ncand > 0 ? S.hR[0] : 0.f, a0Z = ncand > 0 ? S.hZ[0] : 0.f, a00 = ncand > 0 ? S.h0[0] : 1.f, a0m = ncand > 0 ? S.hm[0] : 0.f;
    const float a1R = ncand > 1 ? S.hR[1] : 0.f, a1Z = ncand > 1 ? S.hZ[1] : 0.f, a10 = ncand > 1 ? S.h0[1] : 1.f, a1m = ncand > 1 ? S.hm[1] : 0.f;
    int k = warp;
    int wc = k < WL.n_lim ? WL.lim[k] : 0;
    unsigned lbc = lbits[wc];
    float vc = psi[((lbc >> lane) & 1u) ? (wc << 5) + lane : 0];
    while (k < WL.n_lim) {                            // word index, mask word and flux of the next iteration are fetched one iteration ahead
      const int w = wc, n = (w << 5) + lane;
      const bool bit = (lbc >> lane) & 1u;
      const float v = vc;
      k += nwarp;
      wc = k < WL.n_lim ? WL.lim[k] : 0;
      lbc = lbits[wc];
      vc = psi[((lbc >> lane) & 1u) ? (wc << 5) + lane : 0];     // read before this iteration's store to psi: different words
      bool in = bit && (sgf * v > thr);
      if (!__any_sync(0xffffffffu, in)) {             // no plasma node in this word (warp-uniform): nothing to evaluate
        if (n < N) { xn[n] = -1.f; psi[n] = pc ? 0.f : -1.f; }
        continue;
      }
      const int j = __float2int_rd(((float)n + 0.5f) * inv_nr);     // exact: (n + 0.5)/nr is >= 0.5/nr away from an integer
      const int i = n - j * nr;
      const float fi = (float)i, fj = (float)j;
      {
        const float v0 = fmaf(a0R, fi, fmaf(a0Z, fj, a00)), v1 = fmaf(a1R, fi, fmaf(a1Z, fj, a10));
        bool ok0 = v0 > 0.f, ok1 = v1 > 0.f;
        if (in && (!(fabsf(v0) > a0m) || !(fabsf(v1) > a1m))) {     // inside the FP32 error margin: the FP64 expression decides (rare)
          const double R = D.rmin + i * D.dr, Z = D.zmin + j * D.dz;
          if (!(fabsf(v0) > a0m)) ok0 = ((R - S.cR[0]) * (Ra - S.cR[0]) + (Z - S.cZ[0]) * (Za - S.cZ[0])) > 0.0;
          if (!(fabsf(v1) > a1m)) ok1 = ((R - S.cR[1]) * (Ra - S.cR[1]) + (Z - S.cZ[1]) * (Za - S.cZ[1])) > 0.0;
        }
        in = in && ok0 && ok1;
      }
      if (ncand > 2) {                                // uniform branch
        for (int c = 2; c < ncand; ++c) {
          const float val = fmaf(S.hR[c], fi, fmaf(S.hZ[c], fj, S.h0[c]));
          bool ok = val > 0.f;
          if (in && !(fabsf(val) > S.hm[c])) {
            const double R = D.rmin + i * D.dr, Z = D.zmin + j * D.dz;
            ok = ((R - S.cR[c]) * (Ra - S.cR[c]) + (Z - S.cZ[c]) * (Za - S.cZ[c])) > 0.0;
          }
          in = in && ok;
        }
      }
      const float d = (v - pa_hi) - pa_lo;
      const float x = fminf(fmaxf(fmaf(d, inv_lo, d * inv_hi), 0.f), 1.f);
      const float out = in ? x : -1.f;
      cnt += in;
      if (n < N) xn[n] = out;
      float lv = out;
      if (pc) {                                       // I'(x) = rdA P(x) + fdA Q(x) by Horner (delz column); uniform branch
        float hp, hq;
        if (lowdeg) {
          hp = pp[4]; hq = pq[4];
#pragma unroll
          for (int q = 3; q >= 0; --q) { hp = fmaf(hp, x, pp[q]); hq = fmaf(hq, x, pq[q]); }
        } else {
          hp = pc[MD]; hq = pc[2 * MD + 1];
#pragma unroll
          for (int q = MD - 1; q >= 0; --q) { hp = fmaf(hp, x, pc[q]); hq = fmaf(hq, x, pc[MD + 1 + q]); }
        }
        const int ic = min(i, nr - 1);
        lv = fmaf(rdA[ic], hp, fdA[ic] * hq);
        if (spl && in) lv += spline_current(D, Xs, x, rdA[ic], fdA[ic]);
        lv = in ? lv : 0.f;
      }
      if (n < N) psi[n] = lv;
    }
    if (pc)                                           // rows the delz stencil reaches beyond the lim_mask words: I' = 0 there
      for (int k = warp; k < WL.n_zero; k += nwarp) {
        const int w = WL.zero[k];
        if ((d2bits[w] >> lane) & 1u) psi[(w << 5) + lane] = 0.f;
      }
  } else {
    for (int k = warp; k < WL.n_lim; k += nwarp) {
      const int n = (WL.lim[k] << 5) + lane;
      if (n < N) { xn[n] = -1.f; psi[n] = pc ? 0.f : -1.f; }
    }
    if (pc)
      for (int k = warp; k < WL.n_zero; k += nwarp) {
        const int w = WL.zero[k];
        if ((d2bits[w] >> lane) & 1u) psi[(w << 5) + lane] = 0.f;
      }
  }
  LS_T(5);
  cnt = __reduce_add_sync(0xffffffffu, cnt);
  if (lane == 0 && cnt) atomicAdd(&S.count, cnt);
  __syncthreads();
  LS_T(6);
  if (tid == 0) {
    if (status == 0 && S.count == 0) status = 1;
    if (D.status[s] == 0) {
      if (status == 0 || status == 4) D.so[s] = S.so;
      if (status == 1 || status == 2) { SearchOut z = {}; z.axis_i = S.ia; z.axis_j = S.ja; z.xpt_i = z.xpt_j = -1; D.so[s] = z; }
      D.status[s] = status;
    }
  }
}

}  // namespace ptefit
