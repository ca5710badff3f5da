// ptefit.cu -- C ABI (include/ptefit.h) of the B200-native PTEFIT Picard iteration.
// Host side: validation, table upload, DST/tridiagonal factor precompute, launch sequence.
// No CPU compute path exists: without a usable device every entry point returns PTEFIT_ERR_CUDA.
#include "../../include/ptefit.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <type_traits>
#include <vector>

#include "common.cuh"
#include "fit_kernels.cuh"
#include "search_kernels.cuh"
#include "solve_kernels.cuh"
#include "fused_solve.cuh"
#include "tc_gemm.cuh"
#include "tc_kernels.cuh"
#include "tc_solve.cuh"
#include "dmma_gemm.cuh"
#include "dmma_kernels.cuh"
#include "greens_kernels.cuh"
#include "joint_fit.cuh"
#include "fluxsurf_kernels.cuh"

using namespace ptefit;

static thread_local std::string g_error;

struct GraphKey { int batch, n_iter, warm; };
struct CachedGraph { GraphKey key; cudaGraphExec_t exec; int launches; };

struct ptefit_handle {
  ptefit_precision prec;
  ptefit_gemm_mode gemm;
  int max_batch;
  Dev<float> d32;
  Dev<double> d64;
  std::vector<void *> allocs;
  std::string error;
  int launches = 0;
  int state_batch = 0;                  // slices whose (xn, delz column, X) are those of the last ptefit_reconstruct call (warm_start = 2)
  bool tc = false;                      // tensor-core contractions usable (FP32, 3xTF32 mode)
  TcDev Tc{};
  const float *gp_hi = nullptr, *gp_lo = nullptr, *gb_hi = nullptr, *gb_lo = nullptr;
  int pbd_ntiles = 0, max_split_resp = 1, max_split_pbd = 1;
  const float *c_rdA = nullptr, *c_fdA = nullptr;   // Eq. 10 factors on the compact node list
  bool dm = false;                      // FP64 tensor-core (DMMA) contractions usable (FP64 mode, gemm != FFMA)
  DmDev Dm{};
  bool tcs = false;                     // k_solve_tc usable (FP32, N_Z = 129, tensor-core mode)
  TcSolveDev Ts{};
  size_t tcs_smem = 0;
  int nsm = 0;
  CUtensorMap mapTfHi, mapTfLo, mapTiHi, mapTiLo;   // forward / inverse sine tables of k_solve_tc
  int flags = 0, tc_split_k = 0;
  CallArgs *ca_dev = nullptr;           // device copy of the caller's pointers, rewritten per call
  int std_np = 0;                       // > 0: standard term list, basis generated inside the response GEMM
  CUtensorMap mapJbHi, mapJbLo, mapGpHi, mapGpLo, mapCurHi, mapCurLo, mapGbHi, mapGbLo;
  bool use_graph = true;                // replay the launch sequence as a CUDA graph (PTEFIT_OPT_NO_GRAPH disables)
  std::vector<CachedGraph> graphs;
  cudaStream_t gstream = nullptr;       // capture stream
  bool fused = false;                   // k_solve_fused usable (slice fits shared memory)
  int fused_grid = 0;                   // resident CTAs of k_solve_fused
  size_t fused_smem = 0;
  bool profiling = false;
  std::vector<cudaEvent_t> ev;          // stage boundaries of the last call
  std::vector<int> ev_stage;
  // staging buffers of ptefit_reconstruct_host
  void *hb = nullptr, *hic = nullptr, *hpsi = nullptr, *hco = nullptr, *hax = nullptr, *hxp = nullptr,
       *hpb = nullptr, *hchi = nullptr;
  int *haxij = nullptr, *hxpij = nullptr, *hlim = nullptr, *hst = nullptr;
  cudaStream_t hstream = nullptr;
};

#define CK(call)                                                                          \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) {                                                              \
      char buf_[512];                                                                     \
      snprintf(buf_, sizeof buf_, "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
      if (h) h->error = buf_;                                                             \
      g_error = buf_;                                                                     \
      return e_ == cudaErrorMemoryAllocation ? PTEFIT_ERR_NOMEM : PTEFIT_ERR_CUDA;        \
    }                                                                                     \
  } while (0)

static ptefit_status fail(ptefit_handle *h, ptefit_status st, const char *msg) {
  g_error = msg;
  if (h) h->error = msg;
  return st;
}

template <typename T>
static ptefit_status dev_alloc(ptefit_handle *h, T **p, size_t count) {
  void *q = nullptr;
  CK(cudaMalloc(&q, count * sizeof(T) + 256));
  CK(cudaMemset(q, 0, count * sizeof(T) + 256));
  h->allocs.push_back(q);
  *p = reinterpret_cast<T *>(q);
  return PTEFIT_OK;
}

template <typename T, typename S>
static ptefit_status upload(ptefit_handle *h, const T **p, const S *src, size_t count) {
  std::vector<T> tmp(count);
  for (size_t k = 0; k < count; ++k) tmp[k] = (T)src[k];   // round to nearest (FP32 mode)
  T *q = nullptr;
  ptefit_status st = dev_alloc(h, &q, count);
  if (st != PTEFIT_OK) return st;
  CK(cudaMemcpy(q, tmp.data(), count * sizeof(T), cudaMemcpyHostToDevice));
  *p = q;
  return PTEFIT_OK;
}

#define TRY(x)                        \
  do {                                \
    ptefit_status st_ = (x);          \
    if (st_ != PTEFIT_OK) return st_; \
  } while (0)

template <typename T>
static ptefit_status build(ptefit_handle *h, Dev<T> &D, const ptefit_grid *g, const ptefit_geometry *ge,
                           const ptefit_tables *tb, const ptefit_basis *ba, int B) {
  D.nr = g->nr; D.nz = g->nz; D.N = g->nr * g->nz; D.nri = g->nr - 2; D.nzi = g->nz - 2;
  D.nbnd = 2 * (g->nr + g->nz) - 4; D.M = ge->n_meas; D.nc = ge->n_coil; D.nt = ba->n_terms;
  D.nlim = ge->n_lim; D.ip_sign = ge->ip_sign;
  D.rmin = g->rmin; D.zmin = g->zmin;
  D.dr = (g->rmax - g->rmin) / (g->nr - 1); D.dz = (g->zmax - g->zmin) / (g->nz - 1);
  D.dA = D.dr * D.dz; D.lambda_reg = ba->lambda_reg; D.relax = ba->relax;
  D.cold_rc = ge->cold_rc; D.cold_zc = ge->cold_zc; D.cold_a = ge->cold_a; D.cold_b = ge->cold_b;
  D.npoly = 0; D.has_delz = 0; D.nspl = 0; D.maxdeg = 0; D.spl = nullptr; D.lsq_method = ba->lsq_method; D.fit_coils = ba->fit_coils;
  const ptefit_term *spl_term = nullptr;
  for (int l = 0; l < ba->n_terms; ++l) {
    const ptefit_term &t = ba->terms[l];
    D.terms[l].kind = t.kind; D.terms[l].family = t.kind == 2 ? 0 : t.family; D.terms[l].i = t.i; D.terms[l].N = t.N;
    if (t.kind == 2) { D.has_delz = 1; continue; }
    D.npoly++;
    if (t.family == 1) { D.nspl++; spl_term = &t; }
    else if (t.N > D.maxdeg) D.maxdeg = t.N;
  }
  if (spl_term) {
    // cardinal tension splines (reading O4c): second derivatives m[r][q] at the knots from the
    // tridiagonal system that makes the first derivative continuous (natural ends), solved in FP64
    SplineDev sp{};
    const int nk = spl_term->n_knots;
    const double tau = spl_term->tension;
    sp.nk = nk; sp.tau = tau; sp.inv_tau2 = 1.0 / (tau * tau);
    std::vector<double> a(nk, 0.0), b(nk, 0.0);
    for (int r = 0; r < nk; ++r) sp.knot[r] = spl_term->knots[r];
    for (int r = 0; r + 1 < nk; ++r) {
      const double hh = sp.knot[r + 1] - sp.knot[r];
      sp.inv_h[r] = 1.0 / hh; sp.tau_h[r] = tau * hh; sp.inv_sinh[r] = 1.0 / sinh(tau * hh);
      a[r] = (1.0 / hh - tau / sinh(tau * hh)) / (tau * tau);
      b[r] = (tau * cosh(tau * hh) / sinh(tau * hh) - 1.0 / hh) / (tau * tau);
    }
    for (int q = 0; q < nk; ++q) {                       // one Thomas solve per cardinal function
      std::vector<double> lo(nk, 0.0), di(nk, 1.0), up(nk, 0.0), rh(nk, 0.0);
      for (int r = 1; r + 1 < nk; ++r) {
        lo[r] = a[r - 1]; di[r] = b[r - 1] + b[r]; up[r] = a[r];
        const double y0 = (r - 1 == q), y1 = (r == q), y2 = (r + 1 == q);
        rh[r] = (y2 - y1) * sp.inv_h[r] - (y1 - y0) * sp.inv_h[r - 1];
      }
      for (int r = 1; r < nk; ++r) { const double w = lo[r] / di[r - 1]; di[r] -= w * up[r - 1]; rh[r] -= w * rh[r - 1]; }
      std::vector<double> mm(nk, 0.0);
      mm[nk - 1] = rh[nk - 1] / di[nk - 1];
      for (int r = nk - 2; r >= 0; --r) mm[r] = (rh[r] - up[r] * mm[r + 1]) / di[r];
      for (int r = 0; r < nk; ++r) sp.m[r][q] = mm[r];
    }
    SplineDev *dsp = nullptr;
    TRY(dev_alloc(h, &dsp, 1));
    CK(cudaMemcpy(dsp, &sp, sizeof sp, cudaMemcpyHostToDevice));
    D.spl = dsp;
  }
  TRY(dev_alloc(h, &h->ca_dev, 1));
  D.ca = h->ca_dev;
  const size_t N = D.N;
  // tables; edge-node columns of gp / gb are zeroed (edge nodes never carry current)
  {
    std::vector<double> t(tb->gp, tb->gp + (size_t)D.M * N);
    std::vector<double> u(tb->gb, tb->gb + (size_t)D.nbnd * N);
    for (int j = 0; j < D.nz; ++j)
      for (int i = 0; i < D.nr; ++i)
        if (i == 0 || j == 0 || i == D.nr - 1 || j == D.nz - 1) {
          for (int m = 0; m < D.M; ++m) t[(size_t)m * N + j * D.nr + i] = 0.0;
          for (int k = 0; k < D.nbnd; ++k) u[(size_t)k * N + j * D.nr + i] = 0.0;
        }
    TRY(upload(h, &D.gp, t.data(), t.size()));
    TRY(upload(h, &D.gb, u.data(), u.size()));
  }
  TRY(upload(h, &D.gc, tb->gc, (size_t)D.M * D.nc));
  TRY(upload(h, &D.ggc, tb->ggc, N * D.nc));
  {
    std::vector<double> t((size_t)D.nc * N);
    for (size_t n = 0; n < N; ++n)
      for (int c = 0; c < D.nc; ++c) t[(size_t)c * N + n] = tb->ggc[n * D.nc + c];
    TRY(upload(h, &D.ggc_t, t.data(), t.size()));
  }
  {
    std::vector<double> w(D.M);
    for (int m = 0; m < D.M; ++m) w[m] = 1.0 / ge->sigma[m];
    TRY(upload(h, &D.inv_sigma, w.data(), w.size()));
  }
  if (ba->fit_coils) {
    // constants of the joint fit (Eq. 7): W G_C, and the coil-coil block G_C^T W^2 G_C + diag(1/sigma_ic^2)
    // scaled to a unit diagonal, FP64, from the table values the kernels see (rounded to T first)
    const int M = D.M, nc = D.nc;
    std::vector<double> gw((size_t)M * nc), c22((size_t)nc * nc, 0.0), tc(nc), is2(nc);
    for (int m = 0; m < M; ++m)
      for (int c = 0; c < nc; ++c) gw[(size_t)m * nc + c] = (double)(T)tb->gc[(size_t)m * nc + c] / ge->sigma[m];
    for (int c = 0; c < nc; ++c) is2[c] = 1.0 / (ba->sigma_ic[c] * ba->sigma_ic[c]);
    for (int c = 0; c < nc; ++c)
      for (int e = 0; e <= c; ++e) {
        double acc = 0.0;
        for (int m = 0; m < M; ++m) acc += gw[(size_t)m * nc + c] * gw[(size_t)m * nc + e];
        if (e == c) acc += is2[c];
        c22[(size_t)c * nc + e] = c22[(size_t)e * nc + c] = acc;
      }
    for (int c = 0; c < nc; ++c) tc[c] = sqrt(c22[(size_t)c * nc + c]);
    for (int c = 0; c < nc; ++c)
      for (int e = 0; e < nc; ++e) c22[(size_t)c * nc + e] /= tc[c] * tc[e];
    TRY(upload(h, &D.gcw, gw.data(), gw.size()));
    TRY(upload(h, &D.c22s, c22.data(), c22.size()));
    TRY(upload(h, &D.tcoil, tc.data(), tc.size()));
    TRY(upload(h, &D.inv_sic2, is2.data(), is2.size()));
    TRY(dev_alloc(h, &D.icf, (size_t)B * nc));
    TRY(dev_alloc(h, &D.icm, (size_t)B * nc));
    CK(cudaFuncSetAttribute(k_lsq_joint<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)joint_smem_bytes(M, D.nt, nc)));
  }
  TRY(upload(h, &D.lim_mask, ge->lim_mask, N));
  TRY(upload(h, &D.xpt_mask, ge->xpt_mask ? ge->xpt_mask : ge->lim_mask, N));
  {
    const unsigned char *xm = ge->xpt_mask ? ge->xpt_mask : ge->lim_mask;
    std::vector<unsigned> lb((N + 31) / 32, 0u), xb((N + 31) / 32, 0u);
    for (size_t n = 0; n < N; ++n) {
      if (ge->lim_mask[n]) lb[n >> 5] |= 1u << (n & 31);
      if (xm[n]) xb[n >> 5] |= 1u << (n & 31);
    }
    TRY(upload(h, &D.lim_bits, lb.data(), lb.size()));
    TRY(upload(h, &D.xpt_bits, xb.data(), xb.size()));
    std::vector<unsigned> eb((N + 31) / 32, 0u);
    for (int j = 0; j < D.nz; ++j)
      for (int i = 0; i < D.nr; ++i)
        if (i == 0 || j == 0 || i == D.nr - 1 || j == D.nz - 1) { const size_t n = (size_t)j * D.nr + i; eb[n >> 5] |= 1u << (n & 31); }
    TRY(upload(h, &D.edge_bits, eb.data(), eb.size()));
    std::vector<unsigned> db((N + 31) / 32, 0u);
    for (int j = 1; j < D.nz - 1; ++j)
      for (int i = 1; i < D.nr - 1; ++i) {
        const size_t n = (size_t)j * D.nr + i;
        if (ge->lim_mask[n] || ge->lim_mask[n + D.nr] || ge->lim_mask[n - D.nr]) db[n >> 5] |= 1u << (n & 31);
      }
    TRY(upload(h, &D.dil_bits, db.data(), db.size()));
    std::vector<unsigned> d2((N + 31) / 32, 0u);
    for (int j = 0; j < D.nz; ++j)
      for (int i = 0; i < D.nr; ++i) {
        bool any = false;
        for (int dj = -2; dj <= 2; ++dj)
          if (j + dj >= 0 && j + dj < D.nz && ge->lim_mask[(size_t)(j + dj) * D.nr + i]) any = true;
        const size_t n = (size_t)j * D.nr + i;
        if (any) d2[n >> 5] |= 1u << (n & 31);
      }
    TRY(upload(h, &D.dil2_bits, d2.data(), d2.size()));
  }
  TRY(upload(h, &D.lim_r, ge->lim_r, (size_t)D.nlim));
  TRY(upload(h, &D.lim_z, ge->lim_z, (size_t)D.nlim));
  {
    // bilinear cell and weights of every limiter vertex (same FP64 expressions as search_body)
    std::vector<int> n0(D.nlim);
    std::vector<double> tx(D.nlim), ty(D.nlim);
    for (int v = 0; v < D.nlim; ++v) {
      const double fi = (ge->lim_r[v] - D.rmin) / D.dr, fj = (ge->lim_z[v] - D.zmin) / D.dz;
      int i0 = (int)floor(fi), j0 = (int)floor(fj);
      i0 = i0 < 0 ? 0 : (i0 > D.nr - 2 ? D.nr - 2 : i0);
      j0 = j0 < 0 ? 0 : (j0 > D.nz - 2 ? D.nz - 2 : j0);
      n0[v] = j0 * D.nr + i0; tx[v] = fi - i0; ty[v] = fj - j0;
    }
    TRY(upload(h, &D.lim_n0, n0.data(), n0.size()));
    TRY(upload(h, &D.lim_tx, tx.data(), tx.size()));
    TRY(upload(h, &D.lim_ty, ty.data(), ty.size()));
  }
  // Delta* factors ("the coefficient matrices can be pre-computed"): for each DST
  // mode m the tridiagonal [cw_i, -2/dR^2 + lam_m, ce_i] is LU-factored in FP64 on the host.
  {
    const int nri = D.nri, nzi = D.nzi;
    std::vector<double> w((size_t)nri * nzi), ib((size_t)nri * nzi), ce(nri), cw(nri);
    for (int i = 0; i < nri; ++i) {
      const double R = D.rmin + (i + 1) * D.dr;
      cw[i] = (1.0 + D.dr / (2.0 * R)) / (D.dr * D.dr);
      ce[i] = (1.0 - D.dr / (2.0 * R)) / (D.dr * D.dr);
    }
    const double pi = 3.14159265358979323846;
    for (int mm = 0; mm < nzi; ++mm) {
      const double sn = sin(pi * (mm + 1) / (2.0 * (D.nz - 1)));
      const double diag = -2.0 / (D.dr * D.dr) - 4.0 / (D.dz * D.dz) * sn * sn;
      double piv = diag;
      w[mm] = 0.0; ib[mm] = 1.0 / piv;
      for (int i = 1; i < nri; ++i) {
        const double wi = cw[i] / piv;
        piv = diag - wi * ce[i - 1];
        w[(size_t)i * nzi + mm] = wi;
        ib[(size_t)i * nzi + mm] = 1.0 / piv;
      }
    }
    ce[nri - 1] = ce[nri - 1];  // multiplies x_{nri} = 0 in the back substitution
    TRY(upload(h, &D.tri_w, w.data(), w.size()));
    TRY(upload(h, &D.tri_invb, ib.data(), ib.size()));
    TRY(upload(h, &D.tri_ce, ce.data(), ce.size()));
    // Twisted (two-sided) factorisation of the same systems for k_solve_fused: rows 0..k-1 are
    // eliminated downwards, rows n-1..k+1 upwards, row k = n/2 couples both halves, so two threads
    // per mode walk chains of half the length.  tw2[i][m]: multiplier of row i (towards the
    // previous row of its half; row k: the left one), tw2k[m]: right multiplier of row k,
    // tib2[i][m]: inverse pivots, tod2[i]: off-diagonal used in the back substitution of row i.
    {
      const int n = nri, k = n / 2;
      std::vector<double> w2((size_t)n * nzi, 0.0), ib2((size_t)n * nzi, 0.0), wk(nzi, 0.0), od(n, 0.0);
      for (int i = 0; i < n; ++i) od[i] = (i < k) ? ce[i] : cw[i];
      for (int mm = 0; mm < nzi; ++mm) {
        const double sn = sin(pi * (mm + 1) / (2.0 * (D.nz - 1)));
        const double diag = -2.0 / (D.dr * D.dr) - 4.0 / (D.dz * D.dz) * sn * sn;
        std::vector<double> piv(n, diag);
        for (int i = 1; i < k; ++i) { const double wl = cw[i] / piv[i - 1]; w2[(size_t)i * nzi + mm] = wl; piv[i] = diag - wl * ce[i - 1]; }
        for (int i = n - 2; i > k; --i) { const double wr = ce[i] / piv[i + 1]; w2[(size_t)i * nzi + mm] = wr; piv[i] = diag - wr * cw[i + 1]; }
        double pk = diag;
        if (k >= 1) { const double wl = cw[k] / piv[k - 1]; w2[(size_t)k * nzi + mm] = wl; pk -= wl * ce[k - 1]; }
        if (k + 1 < n) { const double wr = ce[k] / piv[k + 1]; wk[mm] = wr; pk -= wr * cw[k + 1]; }
        piv[k] = pk;
        for (int i = 0; i < n; ++i) ib2[(size_t)i * nzi + mm] = 1.0 / piv[i];
      }
      TRY(upload(h, &D.tw2, w2.data(), w2.size()));
      TRY(upload(h, &D.tib2, ib2.data(), ib2.size()));
      TRY(upload(h, &D.tw2k, wk.data(), wk.size()));
      TRY(upload(h, &D.tod2, od.data(), od.size()));
    }
    const int period = 2 * (D.nz - 1);
    std::vector<double> st(period);
    for (int k = 0; k < period; ++k) st[k] = sin(pi * k / (D.nz - 1));
    st[D.nz - 1] = 0.0;
    TRY(upload(h, &D.sintab, st.data(), st.size()));
    // folded DST matrices, transposed so that four consecutive modes are one vector load:
    // So[j][p] = sin(pi (j+1)(2p+1)/Nz), Se[j][p] = sin(pi (j+1)(2p+2)/Nz) (0 beyond Nz/2-1)
    const int Nz = D.nz - 1, n2 = Nz / 2;
    std::vector<double> tab(2 * (size_t)n2 * n2, 0.0);
    for (int j = 0; j < n2; ++j)
      for (int q = 0; q < n2; ++q) {
        tab[(size_t)j * n2 + q] = sin(pi * (double)((j + 1) * (2 * q + 1) % (2 * Nz)) / Nz);
        if (j < n2 - 1 && q < n2 - 1)
          tab[(size_t)n2 * n2 + (size_t)j * n2 + q] = sin(pi * (double)((j + 1) * (2 * q + 2) % (2 * Nz)) / Nz);
      }
    TRY(upload(h, &D.dst_tab, tab.data(), tab.size()));
  }
  // workspaces
  TRY(dev_alloc(h, &D.xn, (size_t)B * N));
  {   // -1 = outside the plasma: the lean search kernels rewrite the lim_mask words only
    std::vector<T> m1(N, T(-1));
    for (int q = 0; q < B; ++q) CK(cudaMemcpy(D.xn + (size_t)q * N, m1.data(), N * sizeof(T), cudaMemcpyHostToDevice));
  }
  TRY(dev_alloc(h, &D.psi_coil, (size_t)B * N));
  TRY(dev_alloc(h, &D.dred, (size_t)B * D.M));
  TRY(dev_alloc(h, &D.resp, (size_t)B * D.M * D.nt));
  TRY(dev_alloc(h, &D.cur, (size_t)B * N));
  TRY(dev_alloc(h, &D.dzc, (size_t)B * N));
  TRY(dev_alloc(h, &D.psi_bdry, (size_t)B * D.nbnd));
  TRY(dev_alloc(h, &D.fhat, (size_t)B * D.nri * D.nzi));
  TRY(dev_alloc(h, &D.ytmp, (size_t)B * D.nri * D.nzi));
  TRY(dev_alloc(h, &D.X, (size_t)B * D.nt));
  TRY(dev_alloc(h, &D.pco, (size_t)B * PCO_STRIDE));
  TRY(dev_alloc(h, &D.Xprev, (size_t)B * D.nt));
  TRY(dev_alloc(h, &D.chi2, (size_t)B));
  TRY(dev_alloc(h, &D.so, (size_t)B));
  TRY(dev_alloc(h, &D.status, (size_t)B));
  return PTEFIT_OK;
}

#include "tc_host.inc"
#include "dm_host.inc"

extern "C" ptefit_status ptefit_create(const ptefit_grid *g, const ptefit_geometry *ge,
                                       const ptefit_tables *tb, const ptefit_basis *ba,
                                       const ptefit_options *op, ptefit_handle **out) {
  ptefit_handle *h = nullptr;
  if (out) *out = nullptr;
  if (!g || !ge || !tb || !ba || !op || !out) return fail(h, PTEFIT_ERR_INVALID_ARG, "null argument");
  int p2 = g->nz - 1;
  if (g->nz < 9 || g->nz > 257 || (p2 & (p2 - 1)) != 0) return fail(h, PTEFIT_ERR_INVALID_ARG, "nz-1 must be a power of two in [8,256]");
  if (g->nr < 5 || g->nr > 257) return fail(h, PTEFIT_ERR_INVALID_ARG, "nr must be in [5,257]");
  if (!(g->rmin > 0.0) || !(g->rmax > g->rmin) || !(g->zmax > g->zmin)) return fail(h, PTEFIT_ERR_INVALID_ARG, "bad grid extents");
  if (ge->n_meas < 1 || ge->n_coil < 1 || ge->n_coil > 768 || !ge->sigma || !ge->lim_mask || !ge->lim_r || !ge->lim_z)
    return fail(h, PTEFIT_ERR_INVALID_ARG, "bad geometry");
  if (ge->n_lim < 1 || ge->n_lim > PTEFIT_MAX_LIM) return fail(h, PTEFIT_ERR_INVALID_ARG, "n_lim must be in [1,256]");
  if (ge->ip_sign != 1 && ge->ip_sign != -1) return fail(h, PTEFIT_ERR_INVALID_ARG, "ip_sign must be +-1");
  if (!(ge->cold_a > 0.0) || !(ge->cold_b > 0.0)) return fail(h, PTEFIT_ERR_INVALID_ARG, "bad cold-start ellipse");
  for (int m = 0; m < ge->n_meas; ++m)
    if (!(ge->sigma[m] > 0.0)) return fail(h, PTEFIT_ERR_INVALID_ARG, "sigma must be > 0");
  for (int v = 0; v < ge->n_lim; ++v)
    if (ge->lim_r[v] < g->rmin || ge->lim_r[v] > g->rmax || ge->lim_z[v] < g->zmin || ge->lim_z[v] > g->zmax)
      return fail(h, PTEFIT_ERR_INVALID_ARG, "limiter vertex outside the grid");
  for (int j = 0; j < g->nz; ++j)
    for (int i = 0; i < g->nr; ++i)
      if (i == 0 || j == 0 || i == g->nr - 1 || j == g->nz - 1) {
        if (ge->lim_mask[j * g->nr + i] || (ge->xpt_mask && ge->xpt_mask[j * g->nr + i]))
          return fail(h, PTEFIT_ERR_INVALID_ARG, "lim_mask / xpt_mask must be 0 on edge nodes");
      }
  if (!tb->gp || !tb->gc || !tb->gb || !tb->ggc) return fail(h, PTEFIT_ERR_INVALID_ARG, "null table");
  if (ba->n_terms < 1 || ba->n_terms > PTEFIT_MAX_TERMS || !ba->terms) return fail(h, PTEFIT_ERR_INVALID_ARG, "n_terms must be in [1,16]");
  {
    const ptefit_term *sp0 = nullptr;
    for (int l = 0; l < ba->n_terms; ++l) {
      const ptefit_term &t = ba->terms[l];
      if (t.kind < 0 || t.kind > 2) return fail(h, PTEFIT_ERR_UNSUPPORTED, "unknown basis term kind");
      if (t.kind == 2 && l != ba->n_terms - 1) return fail(h, PTEFIT_ERR_INVALID_ARG, "the vertical-shift term must be last");
      if (t.kind == 2) continue;
      if (t.family < 0 || t.family > 1) return fail(h, PTEFIT_ERR_UNSUPPORTED, "unknown basis term family");
      if (t.family == 0 && (t.i < 0 || t.N <= t.i || t.N > 8)) return fail(h, PTEFIT_ERR_INVALID_ARG, "term exponents need 0 <= i < N <= 8");
      if (t.family == 1) {
        if (t.n_knots < 3 || t.n_knots > PTEFIT_MAX_KNOTS || !t.knots || !(t.tension > 0.0) || t.i < 0 || t.i >= t.n_knots)
          return fail(h, PTEFIT_ERR_INVALID_ARG, "spline term needs 3..16 knots, tension > 0 and 0 <= i < n_knots");
        for (int r = 0; r + 1 < t.n_knots; ++r)
          if (!(t.knots[r + 1] > t.knots[r])) return fail(h, PTEFIT_ERR_INVALID_ARG, "spline knots must be strictly increasing");
        if (sp0 && (sp0->n_knots != t.n_knots || sp0->tension != t.tension || memcmp(sp0->knots, t.knots, sizeof(double) * t.n_knots) != 0))
          return fail(h, PTEFIT_ERR_UNSUPPORTED, "all spline terms must share one knot set and tension");
        sp0 = &t;
      }
    }
  }
  if (ba->lsq_method != 0 && ba->lsq_method != 1) return fail(h, PTEFIT_ERR_INVALID_ARG, "lsq_method must be 0 (normal equations) or 1 (Gram-Schmidt QR)");
  if (ba->fit_coils != 0 && ba->fit_coils != 1) return fail(h, PTEFIT_ERR_INVALID_ARG, "fit_coils must be 0 or 1");
  if (ba->lsq_method == 1 || ba->n_terms > 12) {
    const size_t sm = ((size_t)(ge->n_meas + ba->n_terms) * (ba->n_terms + 1) + (size_t)ba->n_terms * (ba->n_terms + 1) + ba->n_terms) * sizeof(double);
    if (sm > 48 * 1024) return fail(h, PTEFIT_ERR_UNSUPPORTED, "lsq_method 1: (n_meas + n_terms)(n_terms + 1) doubles must fit 48 KB of shared memory");
  }
  if (ba->fit_coils) {
    if (!ba->sigma_ic) return fail(h, PTEFIT_ERR_INVALID_ARG, "fit_coils needs sigma_ic");
    for (int c = 0; c < ge->n_coil; ++c)
      if (!(ba->sigma_ic[c] > 0.0)) return fail(h, PTEFIT_ERR_INVALID_ARG, "sigma_ic must be > 0");
    if (ba->n_terms + ge->n_coil > JOINT_MAX_N || joint_smem_bytes(ge->n_meas, ba->n_terms, ge->n_coil) > 200 * 1024)
      return fail(h, PTEFIT_ERR_UNSUPPORTED, "fit_coils: n_terms + n_coil must be <= 96 and the normal matrix must fit 200 KB of shared memory");
    if (ba->lsq_method != 0) return fail(h, PTEFIT_ERR_UNSUPPORTED, "fit_coils uses the normal-equation driver (lsq_method 0)");
  }
  if (op->gemm != PTEFIT_GEMM_3XTF32 && op->gemm != PTEFIT_GEMM_FFMA) return fail(h, PTEFIT_ERR_INVALID_ARG, "gemm must be PTEFIT_GEMM_3XTF32 or PTEFIT_GEMM_FFMA");
  if (op->flags & ~(PTEFIT_OPT_NO_GRAPH | PTEFIT_OPT_NO_FUSED_BASIS | PTEFIT_OPT_SOLVE_FFMA)) return fail(h, PTEFIT_ERR_INVALID_ARG, "unknown option flag");
  if (op->tc_split_k < 0) return fail(h, PTEFIT_ERR_INVALID_ARG, "tc_split_k must be >= 0");
  if (op->gemm == PTEFIT_GEMM_FFMA && ba->n_terms > 12) return fail(h, PTEFIT_ERR_UNSUPPORTED, "PTEFIT_GEMM_FFMA supports at most 12 terms");
  if (ba->fit_coils && ba->n_terms > 12) return fail(h, PTEFIT_ERR_UNSUPPORTED, "fit_coils supports at most 12 terms");
  if (ba->n_terms == 1 && ba->terms[0].kind == 2) return fail(h, PTEFIT_ERR_INVALID_ARG, "need at least one P'/FF' term");
  if (!(ba->lambda_reg >= 0.0) || !(ba->relax > 0.0) || ba->relax > 1.0) return fail(h, PTEFIT_ERR_INVALID_ARG, "need lambda_reg >= 0 and 0 < relax <= 1");
  if (op->max_batch < 1 || op->max_batch > 65535) return fail(h, PTEFIT_ERR_INVALID_ARG, "max_batch must be in [1,65535]");
  if (op->precision != PTEFIT_FP32 && op->precision != PTEFIT_FP64) return fail(h, PTEFIT_ERR_INVALID_ARG, "bad precision");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return fail(h, PTEFIT_ERR_CUDA, "no CUDA device (there is no CPU fallback)");
  {
    int dev = 0, major = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (major != 10) return fail(h, PTEFIT_ERR_CUDA, "device is not sm_100 (the library is built for sm_100a only)");
  }
  h = new ptefit_handle();
  h->prec = op->precision; h->gemm = op->gemm; h->max_batch = op->max_batch;
  h->flags = op->flags; h->tc_split_k = op->tc_split_k;
  h->use_graph = !(op->flags & PTEFIT_OPT_NO_GRAPH);
  { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&h->nsm, cudaDevAttrMultiProcessorCount, dev); }
  ptefit_status st = (h->prec == PTEFIT_FP32) ? build(h, h->d32, g, ge, tb, ba, op->max_batch)
                                              : build(h, h->d64, g, ge, tb, ba, op->max_batch);
  if (st == PTEFIT_OK && h->prec == PTEFIT_FP32 && h->gemm != PTEFIT_GEMM_FFMA) { st = build_tc(h, h->d32, ge, tb, op->max_batch); if (st == PTEFIT_OK) st = build_tcsolve(h, h->d32); }
  if (st == PTEFIT_OK && h->prec == PTEFIT_FP64 && h->gemm != PTEFIT_GEMM_FFMA) st = build_dm(h, h->d64, ge, tb, op->max_batch);
  if (st != PTEFIT_OK) { std::string e = h->error; ptefit_destroy(h); g_error = e; return st; }
  *out = h;
  return PTEFIT_OK;
}

extern "C" void ptefit_destroy(ptefit_handle *h) {
  if (!h) return;
  for (void *p : h->allocs) cudaFree(p);
  for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
  void *hp[] = {h->hb, h->hic, h->hpsi, h->hco, h->hax, h->hxp, h->hpb, h->hchi, h->haxij, h->hxpij, h->hlim, h->hst};
  for (void *p : hp) if (p) cudaFree(p);
  for (auto &g : h->graphs) cudaGraphExecDestroy(g.exec);
  if (h->gstream) cudaStreamDestroy(h->gstream);
  if (h->hstream) cudaStreamDestroy(h->hstream);
  delete h;
}

extern "C" ptefit_status ptefit_greens_table(int n_fld, const double *fr, const double *fz, const double *fcos, const double *fsin,
                                             int n_src, const double *sr, const double *sz, const double *sw, double *out,
                                             int transpose, void *cuda_stream) {
  ptefit_handle *h = nullptr;
  if (n_fld < 1 || n_src < 1 || n_fld > 65535 || !fr || !fz || !sr || !sz || !out || (!fcos) != (!fsin))
    return fail(h, PTEFIT_ERR_INVALID_ARG, "ptefit_greens_table: bad arguments (1 <= n_fld <= 65535, n_src >= 1, non-null points)");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return fail(h, PTEFIT_ERR_CUDA, "no CUDA device (there is no CPU fallback)");
  k_greens_table<<<dim3((n_src + 255) / 256, n_fld), 256, 0, (cudaStream_t)cuda_stream>>>(n_fld, fr, fz, fcos, fsin, n_src, sr, sz, sw, out,
                                                                                        transpose ? 1 : 0);
  CK(cudaGetLastError());
  return PTEFIT_OK;
}

namespace {
template <typename T>
ptefit_status flux_surfaces(ptefit_handle *h, Dev<T> &D, int B, const ptefit_profile_spec *sp, const T *psi, T *Q, T *q, T *geom, T *vert,
                            int *fstat, cudaStream_t st) {
  FsSpec S{};
  S.n_prof = sp->n_prof; S.n_chord = sp->n_chord; S.n_bisect = sp->n_bisect; S.n_q = sp->n_q; S.f_vac = sp->f_vac; S.q_index = -1;
  for (int e = 0; e < sp->n_q; ++e) { S.mu[e] = sp->mu[e]; S.nu[e] = sp->nu[e]; if (sp->mu[e] == -1 && sp->nu[e] == -1) S.q_index = e; }
  S.ff0 = -1; S.n_ff = 0;
  for (int l = 0; l < D.nt; ++l)
    if (D.terms[l].kind == 1 && D.terms[l].family == 0) { if (S.ff0 < 0) S.ff0 = l; S.n_ff++; }
  if (S.ff0 < 0) S.ff0 = 0;
  const size_t sm = ((size_t)S.n_chord + 2 * (size_t)S.n_prof * S.n_chord) * sizeof(double);
  CK(cudaFuncSetAttribute(k_flux_surfaces<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
  // few slices: spread the levels of a slice over several CTAs
  int G = B >= 2 * h->nsm ? 1 : (2 * h->nsm + B - 1) / B;
  if (G > S.n_prof) G = S.n_prof;
  if (G > 16) G = 16;
  k_flux_surfaces<T><<<dim3(B, G), FS_THREADS, sm, st>>>(D, S, psi, Q, q, geom, vert, fstat);
  CK(cudaGetLastError());
  return PTEFIT_OK;
}
}  // namespace

extern "C" ptefit_status ptefit_flux_surfaces(ptefit_handle *h, int batch, const ptefit_profile_spec *sp, const void *d_psi, void *d_Q,
                                              void *d_q, void *d_geom, void *d_vert, int *d_status, void *cuda_stream) {
  if (!h || !sp || !d_psi || !d_Q || !d_q || !d_geom || batch < 1 || batch > h->max_batch)
    return fail(h, PTEFIT_ERR_INVALID_ARG, "ptefit_flux_surfaces: bad arguments");
  if (sp->n_prof < 1 || sp->n_chord < 3 || sp->n_chord > 1024 || (long long)sp->n_prof * sp->n_chord > 12288 || sp->n_bisect < 0 || sp->n_bisect > 60 ||
      sp->n_q < 1 || sp->n_q > FS_MAX_Q || !sp->mu || !sp->nu)
    return fail(h, PTEFIT_ERR_INVALID_ARG, "ptefit_flux_surfaces: need 1 <= n_prof, 3 <= n_chord <= 1024, n_prof n_chord <= 12288, 0 <= n_bisect <= 60, 1 <= n_q <= 8");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (h->prec == PTEFIT_FP32)
    return flux_surfaces<float>(h, h->d32, batch, sp, (const float *)d_psi, (float *)d_Q, (float *)d_q, (float *)d_geom, (float *)d_vert, d_status, st);
  return flux_surfaces<double>(h, h->d64, batch, sp, (const double *)d_psi, (double *)d_Q, (double *)d_q, (double *)d_geom, (double *)d_vert, d_status, st);
}

extern "C" ptefit_status ptefit_get_coil_currents(ptefit_handle *h, int batch, void *d_out, void *cuda_stream) {
  if (!h || !d_out || batch < 1 || batch > h->max_batch) return fail(h, PTEFIT_ERR_INVALID_ARG, "ptefit_get_coil_currents: bad arguments");
  const bool on = h->prec == PTEFIT_FP32 ? h->d32.fit_coils : h->d64.fit_coils;
  if (!on) return fail(h, PTEFIT_ERR_INVALID_ARG, "ptefit_get_coil_currents: the handle was created without fit_coils");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (h->prec == PTEFIT_FP32) k_export_ic<float><<<(batch * h->d32.nc + 255) / 256, 256, 0, st>>>(h->d32, batch, (float *)d_out);
  else k_export_ic<double><<<(batch * h->d64.nc + 255) / 256, 256, 0, st>>>(h->d64, batch, (double *)d_out);
  CK(cudaGetLastError());
  return PTEFIT_OK;
}

extern "C" const char *ptefit_last_error(const ptefit_handle *h) { return h ? h->error.c_str() : g_error.c_str(); }
extern "C" const char *ptefit_global_error(void) { return g_error.c_str(); }
extern "C" int ptefit_last_launch_count(const ptefit_handle *h) { return h ? h->launches : 0; }

#include "launch.inc"

// ---------------------------------------------------------------------------------------------------------
// ptefit_gs_solve_noalloc (include/ptefit.h): the GEMM-based FP64 Delta* solve (launch_solve_dm's sequence:
// PAPER.md:33 Eq. 1) with its whole workspace in one file-scope device array instead of the
// handle's cudaMalloc'ed buffers.  Every GPU that loads the library holds the array until exit; all calls
// share it and it keeps the last call's contents.
// ---------------------------------------------------------------------------------------------------------
#include <mutex>

static __device__ __align__(256) unsigned char g_noalloc_scratch[PTEFIT_NOALLOC_SCRATCH_BYTES];

namespace ptefit {
// k_tridiag_ld with both of its work arrays passed in: Thomas sweeps along R in FP64, one thread per
// (slice, mode), in place on fh[(s, i)][m] (row length ld); forward-sweep values in y[(s, i)][m] (row length
// nzi).  grid (ceil(nzi/128), B), block 128.
__global__ void k_tridiag_ld_scratch(Dev<double> D, int ld, double *__restrict__ fh_all, double *__restrict__ y_all) {
  const int s = blockIdx.y, mm = blockIdx.x * blockDim.x + threadIdx.x;
  if (mm >= D.nzi) return;
  const int nri = D.nri, nzi = D.nzi;
  double *fh = fh_all + (size_t)s * nri * ld;
  double *y = y_all + (size_t)s * nri * nzi;
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
}  // namespace ptefit

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mu;
void *g_noalloc_ptr[NOALLOC_MAX_DEVICES];      // device address of g_noalloc_scratch on device d (0 = not resolved yet)

// In host code `g_noalloc_scratch` is only a stand-in for the symbol, not a device address: resolve it once per
// device, with that device current.
ptefit_status noalloc_scratch(ptefit_handle *h, double **out) {
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(h, PTEFIT_ERR_UNSUPPORTED, "ptefit_gs_solve_noalloc: device ordinal beyond 63");
  std::lock_guard<std::mutex> lk(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    void *p = nullptr;
    CK(cudaGetSymbolAddress(&p, g_noalloc_scratch));
    if (!p) return fail(h, PTEFIT_ERR_CUDA, "ptefit_gs_solve_noalloc: cudaGetSymbolAddress returned a null address");
    g_noalloc_ptr[dev] = p;
  }
  *out = reinterpret_cast<double *>(g_noalloc_ptr[dev]);
  return PTEFIT_OK;
}
}  // namespace

extern "C" ptefit_status ptefit_gs_solve_noalloc(ptefit_handle *h, int batch, const double *d_I, const double *d_pbd, double *d_psi,
                                                 void *cuda_stream) {
  if (!h) return fail(h, PTEFIT_ERR_INVALID_ARG, "null handle");
  if (batch < 1) return fail(h, PTEFIT_ERR_INVALID_ARG, "batch must be >= 1");
  if (!d_I || !d_pbd || !d_psi) return fail(h, PTEFIT_ERR_INVALID_ARG, "null buffer");
  if (h->prec != PTEFIT_FP64 || !h->dm)
    return fail(h, PTEFIT_ERR_UNSUPPORTED, "ptefit_gs_solve_noalloc needs an FP64 handle whose contractions are not FFMA");
  const Dev<double> &D = h->d64;
  DmDev T = h->Dm;                                   // copy: the three transposed maps move into the static array
  const size_t n_t = (size_t)batch * D.nri * T.ldS;  // doubles per transposed map (even: 16-byte rows for cp.async)
  const size_t n_y = (size_t)batch * D.nri * D.nzi;
  const size_t need = (3 * n_t + n_y) * sizeof(double);
  if (need > (size_t)PTEFIT_NOALLOC_SCRATCH_BYTES) {
    char msg[256];
    snprintf(msg, sizeof msg, "ptefit_gs_solve_noalloc: batch %d on a %d x %d grid needs %zu bytes of scratch, the static array holds %u "
             "(at most %zu slices of this grid per call)", batch, D.nr, D.nz, need, (unsigned)PTEFIT_NOALLOC_SCRATCH_BYTES,
             (size_t)PTEFIT_NOALLOC_SCRATCH_BYTES / (((size_t)3 * T.ldS + D.nzi) * D.nri * sizeof(double)));
    return fail(h, PTEFIT_ERR_INVALID_ARG, msg);
  }
  double *s = nullptr;
  TRY(noalloc_scratch(h, &s));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // the array keeps the previous call's contents: the padding column of the transposed maps (never written by
  // the kernels below) must read as zero, so the part this call uses is cleared
  CK(cudaMemsetAsync(s, 0, need, st));
  T.ft = s; T.fh = s + n_t; T.gt = s + 2 * n_t;
  double *y = s + 3 * n_t;
  const dim3 gt((D.nri + 31) / 32, (D.nzi + 31) / 32, batch), bt(32, 8);
  k_rhs_t<<<gt, bt, 0, st>>>(D, T, d_I, d_pbd);
  gemm_dmma(T.ft, T.ldS, T.S, T.ldS, T.fh, T.ldS, batch * D.nri, D.nzi, D.nzi, 1, 0, 1.0, st);
  k_tridiag_ld_scratch<<<dim3((D.nzi + 127) / 128, batch), 128, 0, st>>>(D, T.ldS, T.fh, y);
  gemm_dmma(T.fh, T.ldS, T.S, T.ldS, T.gt, T.ldS, batch * D.nri, D.nzi, D.nzi, 1, 0, 2.0 / (D.nz - 1), st);
  k_total_t<<<gt, bt, 0, st>>>(D, T, d_psi, 0, 0);
  k_edge_total<double><<<dim3((D.nbnd + 255) / 256, batch), 256, 0, st>>>(D, d_psi, d_pbd, 0, 0);
  CK(cudaGetLastError());
  return PTEFIT_OK;
}
