// fused_solve.cuh -- A7 + A8 + A1 (+ the vertical-shift column) of one slice in ONE CTA, flux map
// resident in shared memory:
//   rhs assembly -> DST-I in Z -> FP64 Thomas in R -> DST-I in Z -> psi = psi_pl + psi_coil with
//   relaxation -> axis / X-point / LCFS search and normalisation -> -dI'/dZ column.
// Delta* psi = -mu0 R J_phi on the 5-point stencil (Eq. 1, 118-120); search per
// PAPER.md:122-136.  The DST is a folded dense product: sin(pi (Nz-j) m / Nz) = (-1)^(m+1)
// sin(pi j m / Nz), so odd modes see f_j + f_{Nz-j} and even modes f_j - f_{Nz-j}: two
// (Nz/2)^2 products instead of one (Nz-1)^2.  Used when the slice fits shared memory
// (e.g. 129x129 FP32 = 108 KB, two CTAs per SM); larger grids take the three-kernel path of
// solve_kernels.cuh.  Persistent: CTA b handles slices b, b + gridDim.x, ...
#pragma once
#include "common.cuh"
#include "search_kernels.cuh"

namespace ptefit {

constexpr int FUSED_THREADS = 256;
constexpr int FUSED_CW = 16;       // columns per DST chunk

template <typename T> struct Vec4 { T v[4]; };
__device__ __forceinline__ Vec4<float> load4(const float *p) {
  const float4 q = *reinterpret_cast<const float4 *>(p);
  return {{q.x, q.y, q.z, q.w}};
}
__device__ __forceinline__ Vec4<double> load4(const double *p) {
  const double2 a = *reinterpret_cast<const double2 *>(p), b = *reinterpret_cast<const double2 *>(p + 2);
  return {{a.x, a.y, b.x, b.y}};
}
template <typename T> struct Vec2 { T v[2]; };
__device__ __forceinline__ Vec2<float> load2(const float *p) {
  const float2 q = *reinterpret_cast<const float2 *>(p);
  return {{q.x, q.y}};
}
__device__ __forceinline__ Vec2<double> load2(const double *p) {
  const double2 q = *reinterpret_cast<const double2 *>(p);
  return {{q.x, q.y}};
}

// Shared-memory bytes of k_solve_fused for a grid (host and device agree through this).
template <typename T>
__host__ __device__ inline size_t fused_smem_bytes(int nr, int nz) {
  const int n2 = (nz - 1) / 2;
  const size_t g = ((size_t)nz * nr + 3) & ~(size_t)3;          // 16-byte aligned sub-arrays
  size_t e = 2 * (size_t)n2 * FUSED_CW * sizeof(T);              // fold buffer, reused for the bit masks
  const size_t mb = 3 * (((size_t)nz * nr + 31) / 32) * sizeof(unsigned);   // lim, xpt, edge bit masks
  if (mb > e) e = mb;
  const size_t pbb = (size_t)(2 * (nr + nz) - 4) * sizeof(T);   // ... and for the boundary flux
  if (pbb > e) e = pbb;
  const size_t exb = 2 * (size_t)(FUSED_THREADS / 2) * sizeof(double);   // ... and for the twisted-Thomas hand-over
  if (exb > e) e = exb;
  e = (e + 15) & ~(size_t)15;
  return (g + 2 * (size_t)n2 * n2) * sizeof(T) + e;
}

// In-place DST-I along Z of the interior columns of G[nz][nr] (rows 1..nz-2 <-> modes 1..nz-2),
// unnormalised: G[m][i] <- sum_j sin(pi j m / (nz-1)) G[j][i].
template <typename T>
__device__ void dst_columns(T *G, const T *So, const T *Se, T *E, int nr, int nz) {
  const int Nz = nz - 1, n2 = Nz / 2, nri = nr - 2, nzi = nz - 2;
  const int nq = n2 / 4, ncq = FUSED_CW / 4;
  const int items = 2 * nq * ncq;                              // 4 modes x 4 columns per item
  const int tid = threadIdx.x, nth = blockDim.x;
  for (int c0 = 0; c0 < nri; c0 += FUSED_CW) {
    for (int e = tid; e < n2 * FUSED_CW; e += nth) {          // fold rows j and Nz-j
      const int jj = e / FUSED_CW, c = e - jj * FUSED_CW;
      const int i = 1 + c0 + c;
      T a = T(0), b = T(0);
      if (i <= nri) {
        const T lo = G[(jj + 1) * nr + i];
        if (jj + 1 < n2) { const T hi = G[(Nz - jj - 1) * nr + i]; a = lo + hi; b = lo - hi; }
        else a = lo;                                           // centre row j = Nz/2
      }
      E[e] = a;
      E[n2 * FUSED_CW + e] = b;
    }
    __syncthreads();
    for (int it = tid; it < items; it += nth) {
      const int cq = it % ncq, q = (it / ncq) % nq, par = it / (ncq * nq);
      const T *St = (par ? Se : So) + 4 * q;
      const T *Ep = E + par * n2 * FUSED_CW + 4 * cq;
      T acc[4][4];
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int t = 0; t < 4; ++t) acc[r][t] = T(0);
#pragma unroll 4
      for (int j = 0; j < n2; ++j) {
        const Vec4<T> sv = load4(St + j * n2);
        const Vec4<T> ev = load4(Ep + j * FUSED_CW);
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
          for (int t = 0; t < 4; ++t) acc[r][t] = fma(sv.v[r], ev.v[t], acc[r][t]);
      }
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const int m = 2 * (4 * q + r) + 1 + par;
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          const int i = 1 + c0 + 4 * cq + t;
          if (m <= nzi && i <= nri) G[m * nr + i] = acc[r][t];
        }
      }
    }
    __syncthreads();
  }
}


__device__ __forceinline__ void cp_async4(void *smem, const void *gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(sa), "l"(gmem));
}
__device__ __forceinline__ void cp_async8(void *smem, const void *gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(sa), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p)); }

// grid min(B, resident CTAs), block FUSED_THREADS, dyn smem fused_smem_bytes<T>(nr, nz).
// cur[B][N] node currents (A), pbd[B][nbnd] boundary flux, psi[B][N] in/out.
// do_search = 0: Delta* solve only (debug hook); 1: also search + xn (+ dzc when has_delz).
template <typename T>
__global__ void __launch_bounds__(FUSED_THREADS, 2) k_solve_fused(Dev<T> D, int B, const T *__restrict__ cur_all,
                                                                const T *__restrict__ pbd_all, T *__restrict__ psi_all,
                                                                T *__restrict__ xn_all, int use_relax, int add_coil,
                                                                int do_search) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  if (!psi_all) psi_all = reinterpret_cast<T *>(D.ca->psi);
  const int nr = D.nr, nz = D.nz, N = D.N, nri = D.nri, nzi = D.nzi, Nz = nz - 1, n2 = Nz / 2;
  const int tid = threadIdx.x, nth = blockDim.x, warp = tid >> 5, lane = tid & 31, nwarp = nth >> 5;
  T *G = reinterpret_cast<T *>(smem_raw);
  T *So = G + ((N + 3) & ~3);
  T *Se = So + n2 * n2;
  T *E = Se + n2 * n2;
  unsigned *mbits = reinterpret_cast<unsigned *>(E);        // during the search: lim bits, then xpt bits
  const int nwords = (N + 31) >> 5;
  for (int e = tid; e < 2 * n2 * n2; e += nth) So[e] = D.dst_tab[e];    // So then Se, contiguous
  // per-column constants (same expressions as the unfused kernels, evaluated once per CTA)
  __shared__ T c_rhs[PTEFIT_MAX_NR], c_rdA[PTEFIT_MAX_NR], c_fdA[PTEFIT_MAX_NR];
  __shared__ T pcoef[2 * (PTEFIT_MAX_DEG + 1)];              // I'(x) = rdA P(x) + fdA Q(x)
  __shared__ T c_edge[2];
  for (int i = tid; i < nr; i += nth) {
    const double Rd = D.rmin + i * D.dr;
    c_rhs[i] = T(-kMu0 * Rd / D.dA);
    const T R = T(Rd);
    c_rdA[i] = R * T(D.dA);
    c_fdA[i] = T(kMu0 * D.dA) / R;
    if (i == 1) c_edge[0] = T((1.0 + D.dr / (2.0 * Rd)) / (D.dr * D.dr));
    if (i == nri) c_edge[1] = T((1.0 - D.dr / (2.0 * Rd)) / (D.dr * D.dr));
  }
  const T cz = T(1.0 / (D.dz * D.dz));
  const T scale = T(2.0 / Nz);
  const T esc = scale;
  const T om = T(D.relax);
  const double sg = (double)D.ip_sign;
  for (int s = blockIdx.x; s < B; s += gridDim.x) {
    const T *I = cur_all + (size_t)s * N;
    const T *pbg = pbd_all + (size_t)s * D.nbnd;          // bottom[nr], top[nr], left[nzi], right[nzi]
    const T *pb = E;                                       // staged in the fold buffer (free until the DST)
    T *psi = psi_all + (size_t)s * N;
    const T *pc = D.psi_coil + (size_t)s * N;
    __syncthreads();                                       // previous slice done with G; tables loaded
    // ---- node currents straight into shared memory (asynchronous copies, no register staging)
    for (int k = tid; k < D.nbnd; k += nth) E[k] = pbg[k];
    for (int n = tid; n < N; n += nth) {
      if (sizeof(T) == 4) cp_async4(G + n, I + n); else cp_async8(G + n, I + n);
    }
    // inputs of the later phases: pull them into L2 while the solve runs
    {
      const int lines = (int)(((size_t)N * sizeof(T) + 127) / 128);
      for (int l = tid; l < lines; l += nth) {
        if (add_coil) prefetch_l2(reinterpret_cast<const char *>(pc) + (size_t)l * 128);
        if (use_relax) prefetch_l2(reinterpret_cast<const char *>(psi) + (size_t)l * 128);
      }
    }
    if (do_search && D.has_delz && tid < 2 * (PTEFIT_MAX_DEG + 1)) {
      // the P'/FF' sums of I' = J_b(x) X are polynomials in x: collect their coefficients
      const int kind = tid / (PTEFIT_MAX_DEG + 1), k = tid - kind * (PTEFIT_MAX_DEG + 1);
      const double *Xp = D.X + (size_t)s * D.nt;
      double c = 0.0;
      for (int l = 0; l < D.npoly; ++l)
        if (D.terms[l].kind == kind && D.terms[l].family == 0) c += Xp[l] * ((D.terms[l].i == k ? 1.0 : 0.0) - (D.terms[l].N == k ? 1.0 : 0.0));
      pcoef[tid] = T(c);
    }
    cp_async_wait_all();
    __syncthreads();
    {
    // ---- right-hand side -mu0 R I / dA with the Dirichlet data moved over (interior), edge data (edges)
    // (one warp per grid row: the row tests are warp-uniform, the column tests plain selects)
    for (int j = warp; j < nz; j += nwarp) {
      T *row = G + j * nr;
      if (j == 0 || j == nz - 1) {
        const T *src = pb + (j ? nr : 0);
        for (int i = lane; i < nr; i += 32) row[i] = src[i];
        continue;
      }
      const T pl = pb[2 * nr + j - 1], pr = pb[2 * nr + nzi + j - 1];
      const T el = c_edge[0] * pl, er = c_edge[1] * pr;
      for (int i = lane; i < nr; i += 32) {
        T v = c_rhs[i] * row[i];
        if (i == 1) v -= el;
        if (i == nri) v -= er;
        if (j == 1) v -= cz * pb[i];
        if (j == nzi) v -= cz * pb[nr + i];
        if (i == 0) v = pl;
        if (i == nr - 1) v = pr;
        row[i] = v;
      }
    }
    __syncthreads();
    dst_columns<T>(G, So, Se, E, nr, nz);
    // ---- Thomas sweeps along R in FP64, one thread per mode (precomputed factors).
    // The dependent chain is one DFMA per step.
    if (2 * nzi <= nth && nri >= 3) {
      // twisted factorisation: threads [0, nth/2) eliminate rows 0..k-1 downwards, threads
      // [nth/2, nth) rows n-1..k+1 upwards; row k couples the halves; both substitute outwards.
      const int half = nth >> 1, side = tid >= half, mm = tid - side * half;
      const int n = nri, k = n / 2, len = side ? n - 1 - k : k;
      double *ex = reinterpret_cast<double *>(E);          // [2][half] elimination results next to row k
      const bool act = mm < nzi;
      T *row = G + (mm + 1) * nr + 1;
      double *__restrict__ y = D.ytmp + (size_t)blockIdx.x * nri * nzi + mm;
      const double *__restrict__ tw = D.tw2 + mm;
      const double *__restrict__ tb = D.tib2 + mm;
      const double *__restrict__ tod = D.tod2;
      constexpr int U = 8;
      double prev = 0.0;
      if (act) {
        for (int t0 = 0; t0 < len; t0 += U) {
          double w[U];
#pragma unroll
          for (int u = 0; u < U; ++u) {
            const int t = t0 + u, i = side ? n - 1 - t : t;
            w[u] = (t < len) ? __ldg(tw + (size_t)i * nzi) : 0.0;
          }
#pragma unroll
          for (int u = 0; u < U; ++u) {
            const int t = t0 + u, i = side ? n - 1 - t : t;
            if (t < len) {
              const double v = fma(-w[u], prev, (double)row[i]);
              y[(size_t)i * nzi] = v;
              prev = v;
            }
          }
        }
        ex[side * half + mm] = prev;                       // y_{k-1} (left) or y_{k+1} (right)
      }
      // both threads of a mode need the right-hand side of row k; the left one overwrites it below,
      // so it is read before the barrier
      const double gk = act ? (double)row[k] : 0.0;
      __syncthreads();
      double x = 0.0;
      if (act) {
        const double yk = gk - __ldg(tw + (size_t)k * nzi) * ex[mm] - __ldg(D.tw2k + mm) * ex[half + mm];
        x = yk * __ldg(tb + (size_t)k * nzi);
        if (!side) row[k] = T(x);
        for (int t0 = len - 1; t0 >= 0; t0 -= U) {
          double a[U], b[U];
#pragma unroll
          for (int u = 0; u < U; ++u) {
            const int t = t0 - u, i = side ? n - 1 - t : t;
            const double ib = t >= 0 ? __ldg(tb + (size_t)i * nzi) : 0.0;
            a[u] = t >= 0 ? y[(size_t)i * nzi] * ib : 0.0;
            b[u] = t >= 0 ? __ldg(tod + i) * ib : 0.0;
          }
#pragma unroll
          for (int u = 0; u < U; ++u) {
            const int t = t0 - u, i = side ? n - 1 - t : t;
            if (t >= 0) {
              x = fma(-b[u], x, a[u]);                     // x_i = (y_i - offdiag_i x_neighbour) / piv_i
              row[i] = T(x);
            }
          }
        }
      }
    } else     if (tid < nzi) {
      const int mm = tid;
      T *row = G + (mm + 1) * nr + 1;
      double *__restrict__ y = D.ytmp + (size_t)blockIdx.x * nri * nzi + mm;
      const double *__restrict__ tw = D.tri_w + mm;
      const double *__restrict__ tb = D.tri_invb + mm;
      const double *__restrict__ tce = D.tri_ce;
      constexpr int U = 8;                     // loads of U steps are issued before the dependent chain
      double prev = 0.0;
      for (int i0 = 0; i0 < nri; i0 += U) {
        double w[U];
#pragma unroll
        for (int u = 0; u < U; ++u) w[u] = (i0 + u < nri) ? __ldg(tw + (size_t)(i0 + u) * nzi) : 0.0;
#pragma unroll
        for (int u = 0; u < U; ++u)
          if (i0 + u < nri) {
            const double v = fma(-w[u], prev, (double)row[i0 + u]);
            y[(size_t)(i0 + u) * nzi] = v;
            prev = v;
          }
      }
      double x = 0.0;
      for (int i0 = nri - 1; i0 >= 0; i0 -= U) {
        double a[U], b[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const int i = i0 - u;
          const double ib = i >= 0 ? __ldg(tb + (size_t)i * nzi) : 0.0;
          a[u] = i >= 0 ? y[(size_t)i * nzi] * ib : 0.0;
          b[u] = i >= 0 ? __ldg(tce + i) * ib : 0.0;
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
          if (i0 - u >= 0) {
            x = fma(-b[u], x, a[u]);                       // x_i = (y_i - ce_i x_{i+1}) / piv_i
            row[i0 - u] = T(x);
          }
      }
    }
    __syncthreads();
    dst_columns<T>(G, So, Se, E, nr, nz);
    }
    // ---- bit masks of the search into the (now free) fold buffer
    for (int w = tid; w < 3 * nwords; w += nth)
      mbits[w] = (w < nwords) ? D.lim_bits[w] : (w < 2 * nwords) ? D.xpt_bits[w - nwords] : D.edge_bits[w - 2 * nwords];
    __syncthreads();
    // ---- total flux + relaxation; psi goes to global memory and stays in G for the search.
    // Global loads are issued in batches of EB before use; pass 0 of the search (finiteness and
    // arg-max over the limiter mask) rides along.
    SearchOpt<T> so_opt;
    so_opt.am.v = -INFINITY; so_opt.am.n = 0x7fffffff;
    {
      // flat over the nodes (coalesced, no index arithmetic: edge nodes from a bit mask); the global
      // loads of a batch are issued before use; the arg-max key is kept in T (exact) and widened below
      constexpr int EB = 8;
      const unsigned *ebits = mbits + 2 * nwords;
      const T sgT = T(D.ip_sign);
      T am_v = -INFINITY;
      int am_n = 0x7fffffff;
      for (int n0 = tid; n0 < N; n0 += EB * nth) {
        T cv[EB], ov[EB];
#pragma unroll
        for (int u = 0; u < EB; ++u) {
          const int n = n0 + u * nth;
          cv[u] = (add_coil && n < N) ? pc[n] : T(0);
          ov[u] = (use_relax && n < N) ? psi[n] : T(0);
        }
#pragma unroll
        for (int u = 0; u < EB; ++u) {
          const int n = n0 + u * nth;
          if (n < N) {
            const unsigned bit = 1u << (n & 31);
            const T g = G[n];
            T v = (ebits[n >> 5] & bit) ? g : g * esc;
            v += cv[u];
            if (use_relax) v = ov[u] + om * (v - ov[u]);
            psi[n] = v;
            G[n] = v;
            if (do_search) {
              so_opt.bad |= !isfinite(v);
              const T key = sgT * v;
              if ((mbits[n >> 5] & bit) && (key > am_v || (key == am_v && n < am_n))) { am_v = key; am_n = n; }
            }
          }
        }
      }
      so_opt.am.v = (double)am_v;
      so_opt.am.n = am_n;
    }
    __syncthreads();
    if (do_search) {
      T *xn = xn_all + (size_t)s * N;
      so_opt.lbits = mbits; so_opt.xbits = mbits + nwords; so_opt.have_am = true;
      so_opt.local = G;
      if (D.has_delz) { so_opt.pc = pcoef; so_opt.rdA = c_rdA; so_opt.fdA = c_fdA; so_opt.Xs = D.X + (size_t)s * D.nt; }
      search_body<T>(D, s, G, xn, so_opt);                 // G now holds I'(xn) (delz) or xn
      if (D.has_delz) {
        // -dI'/dZ column for the NEXT fit (I' = J_b(xn) X with the coefficients of this fit)
        __syncthreads();
        T *dzc = D.dzc + (size_t)s * N;
        const T hz = T(0.5 / D.dz);
        const unsigned *ebits = mbits + 2 * nwords;        // the masks are still in the fold buffer
#pragma unroll 4
        for (int n = tid; n < N; n += nth) {
          const bool edge = (ebits[n >> 5] >> (n & 31)) & 1u;
          const int up = edge ? n : n + nr, dn = edge ? n : n - nr;
          dzc[n] = edge ? T(0) : -(G[up] - G[dn]) * hz;
        }
      }
    }
  }
}

}  // namespace ptefit
