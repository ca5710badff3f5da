// fluxsurf_kernels.cuh -- NEXT-2: flux-surface post-processing (PAPER.md:138-148,
// Sec. II.E, Eq. 12, Fig. 1).  One CTA per slice.  Phase 1: one thread per chord marches outwards from the
// refined axis to the first point of the filtered flux with F >= 1 (the boundary end of the chord).
// Phase 2: one thread per (level, chord): n_bisect halvings of [0, t_b] on F(t) - x_p, then one linear
// interpolation ("about 10 iterations").  Phase 3: per level, trapezoid rule of
// |grad psi|^mu R^nu dl over the closed polygon of the chord vertices (one warp per level), the safety
// factor q = (mu0 F / 2 pi) Q_{-1,-1} with F(x)^2 = F_vac^2 - 2 (psi_b - psi_a) int_x^1 FF', and the LCFS
// geometry.  Readings as in DESIGN.md O8: F = psi_N inside the plasma mask, max(1, raw psi_N) outside;
// |grad psi| from the bilinear interpolant of the vertex's cell.  All arithmetic in FP64 on the T-typed
// flux maps (a few thousand bisections per slice: not worth an FP32 variant).
#pragma once
#include "common.cuh"

namespace ptefit {

constexpr int FS_THREADS = 256;
constexpr int FS_MAX_Q = 8;

struct FsSpec {
  int n_prof, n_chord, n_bisect, n_q, n_ff, ff0;      // ff0 = index of the first FF' polynomial term in X
  int mu[FS_MAX_Q], nu[FS_MAX_Q];
  int q_index;                                        // which (mu, nu) pair is (-1, -1), or -1
  double f_vac;
};

// x^e for a small integer exponent (Eq. 12's mu, nu): multiplications and one reciprocal instead of pow().
__device__ __forceinline__ double fs_ipow(double x, int e) {
  double p = 1.0;
  const int n = e < 0 ? -e : e;
  for (int k = 0; k < n; ++k) p *= x;
  return e < 0 ? 1.0 / p : p;
}

template <typename T>
struct FsField {
  const T *psi, *xn;
  int nr, nz;
  double rmin, zmin, dr, dz, rmax, zmax, pa, inv, idr, idz;
  __device__ __forceinline__ double F(int n) const {
    const double x = (double)xn[n];
    return x >= 0.0 ? x : fmax(((double)psi[n] - pa) * inv, 1.0);
  }
  __device__ __forceinline__ void cell(double R, double Z, int &n0, double &tx, double &ty) const {
    const double fi = (R - rmin) / dr, fj = (Z - zmin) / dz;
    int i0 = (int)floor(fi), j0 = (int)floor(fj);
    i0 = max(0, min(i0, nr - 2)); j0 = max(0, min(j0, nz - 2));
    tx = fi - i0; ty = fj - j0; n0 = j0 * nr + i0;
  }
  // the filtered field is continuous across cell edges, so the cell may be found with reciprocal spacings here
  // (cell() keeps the divisions: the gradient of the interpolant is not continuous)
  __device__ __forceinline__ double Fat(double R, double Z) const {
    const double fi = (R - rmin) * idr, fj = (Z - zmin) * idz;
    int i0 = (int)floor(fi), j0 = (int)floor(fj);
    i0 = max(0, min(i0, nr - 2)); j0 = max(0, min(j0, nz - 2));
    const double tx = fi - i0, ty = fj - j0;
    const int n0 = j0 * nr + i0;
    return (1.0 - ty) * ((1.0 - tx) * F(n0) + tx * F(n0 + 1)) + ty * ((1.0 - tx) * F(n0 + nr) + tx * F(n0 + nr + 1));
  }
  __device__ __forceinline__ bool inside(double R, double Z) const { return R > rmin && R < rmax && Z > zmin && Z < zmax; }
};

// grid (B, G): CTA (s, g) handles the levels p = g, g + G, ... of slice s (every CTA repeats the cheap marching
// phase; the CTA that owns the last level writes the geometry).  block FS_THREADS, dyn smem (n_chord + 2 n_prof n_chord) doubles.
// Q[B][n_prof][n_q], q[B][n_prof], geom[B][6], vert[B][n_prof][n_chord][2] (may be nullptr), fstat[B].
template <typename T>
__global__ void __launch_bounds__(FS_THREADS) k_flux_surfaces(Dev<T> D, FsSpec S, const T *__restrict__ psi_all, T *__restrict__ Qo,
                                                              T *__restrict__ qo, T *__restrict__ geom, T *__restrict__ vert,
                                                              int *__restrict__ fstat) {
  extern __shared__ __align__(16) unsigned char fs_raw[];
  double *tb = reinterpret_cast<double *>(fs_raw);                 // [n_chord] boundary end of every chord
  double *vr = tb + S.n_chord;                                     // [n_prof][n_chord] vertex R
  double *vz = vr + (size_t)S.n_prof * S.n_chord;                  // [n_prof][n_chord] vertex Z
  __shared__ int sh_bad;
  const int s = blockIdx.x, tid = threadIdx.x, nth = blockDim.x, lane = tid & 31, warp = tid >> 5;
  const int G = gridDim.y, g0 = blockIdx.y;
  const int npl = g0 < S.n_prof ? (S.n_prof - 1 - g0) / G + 1 : 0;          // levels of this CTA: p = g0 + k G, k < npl
  const SearchOut so = D.so[s];
  FsField<T> f;
  f.psi = psi_all + (size_t)s * D.N; f.xn = D.xn + (size_t)s * D.N; f.nr = D.nr; f.nz = D.nz;
  f.rmin = D.rmin; f.zmin = D.zmin; f.dr = D.dr; f.dz = D.dz; f.idr = 1.0 / D.dr; f.idz = 1.0 / D.dz;
  f.rmax = D.rmin + (D.nr - 1) * D.dr; f.zmax = D.zmin + (D.nz - 1) * D.dz;
  f.pa = so.axis_psi; f.inv = 1.0 / (so.psi_b - so.axis_psi);
  const double Ra = so.axis_r, Za = so.axis_z;
  const double h = 0.5 * fmin(D.dr, D.dz);
  const double two_pi = 6.283185307179586476925;
  if (tid == 0) sh_bad = D.status[s] != 0 ? 1 : 0;
  __syncthreads();
  const bool dead = sh_bad != 0;
  if (!dead)                                           // one warp per chord: 32 marching steps at a time, first hit by ballot
    for (int c = warp; c < S.n_chord; c += nth >> 5) {
      const double th = two_pi * c / S.n_chord, ct = cos(th), st = sin(th);
      int k = 0;
      for (int base = 1; k == 0; base += 32) {
        const int kk = base + lane;
        const double R = Ra + kk * h * ct, Z = Za + kk * h * st;
        const bool hit = !f.inside(R, Z) || f.Fat(R, Z) >= 1.0;
        const unsigned m = __ballot_sync(0xffffffffu, hit);
        if (m) k = base + __ffs(m) - 1;
      }
      if (lane == 0) {
        tb[c] = k * h;
        if (k == 1 && f.Fat(Ra, Za) >= 1.0) sh_bad = 2;
      }
    }
  __syncthreads();
  if (!dead)
    for (int e0 = tid; e0 < npl * S.n_chord; e0 += nth) {
      const int pk = e0 / S.n_chord, c = e0 - pk * S.n_chord, p = g0 + pk * G, e = p * S.n_chord + c;
      const double th = two_pi * c / S.n_chord, ct = cos(th), st = sin(th);
      const double x = (p + 1.0) / S.n_prof;
      double lo = 0.0, hi = tb[c];
      for (int it = 0; it < S.n_bisect; ++it) {
        const double mid = 0.5 * (lo + hi);
        const double R = Ra + mid * ct, Z = Za + mid * st;
        const double fm = f.inside(R, Z) ? f.Fat(R, Z) : 1.0;
        if (fm < x) lo = mid; else hi = mid;
      }
      const double fl = f.Fat(Ra + lo * ct, Za + lo * st);
      const double Rh = Ra + hi * ct, Zh = Za + hi * st;
      const double fh = f.inside(Rh, Zh) ? f.Fat(Rh, Zh) : 1.0;
      double w = fh > fl ? (x - fl) / (fh - fl) : 0.5;
      w = fmin(fmax(w, 0.0), 1.0);
      const double t = lo + w * (hi - lo);
      vr[e] = Ra + t * ct; vz[e] = Za + t * st;
      if (vert) { vert[((size_t)s * S.n_prof * S.n_chord + e) * 2] = T(vr[e]); vert[((size_t)s * S.n_prof * S.n_chord + e) * 2 + 1] = T(vz[e]); }
    }
  __syncthreads();
  // closed integrals: one warp per level, lanes over polygon edges
  const double *X = D.X + (size_t)s * D.nt;
  for (int pk = warp; pk < npl; pk += nth >> 5) {
    const int p = g0 + pk * G;
    double acc[FS_MAX_Q];
#pragma unroll
    for (int e = 0; e < FS_MAX_Q; ++e) acc[e] = 0.0;
    if (!dead)
      for (int c = lane; c < S.n_chord; c += 32) {
        const int c1 = c + 1 == S.n_chord ? 0 : c + 1;
        double gv[2], Rv[2];
        for (int k = 0; k < 2; ++k) {
          const int cc = k ? c1 : c;
          const double R = vr[p * S.n_chord + cc], Z = vz[p * S.n_chord + cc];
          int n0; double tx, ty;
          f.cell(R, Z, n0, tx, ty);
          const double p0 = (double)f.psi[n0], p1 = (double)f.psi[n0 + 1], p2 = (double)f.psi[n0 + f.nr], p3 = (double)f.psi[n0 + f.nr + 1];
          const double gR = ((1.0 - ty) * (p1 - p0) + ty * (p3 - p2)) / f.dr;
          const double gZ = ((1.0 - tx) * (p2 - p0) + tx * (p3 - p1)) / f.dz;
          gv[k] = sqrt(gR * gR + gZ * gZ); Rv[k] = R;
        }
        const double dRl = vr[p * S.n_chord + c1] - vr[p * S.n_chord + c], dZl = vz[p * S.n_chord + c1] - vz[p * S.n_chord + c];
        const double dl = sqrt(dRl * dRl + dZl * dZl);
#pragma unroll
        for (int e = 0; e < FS_MAX_Q; ++e)
          if (e < S.n_q) acc[e] += 0.5 * (fs_ipow(gv[0], S.mu[e]) * fs_ipow(Rv[0], S.nu[e]) + fs_ipow(gv[1], S.mu[e]) * fs_ipow(Rv[1], S.nu[e])) * dl;
      }
#pragma unroll
    for (int e = 0; e < FS_MAX_Q; ++e) acc[e] = warp_sum(acc[e]);
    if (lane == 0) {
      for (int e = 0; e < S.n_q; ++e) Qo[((size_t)s * S.n_prof + p) * S.n_q + e] = dead ? T(0) : T(acc[e]);
      double qv = nan("");
      if (!dead && S.q_index >= 0) {
        const double x = (p + 1.0) / S.n_prof;
        double integ = 0.0;
        for (int j = 0; j < S.n_ff; ++j)
          integ += X[S.ff0 + j] * ((1.0 - pow(x, j + 1.0)) / (j + 1.0) - (1.0 - pow(x, S.n_ff + 1.0)) / (S.n_ff + 1.0));
        const double f2 = S.f_vac * S.f_vac - 2.0 * (so.psi_b - so.axis_psi) * integ;
        qv = kMu0 * sqrt(fmax(f2, 0.0)) / two_pi * acc[S.q_index];
      }
      qo[(size_t)s * S.n_prof + p] = T(qv);
    }
  }
  // LCFS geometry (last level): R_min, R_max, Z_min, Z_max, a, kappa
  if (warp == 0 && (S.n_prof - 1) % G == g0) {
    double rmin = INFINITY, rmax = -INFINITY, zmin = INFINITY, zmax = -INFINITY;
    if (!dead)
      for (int c = lane; c < S.n_chord; c += 32) {
        const double R = vr[(S.n_prof - 1) * S.n_chord + c], Z = vz[(S.n_prof - 1) * S.n_chord + c];
        rmin = fmin(rmin, R); rmax = fmax(rmax, R); zmin = fmin(zmin, Z); zmax = fmax(zmax, Z);
      }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      rmin = fmin(rmin, __shfl_xor_sync(0xffffffffu, rmin, o)); rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, o));
      zmin = fmin(zmin, __shfl_xor_sync(0xffffffffu, zmin, o)); zmax = fmax(zmax, __shfl_xor_sync(0xffffffffu, zmax, o));
    }
    if (lane == 0) {
      T *g = geom + (size_t)s * 6;
      if (dead) { for (int k = 0; k < 6; ++k) g[k] = T(0); }
      else { g[0] = T(rmin); g[1] = T(rmax); g[2] = T(zmin); g[3] = T(zmax); g[4] = T(0.5 * (rmax - rmin)); g[5] = T((zmax - zmin) / (rmax - rmin)); }
      if (fstat) fstat[s] = dead ? 1 : (sh_bad == 2 ? 1 : 0);
    }
  }
}

}  // namespace ptefit
