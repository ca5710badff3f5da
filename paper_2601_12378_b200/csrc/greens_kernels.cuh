// greens_kernels.cuh -- NEXT-3: Green's-function tables on the GPU (Sec. II.A, Eq. 3-5).
// Flux per radian and field of a unit toroidal filament in closed form with complete elliptic
// integrals K, E evaluated by the arithmetic-geometric mean (FP64, ALU bound; one thread per
// (field point, source) pair).  Reading of the garbled Eq. 3-4: Biot-Savart with the power 3/2
// (O1).  COCOS 7: B_R = -(1/R) dpsi/dZ, B_Z = +(1/R) dpsi/dR.
#pragma once
#include "common.cuh"

namespace ptefit {

// K(m), E(m), parameter m = k^2 in [0, 1): a_0 = 1, b_0 = sqrt(1 - m), c_0^2 = m;
// K = pi / (2 a_N), E = K (1 - sum_n 2^(n-1) c_n^2).
__device__ __forceinline__ void agm_ke(double m, double &K, double &E) {
  double a = 1.0, b = sqrt(1.0 - m), s = 0.5 * m, pw = 0.5;
#pragma unroll 1
  for (int it = 0; it < 16; ++it) {
    const double c = 0.5 * (a - b);
    const double an = 0.5 * (a + b);
    b = sqrt(a * b);
    a = an;
    pw *= 2.0;
    s = fma(pw * c, c, s);
    if (fabs(c) <= 1e-17 * a) break;
  }
  K = 1.5707963267948966 / a;
  E = K * (1.0 - s);
}

// out[k][c] (or out[c][k] if transpose) = w_c * g(field point k, source c), where g = psi (flux row:
// fcos[k] = fsin[k] = 0 or fcos == nullptr) or cos a B_R + sin a B_Z (probe row).  Coincident points give 0.
// grid (ceil(n_src/256), n_fld), block 256.
__global__ void __launch_bounds__(256) k_greens_table(int n_fld, const double *__restrict__ fr, const double *__restrict__ fz,
                                                      const double *__restrict__ fcos, const double *__restrict__ fsin, int n_src,
                                                      const double *__restrict__ sr, const double *__restrict__ sz,
                                                      const double *__restrict__ sw, double *__restrict__ out, int transpose) {
  const int k = blockIdx.y, c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_src) return;
  const double rho = fr[k], zf = fz[k], a = sr[c], z = zf - sz[c];
  const double ca = fcos ? fcos[k] : 0.0, sa = fsin ? fsin[k] : 0.0;
  const double s2 = (a + rho) * (a + rho) + z * z, d2 = (a - rho) * (a - rho) + z * z;
  double v = 0.0;
  if (d2 > 0.0 && rho > 0.0 && a > 0.0) {
    const double k2 = 4.0 * a * rho / s2;
    double K, E;
    agm_ke(k2, K, E);
    const double c0 = kMu0 / (2.0 * 3.14159265358979323846);
    if (ca == 0.0 && sa == 0.0) {
      v = c0 * sqrt(a * rho) * ((2.0 - k2) * K - 2.0 * E) / sqrt(k2);                 // Eq. 5
    } else {
      const double pref = c0 / sqrt(s2);
      const double bz = pref * (K + (a * a - rho * rho - z * z) / d2 * E);
      const double br = pref * z / rho * (-K + (a * a + rho * rho + z * z) / d2 * E);
      v = ca * br + sa * bz;
    }
  }
  if (sw) v *= sw[c];
  out[transpose ? (size_t)c * n_fld + k : (size_t)k * n_src + c] = v;
}

}  // namespace ptefit
