// tc_solve.cuh -- A7 + A8 + A1 of one slice per CTA with both DSTs on the 5th-generation tensor
// cores.  FP32 path, grids with N_Z = 129 (DST length 127) and N_R <= 129.
//
//   Delta* psi = -mu0 R J_phi on the 5-point stencil (Eq. 1, 118-120 Sec. II.C) is solved
//   as DST-I in Z -> N_Z-2 tridiagonal systems in R (FP64, precomputed factors: "the coefficient
//   matrices can be pre-computed") -> DST-I in Z.  sin(pi (Nz-j) m / Nz) = (-1)^(m+1)
//   sin(pi j m / Nz) folds each 127-point transform into two 64 x 64 products:
//     forward  Y[m][i] = sum_jj S[jj][m] (F[jj+1][i] +- F[127-jj][i])   (+ odd m, - even m)
//     inverse  psi[jj+1][i], psi[127-jj][i] = U_odd[jj][i] +- U_even[jj][i]
//   Both run as tcgen05.mma kind::tf32 with the 3xTF32 split (a = a_hi + a_lo), accumulators in TMEM:
//     forward:  A = sine table [128 modes][64] (TMA, SWIZZLE_128B), B = folded right-hand side written
//               K-major by the CTA -> D[mode][column]: TMEM lane = mode, exactly the layout a
//               thread-per-mode Thomas sweep wants (tcgen05.ld of 16 columns at a time);
//     Thomas :  4 warps, one thread per mode, FP64 recurrences, the forward-sweep results parked in TMEM
//               (tcgen05.st) instead of global memory; the solution is written hi / lo split, K-major,
//               straight into the A operand tiles of the inverse product;
//     inverse:  A = X [128 columns][64 modes], B = sine table -> D[column][row]: TMEM lane = grid column,
//               so that the epilogue's shared-memory stores are conflict free.
//   The flux map then stays in shared memory for total flux + relaxation + search (search_body) + the
//   vertical-shift column, as in k_solve_fused.  One CTA per SM (192 KB of operands and tables, all 512
//   TMEM columns), persistent over slices.
#pragma once
#include "common.cuh"
#include "search_kernels.cuh"
#include "fused_solve.cuh"
#include "search_lean.cuh"
#include "tc_gemm.cuh"

namespace ptefit {

#ifdef PTEFIT_TUNING   // phase timers of the tuning build only (python -m paper_2601_12378_b200.build --tuning): printed by CTA 0
#define TCS_T(k) do { if (tid == 0 && blockIdx.x == 0) { const long long t_ = clock64(); tcs_clk[k] += t_ - tcs_t0; tcs_t0 = t_; } } while (0)
#else
#define TCS_T(k) do { } while (0)
#endif

constexpr int TCS_THREADS = 512;
constexpr int TCS_NZ = 129;                 // the only DST length this kernel is built for
constexpr int TCS_TAB_BYTES = 65536;        // sine table hi + lo: 2 x [128][64] floats
constexpr int TCS_OP_BYTES = 131072;        // operand tiles: 4 x [128][64] floats (hi / lo x odd / even)

struct TcSolveDev {
  const double *tcib;         // [128][128] inverse pivots of the twisted Thomas factorisation, [row i][TMEM lane]; rows >= nri are 1
  const double *tcw, *tce;    // [nri] sub- and super-diagonal of the tridiagonal systems (cw_i, ce_i)
  int mid;                    // meeting row of the twisted factorisation (top rows < mid, bottom rows > mid)
  const unsigned short *wl;   // [4][nwords] indices of the non-zero words of the lim / xpt / dilated / zero-only masks (WordLists)
  int n_lim, n_xpt, n_dil, n_zero;
};

__host__ __device__ inline size_t tcs_smem_bytes(int nr, int nz) {
  const size_t N = (size_t)nr * nz, nwords = (N + 31) / 32;
  size_t b = 1024 + TCS_TAB_BYTES + TCS_OP_BYTES;          // alignment slack + tables + operands (flux map aliases the operands)
  b += 4 * nwords * sizeof(unsigned);                      // lim / xpt / dilated lim (1 and 2 rows) bit masks
  b += (size_t)(2 * (nr + nz)) * sizeof(float);            // boundary flux
  b += 2 * (size_t)nr * sizeof(double);                    // sub- and super-diagonal
  b += 4 * nwords * sizeof(unsigned short) + 16;           // word lists of the search
  return b + 64;
}

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t *r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};\n" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
      "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void tmem_ld16u(uint32_t taddr, uint32_t *r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
}
// a = hi + lo for the 3xTF32 products: hi = a rounded to TF32 (nearest, ties away: add half an ulp of the
// 10-bit mantissa, clear the low 13 bits -- cvt.rna.tf32.f32 costs four instructions on sm_100a, this
// two), lo = a - hi exactly; the tensor core ignores the low 13 bits of lo itself.
__device__ __forceinline__ void tf32_split(float v, uint32_t &hi, uint32_t &lo) {
  hi = (__float_as_uint(v) + 0x1000u) & 0xffffe000u;
  lo = __float_as_uint(v - __uint_as_float(hi));
}

// Byte offset of element (row n, k) inside a [128 rows][64 k] FP32 operand stored as two K-blocks of
// [128 rows][128 bytes] with the 128-byte swizzle (16-byte chunk index XOR row % 8).
__device__ __forceinline__ uint32_t tcs_off(int n, int k) {
  return (uint32_t)((k >> 5) * 16384 + (n >> 3) * 1024 + (n & 7) * 128 + ((((k & 31) >> 2) ^ (n & 7)) << 4) + (k & 3) * 4);
}

// 3xTF32 product of two [rows][64] operands (hi / lo tiles 32 KB apart): 8 K steps x 3 MMAs.
// a_rowoff / b_rowoff: byte offsets of the first row inside each K-block (multiples of 1024).
__device__ __forceinline__ void tcs_mma64(uint32_t tacc, uint32_t a_hi, uint32_t a_lo, uint32_t b_hi, uint32_t b_lo, uint32_t idesc) {
#pragma unroll
  for (int kb = 0; kb < 2; ++kb) {
    const uint64_t dAh = tc::smem_desc_sw128(a_hi + kb * 16384), dAl = tc::smem_desc_sw128(a_lo + kb * 16384);
    const uint64_t dBh = tc::smem_desc_sw128(b_hi + kb * 16384), dBl = tc::smem_desc_sw128(b_lo + kb * 16384);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint64_t adv = (uint64_t)((k * 32) >> 4);
      tc::mma_tf32(tacc, dAl + adv, dBh + adv, idesc, (kb | k) ? 1u : 0u);     // small terms first
      tc::mma_tf32(tacc, dAh + adv, dBl + adv, idesc, 1u);
      tc::mma_tf32(tacc, dAh + adv, dBh + adv, idesc, 1u);
    }
  }
}

// grid min(B, #SM), block TCS_THREADS, dyn smem tcs_smem_bytes(nr, nz).  Arguments as k_solve_fused.
// mapF*: forward sine table  [128 lanes][64]: lane L < 64 -> odd mode 2L+1, L >= 64 -> even mode 2(L-64)+2;
// mapI*: inverse sine table  [128][64]: rows 0-63 = So[jj][p], rows 64-127 = Se[jj][q].
__global__ void __launch_bounds__(TCS_THREADS, 1)
k_solve_tc(const __grid_constant__ CUtensorMap mapFhi, const __grid_constant__ CUtensorMap mapFlo,
           const __grid_constant__ CUtensorMap mapIhi, const __grid_constant__ CUtensorMap mapIlo, Dev<float> D, TcSolveDev S,
           int B, const float *__restrict__ cur_all, const float *__restrict__ pbd_all, float *__restrict__ psi_all,
           float *__restrict__ xn_all, int use_relax, int add_coil, int do_search) {
  using T = float;
  extern __shared__ unsigned char smem_dyn[];
  if (!psi_all) psi_all = reinterpret_cast<T *>(D.ca->psi);
  unsigned char *base = smem_dyn + ((1024u - (tc::smem_u32(smem_dyn) & 1023u)) & 1023u);   // pointer arithmetic only: keeps the shared address space
  unsigned char *tab = base;                               // [hi kb0][hi kb1][lo kb0][lo kb1], 16 KB each
  unsigned char *op = base + TCS_TAB_BYTES;                // forward: E+ hi, E+ lo, E- hi, E- lo; inverse: Xo hi, Xo lo, Xe hi, Xe lo
  T *Gb = reinterpret_cast<T *>(op);                       // flux map, aliases the operand tiles once they are consumed
  const bool vec_ok = ((reinterpret_cast<uintptr_t>(psi_all) | reinterpret_cast<uintptr_t>(D.psi_coil)) & 15) == 0;
  const int nr = D.nr, nz = D.nz, N = D.N, nri = D.nri, nzi = D.nzi, Nz = nz - 1;
  const int nwords = (N + 31) >> 5;
  unsigned *mbits = reinterpret_cast<unsigned *>(op + TCS_OP_BYTES);   // lim, xpt, dilated-lim bit masks
  T *pb = reinterpret_cast<T *>(mbits + 4 * nwords);       // bottom[nr], top[nr], left[nzi], right[nzi]
  double *ce_s = reinterpret_cast<double *>(reinterpret_cast<unsigned char *>(pb + 2 * (nr + nz)) + ((8u - (tc::smem_u32(pb + 2 * (nr + nz)) & 7u)) & 7u));
  double *cw_s = ce_s + nr;
  unsigned short *wls = reinterpret_cast<unsigned short *>(cw_s + nr);   // [4][nwords]
  const double *ibs = reinterpret_cast<const double *>(op);   // Thomas phase: inverse pivots [i][lane], staged by bulk copies
  __shared__ uint64_t bar_tab, bar_mma, bar_ib[8];
  __shared__ uint32_t tmem_slot;
  __shared__ T c_rhs[PTEFIT_MAX_NR], c_rdA[PTEFIT_MAX_NR], c_fdA[PTEFIT_MAX_NR];
  __shared__ T pcoef[2 * (PTEFIT_MAX_DEG + 1)];
  __shared__ T c_edge[2];
  __shared__ double xch[256];                              // Thomas: what the two halves of a mode exchange in the meeting row
  __shared__ LeanShared lean;
  const int tid = threadIdx.x, nth = blockDim.x, warp = tid >> 5, lane = tid & 31;
  const bool elected = (tid == 8 * 32);                    // lane 0 of warp 8: TMA + MMA issue (warps 0-7 run the Thomas sweeps)

  if (elected) {
    tc::tma_prefetch_desc(&mapFhi); tc::tma_prefetch_desc(&mapFlo); tc::tma_prefetch_desc(&mapIhi); tc::tma_prefetch_desc(&mapIlo);
    tc::mbar_init(&bar_tab, 1);
    tc::mbar_init(&bar_mma, 1);
    for (int c = 0; c < 8; ++c) tc::mbar_init(&bar_ib[c], 1);
    tc::fence_barrier_init();
  }
  if (warp == 0) tc::tmem_alloc<512>(&tmem_slot);
  for (int w = tid; w < 4 * nwords; w += nth)
    mbits[w] = (w < nwords) ? D.lim_bits[w] : (w < 2 * nwords) ? D.xpt_bits[w - nwords] : (w < 3 * nwords) ? D.dil_bits[w - 2 * nwords] : D.dil2_bits[w - 3 * nwords];
  for (int w = tid; w < 4 * nwords; w += nth) wls[w] = S.wl[w];
  WordLists WL;
  WL.lim = wls; WL.xpt = wls + nwords; WL.dil = wls + 2 * nwords; WL.zero = wls + 3 * nwords;
  WL.n_lim = S.n_lim; WL.n_xpt = S.n_xpt; WL.n_dil = S.n_dil; WL.n_zero = S.n_zero;
  for (int i = tid; i < nr; i += nth) {
    const double Rd = D.rmin + i * D.dr;
    c_rhs[i] = T(-kMu0 * Rd / D.dA);
    const T R = T(Rd);
    c_rdA[i] = R * T(D.dA);
    c_fdA[i] = T(kMu0 * D.dA) / R;
    if (i == 1) c_edge[0] = T((1.0 + D.dr / (2.0 * Rd)) / (D.dr * D.dr));
    if (i == nri) c_edge[1] = T((1.0 - D.dr / (2.0 * Rd)) / (D.dr * D.dr));
    ce_s[i] = (i < nri) ? S.tce[i] : 0.0;
    cw_s[i] = (i < nri) ? S.tcw[i] : 0.0;
  }
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem_base = tmem_slot;
  const uint32_t tab_a = tc::smem_u32(tab), op_a = tc::smem_u32(op);
  uint32_t ph_tab = 0, ph_mma = 0, ph_ib = 0;
  auto load_tables = [&](const CUtensorMap *mh, const CUtensorMap *ml) {     // elected thread only
    tc::mbar_expect_tx(&bar_tab, TCS_TAB_BYTES);
    tc::tma_load_2d(tab, mh, &bar_tab, 0, 0);
    tc::tma_load_2d(tab + 16384, mh, &bar_tab, 32, 0);
    tc::tma_load_2d(tab + 32768, ml, &bar_tab, 0, 0);
    tc::tma_load_2d(tab + 49152, ml, &bar_tab, 32, 0);
  };
  if (elected && (int)blockIdx.x < B) load_tables(&mapFhi, &mapFlo);

  const T cz = T(1.0 / (D.dz * D.dz));
  const T scale = T(2.0 / Nz);
  const T om = T(D.relax);
  constexpr uint32_t idesc128 = tc::idesc_tf32(128, 128), idesc64 = tc::idesc_tf32(128, 64);

#ifdef PTEFIT_TUNING
  if (tid == 0) for (int k = 0; k < 8; ++k) lean.clk[k] = 0;
  long long tcs_clk[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, tcs_t0 = clock64();
#endif
  for (int s = blockIdx.x; s < B; s += gridDim.x) {
    const T *I = cur_all + (size_t)s * N;
    const T *pbg = pbd_all + (size_t)s * D.nbnd;
    T *psi = psi_all + (size_t)s * N;
    const T *pc = D.psi_coil + (size_t)s * N;
    T *G = Gb + (vec_ok ? (int)(((size_t)s * N) & 3) : 0);     // G + n is 16-byte aligned exactly when psi + n is
    __syncthreads();                                       // previous slice done with G and pb
    for (int k = tid; k < D.nbnd; k += nth) pb[k] = pbg[k];
    if (do_search && D.has_delz && tid < 2 * (PTEFIT_MAX_DEG + 1)) pcoef[tid] = D.pco[(size_t)s * PCO_STRIDE + tid];   // written by the fit kernel (emit_pco)
    // ---- A. right-hand side -mu0 R I / dA with the Dirichlet data moved over, folded about the mid
    // row and written K-major (row = grid column, k = folded grid row) as hi / lo TF32 tiles.
    // Work item = one grid column n x four consecutive folded rows jj0..jj0+3 (one 16-byte chunk).
    {
      constexpr int ITEMS = (128 * 16) / TCS_THREADS;      // 4
      float lo_v[ITEMS][4], hi_v[ITEMS][4];
#pragma unroll
      for (int u = 0; u < ITEMS; ++u) {
        const int it = tid + u * TCS_THREADS, n = it & 127, q = it >> 7, gi = n + 1;
        const bool valid = n < nri;
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          const int jj = 4 * q + t, j = jj + 1, jp = Nz - j;
          lo_v[u][t] = valid ? __ldg(I + j * nr + gi) : 0.f;
          hi_v[u][t] = (valid && jj < 63) ? __ldg(I + jp * nr + gi) : 0.f;
        }
      }
      // inputs of the later phases: pull them towards L2 while the solve runs
      {
        const int lines = (int)(((size_t)N * sizeof(T) + 127) / 128);
        for (int l = tid; l < lines; l += nth) {
          if (add_coil) prefetch_l2(reinterpret_cast<const char *>(pc) + (size_t)l * 128);
          if (use_relax) prefetch_l2(reinterpret_cast<const char *>(psi) + (size_t)l * 128);
        }
      }
      __syncthreads();                                     // pb staged
#pragma unroll
      for (int u = 0; u < ITEMS; ++u) {
        const int it = tid + u * TCS_THREADS, n = it & 127, q = it >> 7, gi = n + 1;
        const bool valid = n < nri;
        uint32_t ph[4], pl[4], mh[4], ml[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          const int jj = 4 * q + t, j = jj + 1, jp = Nz - j;
          float a = c_rhs[gi] * lo_v[u][t], b = c_rhs[gi] * hi_v[u][t];
          if (gi == 1) { a -= c_edge[0] * pb[2 * nr + j - 1]; b -= c_edge[0] * pb[2 * nr + jp - 1]; }
          if (gi == nri) { a -= c_edge[1] * pb[2 * nr + nzi + j - 1]; b -= c_edge[1] * pb[2 * nr + nzi + jp - 1]; }
          if (j == 1) { a -= cz * pb[gi]; b -= cz * pb[nr + gi]; }          // jp = nzi: top row data
          if (!valid) { a = 0.f; b = 0.f; }
          if (jj >= 63) b = 0.f;                            // mid row has no partner
          const float ep = a + b, em = a - b;
          tf32_split(ep, ph[t], pl[t]);
          tf32_split(em, mh[t], ml[t]);
        }
        const uint32_t off = tcs_off(n, 4 * q);
        *reinterpret_cast<uint4 *>(op + off) = make_uint4(ph[0], ph[1], ph[2], ph[3]);
        *reinterpret_cast<uint4 *>(op + 32768 + off) = make_uint4(pl[0], pl[1], pl[2], pl[3]);
        *reinterpret_cast<uint4 *>(op + 65536 + off) = make_uint4(mh[0], mh[1], mh[2], mh[3]);
        *reinterpret_cast<uint4 *>(op + 98304 + off) = make_uint4(ml[0], ml[1], ml[2], ml[3]);
      }
    }
    tc::fence_proxy_async();
    __syncthreads();
    TCS_T(0);
    // ---- B. forward DST on the tensor cores: D1 = Tab x E+ (lanes 0-63 = odd modes), D2 = Tab x E- (lanes 64-127 = even modes)
    if (elected) {
      tc::mbar_wait(&bar_tab, ph_tab);
      tc::tc_fence_after();
      tcs_mma64(tmem_base + 0, tab_a, tab_a + 32768, op_a, op_a + 32768, idesc128);
      tcs_mma64(tmem_base + 128, tab_a, tab_a + 32768, op_a + 65536, op_a + 98304, idesc128);
      tc::tc_commit(&bar_mma);
    }
    ph_tab ^= 1u;
    // ---- C. Thomas sweeps along R in FP64 on the twisted factorisation: two threads per mode (TMEM lane L),
    // warps 0-3 eliminate downwards from row 0 to row mid-1, warps 4-7 upwards from row nri-1 to row mid+1
    // (both halves of a lane quarter may touch its TMEM lanes: warp % 4 selects the quarter); they meet in
    // row mid and substitute back outwards.  Normalised form (unit off-diagonal), ib = inverse pivots of the
    // respective sweep (row mid: of the meeting row):
    //   top     z_i = ib_i f_i - (ib_i cw_i) z_{i-1},   x_i = z_i - (ce_i ib_i) x_{i+1}
    //   bottom  y_i = ib_i f_i - (ib_i ce_i) y_{i+1},   x_i = y_i - (cw_i ib_i) x_{i-1}
    //   mid     x_m = ib_m (f_m - cw_m z_{m-1} - ce_m y_{m+1}).
    // The pivot table is staged in the (now free) operand region by eight bulk copies of 16 rows; z / y and
    // then x are parked in TMEM columns 256-511.  mid + 1 is a multiple of 16 (or mid = nri - 1: no bottom half).
    if (warp < 8) {
      tc::mbar_wait(&bar_mma, ph_mma);
      tc::tc_fence_after();
      TCS_T(7);
      const int L = tid & 127, half = tid >> 7, mid = S.mid;
      const bool two = mid + 1 < nri;
      const uint32_t tl = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
      const uint32_t src = tl + (L < 64 ? 0u : 128u), ya = tl + 256u;
      const int cm = mid >> 4, c_lo = (mid + 1) >> 4, c_hi = (nri - 1) >> 4;
      if (half == 0) {
        double z = 0.0, tmid = 0.0;
        for (int c = 0; c <= cm; ++c) {
          const int i0 = 16 * c;
          uint32_t f[16], zlo[16], zhi[16];
          tmem_ld16u(src + i0, f);
          tc::mbar_wait(&bar_ib[c], ph_ib);
#pragma unroll
          for (int u = 0; u < 16; ++u) {
            const int i = i0 + u;
            const double ib = ibs[i * 128 + L], fi = (double)__uint_as_float(f[u]);
            const double v = fma(-(ib * cw_s[i]), z, ib * fi);
            if (i == mid) tmid = fma(-cw_s[i], z, fi);
            z = (i < mid) ? v : z;
            zlo[u] = (uint32_t)__double2loint(v);
            zhi[u] = (uint32_t)__double2hiint(v);
          }
          tmem_st16(ya + i0, zlo);
          tmem_st16(ya + 128 + i0, zhi);
        }
        xch[L] = tmid;
      } else {
        double y = 0.0;
        if (two)
          for (int c = c_hi; c >= c_lo; --c) {
            const int i0 = 16 * c;
            uint32_t f[16], zlo[16], zhi[16];
            tmem_ld16u(src + i0, f);
            tc::mbar_wait(&bar_ib[c], ph_ib);
#pragma unroll
            for (int u = 15; u >= 0; --u) {
              const int i = i0 + u;
              const double ib = ibs[i * 128 + L];
              const double v = fma(-(ib * ce_s[i]), y, ib * (double)__uint_as_float(f[u]));
              y = (i < nri) ? v : y;
              zlo[u] = (uint32_t)__double2loint(v);
              zhi[u] = (uint32_t)__double2hiint(v);
            }
            tmem_st16(ya + i0, zlo);
            tmem_st16(ya + 128 + i0, zhi);
          }
        xch[128 + L] = y;
        tc::mbar_wait(&bar_ib[cm], ph_ib);                 // the meeting row's pivot
      }
      tmem_wait_st();
      asm volatile("bar.sync %0, 64;\n" ::"r"(1 + (warp & 3)) : "memory");      // the two warps of this lane quarter
      TCS_T(8);
      double x = ibs[mid * 128 + L] * fma(-ce_s[mid], xch[128 + L], xch[L]);     // x_mid (y = 0 when there is no bottom half)
      if (half == 0) {
        for (int c = cm; c >= 0; --c) {
          const int i0 = 16 * c;
          uint32_t zlo[16], zhi[16];
          tmem_ld16u(ya + i0, zlo);
          tmem_ld16u(ya + 128 + i0, zhi);
#pragma unroll
          for (int u = 15; u >= 0; --u) {
            const int i = i0 + u;
            if (i < mid) x = fma(-(ce_s[i] * ibs[i * 128 + L]), x, __hiloint2double((int)zhi[u], (int)zlo[u]));
            zlo[u] = __float_as_uint(i <= mid ? (float)x : 0.f);
          }
          tmem_st16(ya + i0, zlo);                         // x (FP32) over z's low words; split hi / lo by all warps below
        }
      } else if (two) {
        for (int c = c_lo; c <= c_hi; ++c) {
          const int i0 = 16 * c;
          uint32_t zlo[16], zhi[16];
          tmem_ld16u(ya + i0, zlo);
          tmem_ld16u(ya + 128 + i0, zhi);
#pragma unroll
          for (int u = 0; u < 16; ++u) {
            const int i = i0 + u;
            float xf = 0.f;
            if (i < nri) {
              x = fma(-(cw_s[i] * ibs[i * 128 + L]), x, __hiloint2double((int)zhi[u], (int)zlo[u]));
              xf = (float)x;
            }
            zlo[u] = __float_as_uint(xf);
          }
          tmem_st16(ya + i0, zlo);
        }
      }
      tmem_wait_st();
      tc::tc_fence_before();
      TCS_T(9);
    } else if (elected) {
      // the forward products have completed: operand tiles and the forward table are dead.  Stage the
      // inverse pivots (rows of 128 lanes x 8 bytes, 16 rows per copy; outermost chunks first, as the two
      // sweeps consume them) and fetch the inverse table.
      tc::mbar_wait(&bar_mma, ph_mma);
      for (int cc = 0; cc < 8; ++cc) {
        const int c = (cc & 1) ? 7 - (cc >> 1) : (cc >> 1);
        tc::mbar_expect_tx(&bar_ib[c], 16384);
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(op_a + c * 16384),
                     "l"(S.tcib + (size_t)c * 16 * 128), "r"(16384), "r"(tc::smem_u32(&bar_ib[c]))
                     : "memory");
      }
      load_tables(&mapIhi, &mapIlo);
    }
    ph_mma ^= 1u;
    ph_ib ^= 1u;
    __syncthreads();
    // solution out of TMEM into the A tiles of the inverse DST (all warps: lane quarter q, 32 columns each)
    {
      tc::tc_fence_after();
      const int q = warp & 3, g = warp >> 2, L = q * 32 + lane, kx = L & 63;
      const uint32_t tl = tmem_base + ((uint32_t)(q * 32) << 16) + 256u;
      unsigned char *xt = op + (L < 64 ? 0 : 65536);
      constexpr int CPG = 128 / (TCS_THREADS / 128);         // columns per group of four warps
#pragma unroll
      for (int hf = 0; hf < CPG / 16; ++hf) {
        const int i0 = CPG * g + 16 * hf;
        uint32_t xv[16];
        tmem_ld16u(tl + i0, xv);
#pragma unroll
        for (int u = 0; u < 16; ++u) {
          const uint32_t off = tcs_off(i0 + u, kx);
          const float xf = __uint_as_float(xv[u]);
          uint32_t xh, xl;
          tf32_split(xf, xh, xl);
          *reinterpret_cast<uint32_t *>(xt + off) = xh;
          *reinterpret_cast<uint32_t *>(xt + 32768 + off) = xl;
        }
      }
      tc::fence_proxy_async();
      tc::tc_fence_before();
    }
    __syncthreads();
    TCS_T(1);
    // ---- D. inverse DST: D[column][jj] = Xo x So (TMEM columns 0-63), D[column][64 + jj] = Xe x Se (columns 64-127)
    if (elected) {
      tc::mbar_wait(&bar_tab, ph_tab);
      tc::tc_fence_after();
      tcs_mma64(tmem_base + 0, op_a, op_a + 32768, tab_a, tab_a + 32768, idesc64);
      tcs_mma64(tmem_base + 64, op_a + 65536, op_a + 98304, tab_a + 8192, tab_a + 32768 + 8192, idesc64);
      tc::tc_commit(&bar_mma);
    }
    ph_tab ^= 1u;
    tc::mbar_wait(&bar_mma, ph_mma);
    ph_mma ^= 1u;
    tc::tc_fence_after();
    TCS_T(2);
    if (elected && s + (int)gridDim.x < B) load_tables(&mapFhi, &mapFlo);    // for the next slice of this CTA
    // ---- E. unfold into the flux map (plasma flux, scaled): lane = grid column, 16 folded rows per warp
    {
      const int q = warp & 3, g = warp >> 2, n = q * 32 + lane, gi = n + 1;
      const uint32_t tl = tmem_base + ((uint32_t)(q * 32) << 16);
      uint32_t a[16], b[16];
      if (g < 4) {
        tmem_ld16u(tl + 16 * g, a);
        tmem_ld16u(tl + 64 + 16 * g, b);
      }
      if (g < 4 && n < nri) {
#pragma unroll
        for (int t = 0; t < 16; ++t) {
          const int jj = 16 * g + t, j = jj + 1;
          const float uo = __uint_as_float(a[t]), ue = __uint_as_float(b[t]);
          G[j * nr + gi] = (uo + ue) * scale;
          if (jj < 63) G[(Nz - j) * nr + gi] = (uo - ue) * scale;
        }
      }
      for (int k = tid; k < D.nbnd; k += nth) {            // Dirichlet data on the edge nodes
        int e;
        if (k < nr) e = k;
        else if (k < 2 * nr) e = (nz - 1) * nr + (k - nr);
        else if (k < 2 * nr + nzi) e = (k - 2 * nr + 1) * nr;
        else e = (k - 2 * nr - nzi + 1) * nr + nr - 1;
        G[e] = pb[k];
      }
    }
    tc::tc_fence_before();
    __syncthreads();
    TCS_T(3);
    // ---- total flux + relaxation; psi goes to global memory and stays in G for the search.  Flat over the
    // nodes in 16-byte vectors (G is offset inside its buffer so that G + n and psi + n are aligned together);
    // pass 0 of the search (finiteness, arg-max of s psi over lim_mask) rides along.
    float am_v = -INFINITY;
    int am_n = 0x7fffffff;
    bool bad0 = false;
    {
      const float sgT = float(D.ip_sign);
      float chk = 0.f;                                      // stays 0 unless a flux value is Inf / NaN
      const int a0 = vec_ok ? min(N, (4 - (int)(((size_t)s * N) & 3)) & 3) : N;      // scalar head up to the first aligned node
      const int nq = (N - a0) >> 2, t0 = a0 + 4 * nq;
      // 16-byte body first (strict > keeps the smallest n of equal keys: a thread sees its nodes in increasing n)
      constexpr int EB = 3;
      for (int q0 = tid; q0 < nq; q0 += EB * nth) {
        float4 cv[EB], ov[EB];
#pragma unroll
        for (int u = 0; u < EB; ++u) {
          const int q = q0 + u * nth;
          cv[u] = (add_coil && q < nq) ? *reinterpret_cast<const float4 *>(pc + a0 + 4 * q) : make_float4(0.f, 0.f, 0.f, 0.f);
          ov[u] = (use_relax && q < nq) ? *reinterpret_cast<const float4 *>(psi + a0 + 4 * q) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < EB; ++u) {
          const int q = q0 + u * nth, n = a0 + 4 * q;
          if (q < nq) {
            const float4 g = *reinterpret_cast<const float4 *>(G + n);
            const unsigned lb = __funnelshift_r(mbits[n >> 5], mbits[(n >> 5) + 1], n & 31);   // lim bits of nodes n..n+3
            float v[4] = {g.x + cv[u].x, g.y + cv[u].y, g.z + cv[u].z, g.w + cv[u].w};
            const float o[4] = {ov[u].x, ov[u].y, ov[u].z, ov[u].w};
#pragma unroll
            for (int t = 0; t < 4; ++t) {
              if (use_relax) v[t] = fmaf(om, v[t] - o[t], o[t]);
              chk = fmaf(v[t], 0.f, chk);
              const float key = sgT * v[t];
              if (((lb >> t) & 1u) && key > am_v) { am_v = key; am_n = n + t; }
            }
            const float4 r = make_float4(v[0], v[1], v[2], v[3]);
            *reinterpret_cast<float4 *>(psi + n) = r;
            *reinterpret_cast<float4 *>(G + n) = r;
          }
        }
      }
      for (int n = tid; n < a0 + (N - t0); n += nth) {     // unaligned head and tail nodes
        const int m = n < a0 ? n : t0 + (n - a0);
        float v = G[m] + (add_coil ? pc[m] : 0.f);
        if (use_relax) { const float o = psi[m]; v = fmaf(om, v - o, o); }
        psi[m] = v; G[m] = v;
        chk = fmaf(v, 0.f, chk);
        const float key = sgT * v;
        if (((mbits[m >> 5] >> (m & 31)) & 1u) && (key > am_v || (key == am_v && m < am_n))) { am_v = key; am_n = m; }
      }
      bad0 = !(chk == 0.f);
    }
    __syncthreads();
    TCS_T(4);
    if (do_search) {
      float *xn = xn_all + (size_t)s * N;
      search_lean(D, lean, s, G, xn, mbits, mbits + nwords, mbits + 3 * nwords, WL, am_v, am_n, bad0, D.has_delz ? pcoef : nullptr, c_rdA, c_fdA,
                  D.X + (size_t)s * D.nt);                 // G now holds I'(xn) (delz) or xn on the lim_mask words
      TCS_T(5);
      if (D.has_delz) {
        // -dI'/dZ column for the NEXT fit, on the nodes of the compact list only (lim_mask dilated by one row;
        // everything else keeps the zero of the memset at the start of the call)
        __syncthreads();
        float *__restrict__ dzc = D.dzc + (size_t)s * N;
        const float hz = float(0.5 / D.dz);
        const unsigned *dbits = mbits + 2 * nwords;
        const int nwarp = nth >> 5;
        int k = warp;
        int wc = k < WL.n_dil ? WL.dil[k] : 0;
        unsigned dbc = dbits[wc];
        while (k < WL.n_dil) {                             // word index and mask word fetched one iteration ahead
          const int w = wc;
          const unsigned db = dbc;
          k += nwarp;
          wc = k < WL.n_dil ? WL.dil[k] : 0;
          dbc = dbits[wc];
          const int n = (w << 5) + lane;
          if ((db >> lane) & 1u) dzc[n] = -(G[n + nr] - G[n - nr]) * hz;     // G = 0 off the lim_mask nodes (search_lean)
        }
      }
      TCS_T(6);
    }
  }
#ifdef PTEFIT_TUNING
  if (tid == 0 && blockIdx.x == 0 && do_search)
    printf("k_solve_tc cycles: rhs %lld fwd+thomas %lld inv %lld unfold %lld total-flux %lld search %lld delz %lld | mma-wait %lld fwd-sweep %lld bwd-sweep %lld (tmem-ld %lld ib-wait %lld)\n", tcs_clk[0], tcs_clk[1],
           tcs_clk[2], tcs_clk[3], tcs_clk[4], tcs_clk[5], tcs_clk[6], tcs_clk[7], tcs_clk[8], tcs_clk[9], tcs_clk[10], tcs_clk[11]);
  if (tid == 0 && blockIdx.x == 0 && do_search)
    printf("  search_lean cycles: argmax+axis %lld scan %lld decide %lld limiter %lld pb %lld mask %lld tail %lld nlist %d ncand %d\n", lean.clk[0], lean.clk[1], lean.clk[2],
           lean.clk[3], lean.clk[4], lean.clk[5], lean.clk[6], lean.nlist, lean.ncand);
#endif
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 0) tc::tmem_dealloc<512>(tmem_base);
}

// Stand-alone lean search for warm starts on the FP32 tensor-core path: flux map into shared memory, then
// search_lean (normalised flux on the lim_mask words; the rest of xn keeps the -1 written at create).
// grid B, block TCS_THREADS, dyn smem tcs_search_smem_bytes.
__host__ __device__ inline size_t tcs_search_smem_bytes(int nr, int nz) {
  const size_t N = (size_t)nr * nz, nwords = (N + 31) / 32;
  return (N + 4) * sizeof(float) + 4 * nwords * sizeof(unsigned) + 4 * nwords * sizeof(unsigned short) + 64;
}
__global__ void __launch_bounds__(TCS_THREADS, 1) k_search_tc(Dev<float> D, TcSolveDev S, const float *__restrict__ psi_all, float *__restrict__ xn_all) {
  extern __shared__ __align__(16) unsigned char smem_dyn[];
  __shared__ LeanShared lean;
  if (!psi_all) psi_all = reinterpret_cast<const float *>(D.ca->psi);
  const int s = blockIdx.x, tid = threadIdx.x, nth = blockDim.x, N = D.N, nwords = (N + 31) >> 5;
  float *G = reinterpret_cast<float *>(smem_dyn);
  unsigned *mbits = reinterpret_cast<unsigned *>(G + ((N + 3) & ~3));
  unsigned short *wls = reinterpret_cast<unsigned short *>(mbits + 4 * nwords);
  for (int w = tid; w < 4 * nwords; w += nth) {
    mbits[w] = (w < nwords) ? D.lim_bits[w] : (w < 2 * nwords) ? D.xpt_bits[w - nwords] : (w < 3 * nwords) ? D.dil_bits[w - 2 * nwords] : D.dil2_bits[w - 3 * nwords];
    wls[w] = S.wl[w];
  }
  WordLists WL;
  WL.lim = wls; WL.xpt = wls + nwords; WL.dil = wls + 2 * nwords; WL.zero = wls + 3 * nwords;
  WL.n_lim = S.n_lim; WL.n_xpt = S.n_xpt; WL.n_dil = S.n_dil; WL.n_zero = S.n_zero;
  __syncthreads();
  const float *psi = psi_all + (size_t)s * N;
  const float sgT = float(D.ip_sign);
  float am_v = -INFINITY, chk = 0.f;
  int am_n = 0x7fffffff;
  for (int n = tid; n < N; n += nth) {
    const float v = psi[n];
    G[n] = v;
    chk = fmaf(v, 0.f, chk);
    const float key = sgT * v;
    if (((mbits[n >> 5] >> (n & 31)) & 1u) && key > am_v) { am_v = key; am_n = n; }      // n increases per thread: ties keep the smallest
  }
  __syncthreads();
  search_lean(D, lean, s, G, xn_all + (size_t)s * N, mbits, mbits + nwords, mbits + 3 * nwords, WL, am_v, am_n, !(chk == 0.f), nullptr, nullptr,
              nullptr, nullptr);
}

}  // namespace ptefit
