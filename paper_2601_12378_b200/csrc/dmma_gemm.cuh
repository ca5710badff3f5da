// dmma_gemm.cuh -- FP64 contractions on the FP64 tensor-core path (mma.sync.m8n8k4.f64, "DMMA"):
//   response  R = G_P J_b             (Eq. 6)    rows = (slice, term), cols = channels
//   boundary  psi_bdry = G_B I        (Dirichlet data)  rows = slices, cols = edge nodes
//   DST-I in Z of the Delta* solve         rows = (slice, grid column), cols = modes
// All are C[M][N] = alpha * sum_k A[m][k] B[n][k] with both operands K-major (row-major [rows][K]).
// One kernel: 64 x 64 x 16 CTA tile, four warps of 32 x 32 (16 DMMA accumulators each), three cp.async
// stages, optional split-K over blockIdx.z (each split writes its own partial; consumers add them in a
// fixed order, so results are bit-reproducible).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ptefit {
namespace dm {

constexpr int BM = 64, BN = 64, BK = 16, STAGES = 3, THREADS = 128;
constexpr int LD = BK + 4;          // padded row length (doubles): 20 = 4 mod 16 -> conflict-free fragment loads
constexpr int TILE = BM * LD;       // doubles per operand tile
constexpr int SMEM_BYTES = STAGES * 2 * TILE * 8;

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, int src_bytes) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sa), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// grid (ceil(M/64), ceil(N/64), splits), block 128, dyn smem SMEM_BYTES.
// A[M][lda], B[N][ldb]: lda, ldb even, bases 16-byte aligned.  C + z * split_stride receives split z:
// C[m][n] at m * ldc + n.
__global__ void __launch_bounds__(THREADS) k_gemm_dmma(const double *__restrict__ A, int lda, const double *__restrict__ B, int ldb,
                                                       double *__restrict__ C, int ldc, int M, int N, int K, size_t split_stride,
                                                       double alpha) {
  extern __shared__ __align__(16) unsigned char dm_smem[];
  double *sm = reinterpret_cast<double *>(dm_smem);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN;
  const int kblocks = (K + BK - 1) / BK, nsplit = gridDim.z, z = blockIdx.z;
  const int kb0 = (int)(((long long)kblocks * z) / nsplit), kb1 = (int)(((long long)kblocks * (z + 1)) / nsplit);
  const int wm = warp >> 1, wn = warp & 1;

  auto load_stage = [&](int st, int kb) {
    double *As = sm + st * 2 * TILE, *Bs = As + TILE;
    const int k0 = kb * BK;
#pragma unroll
    for (int u = 0; u < (BM * BK / 2) / THREADS; ++u) {            // 16-byte chunks: 8 per row
      const int e = tid + u * THREADS, r = e >> 3, c = (e & 7) * 2;
      const int k = k0 + c;
      int bytes = (K - k) * 8;
      bytes = bytes < 0 ? 0 : (bytes > 16 ? 16 : bytes);
      const int ra = m0 + r, rb = n0 + r;
      const int ba = ra < M ? bytes : 0, bb = rb < N ? bytes : 0;
      cp_async16(As + r * LD + c, A + (size_t)(ra < M ? ra : 0) * lda + (ba ? k : 0), ba);
      cp_async16(Bs + r * LD + c, B + (size_t)(rb < N ? rb : 0) * ldb + (bb ? k : 0), bb);
    }
  };

  double acc[4][4][2];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;

  const int nkb = kb1 - kb0;
#pragma unroll
  for (int p = 0; p < STAGES - 1; ++p) {
    if (p < nkb) load_stage(p, kb0 + p);
    cp_commit();
  }
  for (int it = 0; it < nkb; ++it) {
    cp_wait<STAGES - 2>();
    __syncthreads();
    if (it + STAGES - 1 < nkb) load_stage((it + STAGES - 1) % STAGES, kb0 + it + STAGES - 1);
    cp_commit();
    const double *As = sm + (it % STAGES) * 2 * TILE, *Bs = As + TILE;
    const double *ap = As + (wm * 32 + (lane >> 2)) * LD + (lane & 3);
    const double *bp = Bs + (wn * 32 + (lane >> 2)) * LD + (lane & 3);
#pragma unroll
    for (int kk = 0; kk < BK / 4; ++kk) {
      double a[4], b[4];
#pragma unroll
      for (int t = 0; t < 4; ++t) { a[t] = ap[t * 8 * LD + kk * 4]; b[t] = bp[t * 8 * LD + kk * 4]; }
#pragma unroll
      for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) dmma(acc[mt][nt][0], acc[mt][nt][1], a[mt], b[nt]);
    }
  }
  cp_wait<0>();
  double *Cz = C + (size_t)z * split_stride;
#pragma unroll
  for (int mt = 0; mt < 4; ++mt) {
    const int row = m0 + wm * 32 + mt * 8 + (lane >> 2);
    if (row >= M) continue;
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
      const int col = n0 + wn * 32 + nt * 8 + 2 * (lane & 3);
      double *o = Cz + (size_t)row * ldc + col;
      if (col < N) o[0] = alpha * acc[mt][nt][0];
      if (col + 1 < N) o[1] = alpha * acc[mt][nt][1];
    }
  }
}

}  // namespace dm
}  // namespace ptefit
