// tc_gemm.cuh -- the two dense contractions of the Picard iteration on the 5th-generation tensor
// cores (tcgen05.mma kind::tf32, accumulators in TMEM, operands staged by TMA):
//   response  R = G_P J_b            (Eq. 6)   rows = (slice, term), cols = channels
//   boundary  psi_bdry = G_B I       (Dirichlet data)   rows = slices, cols = edge nodes
// Both are D[M][N] = A[M][K] B[N][K]^T with K = the compacted list of nodes that may carry current
// (lim_mask = 1), A = per-slice data, B = a Green's table.  FP32 accuracy comes from the 3xTF32
// split a = a_hi + a_lo (a_hi = a rounded to TF32):  D += A_hi B_hi + A_hi B_lo + A_lo B_hi.
// K is split over blockIdx.z; each split writes its own partial (summed in a fixed order by the
// consumer, so results are bit-reproducible).  DESIGN.md "k_gemm_3xtf32".
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace ptefit {
namespace tc {

constexpr int BM = 128;          // rows of A per CTA (TMEM lanes)
constexpr int BK = 32;           // K per stage: 32 floats = one 128-byte swizzle row
constexpr int UMMA_K = 8;        // K of one tcgen05.mma kind::tf32
constexpr int GEMM_THREADS = 320;  // warp 0: TMA, warp 1: MMA, warps 2-9: accumulate + epilogue
constexpr int DRAIN = 4;         // K blocks accumulated in TMEM before promotion to FP32 registers

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

// 2-D TMA tile load: coordinates (c0 = innermost = k, c1 = row), completion on an mbarrier.
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];\n" ::"r"(smem_u32(dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap *map) {
  asm volatile("prefetch.tensormap [%0];\n" ::"l"(map) : "memory");
}

// TMEM allocation (one warp), columns = power of two >= 32.
template <int COLS>
__device__ __forceinline__ void tmem_alloc(uint32_t *slot) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(slot)), "n"(COLS));
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
}
template <int COLS>
__device__ __forceinline__ void tmem_dealloc(uint32_t addr) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(addr), "n"(COLS));
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}

// Shared-memory matrix descriptor, K-major operand, 128-byte swizzle: rows are 128 bytes, groups of
// 8 rows (1024 bytes) follow each other (stride byte offset 1024); sm_100 descriptor version 1.
__device__ __forceinline__ uint64_t smem_desc_sw128(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFF) >> 4);            // start address, bits [0,14)
  d |= (uint64_t)1 << 16;                              // leading byte offset (unused with swizzle)
  d |= (uint64_t)(1024 >> 4) << 32;                    // stride byte offset, bits [32,46)
  d |= (uint64_t)1 << 46;                              // version = 1 (Blackwell)
  d |= (uint64_t)2 << 61;                              // layout: SWIZZLE_128B
  return d;
}
// Instruction descriptor: D = F32, A = B = TF32, both K-major, shape M x N.
__host__ __device__ constexpr uint32_t idesc_tf32(int M, int N) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void mma_tf32(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(tmem_d),
      "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
// TMEM -> registers: this warp's 32 lanes x 16 consecutive 32-bit columns.
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float *v) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
#pragma unroll
  for (int k = 0; k < 16; ++k) v[k] = __uint_as_float(r[k]);
}


template <int BN, int STAGES>
struct GemmSmem {
  static constexpr int A_BYTES = BM * BK * 4;            // 16 KB per hi / lo tile
  static constexpr int B_BYTES = BN * BK * 4;
  static constexpr int STAGE_BYTES = 2 * A_BYTES + 2 * B_BYTES;
  static constexpr int BYTES = STAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 256 /*barriers*/;
};

// D partial[z][m][n] = sum over the K blocks of split z of A[m][k] B[n][k]  (3xTF32).
// The tensor core adds into its TMEM accumulator with truncation, so long accumulation chains drift
// (measured: 1e-5 relative after ~700 MMAs).  The chain is therefore cut every DRAIN K blocks: the
// MMA warp alternates between two TMEM accumulators, and the eight accumulate warps add each
// finished chunk into FP32 registers (round-to-nearest) while the next chunk is being multiplied.
// grid (M tiles, N tiles, splits), block GEMM_THREADS, dyn smem GemmSmem<BN,STAGES>::BYTES.
// out: [splits][m_rows][ldo] floats, m_rows = gridDim.x * BM, ldo >= gridDim.y * BN.
// With NP > 0 the A operand (basis columns of Eq. 10, for the standard term list
// NP P' terms x^i - x^NP, NFF FF' terms x^j - x^NFF, optional delz column; 8 rows per slice) is
// generated by four producer warps straight into the swizzled shared-memory tiles instead of
// being loaded by TMA: J_b is never materialised in HBM.
struct AProd {
  const float *xn, *dzc;      // [B][N] normalised flux (-1 outside the mask), delz column
  const int *cnode;           // [Kc] compact node list
  const float *rdA, *fdA;     // [Kc] R dA and mu0 dA / R of the compact nodes
  int N, B, has_delz;
  // epilogue of the DST products (split solve path): epi = 1 stores D[(s, i)][c] * scale transposed
  // into the flux grid, out[s][(c + 1) nr + i + 1], rows r = s RS + i; epi = 0: plain partials
  int epi, RS, nri, nzi, nr;
  float scale;
};
constexpr int PROD_GROUPS = 2;   // groups of four basis-producer warps; group g fills the K blocks kb0 + g, kb0 + g + PROD_GROUPS, ...
template <int NP> constexpr int gemm_threads() { return NP > 0 ? GEMM_THREADS + 128 * PROD_GROUPS : GEMM_THREADS; }

template <int BN, int STAGES, int NP = 0, int NFF = 0>
__global__ void __launch_bounds__(gemm_threads<NP>(), 1)
k_gemm_3xtf32(const __grid_constant__ CUtensorMap mapAhi, const __grid_constant__ CUtensorMap mapAlo,
              const __grid_constant__ CUtensorMap mapBhi, const __grid_constant__ CUtensorMap mapBlo,
              float *__restrict__ out, int ldo, int kblocks, const AProd ap) {
  using L = GemmSmem<BN, STAGES>;
  static_assert(BN % 16 == 0 && BN <= 256, "N tile");
  extern __shared__ unsigned char smem_raw[];
  unsigned char *base = reinterpret_cast<unsigned char *>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint64_t *full = reinterpret_cast<uint64_t *>(base + STAGES * L::STAGE_BYTES);
  uint64_t *empty = full + STAGES;
  uint64_t *tfull = empty + STAGES;                    // [2] accumulator chunk ready
  uint64_t *tempty = tfull + 2;                        // [2] accumulator drained
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + 2);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN;
  const int nsplit = gridDim.z, z = blockIdx.z;
  const int kb0 = (int)(((long long)kblocks * z) / nsplit), kb1 = (int)(((long long)kblocks * (z + 1)) / nsplit);
  const int nchunks = (kb1 - kb0 + DRAIN - 1) / DRAIN;
  constexpr int ACC_COLS = BN <= 64 ? 64 : BN <= 128 ? 128 : 256;      // column stride between the two accumulators
  constexpr int TMEM_COLS = 2 * ACC_COLS;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&mapAhi); tma_prefetch_desc(&mapAlo); tma_prefetch_desc(&mapBhi); tma_prefetch_desc(&mapBlo);
    for (int s = 0; s < STAGES; ++s) { mbar_init(full + s, NP > 0 ? 5 : 1); mbar_init(empty + s, 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tfull + b, 1); mbar_init(tempty + b, 8); }
    fence_barrier_init();
  }
  if (NP > 0) {                                        // rows of unused terms stay zero for the whole kernel
    for (int e = threadIdx.x; e < STAGES * 2 * L::A_BYTES / 16; e += blockDim.x) {
      const int st = e / (2 * L::A_BYTES / 16), w = e - st * (2 * L::A_BYTES / 16);
      reinterpret_cast<uint4 *>(base + st * L::STAGE_BYTES)[w] = make_uint4(0, 0, 0, 0);
    }
    fence_proxy_async();
  }
  if (warp == 1) tmem_alloc<TMEM_COLS>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {                                   // ---- TMA producer
      for (int kb = kb0, it = 0; kb < kb1; ++kb, ++it) {
        const int s = it % STAGES;
        const uint32_t ph = (uint32_t)(it / STAGES) & 1u;
        mbar_wait(empty + s, ph ^ 1u);
        unsigned char *st = base + s * L::STAGE_BYTES;
        mbar_expect_tx(full + s, (uint32_t)(NP > 0 ? 2 * L::B_BYTES : L::STAGE_BYTES));
        if (NP == 0) {
          tma_load_2d(st, &mapAhi, full + s, kb * BK, m0);
          tma_load_2d(st + L::A_BYTES, &mapAlo, full + s, kb * BK, m0);
        }
        tma_load_2d(st + 2 * L::A_BYTES, &mapBhi, full + s, kb * BK, n0);
        tma_load_2d(st + 2 * L::A_BYTES + L::B_BYTES, &mapBlo, full + s, kb * BK, n0);
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {                                   // ---- MMA issuer
      constexpr uint32_t idesc = idesc_tf32(BM, BN);
      int it = 0;
      for (int c = 0; c < nchunks; ++c) {
        const int buf = c & 1;
        mbar_wait(tempty + buf, ((uint32_t)(c >> 1) & 1u) ^ 1u);       // accumulator drained by the register adders
        tc_fence_after();
        const uint32_t tacc = tmem_base + (uint32_t)(buf * ACC_COLS);
        const int kend = min(kb0 + (c + 1) * DRAIN, kb1);
        for (int kb = kb0 + c * DRAIN; kb < kend; ++kb, ++it) {
          const int s = it % STAGES;
          const uint32_t ph = (uint32_t)(it / STAGES) & 1u;
          mbar_wait(full + s, ph);
          tc_fence_after();
          const uint32_t sa = smem_u32(base + s * L::STAGE_BYTES);
          const uint64_t dAhi = smem_desc_sw128(sa), dAlo = smem_desc_sw128(sa + L::A_BYTES);
          const uint64_t dBhi = smem_desc_sw128(sa + 2 * L::A_BYTES), dBlo = smem_desc_sw128(sa + 2 * L::A_BYTES + L::B_BYTES);
#pragma unroll
          for (int k = 0; k < BK / UMMA_K; ++k) {
            const uint64_t adv = (uint64_t)((k * UMMA_K * 4) >> 4);    // +32 bytes per K step inside the swizzle row
            // small terms first, so that they are not absorbed by the large one
            mma_tf32(tacc, dAlo + adv, dBhi + adv, idesc, (kb > kb0 + c * DRAIN || k > 0) ? 1u : 0u);
            mma_tf32(tacc, dAhi + adv, dBlo + adv, idesc, 1u);
            mma_tf32(tacc, dAhi + adv, dBhi + adv, idesc, 1u);
          }
          tc_commit(empty + s);                        // frees the stage once these MMAs have read it
        }
        tc_commit(tfull + buf);                        // chunk complete
      }
    }
  } else if (NP > 0 && warp >= 10) {                   // ---- basis producers (warps 10-17: two groups of four)
    constexpr int NPOLY = NP + NFF;
    constexpr int PMAX = NP > NFF ? NP : NFF;
    // lane -> (slice sq = lane >> 3 of the warp's four, node quad kq = lane & 7 of the block's
    // 32 nodes): four consecutive nodes of one slice per thread, so that every term row is one
    // 16-byte store per hi / lo tile (a quarter warp covers one 128-byte row: conflict free).
    const int pg = (warp - 10) >> 2, pw_ = (warp - 10) & 3, sq = lane >> 3, kq = lane & 7;
    const int sl = min(m0 / 8 + 4 * pw_ + sq, ap.B - 1);
    const float *xs = ap.xn + (size_t)sl * ap.N, *ds = ap.dzc + (size_t)sl * ap.N;
    // software pipeline of the gather: node indices and factors of block kb + 3, flux values of
    // block kb + 2 (their addresses need the indices), arithmetic of block kb
    int4 nidx = make_int4(0, 0, 0, 0);
    float4 nr_ = make_float4(0.f, 0.f, 0.f, 0.f), nf_ = nr_;
    auto fetch_idx = [&](int kb) {
      if (kb >= kb1) return;
      const int kc = kb * BK + 4 * kq;
      nidx = *reinterpret_cast<const int4 *>(ap.cnode + kc);
      nr_ = *reinterpret_cast<const float4 *>(ap.rdA + kc);
      nf_ = *reinterpret_cast<const float4 *>(ap.fdA + kc);
    };
    auto fetch_val = [&](int kb, float *x, float *d, float4 &r, float4 &f) {   // uses nidx = indices of block kb
      if (kb >= kb1) return;
      const int4 n = nidx;
      r = nr_; f = nf_;
      x[0] = xs[n.x]; x[1] = xs[n.y]; x[2] = xs[n.z]; x[3] = xs[n.w];
      if (ap.has_delz) { d[0] = ds[n.x]; d[1] = ds[n.y]; d[2] = ds[n.z]; d[3] = ds[n.w]; }
      else d[0] = d[1] = d[2] = d[3] = 0.f;
    };
    // one K block: consume a register buffer filled two blocks ago, refill it for block kb + 2
    // (gather latency ~ two block times), then write the tiles of block kb
    auto step = [&](int kb, int it, float *xb, float *db, float4 &rb, float4 &fb) {
      const int s = it % STAGES;
      const uint32_t ph = (uint32_t)(it / STAGES) & 1u;
      float d[4];
      const float r[4] = {rb.x, rb.y, rb.z, rb.w}, f[4] = {fb.x, fb.y, fb.z, fb.w};
      float pwv[4][PMAX + 1];
      bool in[4];
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        d[t] = db[t];
        pwv[t][0] = 1.f;
#pragma unroll
        for (int k = 1; k <= PMAX; ++k) pwv[t][k] = pwv[t][k - 1] * xb[t];
        in[t] = !(xb[t] < 0.f);
      }
      fetch_val(kb + 2 * PROD_GROUPS, xb, db, rb, fb);
      fetch_idx(kb + 3 * PROD_GROUPS);
      mbar_wait(empty + s, ph ^ 1u);
      unsigned char *ahi = base + s * L::STAGE_BYTES, *alo = ahi + L::A_BYTES;
      const uint32_t rowbase = (uint32_t)(4 * pw_ + sq) * 1024u;
#pragma unroll
      for (int l = 0; l < NPOLY + 1; ++l) {
        if (l == NPOLY && !ap.has_delz) break;
        uint32_t hr[4], lr[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          float v;
          if (l < NP) v = in[t] ? (pwv[t][l] - pwv[t][NP]) * r[t] : 0.f;
          else if (l < NPOLY) v = in[t] ? (pwv[t][l - NP] - pwv[t][NFF]) * f[t] : 0.f;
          else v = d[t];
          // hi = v rounded to TF32 (add half an ulp of the 10-bit mantissa, clear the low 13 bits: two
          // instructions where cvt.rna.tf32.f32 costs four on sm_100a); lo = v - hi exactly, its low bits
          // are ignored by the tensor core
          hr[t] = (__float_as_uint(v) + 0x1000u) & 0xffffe000u;
          lr[t] = __float_as_uint(v - __uint_as_float(hr[t]));
        }
        const uint32_t off = rowbase + (uint32_t)l * 128u + (((uint32_t)kq ^ (uint32_t)l) << 4);
        *reinterpret_cast<uint4 *>(ahi + off) = make_uint4(hr[0], hr[1], hr[2], hr[3]);
        *reinterpret_cast<uint4 *>(alo + off) = make_uint4(lr[0], lr[1], lr[2], lr[3]);
      }
      fence_proxy_async();                              // generic-proxy writes -> visible to tcgen05.mma
      __syncwarp();
      if (lane == 0) mbar_arrive(full + s);
    };
    float xa[4], da[4], xb2[4], db2[4];
    float4 ra, fa, rb2, fb2;
    const int k0 = kb0 + pg;                             // this group's first K block
    fetch_idx(k0);
    fetch_val(k0, xa, da, ra, fa);
    fetch_idx(k0 + PROD_GROUPS);
    fetch_val(k0 + PROD_GROUPS, xb2, db2, rb2, fb2);
    fetch_idx(k0 + 2 * PROD_GROUPS);
    for (int kb = k0; kb < kb1; kb += 2 * PROD_GROUPS) {
      step(kb, kb - kb0, xa, da, ra, fa);
      if (kb + PROD_GROUPS < kb1) step(kb + PROD_GROUPS, kb + PROD_GROUPS - kb0, xb2, db2, rb2, fb2);
    }
  } else if (warp >= 2 && warp < 10) {                 // ---- promotion to registers + epilogue
    const int q = warp & 3;                            // TMEM lane quarter this warp may access
    const int half = (warp - 2) >> 2;                  // which half of the columns
    constexpr int C0 = ((BN / 16 + 1) / 2) * 16;       // columns of half 0 (multiple of 16)
    constexpr int NCH = C0 / 16;                       // 16-column groups per thread (half 1 may use fewer)
    const int col0 = half ? C0 : 0, ncols = half ? BN - C0 : C0;
    float acc[NCH][16];
#pragma unroll
    for (int g = 0; g < NCH; ++g)
#pragma unroll
      for (int k = 0; k < 16; ++k) acc[g][k] = 0.f;
    for (int c = 0; c < nchunks; ++c) {
      const int buf = c & 1;
      mbar_wait(tfull + buf, (uint32_t)(c >> 1) & 1u);
      tc_fence_after();
      const uint32_t tacc = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * ACC_COLS + col0);
#pragma unroll
      for (int g = 0; g < NCH; ++g) {
        if (g * 16 < ncols) {
          float v[16];
          tmem_ld16(tacc + (uint32_t)(g * 16), v);
#pragma unroll
          for (int k = 0; k < 16; ++k) acc[g][k] += v[k];
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty + buf);
    }
    const int row = q * 32 + lane;
    if (ap.epi == 1) {
      const int r = m0 + row, sl = r / ap.RS, i = r - sl * ap.RS;
      if (sl < ap.B && i < ap.nri) {
        float *o = out + (size_t)sl * ap.N + i + 1;
#pragma unroll
        for (int g = 0; g < NCH; ++g) {
          if (g * 16 < ncols) {
#pragma unroll
            for (int k = 0; k < 16; ++k) {
              const int c = n0 + col0 + g * 16 + k;              // mode / row index c + 1 of the grid
              if (c < ap.nzi) o[(c + 1) * ap.nr] = acc[g][k] * ap.scale;
            }
          }
        }
      }
    } else {
    float *o = out + ((size_t)z * gridDim.x * BM + m0 + row) * ldo + n0 + col0;
#pragma unroll
    for (int g = 0; g < NCH; ++g) {
      if (g * 16 < ncols) {
#pragma unroll
        for (int k = 0; k < 16; k += 4)
          *reinterpret_cast<float4 *>(o + g * 16 + k) = make_float4(acc[g][k], acc[g][k + 1], acc[g][k + 2], acc[g][k + 3]);
      }
    }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc<TMEM_COLS>(tmem_base);
}

}  // namespace tc
}  // namespace ptefit
