// gemm_tc.cu — BF16 node contractions (a3, a5 and their adjoints) on the 5th-generation tensor cores.
//
//   C[M,N] = epi( A[M,K] * Wt[N,K]^T ),  BF16 operands, FP32 accumulation.
//
// One CTA computes a 128 x BN tile (BN = largest of 256/128/64/32 dividing N).  Warp roles:
//   warp 0    TMA producer: cp.async.bulk.tensor.2d of the A tile [128 x 64] and the Wt tile [BN x 64] per k-block into
//             a ring of shared-memory stages (SWIZZLE_128B, K-major), completion on the stage's "full" mbarrier;
//   warp 1    MMA issuer: one thread issues tcgen05.mma.cta_group::1.kind::f16 (M = 128, N = BN, K = 16) four times per
//             k-block, accumulator in TMEM; tcgen05.commit frees the stage ("empty" mbarrier) and finally signals
//             the epilogue ("accumulator full" mbarrier);
//   warps 2-5 epilogue: tcgen05.ld (32 lanes x 32 columns per warp): a thread owns one output row and walks it 32 columns
//             at a time, then bias / SiLU / silu' / accumulate and FP32 / BF16 stores as 32-byte pieces of that row.
//             Warp 2 also allocates and frees the TMEM columns.  The persistent kernel (tc_gemm_pk) runs eight epilogue warps,
//             two per TMEM lane quadrant splitting the tile's columns, and, where the epilogue has bias / activation work
//             (TST), sends the BF16 output through shared memory and the TMA engine instead: a warp stages its 32 rows x 64
//             columns (128-byte swizzle) and one lane issues cp.async.bulk.tensor shared -> global.
// K <= 768 here (at most 12 k-blocks), so a CTA is short; two CTAs share an SM (TMEM 2 x 256 columns, shared memory
// 2 x <= 113 KB) so one tile's epilogue overlaps the other's loads and MMAs.
#include <cuda.h>

#include <algorithm>
#include <cstdlib>
#include <mutex>
#include <unordered_map>

#include "common.cuh"
#include "gemm_tc.cuh"
#include "tc_ptx.cuh"

namespace pnn {

namespace {

constexpr int BM = 128, BK = 64;
constexpr int EPI_PER_Q = 2;                      // persistent kernel: epilogue warps per TMEM lane quadrant
constexpr int NTHREADS_PK = 64 + 128 * EPI_PER_Q; // TMA warp, MMA warp, 4 * EPI_PER_Q epilogue warps

using namespace tc;

// SiLU of the READOUT epilogue: ex2.approx / rcp.approx (relative error ~1e-6) instead of expf and an IEEE division, about 6
// instead of 18 instructions per element.  Only there: the readout sums silu values in FP32 straight into the atom energy, so
// the approximation stays a 1e-6 effect.  In the hidden layers the activation is rounded to BF16 and fed on, and a change
// in the last bits flips BF16 rounding decisions that the network amplifies (cfg3 results move by
// percents under 1e-7 perturbations) -- measured: with the approximate SiLU in the hidden-layer epilogues the cfg4 batch
// gains another 0.3 ms, and the single-structure cfg3 BF16 blended check moves from inside 2e-2 to 3.3e-2.  They keep silu_f.
__device__ __forceinline__ float silu_fast(float x) { return __fdividef(x, 1.0f + __expf(-x)); }

__device__ __forceinline__ void sts128(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
// 32-byte global store (STG.256 on sm_100: one full L2 sector per instruction; a row-owner thread otherwise writes its
// row in 16-byte halves of a sector).  p must be 32-byte aligned.
__device__ __forceinline__ void st256(void* p, uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t a4,
                                      uint32_t a5, uint32_t a6, uint32_t a7) {
  asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "r"(a0), "r"(a1), "r"(a2), "r"(a3),
               "r"(a4), "r"(a5), "r"(a6), "r"(a7)
               : "memory");
}
__device__ __forceinline__ void ld256(const void* p, float (&v)[8]) {
  uint32_t a[8];
  asm volatile("ld.global.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(a[0]), "=r"(a[1]), "=r"(a[2]), "=r"(a[3]), "=r"(a[4]), "=r"(a[5]), "=r"(a[6]), "=r"(a[7])
               : "l"(p)
               : "memory");
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(a[i]);
}
__device__ __forceinline__ bool al32(const void* p, int64_t ld_bytes) {
  return ((reinterpret_cast<uintptr_t>(p) | (uintptr_t)ld_bytes) & 31) == 0;
}

// Epilogue of one output row segment: 32 accumulator columns of row m starting at column n (bias, activation, optional
// pre-activation store / silu' factor / accumulate, FP32 and / or BF16 stores as 16-byte vectors of the row).
template <bool KEEP_CB = false>
__device__ __forceinline__ void epi_chunk(const TcEpi& epi, int64_t m, int n, const uint32_t (&r)[32], uint32_t* hout = nullptr) {
  float x[32];
#pragma unroll
  for (int j = 0; j < 32; ++j) x[j] = __uint_as_float(r[j]);
  if (epi.bias) {
#pragma unroll
    for (int j = 0; j < 32; j += 4) {
      const float4 bv = __ldg(reinterpret_cast<const float4*>(epi.bias + n + j));
      x[j] += bv.x; x[j + 1] += bv.y; x[j + 2] += bv.z; x[j + 3] += bv.w;
    }
  }
  if (epi.act == ACT_SILU) {
    if (epi.pre) {
      float* pp = epi.pre + m * epi.ldpre + n;
      if (al32(epi.pre, epi.ldpre * 4)) {
#pragma unroll
        for (int j = 0; j < 32; j += 8)
          st256(pp + j, __float_as_uint(x[j]), __float_as_uint(x[j + 1]), __float_as_uint(x[j + 2]),
                __float_as_uint(x[j + 3]), __float_as_uint(x[j + 4]), __float_as_uint(x[j + 5]),
                __float_as_uint(x[j + 6]), __float_as_uint(x[j + 7]));
      } else {
#pragma unroll
        for (int j = 0; j < 32; j += 4)
          reinterpret_cast<float4*>(pp)[j >> 2] = make_float4(x[j], x[j + 1], x[j + 2], x[j + 3]);
      }
    }
#pragma unroll
    for (int j = 0; j < 32; ++j) x[j] = silu_f<float>(x[j]);
  } else if (epi.act == ACT_MUL_DSILU) {
    const float* ap = epi.aux + m * epi.ldaux + n;
    if (al32(epi.aux, epi.ldaux * 4)) {
#pragma unroll
      for (int j = 0; j < 32; j += 8) {
        float av[8];
        ld256(ap + j, av);
#pragma unroll
        for (int i = 0; i < 8; ++i) x[j + i] *= dsilu_f<float>(av[i]);
      }
    } else {
#pragma unroll
      for (int j = 0; j < 32; j += 4) {
        const float4 av = reinterpret_cast<const float4*>(ap)[j >> 2];
        x[j] *= dsilu_f<float>(av.x); x[j + 1] *= dsilu_f<float>(av.y);
        x[j + 2] *= dsilu_f<float>(av.z); x[j + 3] *= dsilu_f<float>(av.w);
      }
    }
  }
  if (epi.C) {
    float4* cp = reinterpret_cast<float4*>(epi.C + m * epi.ldc + n);
    if (epi.accumulate) {
      if (al32(epi.C, epi.ldc * 4)) {
#pragma unroll
        for (int j = 0; j < 32; j += 8) {
          float cv[8];
          ld256(reinterpret_cast<const float*>(cp) + j, cv);
#pragma unroll
          for (int i = 0; i < 8; ++i) x[j + i] += cv[i];
        }
      } else {
#pragma unroll
        for (int j = 0; j < 32; j += 4) {
          const float4 cv = cp[j >> 2];
          x[j] += cv.x; x[j + 1] += cv.y; x[j + 2] += cv.z; x[j + 3] += cv.w;
        }
      }
    }
    if (al32(epi.C, epi.ldc * 4)) {
#pragma unroll
      for (int j = 0; j < 32; j += 8)
        st256(reinterpret_cast<float*>(cp) + j, __float_as_uint(x[j]), __float_as_uint(x[j + 1]),
              __float_as_uint(x[j + 2]), __float_as_uint(x[j + 3]), __float_as_uint(x[j + 4]),
              __float_as_uint(x[j + 5]), __float_as_uint(x[j + 6]), __float_as_uint(x[j + 7]));
    } else {
#pragma unroll
      for (int j = 0; j < 32; j += 4) cp[j >> 2] = make_float4(x[j], x[j + 1], x[j + 2], x[j + 3]);
    }
  }
  if (KEEP_CB) { // TMA-store epilogue: the BF16 words go to the caller, which stages them in shared memory
#pragma unroll
    for (int j = 0; j < 32; j += 2) {
      __nv_bfloat162 t = __floats2bfloat162_rn(x[j], x[j + 1]);
      hout[j >> 1] = *reinterpret_cast<uint32_t*>(&t);
    }
  } else if (epi.Cb) {
    uint4* bp = reinterpret_cast<uint4*>(epi.Cb + m * epi.ldcb + n);
    uint32_t h[16];
#pragma unroll
    for (int j = 0; j < 32; j += 2) {
      __nv_bfloat162 t = __floats2bfloat162_rn(x[j], x[j + 1]);
      h[j >> 1] = *reinterpret_cast<uint32_t*>(&t);
    }
    if (al32(epi.Cb, epi.ldcb * 2)) {
      st256(bp, h[0], h[1], h[2], h[3], h[4], h[5], h[6], h[7]);
      st256(bp + 2, h[8], h[9], h[10], h[11], h[12], h[13], h[14], h[15]);
    } else {
#pragma unroll
      for (int q = 0; q < 4; ++q) bp[q] = make_uint4(h[4 * q], h[4 * q + 1], h[4 * q + 2], h[4 * q + 3]);
    }
  }
}

template <int BN, int STAGES>
struct TcSmem {
  static constexpr int A_BYTES = BM * BK * 2;
  static constexpr int B_BYTES = BN * BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int PIPE_BYTES = STAGES * STAGE_BYTES;
  static constexpr int TOTAL = PIPE_BYTES + 1024 /*alignment slack*/ + 256;
};

template <int BN, int STAGES>
__global__ void __launch_bounds__(NTHREADS_PK)
tc_gemm_k(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, int64_t M, int N, int K,
          int n_tiles, TcEpi epi) {
  using L = TcSmem<BN, STAGES>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t tiles = (raw + 1023u) & ~1023u;                 // 1024-byte aligned stage ring
  unsigned char* tiles_ptr = smem_raw + (tiles - raw);
  const uint32_t PIPE = L::PIPE_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(tiles_ptr + PIPE); // full[STAGES], empty[STAGES], accfull
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * STAGES + 1);
  const uint32_t bar0 = smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (STAGES + s); };
  const uint32_t acc_bar = bar0 + 8u * (2 * STAGES);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t m_tile = blockIdx.x / n_tiles;
  const int n_tile = blockIdx.x % n_tiles;
  const int64_t m0 = m_tile * BM;
  const int n0 = n_tile * BN;
  const int nkb = (K + BK - 1) / BK;
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    mbar_init(acc_bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(BN)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % STAGES;
        const uint32_t ph = (kb / STAGES) & 1;
        mbar_wait(empty_bar(s), ph ^ 1u);
        const uint32_t sa = tiles + s * L::STAGE_BYTES;
        mbar_expect_tx(full_bar(s), L::STAGE_BYTES);
        tma_load_2d(sa, &tmA, full_bar(s), kb * BK, (int)m0);
        tma_load_2d(sa + L::A_BYTES, &tmB, full_bar(s), kb * BK, n0);
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      // instruction descriptor: D = F32, A = B = BF16, both K-major, N = BN, M = 128
      const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % STAGES;
        const uint32_t ph = (kb / STAGES) & 1;
        mbar_wait(full_bar(s), ph);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t sa = tiles + s * L::STAGE_BYTES;
        const uint64_t ad = umma_desc_sw128(sa), bd = umma_desc_sw128(sa + L::A_BYTES);
#pragma unroll
        for (int k = 0; k < BK / 16; ++k)
          umma_bf16(tmem_base, ad + (uint64_t)(k * 2), bd + (uint64_t)(k * 2), idesc, (kb | k) ? 1u : 0u);
        umma_commit(empty_bar(s));
      }
      umma_commit(acc_bar);
    }
  } else {
    // epilogue warps 2..5: TMEM lane quadrant = warp % 4; a thread owns one output row and walks it 32 columns at a
    // time (tcgen05.ld 32x32b.x32), so every global access is a 16-byte vector of that row
    // (EPI_PER_Q warps per quadrant split the tile's columns, as in the persistent kernel)
    const int q = warp & 3, part = (warp - 2) >> 2;
    constexpr int PARTS = (BN / 32 >= EPI_PER_Q) ? EPI_PER_Q : (BN >= 64 ? 2 : 1);
    const int c_lo = part < PARTS ? part * (BN / PARTS) : 0, c_hi = part < PARTS ? c_lo + BN / PARTS : 0;
    mbar_wait(acc_bar, 0);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const int64_t m = m0 + q * 32 + lane;
    const bool row_ok = m < M;
#pragma unroll 1
    for (int c0 = c_lo; c0 < c_hi; c0 += 32) {
      uint32_t r[32];
      tmem_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)c0, r);
      if (!row_ok) continue;
      epi_chunk(epi, m, n0 + c0, r);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  }
  __syncthreads();
  if (warp == 2) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(BN) : "memory");
  }
}

// Persistent variant for large M (the screening batches): one CTA per SM slot walks tiles t = blockIdx.x, + gridDim.x, ...
// The shared-memory stage ring runs on across tiles, and the accumulator is double-buffered in TMEM (2 x BN columns), so
// the TMA loads and MMAs of tile i+1 overlap the epilogue (global stores) of tile i: these GEMMs have K <= 768 and are
// bound by HBM traffic, not by the tensor pipe, so what matters is that loads and stores never pause.
// TST: the BF16 output leaves through shared memory and the TMA engine (cp.async.bulk.tensor shared -> global): an epilogue
// warp stages its 32 rows x 64 columns (4 KB, 128-byte swizzle as the tensor map of C expects) and one lane issues the store.
// A row-owner thread's own global stores touch 32 different lines per instruction and kept the L1 / LSU data pipe ~70 % busy on
// the wide-output launches (profiles/r02_bf16_node.md); staged, a warp's 4 KB cost 32 shared-memory wavefronts and one TMA.
constexpr int TST_WARP_BYTES = 32 * 128;
template <int BN, int STAGES, bool TST = false>
__global__ void __launch_bounds__(NTHREADS_PK, 2)
tc_gemm_pk(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
           const __grid_constant__ CUtensorMap tmC, int64_t M, int N, int K, int n_tiles, int64_t total_tiles, TcEpi epi) {
  constexpr int A_BYTES = BM * BK * 2, B_BYTES = BN * BK * 2, STAGE_BYTES = A_BYTES + B_BYTES;
  constexpr int STG_BYTES = TST ? 4 * EPI_PER_Q * TST_WARP_BYTES : 0;
  static_assert(!TST || (BN == 128 && EPI_PER_Q == 2), "TMA-store epilogue: 64 columns per epilogue warp");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t tiles = (raw + 1023u) & ~1023u;
  unsigned char* tiles_ptr = smem_raw + (tiles - raw);
  const uint32_t stg0 = tiles + STAGES * STAGE_BYTES; // TST: one 4 KB staging buffer per epilogue warp (1024-byte aligned)
  uint64_t* bars = reinterpret_cast<uint64_t*>(tiles_ptr + STAGES * STAGE_BYTES + STG_BYTES); // full[S], empty[S], accfull[2], accempty[2]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * STAGES + 4);
  const uint32_t bar0 = smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (STAGES + s); };
  auto accfull_bar = [&](int b) { return bar0 + 8u * (2 * STAGES + b); };
  auto accempty_bar = [&](int b) { return bar0 + 8u * (2 * STAGES + 2 + b); };
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nkb = (K + BK - 1) / BK;

  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(accfull_bar(b), 1); mbar_init(accempty_bar(b), 4 * EPI_PER_Q); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(2 * BN)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_base = *tmem_slot;

  // Tile sequence of this CTA, identical in the three roles.  Plain GEMM: tiles blockIdx.x, + gridDim.x, ... of the
  // (row tile, column tile) grid.  Readout mode: row tiles blockIdx.x, + gridDim.x, ..., and per row tile the heads
  // (column tiles) that occur in it (epi.head_mask).
  const int64_t m_tiles = (M + BM - 1) / BM;
  auto for_each_tile = [&](auto&& body) {
    if (epi.readout) {
      for (int64_t mt = blockIdx.x; mt < m_tiles; mt += gridDim.x) {
        unsigned long long msk = epi.head_mask[mt];
        while (msk) { const int h = __ffsll((long long)msk) - 1; msk &= msk - 1; body(mt, h); }
      }
    } else {
      for (int64_t tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) body(tile / n_tiles, (int)(tile % n_tiles));
    }
  };
  if (warp == 0) {
    if (lane == 0) {
      uint32_t it = 0; // k-blocks issued so far: stage = it % STAGES, parity = (it / STAGES) & 1
      for_each_tile([&](int64_t mt, int nt) {
        const int m0 = (int)(mt * BM), n0 = nt * BN;
        for (int kb = 0; kb < nkb; ++kb, ++it) {
          const int s = it % STAGES;
          mbar_wait(empty_bar(s), ((it / STAGES) & 1u) ^ 1u);
          const uint32_t sa = tiles + s * STAGE_BYTES;
          mbar_expect_tx(full_bar(s), STAGE_BYTES);
          tma_load_2d(sa, &tmA, full_bar(s), kb * BK, m0);
          tma_load_2d(sa + A_BYTES, &tmB, full_bar(s), kb * BK, n0);
        }
      });
    }
  } else if (warp == 1) {
    if (lane == 0) {
      const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
      uint32_t it = 0, j = 0; // j: tiles done by this CTA; accumulator buffer j & 1
      for_each_tile([&](int64_t, int) {
        const uint32_t b = j & 1u;
        mbar_wait(accempty_bar(b), ((j >> 1) & 1u) ^ 1u); // the epilogue has drained this buffer
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t acc = tmem_base + b * BN;
        for (int kb = 0; kb < nkb; ++kb, ++it) {
          const int s = it % STAGES;
          mbar_wait(full_bar(s), (it / STAGES) & 1u);
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
          const uint32_t sa = tiles + s * STAGE_BYTES;
          const uint64_t ad = umma_desc_sw128(sa), bd = umma_desc_sw128(sa + A_BYTES);
#pragma unroll
          for (int k = 0; k < BK / 16; ++k)
            umma_bf16(acc, ad + (uint64_t)(k * 2), bd + (uint64_t)(k * 2), idesc, (kb | k) ? 1u : 0u);
          umma_commit(empty_bar(s));
        }
        umma_commit(accfull_bar(b));
        ++j;
      });
    }
  } else {
    // Several warps share a TMEM lane quadrant (a warp reads the lanes 32 (warp % 4) ...) and split the tile's columns: these
    // GEMMs are bound by the epilogue (a row per thread: bias / activation / conversions and 32-byte stores of 256+ columns),
    // not by the tensor pipe or HBM, so more warps shorten it.  Readout mode sums over ALL columns of a head per row:
    // there (and for narrow tiles) the surplus warps of a quadrant only hand the buffer back.
    const int q = warp & 3, part = (warp - 2) >> 2;
    constexpr int PARTS = (BN / 32 >= EPI_PER_Q) ? EPI_PER_Q : (BN >= 64 ? 2 : 1); // column groups of >= 32
    const int parts = epi.readout ? 1 : PARTS;
    const int c_lo = part < parts ? part * (BN / parts) : 0, c_hi = part < parts ? c_lo + BN / parts : 0;
    uint32_t j = 0;
    for_each_tile([&](int64_t mt, int nt) {
      const uint32_t b = j & 1u;
      const int64_t m = mt * BM + q * 32 + lane;
      const int n0 = nt * BN;
      mbar_wait(accfull_bar(b), (j >> 1) & 1u);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      bool row_ok = m < M;
      int hrow = 0;
      float esum = 0.0f;
      if (epi.readout && row_ok) { // column tile nt = head nt: only the rows of that head are read out
        hrow = epi.head[epi.a2s[m]];
        row_ok = (hrow == nt);
      }
#pragma unroll 1
      for (int c0 = c_lo; c0 < c_hi; c0 += 32) {
        uint32_t r[32];
        tmem_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + b * BN + (uint32_t)c0, r);
        if (!row_ok && !TST) continue;
        if (epi.readout) {
          const int n = n0 + c0;
#pragma unroll
          for (int jj = 0; jj < 32; jj += 4) {
            const float4 bv = __ldg(reinterpret_cast<const float4*>(epi.bias + n + jj));
            const float4 wv = __ldg(reinterpret_cast<const float4*>(epi.w2 + n + jj));
            const float p0 = __uint_as_float(r[jj]) + bv.x, p1 = __uint_as_float(r[jj + 1]) + bv.y,
                        p2 = __uint_as_float(r[jj + 2]) + bv.z, p3 = __uint_as_float(r[jj + 3]) + bv.w;
            if (epi.opre) *reinterpret_cast<float4*>(epi.opre + m * BN + c0 + jj) = make_float4(p0, p1, p2, p3);
            esum = fmaf(wv.x, silu_fast(p0), esum); esum = fmaf(wv.y, silu_fast(p1), esum);
            esum = fmaf(wv.z, silu_fast(p2), esum); esum = fmaf(wv.w, silu_fast(p3), esum);
          }
          if (c0 + 32 >= BN) epi.eatom[m] = esum + epi.b2[hrow];
          continue;
        }
        if (TST) {
          const uint32_t sbuf = stg0 + (uint32_t)(warp - 2) * TST_WARP_BYTES;
          if (c0 == c_lo) { // the previous tile's store must have read this buffer before it is rewritten
            if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            __syncwarp();
          }
          uint32_t h[16];
          if (row_ok) epi_chunk<true>(epi, m, n0 + c0, r, h); // rows beyond M: staged as they are, clipped by the TMA store
          else {
#pragma unroll
            for (int i = 0; i < 16; ++i) h[i] = 0u;
          }
          const uint32_t rowb = sbuf + (uint32_t)lane * 128u, jc0 = (uint32_t)(c0 - c_lo) >> 3; // 16-byte chunk of column c0
#pragma unroll
          for (int i = 0; i < 4; ++i)
            sts128(rowb + (((jc0 + i) ^ ((uint32_t)lane & 7u)) << 4), h[4 * i], h[4 * i + 1], h[4 * i + 2], h[4 * i + 3]);
          if (c0 + 32 >= c_hi) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) {
              asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(
                               reinterpret_cast<uint64_t>(&tmC)),
                           "r"(n0 + c_lo), "r"((int)(mt * BM) + q * 32), "r"(sbuf)
                           : "memory");
              asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
          }
          continue;
        }
        epi_chunk(epi, m, n0 + c0, r);
      }
      // all TMEM reads of this warp are complete (tcgen05.wait::ld in tmem_ld32): hand the buffer back to the MMA warp
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      __syncwarp();
      if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(accempty_bar(b)) : "memory");
      ++j;
    });
  }
  if (TST && warp >= 2 && lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); // stores done before exit
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 2) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(2 * BN) : "memory");
  }
}

__global__ void __launch_bounds__(256) f32_to_bf16_k(int64_t n, const float* __restrict__ src,
                                                     __nv_bfloat16* __restrict__ dst) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = __float2bfloat16_rn(src[i]);
}

// ------------------------------------------------------------------------------------------ TMA descriptors
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  });
  return fn;
}

struct MapKey {
  const void* ptr; int64_t rows, ld; int cols, box_rows;
  bool operator==(const MapKey& o) const {
    return ptr == o.ptr && rows == o.rows && ld == o.ld && cols == o.cols && box_rows == o.box_rows;
  }
};
struct MapKeyHash {
  size_t operator()(const MapKey& k) const {
    size_t h = std::hash<const void*>()(k.ptr);
    h = h * 1000003u ^ std::hash<int64_t>()(k.rows);
    h = h * 1000003u ^ std::hash<int64_t>()(k.ld);
    h = h * 1000003u ^ std::hash<int>()(k.cols * 512 + k.box_rows);
    return h;
  }
};

// BF16 row-major [rows][cols] with row stride ld (elements); box = [box_rows][64], 128-byte swizzle, OOB zero fill.
bool get_tensor_map(const __nv_bfloat16* ptr, int64_t rows, int cols, int64_t ld, int box_rows, CUtensorMap* out) {
  static std::unordered_map<MapKey, CUtensorMap, MapKeyHash> cache;
  static std::mutex mu;
  const MapKey key{ptr, rows, ld, cols, box_rows};
  std::lock_guard<std::mutex> lock(mu);
  auto it = cache.find(key);
  if (it != cache.end()) { *out = it->second; return true; }
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  CUtensorMap tm;
  const cuuint64_t gdim[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  const cuuint64_t gstride[1] = {(cuuint64_t)ld * 2};
  const cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<__nv_bfloat16*>(ptr), gdim, gstride, box,
                        estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  if (cache.size() > 4096) cache.clear();
  cache.emplace(key, tm);
  *out = tm;
  return true;
}

template <int BN, int STAGES, bool TST = false>
int launch_persistent(int64_t M, int N, int K, const CUtensorMap& ta, const CUtensorMap& tb, const TcEpi& epi,
                      cudaStream_t st, const CUtensorMap* tc = nullptr) {
  constexpr int SMEM = STAGES * (BM * BK * 2 + BN * BK * 2) + (TST ? 4 * EPI_PER_Q * TST_WARP_BYTES : 0) + 1024 + 256;
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(tc_gemm_pk<BN, STAGES, TST>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
    attr_set = true;
  }
  const int n_tiles = N / BN;
  const int64_t total = ((M + BM - 1) / BM) * n_tiles;
  const int per_sm = (2 * BN <= 256 && SMEM <= 110 * 1024) ? 2 : 1; // TMEM: 512 columns per SM
  const unsigned grid = (unsigned)std::min<int64_t>(total, 148 * per_sm);
  tc_gemm_pk<BN, STAGES, TST><<<grid, NTHREADS_PK, SMEM, st>>>(ta, tb, tc ? *tc : ta, M, N, K, n_tiles, total, epi);
  PNN_KCHECK("tc_gemm_pk");
  return 1;
}

template <int BN, int STAGES>
int launch_cfg(int64_t M, int N, int K, const CUtensorMap& ta, const CUtensorMap& tb, const TcEpi& epi,
               cudaStream_t st) {
  using L = TcSmem<BN, STAGES>;
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(tc_gemm_k<BN, STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, L::TOTAL);
    attr_set = true;
  }
  const int n_tiles = N / BN;
  const int64_t m_tiles = (M + BM - 1) / BM;
  tc_gemm_k<BN, STAGES><<<(unsigned)(m_tiles * n_tiles), NTHREADS_PK, L::TOTAL, st>>>(ta, tb, M, N, K, n_tiles, epi);
  PNN_KCHECK("tc_gemm_k");
  return 1;
}

} // namespace

int launch_gemm_tc(int64_t M, int N, int K, const __nv_bfloat16* A, int64_t lda, const __nv_bfloat16* Wt, int64_t ldw,
                   const TcEpi& epi, cudaStream_t st) {
  if (M <= 0) return 0;
  // Widest tile that still gives about two waves of CTAs: small problems (a few thousand rows) are bound by the
  // serial load -> MMA -> epilogue latency of one CTA, so they are cut into more, narrower tiles.
  const int64_t m_tiles = (M + BM - 1) / BM;
  int bn = (N % 64 == 0) ? 64 : 32;
  for (int cand = 256; cand > 64; cand >>= 1)
    if (N % cand == 0 && m_tiles * (N / cand) >= 2 * 148) { bn = cand; break; }
  const bool persist = m_tiles * (N / bn) >= 8 * 148;
  // persistent kernel: 128-wide tiles, so that two CTAs (eight epilogue warps) share an SM and its 512 TMEM columns
  if (persist && bn == 256) bn = 128;
  CUtensorMap ta, tb;
  if (!get_tensor_map(A, M, K, lda, BM, &ta) || !get_tensor_map(Wt, N, K, ldw, bn, &tb)) return -1;
  if (persist) { // many tiles per SM: the persistent, double-buffered kernel
    switch (bn) {
      case 256: return launch_persistent<256, 4>(M, N, K, ta, tb, epi, st);
      case 128: {
        // BF16 output, no readout: through shared memory and the TMA store engine (two pipeline stages make room for the
        // staging buffers at two CTAs per SM)
        CUtensorMap tc;
        // Measured on cfg4 (ncu, per launch): N x 768 with bias 264 -> 205 us, N x 256 with bias and SiLU 166 -> 88 us (with the
        // approximate SiLU), but the plain 3N x 512 conversion epilogue 420 -> 440 us (it loses the third stage and had
        // little arithmetic to take the stores away from): staged stores only where the epilogue has bias / activation work
        if (epi.Cb && !epi.readout && (epi.bias || epi.act) && (reinterpret_cast<uintptr_t>(epi.Cb) & 15) == 0 &&
            (epi.ldcb * 2) % 16 == 0 &&
            get_tensor_map(epi.Cb, M, N, epi.ldcb, 32, &tc))
          return launch_persistent<128, 2, true>(M, N, K, ta, tb, epi, st, &tc);
        return launch_persistent<128, 3>(M, N, K, ta, tb, epi, st);
      }
      case 64: return launch_persistent<64, 4>(M, N, K, ta, tb, epi, st);
      default: return launch_persistent<32, 4>(M, N, K, ta, tb, epi, st);
    }
  }
  switch (bn) {
    case 256: return launch_cfg<256, 2>(M, N, K, ta, tb, epi, st);
    case 128: return launch_cfg<128, 3>(M, N, K, ta, tb, epi, st);
    case 64: return launch_cfg<64, 4>(M, N, K, ta, tb, epi, st);
    default: return launch_cfg<32, 4>(M, N, K, ta, tb, epi, st);
  }
}

bool readout_tc_supported(int F, int H) { return (F == 64 || F == 128 || F == 256) && H <= 64; }

// mask[t] = set of heads used by the rows of the 128-row tile t (one warp per tile); bad head indices are flagged
__global__ void __launch_bounds__(256) head_mask_k(int64_t N, int H, const int32_t* __restrict__ a2s,
                                                   const int32_t* __restrict__ head, unsigned long long* mask, int* d_err) {
  const int64_t t = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (t * BM >= N) return;
  unsigned long long m = 0;
  bool bad = false;
  for (int r = lane; r < BM; r += 32) {
    const int64_t row = t * BM + r;
    if (row < N) {
      const int h = head[a2s[row]];
      if (h < 0 || h >= H) bad = true; else m |= 1ull << h;
    }
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) m |= __shfl_xor_sync(0xffffffffu, m, o);
  if (__any_sync(0xffffffffu, bad) && lane == 0) atomicOr(d_err, ERRF_BAD_HEAD);
  if (lane == 0) mask[t] = m;
}

int launch_readout_tc(int64_t N, int F, int H, const __nv_bfloat16* s16, const __nv_bfloat16* W1all, const float* b1,
                      const float* w2, const float* b2, const int32_t* a2s, const int32_t* head, float* opre,
                      float* eatom, int* d_err, unsigned long long* head_mask, cudaStream_t st) {
  if (N <= 0) return 0;
  const int Fh = F / 2;
  if (!readout_tc_supported(F, H)) return -1;
  CUtensorMap ta, tb;
  if (!get_tensor_map(s16, N, F, F, BM, &ta) || !get_tensor_map(W1all, (int64_t)H * Fh, F, F, Fh, &tb)) return -1;
  const int64_t m_tiles = (N + BM - 1) / BM;
  head_mask_k<<<(unsigned)((m_tiles * 32 + 255) / 256), 256, 0, st>>>(N, H, a2s, head, head_mask, d_err);
  PNN_KCHECK("head_mask_k");
  TcEpi e;
  e.bias = b1; e.readout = 1; e.a2s = a2s; e.head = head; e.w2 = w2; e.b2 = b2; e.eatom = eatom; e.opre = opre;
  e.H = H; e.d_err = d_err; e.head_mask = head_mask;
  switch (Fh) {
    case 128: return 1 + launch_persistent<128, 3>(N, H * Fh, F, ta, tb, e, st);
    case 64: return 1 + launch_persistent<64, 4>(N, H * Fh, F, ta, tb, e, st);
    default: return 1 + launch_persistent<32, 4>(N, H * Fh, F, ta, tb, e, st);
  }
}

int launch_f32_to_bf16(int64_t n, const float* src, __nv_bfloat16* dst, cudaStream_t st) {
  if (n <= 0) return 0;
  f32_to_bf16_k<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, src, dst);
  PNN_KCHECK("f32_to_bf16_k");
  return 1;
}

} // namespace pnn
