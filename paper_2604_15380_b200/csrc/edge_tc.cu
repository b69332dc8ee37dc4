// edge_tc.cu — a4 (forward message step) of the BF16 model with the filter contraction on the tcgen05 tensor cores.
//
// SURVEY.md §8(c) B3, per edge e = (i <- j):  w_e = (flt_W g(d_e) + flt_b) c(d_e),  x_e = phi_j o w_e,
//   s'_i = s_i + sum_e x^ss,   v'_i[a] = v_i[a] + sum_e ( x^vs u_e[a] + x^vv o v_j[a] ).
//
// The filter is the small-K GEMM  W^T[3F x edges] = Wf[3F x (K+1)] . G^T[(K+1) x edges]  (SURVEY.md §7 hard part 3), run
// TRANSPOSED on tcgen05.mma so that FEATURES lie on the 128 TMEM lanes and EDGES on the TMEM columns:
//   A (shared memory, resident for the whole kernel): per accumulator a = chunk*2 + parity the 128 filter rows of the
//       features f = 2*lane + parity, K-major, column K = flt_b, zero padded to KP = 16 ceil((K+1)/16);
//   B (shared memory ring): a tile of 16 CONSECUTIVE CSR edges x KP: g_k(d) c(d), c(d) in column K (BF16);
//   D (TMEM): 6 accumulators [128 lanes x 16 columns] FP32 per pipeline (4 in the first block, where v = 0).
// A thread of an epilogue warp owns TMEM lane l of its quadrant = the feature PAIR (2l, 2l+1): one tcgen05.ld gives it
// the filter values of its two features for the 16 edges of the tile; it then walks the edges, gathers the sender's
// phi_j / v_j pair as one 32-bit word per chunk (a warp reads 128 contiguous bytes of the row: one L1 wavefront, the rows
// of a molecule stay in L1 because neighbouring receivers are processed by the same CTA), multiplies with packed
// FP32 FMAs and keeps the receiver's segment sum in registers: no cross-lane reduction, no atomics, and neither the MMA
// nor its operand staging occupy the issue slots of the warps that do the gathers.
//
// One persistent CTA per SM, NGRP independent pipelines, each = 1 producer warp + 4 epilogue warps:
//   producer  (per tile) radial basis x cutoff of 16 edges -> B slot; sender index, unit vector, receiver -> metadata slot;
//             lane 0 then issues the 6 x KP/16 tcgen05.mma of the tile and commits them to the pipeline's "TMEM full"
//             mbarrier; it also prefetches the next atom range's rows into L2 (cp.async.bulk.prefetch);
//   epilogue  waits, tcgen05.ld's the tile into registers, frees the TMEM buffer at once (the next tile's MMAs overlap
//             the arithmetic of this one), runs the edge loop, and at every change of receiver adds the residual row
//             and writes s', v' (FP32) and their BF16 copies with coalesced 8-byte / 4-byte stores.
#include <algorithm>
#include <cstddef>
#include <cstring>
#include <vector>

#include "common.cuh"
#include "edge_tc.cuh"
#include "tc_ptx.cuh"

namespace pnn {

namespace {

using namespace tc;

constexpr int NE = 16;   // edges per tile = N of the UMMA
constexpr int NGRP = 2;  // pipelines per CTA
constexpr int NSLOT = 4; // ring slots (B tile + metadata) per pipeline
constexpr int SPLIT = 2; // epilogue warps per TMEM lane quadrant: they share the features and take alternate receivers
constexpr int EPW = 4 * SPLIT; // epilogue warps per pipeline
constexpr int NPROD = 2; // producer warps per pipeline (tile n is staged and issued by producer n % NPROD)
constexpr int NTHR = NGRP * (EPW + NPROD) * 32;
constexpr int ES = 4;    // edges per epilogue step (TMEM columns per tcgen05.ld)

// A tile = 4 steps of 4 TMEM columns; a step holds up to 4 edges of ONE receiver (a receiver with d edges takes
// ceil(d / 4) steps, the last one ragged), so a step is processed by exactly one epilogue half (receiver % SPLIT).
struct TileMeta {
  float Ux[NE], Uy[NE], Uz[NE]; // per column: unit vector (0 in unused columns)
  uint32_t OFF[NE];             // per column: sender row offset in 16-byte units (row = 3F BF16)
  int2 sinfo[NE / ES];          // per step: (receiver, valid edges; 0 = unused step)
  uint32_t smask[SPLIT];        // bit s: step s is used and belongs to epilogue half h
  uint32_t pad[4 - SPLIT];
};
// explicit shared-space loads from 32-bit shared addresses (no generic-to-shared conversions in the inner loops)
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ float4 lds128f(uint32_t a) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ uint2 lds64(uint32_t a) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ uint32_t lds32(uint32_t a) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
  return v;
}
// backoff for the waits of warps that are ahead of their consumers (their polling would take issue slots)
__device__ __forceinline__ void mbar_wait_backoff(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  for (;;) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    if (ok) break;
    __nanosleep(512);
  }
}

__device__ __forceinline__ float2 bf2(uint32_t x) {
  return make_float2(__uint_as_float(x << 16), __uint_as_float(x & 0xffff0000u));
}
__device__ __forceinline__ uint32_t pack_bf2(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}
__device__ __forceinline__ uint32_t ldg_nc32(const void* p) { return __ldg(reinterpret_cast<const uint32_t*>(p)); }
// streaming accesses that should not displace the gathered rows from L1
__device__ __forceinline__ float2 ld_stream2(const float* p) {
  float2 v;
  asm volatile("ld.global.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ void st_stream2(float* p, float2 v) {
  asm volatile("st.global.cs.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void st_stream1(void* p, uint32_t v) {
  asm volatile("st.global.cs.b32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// NACC accumulators (16 columns apart) x 4 columns from one base address, asynchronous
template <int NACC>
__device__ __forceinline__ void tmem_ld4_accs(uint32_t taddr, float (&r)[NACC][4]) {
  uint32_t u[NACC][4];
  if constexpr (NACC == 6) {
    asm volatile(
        "{\n\t.reg .b32 t1, t2, t3, t4, t5;\n\t"
        "add.u32 t1, %24, 16;\n\tadd.u32 t2, %24, 32;\n\tadd.u32 t3, %24, 48;\n\tadd.u32 t4, %24, 64;\n\tadd.u32 t5, %24, 80;\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%24];\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%4, %5, %6, %7}, [t1];\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%8, %9, %10, %11}, [t2];\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%12, %13, %14, %15}, [t3];\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%16, %17, %18, %19}, [t4];\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%20, %21, %22, %23}, [t5];\n\t}"
        : "=r"(u[0][0]), "=r"(u[0][1]), "=r"(u[0][2]), "=r"(u[0][3]), "=r"(u[1][0]), "=r"(u[1][1]), "=r"(u[1][2]), "=r"(u[1][3]),
          "=r"(u[2][0]), "=r"(u[2][1]), "=r"(u[2][2]), "=r"(u[2][3]), "=r"(u[3][0]), "=r"(u[3][1]), "=r"(u[3][2]), "=r"(u[3][3]),
          "=r"(u[4][0]), "=r"(u[4][1]), "=r"(u[4][2]), "=r"(u[4][3]), "=r"(u[5][0]), "=r"(u[5][1]), "=r"(u[5][2]), "=r"(u[5][3])
        : "r"(taddr)
        : "memory");
  } else {
    asm volatile(
        "{\n\t.reg .b32 t1, t2, t3;\n\t"
        "add.u32 t1, %16, 16;\n\tadd.u32 t2, %16, 32;\n\tadd.u32 t3, %16, 48;\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%16];\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%4, %5, %6, %7}, [t1];\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%8, %9, %10, %11}, [t2];\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%12, %13, %14, %15}, [t3];\n\t}"
        : "=r"(u[0][0]), "=r"(u[0][1]), "=r"(u[0][2]), "=r"(u[0][3]), "=r"(u[1][0]), "=r"(u[1][1]), "=r"(u[1][2]), "=r"(u[1][3]),
          "=r"(u[2][0]), "=r"(u[2][1]), "=r"(u[2][2]), "=r"(u[2][3]), "=r"(u[3][0]), "=r"(u[3][1]), "=r"(u[3][2]), "=r"(u[3][3])
        : "r"(taddr)
        : "memory");
  }
#pragma unroll
  for (int a = 0; a < NACC; ++a)
#pragma unroll
    for (int i = 0; i < 4; ++i) r[a][i] = __uint_as_float(u[a][i]);
}
// 32 TMEM lanes x 4 columns, asynchronous
__device__ __forceinline__ void tmem_ld4_async(uint32_t taddr, float (&r)[4]) {
  uint32_t u[4];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
               : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3])
               : "r"(taddr)
               : "memory");
#pragma unroll
  for (int i = 0; i < 4; ++i) r[i] = __uint_as_float(u[i]);
}
__device__ __forceinline__ void tmem_wait4(float (&r)[4], bool do_wait) {
  if (do_wait) asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(r[0]), "+f"(r[1]), "+f"(r[2]), "+f"(r[3]) : : "memory");
  else asm volatile("" : "+f"(r[0]), "+f"(r[1]), "+f"(r[2]), "+f"(r[3]) : : "memory");
}
__device__ __forceinline__ void mbar_wait_sleep(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}

template <int KP, bool HASV>
struct FwdSmem {
  static constexpr int NACC = HASV ? 6 : 4;
  static constexpr int A_BYTES = NACC * 128 * KP * 2;
  static constexpr int B_TILE = NE * KP * 2;
  static constexpr int GRP_BYTES = NSLOT * B_TILE + NSLOT * (int)sizeof(TileMeta);
  static constexpr int BAR_OFF = A_BYTES + NGRP * GRP_BYTES;
  static constexpr int NBAR_G = 2 * NSLOT + 4; // meta_full[NSLOT], meta_empty[NSLOT], tmem_full[2], tmem_empty[2]
  static constexpr int NBAR = NGRP * NBAR_G;
  static constexpr int TOTAL = BAR_OFF + NBAR * 8 + 32 + 128 /* alignment slack */;
  static constexpr int TMEM_COLS = (NGRP * 2 * NACC * NE <= 256) ? 256 : 512;
};

// FT: the feature width when it is known at compile time (row offsets become immediates), 0 = use a.F
template <int KP, bool HASV, int FT>
__global__ void __launch_bounds__(NTHR, 1)
edge_fwd_tc_k(EdgeMmaArgs a, int RA, const __nv_bfloat16* __restrict__ fltT, const __nv_bfloat16* __restrict__ phi,
              const float* __restrict__ s_in, int64_t ld_sin, const __nv_bfloat16* __restrict__ v_in,
              const float* __restrict__ v_res, float* __restrict__ s1, int64_t ld_s1, float* __restrict__ v1,
              EdgeMirror mir) {
  using L = FwdSmem<KP, HASV>;
  constexpr int NACC = L::NACC, KS = KP / 16, KC = KP / 8;
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 127u) & ~127u;
  unsigned char* sm = smem_raw + (base - raw);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + L::BAR_OFF);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + L::NBAR);
  int* range = reinterpret_cast<int*>(tmem_slot + 1); // [2]: this CTA's atom range
  const uint32_t bar0 = base + L::BAR_OFF;
  auto meta_full = [&](int g, int s) { return bar0 + 8u * (g * L::NBAR_G + s); };
  auto meta_empty = [&](int g, int s) { return bar0 + 8u * (g * L::NBAR_G + NSLOT + s); };
  auto tmem_full = [&](int g, int b) { return bar0 + 8u * (g * L::NBAR_G + 2 * NSLOT + b); };
  auto tmem_empty = [&](int g, int b) { return bar0 + 8u * (g * L::NBAR_G + 2 * NSLOT + 2 + b); };

  // resident A operand: the packed filter image of this block, copied verbatim
  {
    const uint4* src = reinterpret_cast<const uint4*>(fltT);
    uint4* dst = reinterpret_cast<uint4*>(sm);
    for (int i = tid; i < L::A_BYTES / 16; i += NTHR) dst[i] = __ldg(src + i);
  }
  if (tid == 0) {
    for (int g = 0; g < NGRP; ++g) {
      for (int s = 0; s < NSLOT; ++s) { mbar_init(meta_full(g, s), 1); mbar_init(meta_empty(g, s), EPW); }
      for (int b = 0; b < 2; ++b) { mbar_init(tmem_full(g, b), 1); mbar_init(tmem_empty(g, b), EPW); }
    }
    mbar_init_fence();
  }
  if (warp == 0 && lane < 2) {
    // this CTA's contiguous atom range, balanced by edge count: [first atom with rowptr >= b E / nCTA, same for b + 1)
    const int b = blockIdx.x + lane;
    int res;
    if (b == 0) res = 0;
    else if (b >= (int)gridDim.x) res = (int)a.N;
    else {
      const int64_t E = __ldg(a.rowptr + a.N);
      const int target = (int)(E * b / gridDim.x);
      int lo = 0, hi = (int)a.N; // first i in [0, N] with rowptr[i] >= target
      while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(a.rowptr + mid) >= target) hi = mid; else lo = mid + 1;
      }
      res = lo;
    }
    range[lane] = res;
  }
  if (warp == NGRP * EPW) tmem_alloc<L::TMEM_COLS>(tmem_slot);
  fence_proxy_async_smem(); // the A image was written with st.shared and is read by the MMA (async proxy)
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const int c_lo = range[0], c_hi = range[1];

  const int F = FT ? FT : a.F;
  // window w of this CTA = atoms [c_lo + w RA, min(c_lo + (w+1) RA, c_hi)), handled by pipeline w % NGRP

  if (warp >= NGRP * EPW) {
    // ================================================================== producer pp of pipeline g
    const int g = (warp - NGRP * EPW) / NPROD, pp = (warp - NGRP * EPW) % NPROD;
    unsigned char* grp = sm + L::A_BYTES + g * L::GRP_BYTES;
    const uint32_t grp_u = base + L::A_BYTES + g * L::GRP_BYTES;
    const int r = lane & 15, half = lane >> 4;
    const float rc = a.rc;
    const float dmu = (a.K > 1) ? rc / (float)(a.K - 1) : rc;
    const float gamma = 1.0f / (2.0f * dmu * dmu);
    const float pi_rc = 3.14159265358979323846f / rc;
    const float bes_A = sqrtf(2.0f / rc);
    const uint32_t row16 = (uint32_t)(3 * F / 8); // 16-byte units per row of phi / v_in
    constexpr uint32_t idesc = umma_idesc_bf16(128, NE);
    // UMMA shared-memory descriptors (no swizzle, K-major): high word constant, low word = start address >> 4 | LBO field
    const uint32_t d_hi = (uint32_t)(umma_desc_nosw(0, 128, KC * 128) >> 32);
    const uint32_t a_lo0 = (uint32_t)umma_desc_nosw(base, 128, KC * 128);
    uint32_t n = 0; // tiles of this pipeline so far (both producers count all of them)
    for (int64_t a0 = (int64_t)c_lo + (int64_t)g * RA; a0 < c_hi; a0 += (int64_t)NGRP * RA) {
      const int64_t a1 = min(a0 + RA, (int64_t)c_hi);
      const int na = (int)(a1 - a0);
      // lane l < na: receiver a0 + l; so = exclusive prefix sum of its steps (lane na: the window's total)
      const int rp = (lane <= na) ? __ldg(a.rowptr + a0 + lane) : 0;
      const int rp1 = __shfl_down_sync(0xffffffffu, rp, 1);
      const int nst = (lane < na) ? (rp1 - rp + ES - 1) / ES : 0;
      int so = nst;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, so, o); if (lane >= o) so += t; }
      so -= nst;
      const int tot = __shfl_sync(0xffffffffu, so, na);
      for (int s0 = 0; s0 < tot; s0 += NE / ES, ++n) {
        if ((n % NPROD) != (uint32_t)pp) continue;
        const int slot = n % NSLOT;
        mbar_wait_backoff(meta_empty(g, slot), ((n / NSLOT) & 1u) ^ 1u);
        TileMeta* mt = reinterpret_cast<TileMeta*>(grp + NSLOT * L::B_TILE) + slot;
        unsigned char* Bt = grp + slot * L::B_TILE;
        // this lane's column r = step (r / 4), position (r % 4): receiver = last lane l < na with so[l] <= step
        const int S = s0 + (r >> 2);
        int pos = 0;
#pragma unroll
        for (int step = 16; step >= 1; step >>= 1) {
          const int t = pos + step;
          const int val = __shfl_sync(0xffffffffu, so, t & 31);
          if (t < na && val <= S) pos = t;
        }
        const int so_p = __shfl_sync(0xffffffffu, so, pos), rp_p = __shfl_sync(0xffffffffu, rp, pos),
                  rp_n = __shfl_sync(0xffffffffu, rp, pos + 1);
        const int e = rp_p + (S - so_p) * ES + (r & 3);
        const bool ok = S < tot && e < rp_n;
        const int rcv = (int)a0 + pos;
        float4 gq = make_float4(0.f, 0.f, 0.f, 1.f);
        int j = 0;
        if (ok) { gq = __ldg(reinterpret_cast<const float4*>(a.geom) + e); j = __ldg(a.col + e); }
        const float d = gq.w;
        float sn_, cs_;
        __sincosf(pi_rc * d, &sn_, &cs_);
        const float cut = ok ? 0.5f * (cs_ + 1.0f) : 0.0f;
        // this lane's KP/2 columns k = half*KP/2 ... : g_k(d) c(d) (k < K), c(d) (k == K), 0 (k > K)
#pragma unroll
        for (int q = 0; q < KP / 16; ++q) {
          float v[8];
#pragma unroll
          for (int x = 0; x < 8; ++x) {
            const int k = half * (KP / 2) + q * 8 + x;
            float val;
            if (a.rbf == 1) val = bes_A * __sinf((float)(k + 1) * pi_rc * d) / d;
            else { const float dd = d - (float)k * dmu; val = __expf(-gamma * dd * dd); }
            v[x] = (k < a.K) ? val * cut : (k == a.K ? cut : 0.0f);
          }
          const int kc = half * (KP / 16) + q;
          *reinterpret_cast<uint4*>(Bt + (r >> 3) * (KC * 128) + kc * 128 + (r & 7) * 16) =
              make_uint4(pack_bf2(v[0], v[1]), pack_bf2(v[2], v[3]), pack_bf2(v[4], v[5]), pack_bf2(v[6], v[7]));
        }
        const uint32_t okm = __ballot_sync(0xffffffffu, ok && half == 0); // bit r: column r holds an edge
        const int jfirst = __shfl_sync(0xffffffffu, j, lane & ~3);
        if (half == 0) {
          mt->Ux[r] = ok ? gq.x : 0.f; mt->Uy[r] = ok ? gq.y : 0.f; mt->Uz[r] = ok ? gq.z : 0.f;
          mt->OFF[r] = (uint32_t)(ok ? j : jfirst) * row16; // unused columns of a step gather a valid row (weight 0)
          if ((r & 3) == 0) mt->sinfo[r >> 2] = make_int2(rcv, __popc((okm >> r) & 15u));
        }
#pragma unroll
        for (int hh = 0; hh < SPLIT; ++hh) {
          const uint32_t m = __ballot_sync(0xffffffffu, ok && half == 0 && (r & 3) == 0 && (rcv % SPLIT) == hh);
          // bit 4 s of m -> bit s
          if (lane == 0) mt->smask[hh] = (m & 1u) | ((m >> 3) & 2u) | ((m >> 6) & 4u) | ((m >> 9) & 8u);
        }
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(meta_full(g, slot));
          const uint32_t buf = n & 1u;
          mbar_wait_backoff(tmem_empty(g, buf), ((n >> 1) & 1u) ^ 1u); // the epilogue has read tile n - 2 out of this buffer
          tc_fence_after();
          const uint32_t b_lo0 = (uint32_t)umma_desc_nosw(grp_u + slot * L::B_TILE, 128, KC * 128);
          const uint32_t tmem_t = tmem_base + (uint32_t)((g * 2 + buf) * NACC * NE);
#pragma unroll
          for (int acc = 0; acc < NACC; ++acc)
#pragma unroll
            for (int ks = 0; ks < KS; ++ks)
              umma_bf16_lohi(tmem_t + (uint32_t)(acc * NE), a_lo0 + (uint32_t)((acc * (128 * KP * 2) + ks * 256) >> 4), d_hi,
                             b_lo0 + (uint32_t)((ks * 256) >> 4), d_hi, idesc, ks != 0);
          umma_commit(tmem_full(g, buf));
        }
        __syncwarp();
      }
    }
  } else {
    // ================================================================== epilogue warp (pipeline g, TMEM quadrant q)
    const int g = warp / EPW, q = warp % 4, h = (warp % EPW) / 4; // h: takes the receivers with i % SPLIT == h
    const uint32_t grp_u = base + L::A_BYTES + g * L::GRP_BYTES;
    const int p = q * 32 + lane;       // feature pair
    const bool act = FT ? (2 * p < FT) : (2 * p < F);
    const int f0 = act ? 2 * p : 0;    // inactive lanes compute on pair 0 and store nothing
    const char* phi_f = reinterpret_cast<const char*>(phi) + f0 * 2;
    const char* vin_f = reinterpret_cast<const char*>(v_in) + f0 * 2;
    uint32_t n = 0;
    for (int64_t a0 = (int64_t)c_lo + (int64_t)g * RA; a0 < c_hi; a0 += (int64_t)NGRP * RA) {
      const int64_t a1 = min(a0 + RA, (int64_t)c_hi);
      const int na = (int)(a1 - a0);
      int tot; // steps of the window (as the producer counts them)
      {
        const int rp = (lane <= na) ? __ldg(a.rowptr + a0 + lane) : 0;
        const int rp1 = __shfl_down_sync(0xffffffffu, rp, 1);
        tot = (lane < na) ? (rp1 - rp + ES - 1) / ES : 0;
#pragma unroll
        for (int o = 16; o; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
      }
      int cur = (int)a0 + ((h - (int)(a0 % SPLIT) + SPLIT) % SPLIT); // my first atom of the window
      // Segment sums of the current receiver.  The packed FMAs pair two EDGES of one feature (component .x: even
      // columns of the step, .y: odd columns), so that both operands of a packed product are adjacent registers
      // (two TMEM columns of one accumulator; two unpacked halves): [feature parity] for s, [axis][feature parity] for v.
      float2 as[2], av[3][2];
      auto begin_row = [&](int i) { // new receiver: zero sums; pull its residual row (read when it is complete) towards L2
        as[0] = as[1] = make_float2(0.f, 0.f);
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) av[ax][0] = av[ax][1] = make_float2(0.f, 0.f);
        asm volatile("prefetch.global.L2 [%0];" ::"l"(s_in + (int64_t)i * ld_sin + f0));
        if (HASV) {
#pragma unroll
          for (int ax = 0; ax < 3; ++ax) asm volatile("prefetch.global.L2 [%0];" ::"l"(v_res + ((int64_t)i * 3 + ax) * F + f0));
        }
      };
      auto end_row = [&](int i) {
        if (!act) return;
        const float2 rs = ld_stream2(s_in + (int64_t)i * ld_sin + f0);
        float2 rv[3];
#pragma unroll
        for (int ax = 0; ax < 3; ++ax)
          rv[ax] = HASV ? ld_stream2(v_res + ((int64_t)i * 3 + ax) * F + f0) : make_float2(0.f, 0.f);
        const float2 o = make_float2(rs.x + (as[0].x + as[0].y), rs.y + (as[1].x + as[1].y));
        st_stream2(s1 + (int64_t)i * ld_s1 + f0, o);
        if (mir.s1) st_stream1(mir.s1 + (int64_t)i * mir.ld_s1 + f0, pack_bf2(o.x, o.y));
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
          const float2 ov = make_float2(rv[ax].x + (av[ax][0].x + av[ax][0].y), rv[ax].y + (av[ax][1].x + av[ax][1].y));
          const int64_t off = ((int64_t)i * 3 + ax) * F + f0;
          st_stream2(v1 + off, ov);
          if (mir.v1) st_stream1(mir.v1 + off, pack_bf2(ov.x, ov.y));
        }
      };
      begin_row(cur < (int)a1 ? cur : (int)a0);
      for (int s0 = 0; s0 < tot; s0 += NE / ES, ++n) {
        const int slot = n % NSLOT;
        const uint32_t buf = n & 1u;
        uint32_t mt_u = grp_u + NSLOT * L::B_TILE + slot * (uint32_t)sizeof(TileMeta);
        asm volatile("" : "+r"(mt_u)); // keep it in a register (it is otherwise recomputed from scratch at every use)
        mbar_wait_sleep(meta_full(g, slot), (n / NSLOT) & 1u);
        const uint32_t mymask = lds32(mt_u + (uint32_t)offsetof(TileMeta, smask) + 4u * h);
        // (every warp observes every phase of the barrier, also for tiles it has no edge in: a parity wait two phases
        // behind would pass at once)
        mbar_wait_sleep(tmem_full(g, buf), (n >> 1) & 1u);
        if (mymask) {
          tc_fence_after();
          uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)((g * 2 + buf) * NACC * NE);
          asm volatile("" : "+r"(taddr));
#pragma unroll
          for (int si = 0; si < NE / ES; ++si) {
            if ((mymask >> si) & 1u) {
              constexpr uint32_t kOFF = (uint32_t)offsetof(TileMeta, OFF), kINF = (uint32_t)offsetof(TileMeta, sinfo),
                                 kUX = (uint32_t)offsetof(TileMeta, Ux), kUY = (uint32_t)offsetof(TileMeta, Uy),
                                 kUZ = (uint32_t)offsetof(TileMeta, Uz);
              const uint32_t cb = (uint32_t)si * (ES * 4); // byte offset of the step's columns in the per-column arrays
              float W[NACC][ES];
              static_assert(NE == 16, "tmem_ld4_accs assumes accumulators 16 columns apart");
              tmem_ld4_accs<NACC>(taddr + si * ES, W);
              const uint4 oo = lds128(mt_u + kOFF + cb);
              const uint32_t offs[4] = {oo.x, oo.y, oo.z, oo.w};
              // all four columns gather: an unused column of a ragged step reads a valid row and has zero filter values
              uint32_t gw[ES][6];
#pragma unroll
              for (int c = 0; c < ES; ++c) {
                const char* pr = phi_f + (uint64_t)offs[c] * 16u;
                gw[c][0] = ldg_nc32(pr); gw[c][1] = ldg_nc32(pr + 2 * F);
                if (HASV) {
                  gw[c][2] = ldg_nc32(pr + 4 * F);
                  const char* vr = vin_f + (uint64_t)offs[c] * 16u;
                  gw[c][3] = ldg_nc32(vr); gw[c][4] = ldg_nc32(vr + 2 * F); gw[c][5] = ldg_nc32(vr + 4 * F);
                }
              }
              const int i = (int)lds32(mt_u + kINF + 8u * si);
              if (i != cur) { // receiver complete: write it (and any edge-less atoms of mine before the next one)
                end_row(cur);
                for (int k = cur + SPLIT; k < i; k += SPLIT) { begin_row(k); end_row(k); }
                cur = i;
                begin_row(cur);
              }
#pragma unroll
              for (int acc = 0; acc < NACC; ++acc) tmem_wait4(W[acc], acc == 0);
              // columns (0, 1) and (2, 3) of the step as packed pairs
#pragma unroll
              for (int pr2 = 0; pr2 < ES / 2; ++pr2) {
                const int c = 2 * pr2;
                const uint2 u0b = lds64(mt_u + kUX + cb + 8u * pr2), u1b = lds64(mt_u + kUY + cb + 8u * pr2),
                            u2b = lds64(mt_u + kUZ + cb + 8u * pr2);
                const float2 u0 = make_float2(__uint_as_float(u0b.x), __uint_as_float(u0b.y));
                const float2 u1 = make_float2(__uint_as_float(u1b.x), __uint_as_float(u1b.y));
                const float2 u2 = make_float2(__uint_as_float(u2b.x), __uint_as_float(u2b.y));
#pragma unroll
                for (int par = 0; par < 2; ++par) { // feature 2p + par: low / high halves of the gathered words
                  auto half2 = [&](int x) {
                    return par ? make_float2(__uint_as_float(gw[c][x] & 0xffff0000u), __uint_as_float(gw[c + 1][x] & 0xffff0000u))
                               : make_float2(__uint_as_float(gw[c][x] << 16), __uint_as_float(gw[c + 1][x] << 16));
                  };
                  as[par] = __ffma2_rn(half2(0), make_float2(W[par][c], W[par][c + 1]), as[par]);
                  const float2 xvs = __fmul2_rn(half2(1), make_float2(W[2 + par][c], W[2 + par][c + 1]));
                  av[0][par] = __ffma2_rn(xvs, u0, av[0][par]);
                  av[1][par] = __ffma2_rn(xvs, u1, av[1][par]);
                  av[2][par] = __ffma2_rn(xvs, u2, av[2][par]);
                  if (HASV) {
                    const float2 xvv = __fmul2_rn(half2(2), make_float2(W[NACC - 2 + par][c], W[NACC - 2 + par][c + 1]));
                    av[0][par] = __ffma2_rn(xvv, half2(3), av[0][par]);
                    av[1][par] = __ffma2_rn(xvv, half2(4), av[1][par]);
                    av[2][par] = __ffma2_rn(xvv, half2(5), av[2][par]);
                  }
                }
              }
            }
          }
          tc_fence_before();
        }
        __syncwarp();
        if (lane == 0) { mbar_arrive(tmem_empty(g, buf)); mbar_arrive(meta_empty(g, slot)); }
      }
      if (cur < (int)a1) {
        end_row(cur);
        for (int k = cur + SPLIT; k < (int)a1; k += SPLIT) { begin_row(k); end_row(k); }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == NGRP * EPW) {
    tc_fence_after();
    tmem_dealloc<L::TMEM_COLS>(tmem_base);
  }
}

uint16_t to_bf16_host(double x) {
  float f = (float)x;
  uint32_t u;
  std::memcpy(&u, &f, 4);
  const uint32_t r = u + 0x7fffu + ((u >> 16) & 1u); // round to nearest even
  return (uint16_t)(r >> 16);
}

} // namespace

int edge_mma_kp(int K) { return (K + 1 + 15) / 16 * 16; }

// Host-side packing of one block's filter as the resident A operand of edge_fwd_tc_k: 6 accumulator tiles
// a = chunk*2 + parity of 128 rows x KP columns, row l = filter row of feature 2l + parity (zero for 2l + parity >= F),
// column k < K: flt_W, k == K: flt_b, then zeros; stored in the UMMA no-swizzle K-major layout
// [16 row groups][KP/8 column chunks][8 rows][8 elements].
int64_t edge_tc_filter_elems(int K) { return (int64_t)6 * 128 * edge_mma_kp(K); }

void pack_filter_tc(int F, int K, const double* fltW, const double* fltb, uint16_t* out) {
  const int KP = edge_mma_kp(K), KC = KP / 8;
  std::memset(out, 0, sizeof(uint16_t) * (size_t)edge_tc_filter_elems(K));
  for (int c = 0; c < 3; ++c)
    for (int par = 0; par < 2; ++par)
      for (int l = 0; l < 128; ++l) {
        const int f = 2 * l + par;
        if (f >= F) continue;
        const int64_t src = (int64_t)c * F + f;
        uint16_t* tile = out + (size_t)(c * 2 + par) * 128 * KP;
        for (int k = 0; k <= K; ++k) {
          const uint16_t val = k < K ? to_bf16_host(fltW[src * K + k]) : to_bf16_host(fltb[src]);
          tile[((size_t)((l >> 3) * KC + (k >> 3)) * 8 + (l & 7)) * 8 + (k & 7)] = val;
        }
      }
}

int launch_edge_fwd_tc(const EdgeMmaArgs& a, const __nv_bfloat16* fltT, const __nv_bfloat16* phi, const float* s_in,
                       int64_t ld_sin, const __nv_bfloat16* v_in, const float* v_res, float* s1, int64_t ld_s1, float* v1,
                       const EdgeMirror& mir, cudaStream_t st) {
  if (a.N == 0) return 0;
  const int KP = edge_mma_kp(a.K);
  // One persistent CTA per SM takes a contiguous, edge-balanced range of atoms and cuts it into windows of RA atoms that
  // alternate between its pipelines: about 4 windows per pipeline, between 2 and 16 atoms each.
  const int RA = (int)std::min<int64_t>(16, std::max<int64_t>(2, a.N / (148 * NGRP * 8)));
  const unsigned grid = (unsigned)std::min<int64_t>(148, (a.N + RA * NGRP - 1) / (RA * NGRP));
#define PNN_LAUNCH2(KPV, HV, FTV)                                                                                    \
  {                                                                                                                  \
    using L = FwdSmem<KPV, HV>;                                                                                      \
    static bool attr_set = false;                                                                                    \
    if (!attr_set) {                                                                                                 \
      cudaFuncSetAttribute(edge_fwd_tc_k<KPV, HV, FTV>, cudaFuncAttributeMaxDynamicSharedMemorySize, L::TOTAL);      \
      attr_set = true;                                                                                               \
    }                                                                                                                \
    edge_fwd_tc_k<KPV, HV, FTV><<<grid, NTHR, L::TOTAL, st>>>(a, RA, fltT, phi, s_in, ld_sin, v_in, v_res, s1, ld_s1, \
                                                              v1, mir);                                              \
    PNN_KCHECK("edge_fwd_tc_k");                                                                                     \
  }
#define PNN_LAUNCH(KPV, HV) { if (a.F == 256) PNN_LAUNCH2(KPV, HV, 256) else PNN_LAUNCH2(KPV, HV, 0) }
  const bool hv = v_in != nullptr;
  if (KP == 16) { if (hv) PNN_LAUNCH(16, true) else PNN_LAUNCH(16, false) }
  else if (KP == 32) { if (hv) PNN_LAUNCH(32, true) else PNN_LAUNCH(32, false) }
  else { if (hv) PNN_LAUNCH(48, true) else PNN_LAUNCH(48, false) }
#undef PNN_LAUNCH2
#undef PNN_LAUNCH
  return 1;
}

} // namespace pnn
