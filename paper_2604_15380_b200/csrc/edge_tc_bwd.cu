// edge_tc_bwd.cu — a7 (reverse message step, R3 + R4 of SURVEY.md §8(c)) of the BF16 model on the tcgen05 tensor cores.
//
// Same transposed layout as the forward kernel (edge_tc.cu): FEATURES on the 128 TMEM lanes, EDGES on the TMEM columns, an
// epilogue thread owns the feature pair (2l, 2l+1) of its lane.  The sender scatters of the reverse sweep are rewritten as
// gathers over the receiver's own CSR row (note under R4: the edge set is symmetric, w depends only on d, u flips sign), so
// the kernel is again "per receiver i, sum over its edges (i <- j)".  Per tile of 16 columns the tensor core gives BOTH
//   W[f, e]  = sum_k Wf[f, k] G [e, k]     the filter value           (B operand: g_k(d) c(d), column K = c(d))
//   D[f, e]  = sum_k Wf[f, k] G'[e, k]     its derivative dw/dd       (B operand: d/dd of the same columns)
// for the 3 chunks x 2 feature parities (12 accumulators of 16 columns, 8 in the first block where v = 0).  With
//   l = (s-bar'_i, v-bar'_i, v_i, phi_i) the receiver's own rows and (phi_j, s-bar'_j, v-bar'_j, v_j) gathered (BF16), per edge
//   ss   A0 += sb_j w                   x = sb_i phi_j + sb_j phi_i
//   vs   A1 -= (vb_j.u) w               x = (vb_i.u) phi_j - (vb_j.u) phi_i     q[a] = vb_i[a] phi_j - vb_j[a] phi_i
//   vv   A2[a] += vb_j[a] w             Pv += (vb_j.v_i) w                      x = (vb_i.v_j) phi_j + (vb_j.v_i) phi_i
//   dE/dd_e = sum_{chunks, f} x D       force_i += dE/dd_e u_e + sum_f (q_f - x_f^vs u_e) w_f^vs / d_e   (q_f.u = x_f^vs)
// all of it per feature pair in registers (packed FP32 FMAs); the force is linear in the per-feature terms, so a thread
// keeps its own partial force and the 128 threads meet once per receiver (warp shuffle, one force slab per epilogue warp).
// Outputs per receiver: phi-bar (BF16: A0 | A1 | Pv), v-bar_in = v-bar' + phi_i^vv A2 (FP32), force slab partials.
//
// One persistent CTA per SM: NGRP pipelines x (2 producer warps + 4 epilogue warps); a step = 2 TMEM columns = up to 2
// edges of ONE receiver.  The TMEM buffer of a pipeline (12 x 16 columns) is single: the producers' next MMAs wait for the
// epilogue to finish the tile, and the other pipeline fills the gap.
#include <algorithm>
#include <cstddef>
#include <cstring>

#include "common.cuh"
#include "edge_tc.cuh"
#include "tc_ptx.cuh"

namespace pnn {

namespace {

using namespace tc;

constexpr int NE = 16;   // columns per tile = N of the UMMA
constexpr int NGRP = 2;  // pipelines per CTA
constexpr int NSLOT = 4; // ring slots (2 B tiles + metadata) per pipeline
constexpr int EPW = 4;   // epilogue warps per pipeline (one per TMEM lane quadrant)
constexpr int NPROD = 2; // producer warps per pipeline
constexpr int NTHR = NGRP * (EPW + NPROD) * 32;
constexpr int ES = 2;    // columns per step
constexpr int NSTEP = NE / ES;

struct TileMetaB {
  float Ux[NE], Uy[NE], Uz[NE], Id[NE]; // per column: unit vector and 1/d (0 in unused columns)
  uint32_t OFF[NE];                     // per column: sender row offset in 16-byte units for rows of 3F BF16
  uint32_t OFS[NE];                     // ... for rows of F BF16 (s-bar)
  int2 sinfo[NSTEP];                    // per step: (receiver, valid edges; 0 = unused step)
};

__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ uint2 lds64(uint32_t a) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ float2 lds64f(uint32_t a) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
  return v;
}
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
// 32 TMEM lanes x 2 columns, asynchronous
__device__ __forceinline__ void tmem_ld2_async(uint32_t taddr, float (&r)[2]) {
  uint32_t u0, u1;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(u0), "=r"(u1) : "r"(taddr) : "memory");
  r[0] = __uint_as_float(u0); r[1] = __uint_as_float(u1);
}
__device__ __forceinline__ void tmem_wait2(float (&r)[2], bool do_wait) {
  if (do_wait) asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(r[0]), "+f"(r[1]) : : "memory");
  else asm volatile("" : "+f"(r[0]), "+f"(r[1]) : : "memory");
}
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 splat(float x) { return make_float2(x, x); }

struct Gath { uint32_t gp[ES][3], gs[ES], gb[ES][3], gv[ES][3]; }; // gathered words of one step

template <int KP, bool HASV>
struct BwdSmem {
  static constexpr int NCH = HASV ? 3 : 2;
  static constexpr int NACC = 2 * NCH;          // accumulators of W; as many again for D
  static constexpr int A_BYTES = NACC * 128 * KP * 2;
  static constexpr int B_TILE = NE * KP * 2;    // one of the two B tiles (G, G') of a slot
  static constexpr int GRP_BYTES = NSLOT * 2 * B_TILE + NSLOT * (int)sizeof(TileMetaB);
  static constexpr int BAR_OFF = A_BYTES + NGRP * GRP_BYTES;
  static constexpr int NBAR_G = 2 * NSLOT + 3;  // meta_full[NSLOT], meta_empty[NSLOT], tmem_full, tmem_empty[2]
  static constexpr int NBAR = NGRP * NBAR_G;
  static constexpr int TOTAL = BAR_OFF + NBAR * 8 + 32 + 128;
  static constexpr int TMEM_COLS = (NGRP * 2 * NACC * NE <= 256) ? 256 : 512;
};

template <int KP, bool HASV, int FT>
__global__ void __launch_bounds__(NTHR, 1)
edge_bwd_tc_k(EdgeMmaArgs a, int RA, const __nv_bfloat16* __restrict__ fltT, const __nv_bfloat16* __restrict__ phi,
              const __nv_bfloat16* __restrict__ v_in, const __nv_bfloat16* __restrict__ sb16,
              const __nv_bfloat16* __restrict__ vb16, const float* __restrict__ vb1, __nv_bfloat16* __restrict__ phib16,
              float* __restrict__ vb_in, float* __restrict__ fpart, int first_block) {
  using L = BwdSmem<KP, HASV>;
  constexpr int NACC = L::NACC, KS = KP / 16, KC = KP / 8;
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 127u) & ~127u;
  unsigned char* sm = smem_raw + (base - raw);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + L::BAR_OFF);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + L::NBAR);
  int* range = reinterpret_cast<int*>(tmem_slot + 1);
  const uint32_t bar0 = base + L::BAR_OFF;
  auto meta_full = [&](int g, int s) { return bar0 + 8u * (g * L::NBAR_G + s); };
  auto meta_empty = [&](int g, int s) { return bar0 + 8u * (g * L::NBAR_G + NSLOT + s); };
  auto tmem_full = [&](int g) { return bar0 + 8u * (g * L::NBAR_G + 2 * NSLOT); };
  auto tmem_empty = [&](int g, uint32_t b) { return bar0 + 8u * (g * L::NBAR_G + 2 * NSLOT + 1 + b); };

  { // resident A operand: the packed filter image of this block (the first NACC accumulator tiles), copied verbatim
    const uint4* src = reinterpret_cast<const uint4*>(fltT);
    uint4* dst = reinterpret_cast<uint4*>(sm);
    for (int i = tid; i < L::A_BYTES / 16; i += NTHR) dst[i] = __ldg(src + i);
  }
  if (tid == 0) {
    for (int g = 0; g < NGRP; ++g) {
      for (int s = 0; s < NSLOT; ++s) { mbar_init(meta_full(g, s), 1); mbar_init(meta_empty(g, s), EPW); }
      mbar_init(tmem_full(g), 1);
      mbar_init(tmem_empty(g, 0), EPW); mbar_init(tmem_empty(g, 1), EPW);
    }
    mbar_init_fence();
  }
  if (warp == 0 && lane < 2) { // this CTA's contiguous atom range, balanced by edge count
    const int b = blockIdx.x + lane;
    int res;
    if (b == 0) res = 0;
    else if (b >= (int)gridDim.x) res = (int)a.N;
    else {
      const int64_t E = __ldg(a.rowptr + a.N);
      const int target = (int)(E * b / gridDim.x);
      int lo = 0, hi = (int)a.N;
      while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(a.rowptr + mid) >= target) hi = mid; else lo = mid + 1;
      }
      res = lo;
    }
    range[lane] = res;
  }
  if (warp == NGRP * EPW) tmem_alloc<L::TMEM_COLS>(tmem_slot);
  fence_proxy_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const int c_lo = range[0], c_hi = range[1];
  const int F = FT ? FT : a.F;

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
    const uint32_t row16 = (uint32_t)(3 * F / 8), rows16 = (uint32_t)(F / 8);
    constexpr uint32_t idesc = umma_idesc_bf16(128, NE);
    // UMMA shared-memory descriptors (no swizzle, K-major): high word constant, low word = start address >> 4 | LBO field
    const uint32_t d_hi = (uint32_t)(umma_desc_nosw(0, 128, KC * 128) >> 32);
    const uint32_t a_lo0 = (uint32_t)umma_desc_nosw(base, 128, KC * 128);
    const uint32_t tmem_g = tmem_base + (uint32_t)(g * 2 * NACC * NE);
    static_assert(BwdSmem<48, true>::TOTAL < (1 << 18), "descriptor start addresses are 18-bit");
    uint32_t n = 0;
    for (int64_t a0 = (int64_t)c_lo + (int64_t)g * RA; a0 < c_hi; a0 += (int64_t)NGRP * RA) {
      const int64_t a1 = min(a0 + RA, (int64_t)c_hi);
      const int na = (int)(a1 - a0);
      const int rp = (lane <= na) ? __ldg(a.rowptr + a0 + lane) : 0;
      const int rp1 = __shfl_down_sync(0xffffffffu, rp, 1);
      const int nst = (lane < na) ? (rp1 - rp + ES - 1) / ES : 0;
      int so = nst;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, so, o); if (lane >= o) so += t; }
      so -= nst;
      const int tot = __shfl_sync(0xffffffffu, so, na);
      for (int s0 = 0; s0 < tot; s0 += NSTEP, ++n) {
        if ((n % NPROD) != (uint32_t)pp) continue;
        const int slot = n % NSLOT;
        mbar_wait_backoff(meta_empty(g, slot), ((n / NSLOT) & 1u) ^ 1u);
        TileMetaB* mt = reinterpret_cast<TileMetaB*>(grp + NSLOT * 2 * L::B_TILE) + slot;
        unsigned char* Bt = grp + slot * 2 * L::B_TILE;
        const int S = s0 + r / ES;
        int pos = 0;
#pragma unroll
        for (int step = 16; step >= 1; step >>= 1) {
          const int t = pos + step;
          const int val = __shfl_sync(0xffffffffu, so, t & 31);
          if (t < na && val <= S) pos = t;
        }
        const int so_p = __shfl_sync(0xffffffffu, so, pos), rp_p = __shfl_sync(0xffffffffu, rp, pos),
                  rp_n = __shfl_sync(0xffffffffu, rp, pos + 1);
        const int e = rp_p + (S - so_p) * ES + (r % ES);
        const bool ok = S < tot && e < rp_n;
        const int rcv = (int)a0 + pos;
        float4 gq = make_float4(0.f, 0.f, 0.f, 1.f);
        int j = 0;
        if (ok) { gq = __ldg(reinterpret_cast<const float4*>(a.geom) + e); j = __ldg(a.col + e); }
        const float d = gq.w;
        float sn_, cs_;
        __sincosf(pi_rc * d, &sn_, &cs_);
        const float cut = ok ? 0.5f * (cs_ + 1.0f) : 0.0f, cutd = ok ? -0.5f * pi_rc * sn_ : 0.0f;
#pragma unroll
        for (int q = 0; q < KP / 16; ++q) {
          float v[8], vd[8];
#pragma unroll
          for (int x = 0; x < 8; ++x) {
            const int k = half * (KP / 2) + q * 8 + x;
            float val, der;
            if (a.rbf == 1) {
              const float wn = (float)(k + 1) * pi_rc, id = 1.0f / d;
              float s1, c1;
              __sincosf(wn * d, &s1, &c1);
              val = bes_A * s1 * id;
              der = (bes_A * wn * c1 - val) * id;
            } else {
              const float dd = d - (float)k * dmu;
              val = __expf(-gamma * dd * dd);
              der = -2.0f * gamma * dd * val;
            }
            v[x] = (k < a.K) ? val * cut : (k == a.K ? cut : 0.0f);
            vd[x] = (k < a.K) ? der * cut + val * cutd : (k == a.K ? cutd : 0.0f);
          }
          const int kc = half * (KP / 16) + q;
          const int off = (r >> 3) * (KC * 128) + kc * 128 + (r & 7) * 16;
          *reinterpret_cast<uint4*>(Bt + off) =
              make_uint4(pack_bf2(v[0], v[1]), pack_bf2(v[2], v[3]), pack_bf2(v[4], v[5]), pack_bf2(v[6], v[7]));
          *reinterpret_cast<uint4*>(Bt + L::B_TILE + off) =
              make_uint4(pack_bf2(vd[0], vd[1]), pack_bf2(vd[2], vd[3]), pack_bf2(vd[4], vd[5]), pack_bf2(vd[6], vd[7]));
        }
        const uint32_t okm = __ballot_sync(0xffffffffu, ok && half == 0);
        const int jfirst = __shfl_sync(0xffffffffu, j, lane & ~(ES - 1));
        if (half == 0) {
          mt->Ux[r] = ok ? gq.x : 0.f; mt->Uy[r] = ok ? gq.y : 0.f; mt->Uz[r] = ok ? gq.z : 0.f;
          mt->Id[r] = ok ? 1.0f / d : 0.f;
          const uint32_t jj = (uint32_t)(ok ? j : jfirst); // unused columns of a step gather a valid row (weight 0)
          mt->OFF[r] = jj * row16;
          mt->OFS[r] = jj * rows16;
          if ((r % ES) == 0) mt->sinfo[r / ES] = make_int2(rcv, __popc((okm >> r) & ((1u << ES) - 1u)));
        }
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(meta_full(g, slot));
          // the epilogue has finished tile n - 1 (one TMEM buffer per group).  Tiles alternate between two barriers by
          // parity, so that this producer (which owns one parity) sees EVERY phase of the other parity's barrier in order:
          // on a single barrier it would skip every other phase, and a parity wait for a phase two behind the barrier's
          // current one never returns.
          if (n >= 1) mbar_wait_backoff(tmem_empty(g, (n - 1u) & 1u), ((n - 1u) >> 1) & 1u);
          tc_fence_after();
          const uint32_t b_lo0 = (uint32_t)umma_desc_nosw(grp_u + slot * 2 * L::B_TILE, 128, KC * 128);
#pragma unroll
          for (int part = 0; part < 2; ++part) // W from G, D from G'
#pragma unroll
            for (int acc = 0; acc < NACC; ++acc)
#pragma unroll
              for (int ks = 0; ks < KS; ++ks)
                umma_bf16_lohi(tmem_g + (uint32_t)((part * NACC + acc) * NE),
                               a_lo0 + (uint32_t)((acc * (128 * KP * 2) + ks * 256) >> 4), d_hi,
                               b_lo0 + (uint32_t)((part * L::B_TILE + ks * 256) >> 4), d_hi, idesc, ks != 0);
          umma_commit(tmem_full(g));
        }
        __syncwarp();
      }
    }
  } else {
    // ================================================================== epilogue warp (pipeline g, TMEM quadrant q)
    const int g = warp / EPW, q = warp % EPW;
    const uint32_t grp_u = base + L::A_BYTES + g * L::GRP_BYTES;
    const int p = q * 32 + lane;
    const bool act = FT ? (2 * p < FT) : (2 * p < F);
    const int f0 = act ? 2 * p : 0; // inactive lanes compute on pair 0, store nothing and add nothing to the force
    const char* phi_f = reinterpret_cast<const char*>(phi) + f0 * 2;
    const char* vin_f = reinterpret_cast<const char*>(v_in) + f0 * 2;
    const char* vb_f = reinterpret_cast<const char*>(vb16) + f0 * 2;
    const char* sb_f = reinterpret_cast<const char*>(sb16) + f0 * 2;
    const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(g * 2 * NACC * NE);
    uint32_t n = 0;
    for (int64_t a0 = (int64_t)c_lo + (int64_t)g * RA; a0 < c_hi; a0 += (int64_t)NGRP * RA) {
      const int64_t a1 = min(a0 + RA, (int64_t)c_hi);
      const int na = (int)(a1 - a0);
      int tot;
      {
        const int rp = (lane <= na) ? __ldg(a.rowptr + a0 + lane) : 0;
        const int rp1 = __shfl_down_sync(0xffffffffu, rp, 1);
        tot = (lane < na) ? (rp1 - rp + ES - 1) / ES : 0;
#pragma unroll
        for (int o = 16; o; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
      }
      int cur = (int)a0;
      // the receiver's own rows (float2 = the thread's feature pair) and its segment sums
      float2 lph[3], lsb, lvb[3], lvi[3], A0, A1, Pv, A2[3], fpp[3];
      auto begin_row = [&](int i) {
        const char* pr = phi_f + (int64_t)i * 3 * F * 2;
        lph[0] = bf2(ldg_nc32(pr)); lph[1] = bf2(ldg_nc32(pr + 2 * F));
        lph[2] = HASV ? bf2(ldg_nc32(pr + 4 * F)) : make_float2(0.f, 0.f);
        lsb = bf2(ldg_nc32(sb_f + (int64_t)i * F * 2));
        const char* br = vb_f + (int64_t)i * 3 * F * 2;
        lvb[0] = bf2(ldg_nc32(br)); lvb[1] = bf2(ldg_nc32(br + 2 * F)); lvb[2] = bf2(ldg_nc32(br + 4 * F));
        if (HASV) {
          const char* vr = vin_f + (int64_t)i * 3 * F * 2;
          lvi[0] = bf2(ldg_nc32(vr)); lvi[1] = bf2(ldg_nc32(vr + 2 * F)); lvi[2] = bf2(ldg_nc32(vr + 4 * F));
        } else {
          lvi[0] = lvi[1] = lvi[2] = make_float2(0.f, 0.f);
        }
        A0 = A1 = Pv = make_float2(0.f, 0.f);
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) A2[ax] = fpp[ax] = make_float2(0.f, 0.f);
      };
      auto end_row = [&](int i) {
        if (HASV && act) {
          __nv_bfloat16* pb = phib16 + (int64_t)i * 3 * F + f0;
          st_stream1(pb, pack_bf2(A0.x, A0.y));
          st_stream1(pb + F, pack_bf2(A1.x, A1.y));
          st_stream1(pb + 2 * F, pack_bf2(Pv.x, Pv.y));
#pragma unroll
          for (int ax = 0; ax < 3; ++ax) {
            const int64_t off = ((int64_t)i * 3 + ax) * F + f0;
            const float2 res = ld_stream2(vb1 + off);
            st_stream2(vb_in + off, make_float2(res.x + lph[2].x * A2[ax].x, res.y + lph[2].y * A2[ax].y));
          }
        }
        float f3[3];
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
          f3[ax] = act ? fpp[ax].x + fpp[ax].y : 0.0f;
#pragma unroll
          for (int o = 16; o; o >>= 1) f3[ax] += __shfl_xor_sync(0xffffffffu, f3[ax], o);
        }
        if (lane == 0) { // force slab q of receiver i
          float* dst = fpart + ((int64_t)q * a.N + i) * 3;
          if (first_block) { dst[0] = f3[0]; dst[1] = f3[1]; dst[2] = f3[2]; }
          else { dst[0] += f3[0]; dst[1] += f3[1]; dst[2] += f3[2]; }
        }
      };
      begin_row(cur);
      for (int s0 = 0; s0 < tot; s0 += NSTEP, ++n) {
        const int slot = n % NSLOT;
        uint32_t mt_u = grp_u + NSLOT * 2 * L::B_TILE + slot * (uint32_t)sizeof(TileMetaB);
        asm volatile("" : "+r"(mt_u));
        mbar_wait(meta_full(g, slot), (n / NSLOT) & 1u);
        mbar_wait(tmem_full(g), n & 1u);
        tc_fence_after();
        // The gathers of step si + 1 are issued before the arithmetic of step si (two register sets, the loop is unrolled
        // by two steps): with two epilogue warps per scheduler there is little else to hide their latency behind.
        auto load_step = [&](int si, Gath& G) {
          const uint32_t cb = (uint32_t)si * (ES * 4);
          const uint2 oo = lds64(mt_u + (uint32_t)offsetof(TileMetaB, OFF) + cb);
          const uint2 os = lds64(mt_u + (uint32_t)offsetof(TileMetaB, OFS) + cb);
          const uint32_t offs[2] = {oo.x, oo.y}, ofss[2] = {os.x, os.y};
#pragma unroll
          for (int c = 0; c < ES; ++c) {
            const char* pr = phi_f + (uint64_t)offs[c] * 16u;
            G.gp[c][0] = ldg_nc32(pr); G.gp[c][1] = ldg_nc32(pr + 2 * F);
            G.gs[c] = ldg_nc32(sb_f + (uint64_t)ofss[c] * 16u);
            const char* br = vb_f + (uint64_t)offs[c] * 16u;
            G.gb[c][0] = ldg_nc32(br); G.gb[c][1] = ldg_nc32(br + 2 * F); G.gb[c][2] = ldg_nc32(br + 4 * F);
            if (HASV) {
              G.gp[c][2] = ldg_nc32(pr + 4 * F);
              const char* vr = vin_f + (uint64_t)offs[c] * 16u;
              G.gv[c][0] = ldg_nc32(vr); G.gv[c][1] = ldg_nc32(vr + 2 * F); G.gv[c][2] = ldg_nc32(vr + 4 * F);
            }
          }
        };
        auto used = [&](int si) {
          return si < NSTEP && lds64(mt_u + (uint32_t)offsetof(TileMetaB, sinfo) + 8u * si).y != 0u;
        };
        auto process = [&](int si, const Gath& G, bool last) {
          const uint32_t cb = (uint32_t)si * (ES * 4);
          float W[NACC][ES], D[NACC][ES];
#pragma unroll
          for (int acc = 0; acc < NACC; ++acc) {
            tmem_ld2_async(taddr + acc * NE + si * ES, W[acc]);
            tmem_ld2_async(taddr + (NACC + acc) * NE + si * ES, D[acc]);
          }
          const int i = (int)lds64(mt_u + (uint32_t)offsetof(TileMetaB, sinfo) + 8u * si).x;
          if (i != cur) { // receiver complete: write it and any edge-less atoms before the next one
            end_row(cur);
            for (int k = cur + 1; k < i; ++k) { begin_row(k); end_row(k); }
            cur = i;
            begin_row(cur);
          }
          const float2 ux = lds64f(mt_u + (uint32_t)offsetof(TileMetaB, Ux) + cb);
          const float2 uy = lds64f(mt_u + (uint32_t)offsetof(TileMetaB, Uy) + cb);
          const float2 uz = lds64f(mt_u + (uint32_t)offsetof(TileMetaB, Uz) + cb);
          const float2 idd = lds64f(mt_u + (uint32_t)offsetof(TileMetaB, Id) + cb);
#pragma unroll
          for (int acc = 0; acc < NACC; ++acc) { tmem_wait2(W[acc], acc == 0); tmem_wait2(D[acc], false); }
          if (last) { // the tile's last TMEM read is done: hand the buffer back now, so that the next tile's MMAs (there is
                      // ONE buffer per pipeline) run under the arithmetic of this step instead of after it
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tmem_empty(g, n & 1u));
          }
#pragma unroll
          for (int c = 0; c < ES; ++c) {
            const float u0 = c ? ux.y : ux.x, u1 = c ? uy.y : uy.x, u2 = c ? uz.y : uz.x, invd = c ? idd.y : idd.x;
            // ---- ss
            const float2 wss = make_float2(W[0][c], W[1][c]), dss = make_float2(D[0][c], D[1][c]);
            const float2 pj0 = bf2(G.gp[c][0]), sj = bf2(G.gs[c]);
            A0 = __ffma2_rn(sj, wss, A0);
            float2 y = __fmul2_rn(__ffma2_rn(lsb, pj0, __fmul2_rn(sj, lph[0])), dss);
            // ---- vs
            const float2 wvs = make_float2(W[2][c], W[3][c]), dvs = make_float2(D[2][c], D[3][c]);
            const float2 pj1 = bf2(G.gp[c][1]);
            const float2 b0 = bf2(G.gb[c][0]), b1 = bf2(G.gb[c][1]), b2 = bf2(G.gb[c][2]);
            const float2 tj = __ffma2_rn(b2, splat(u2), __ffma2_rn(b1, splat(u1), __fmul2_rn(b0, splat(u0))));
            const float2 ti = __ffma2_rn(lvb[2], splat(u2), __ffma2_rn(lvb[1], splat(u1), __fmul2_rn(lvb[0], splat(u0))));
            const float2 ntj = neg2(tj), nlph = neg2(lph[1]);
            A1 = __ffma2_rn(ntj, wvs, A1);
            const float2 xvs = __ffma2_rn(ti, pj1, __fmul2_rn(ntj, lph[1]));
            y = __ffma2_rn(xvs, dvs, y);
            const float2 wd = __fmul2_rn(wvs, splat(invd));
            const float2 nx = neg2(xvs);
            // tangential part: (q[a] - x u[a]) w / d with q[a] = vb_i[a] phi_j - vb_j[a] phi_i
            fpp[0] = __ffma2_rn(__ffma2_rn(nx, splat(u0), __ffma2_rn(lvb[0], pj1, __fmul2_rn(b0, nlph))), wd, fpp[0]);
            fpp[1] = __ffma2_rn(__ffma2_rn(nx, splat(u1), __ffma2_rn(lvb[1], pj1, __fmul2_rn(b1, nlph))), wd, fpp[1]);
            fpp[2] = __ffma2_rn(__ffma2_rn(nx, splat(u2), __ffma2_rn(lvb[2], pj1, __fmul2_rn(b2, nlph))), wd, fpp[2]);
            // ---- vv
            if (HASV) {
              const float2 wvv = make_float2(W[NACC - 2][c], W[NACC - 1][c]), dvv = make_float2(D[NACC - 2][c], D[NACC - 1][c]);
              const float2 pj2 = bf2(G.gp[c][2]);
              const float2 v0 = bf2(G.gv[c][0]), v1 = bf2(G.gv[c][1]), v2 = bf2(G.gv[c][2]);
              A2[0] = __ffma2_rn(b0, wvv, A2[0]);
              A2[1] = __ffma2_rn(b1, wvv, A2[1]);
              A2[2] = __ffma2_rn(b2, wvv, A2[2]);
              const float2 blv = __ffma2_rn(b2, lvi[2], __ffma2_rn(b1, lvi[1], __fmul2_rn(b0, lvi[0])));
              const float2 liv = __ffma2_rn(lvb[2], v2, __ffma2_rn(lvb[1], v1, __fmul2_rn(lvb[0], v0)));
              Pv = __ffma2_rn(blv, wvv, Pv);
              y = __ffma2_rn(__ffma2_rn(liv, pj2, __fmul2_rn(blv, lph[2])), dvv, y);
            }
            // ---- radial part: dE/dd u
            fpp[0] = __ffma2_rn(y, splat(u0), fpp[0]);
            fpp[1] = __ffma2_rn(y, splat(u1), fpp[1]);
            fpp[2] = __ffma2_rn(y, splat(u2), fpp[2]);
          }
        };
        Gath Ga, Gb;
        load_step(0, Ga); // (the first step of a tile is always used)
#pragma unroll 1
        for (int si = 0; si < NSTEP; si += 2) {
          const bool u1 = used(si + 1);
          if (u1) load_step(si + 1, Gb);
          process(si, Ga, !u1);
          if (!u1) break;
          const bool u2 = used(si + 2);
          if (u2) load_step(si + 2, Ga);
          process(si + 1, Gb, !u2);
          if (!u2) break;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(meta_empty(g, slot)); // (tmem_empty was signalled inside the tile's last step)
      }
      end_row(cur);
      for (int k = cur + 1; k < (int)a1; ++k) { begin_row(k); end_row(k); }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == NGRP * EPW) {
    tc_fence_after();
    tmem_dealloc<L::TMEM_COLS>(tmem_base);
  }
}

} // namespace

int edge_tc_bwd_num_slabs() { return EPW; }

int launch_edge_bwd_tc(const EdgeMmaArgs& a, const __nv_bfloat16* fltT, const __nv_bfloat16* phi, const __nv_bfloat16* v_in,
                       const __nv_bfloat16* sb16, const __nv_bfloat16* vb16, const float* vb1, __nv_bfloat16* phib16,
                       float* vb_in, float* fpart, int first_block, cudaStream_t st) {
  if (a.N == 0) return 0;
  const int KP = edge_mma_kp(a.K);
  const int RA = (int)std::min<int64_t>(16, std::max<int64_t>(2, a.N / (148 * NGRP * 8)));
  const unsigned grid = (unsigned)std::min<int64_t>(148, (a.N + RA * NGRP - 1) / (RA * NGRP));
#define PNN_LAUNCH2(KPV, HV, FTV)                                                                                     \
  {                                                                                                                   \
    using L = BwdSmem<KPV, HV>;                                                                                       \
    static bool attr_set = false;                                                                                     \
    if (!attr_set) {                                                                                                  \
      cudaFuncSetAttribute(edge_bwd_tc_k<KPV, HV, FTV>, cudaFuncAttributeMaxDynamicSharedMemorySize, L::TOTAL);       \
      attr_set = true;                                                                                                \
    }                                                                                                                 \
    edge_bwd_tc_k<KPV, HV, FTV><<<grid, NTHR, L::TOTAL, st>>>(a, RA, fltT, phi, v_in, sb16, vb16, vb1, phib16, vb_in, \
                                                              fpart, first_block);                                    \
    PNN_KCHECK("edge_bwd_tc_k");                                                                                      \
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
