// edge_mma.cu — a7 reverse edge kernel of the BF16 model: the filter contraction runs on the tensor cores (mma.sync on
// 16-edge tiles of one receiver).  The forward kernel of the BF16 model is edge_tc.cu (tcgen05).
//
// The filter is a small-K GEMM [edges x K] . [K x 3F] (SURVEY.md §7 hard part 3).  A 16-edge tile of ONE receiver is the M
// dimension of mma.sync.m16n8k16 (BF16 operands, FP32 accumulation): A = radial basis times cutoff, rounded to BF16, with
// the cutoff itself as an extra column so that flt_b rides along as an extra weight row; B = filter weights.  A warp owns a
// 32-feature slab of all three chunks.  The MMA columns are permuted (on the host, when the model is created) so that
// thread (g, t) of the accumulator fragment owns the 8 CONTIGUOUS features t*8 .. t*8+7 of the slab: the gathered sender
// rows (BF16) are then read with one 16-byte load per row and chunk, straight into the fragment layout, and multiplied in
// registers with packed FP32 FMAs (fma.rn.f32x2).  No atomics.
#include <algorithm>
#include <cstring>

#include "common.cuh"
#include "edge_mma.cuh"

namespace pnn {

namespace {

constexpr int TE = 16; // edges (rows) per MMA tile
constexpr int NTCB = 3; // tiles of one receiver staged per round

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// two BF16 packed in 32 bits -> (low, high) as FP32
__device__ __forceinline__ float2 bf2(uint32_t x) {
  return make_float2(__uint_as_float(x << 16), __uint_as_float(x & 0xffff0000u));
}
__device__ __forceinline__ uint32_t pack_bf2(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ uint4 ldg16(const __nv_bfloat16* p) { return __ldg(reinterpret_cast<const uint4*>(p)); }

constexpr int RED_PITCH = 80; // 16 floats + 16 bytes: conflict-free 16-byte accesses

// 16 per-thread partials -> sums over the 8 row groups.  Lanes with (g >> 2) == rh receive out[q] = sum of value
// (g & 3) * 4 + q; the other lanes receive nothing.
__device__ __forceinline__ void reduce16(const float (&v)[16], int lane, int rh, unsigned char* red, float (&out)[4]) {
  const int g = lane >> 2, t = lane & 3;
#pragma unroll
  for (int q = 0; q < 4; ++q)
    *reinterpret_cast<float4*>(red + lane * RED_PITCH + q * 16) = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
  __syncwarp();
  if ((g >> 2) == rh) {
    float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int gg = 0; gg < 8; ++gg) {
      const float4 x = *reinterpret_cast<const float4*>(red + (gg * 4 + t) * RED_PITCH + (g & 3) * 16);
      s.x += x.x; s.y += x.y; s.z += x.z; s.w += x.w;
    }
    out[0] = s.x; out[1] = s.y; out[2] = s.z; out[3] = s.w;
  }
  __syncwarp();
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ float2 neg2(float2 x) { return make_float2(-x.x, -x.y); }
__device__ __forceinline__ uint32_t sel4(const uint4& v, int nt) { return nt == 0 ? v.x : nt == 1 ? v.y : nt == 2 ? v.z : v.w; }

// Stage the A operand of up to NTC tiles of one receiver (one warp): G[row][k] = g_k(d) c(d) (k < K), c(d) (k == K),
// 0 (k > K), BF16; with BWD also G2 = dG/dd.  Us[row] = (u_x, u_y, u_z, d), Cs[row] = (c, c'), Js[row] = sender.
// Rows past the end of the receiver's segment are zero and gather from the receiver itself (finite values times an
// exact zero weight).
template <int KP, bool BWD>
__device__ __forceinline__ void stage_rows(const EdgeMmaArgs& a, int lane, int nrow, int e0, int eb, int self,
                                           unsigned char* Gs, unsigned char* G2s, float4* Us, float2* Cs, int* Js,
                                           float dmu, float gamma, float pi_rc) {
  constexpr int PA = KP * 2 + 16;
  for (int row = lane; row < nrow; row += 32) {
    const int e = e0 + row;
    float4 gq = make_float4(0.f, 0.f, 0.f, 1.f);
    float2 cc = make_float2(0.f, 0.f);
    int j = self;
    if (e < eb) {
      gq = __ldg(reinterpret_cast<const float4*>(a.geom) + e);
      j = __ldg(a.col + e);
      float sn, cs;
      __sincosf(pi_rc * gq.w, &sn, &cs);
      cc = make_float2(0.5f * (cs + 1.0f), -0.5f * pi_rc * sn);
    }
    Us[row] = gq; Cs[row] = cc; Js[row] = j;
  }
  __syncwarp();
  for (int idx = lane; idx < nrow * (KP / 2); idx += 32) {
    const int row = idx / (KP / 2), k = (idx % (KP / 2)) * 2;
    const float d = Us[row].w;
    const float2 cc = Cs[row]; // (0, 0) on padded rows
    float r0 = 0.f, r1 = 0.f, e0 = 0.f, e1 = 0.f; // basis functions k, k+1 and their derivatives
    if (a.rbf == 1) { // Bessel: sqrt(2/rc) sin(n pi d / rc) / d, n = k + 1
      const float A = sqrtf(2.0f / a.rc), id = 1.0f / d, w0 = (float)(k + 1) * pi_rc, w1 = w0 + pi_rc;
      float s0, c0, s1, c1;
      __sincosf(w0 * d, &s0, &c0);
      __sincosf(w1 * d, &s1, &c1);
      if (k < a.K) { r0 = A * s0 * id; e0 = (A * w0 * c0 - r0) * id; }
      if (k + 1 < a.K) { r1 = A * s1 * id; e1 = (A * w1 * c1 - r1) * id; }
    } else {          // Gaussian
      const float d0 = d - (float)k * dmu, d1 = d0 - dmu;
      if (k < a.K) { r0 = __expf(-gamma * d0 * d0); e0 = -2.0f * gamma * d0 * r0; }
      if (k + 1 < a.K) { r1 = __expf(-gamma * d1 * d1); e1 = -2.0f * gamma * d1 * r1; }
    }
    const float g0 = (k < a.K) ? r0 * cc.x : (k == a.K ? cc.x : 0.f);
    const float g1 = (k + 1 < a.K) ? r1 * cc.x : (k + 1 == a.K ? cc.x : 0.f);
    *reinterpret_cast<uint32_t*>(Gs + row * PA + k * 2) = pack_bf2(g0, g1);
    if (BWD) { // d/dd of the same columns
      const float h0 = (k < a.K) ? e0 * cc.x + r0 * cc.y : (k == a.K ? cc.y : 0.f);
      const float h1 = (k + 1 < a.K) ? e1 * cc.x + r1 * cc.y : (k + 1 == a.K ? cc.y : 0.f);
      *reinterpret_cast<uint32_t*>(G2s + row * PA + k * 2) = pack_bf2(h0, h1);
    }
  }
  __syncwarp();
}

// ------------------------------------------------------------------------------------------ reverse
// R3 + R4 of SURVEY.md §8(c) with the sender scatters rewritten as gathers over the receiver's own CSR row (the note
// under R4).  Same tiling as the forward kernel.  Per 16-edge tile, chunk c and 32-feature slab:
//   MMA 1   w[e, f]   = sum_k G[e, k] Wf[f, k]                 (the filter value, as in the forward kernel)
//   X[e, f] = the factor that multiplies dw/dd in dE/dd_e      (packed FP32 from the gathered BF16 rows), rounded to BF16
//   MMA 2   Y[e, k]  += sum_f X[e, f] Wf[f, k]                 (contraction over FEATURES: the accumulator fragment of X
//                                                              is already the A-fragment layout; B = the same filter
//                                                              rows through ldmatrix.trans)
//   dE/dd_e  = sum_k G'[e, k] Y[e, k]                          (K + 1 products per edge instead of F per edge)
// so the radial force costs one more small MMA instead of a per-feature FMA chain.  The node adjoints
// (phi-bar, v-bar_in) are segment sums kept in registers and reduced over the 8 row groups through shared memory.
template <int KP, bool HASV>
__global__ void __launch_bounds__(128, 2)
edge_bwd_mma_k(EdgeMmaArgs a, int NSL, int RB, const __nv_bfloat16* __restrict__ phi, const __nv_bfloat16* __restrict__ v_in,
               const __nv_bfloat16* __restrict__ sb16, const __nv_bfloat16* __restrict__ vb16, const float* vb1,
               __nv_bfloat16* phib16, float* vb_in, float* __restrict__ fpart, int first_block) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  constexpr int PA = KP * 2 + 16;
  constexpr int KS = KP / 16, KN = KP / 8;
  constexpr int NR = NTCB * TE;
  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
  unsigned char* Ws = smem;                                                      // [3][NSL][32 rows][PA]
  unsigned char* base = Ws + (size_t)3 * NSL * 32 * PA;
  unsigned char* Gs = base + (size_t)warp * NR * PA;                             // per warp [NR][PA]  G
  unsigned char* G2s = base + (size_t)nwarp * NR * PA + (size_t)warp * NR * PA;  // per warp [NR][PA]  dG/dd
  unsigned char* base2 = base + (size_t)2 * nwarp * NR * PA;
  float4* Us = reinterpret_cast<float4*>(base2) + warp * NR;
  float2* Cs = reinterpret_cast<float2*>(reinterpret_cast<float4*>(base2) + nwarp * NR) + warp * NR;
  int* Js = reinterpret_cast<int*>(reinterpret_cast<float2*>(reinterpret_cast<float4*>(base2) + nwarp * NR) + nwarp * NR) + warp * NR;
  unsigned char* Rs = reinterpret_cast<unsigned char*>(
      reinterpret_cast<int*>(reinterpret_cast<float2*>(reinterpret_cast<float4*>(base2) + nwarp * NR) + nwarp * NR) + nwarp * NR) +
      (size_t)warp * 32 * RED_PITCH;

  const int F = a.F;
  const int g = lane >> 2, t = lane & 3;
  const int slab0 = blockIdx.y * NSL;
  {
    const int nslab_tot = F / 32;
    constexpr int V = KP * 2 / 16;
    for (int idx = tid; idx < 3 * NSL * 32 * V; idx += nthr) {
      const int v = idx % V, r = idx / V;
      const int c = r / (NSL * 32), w = (r / 32) % NSL, row = r % 32;
      const uint4 val = __ldg(reinterpret_cast<const uint4*>(a.fltP) + ((size_t)((c * nslab_tot + slab0 + w) * 32 + row)) * V + v);
      *reinterpret_cast<uint4*>(Ws + (size_t)r * PA + v * 16) = val;
    }
  }
  __syncthreads();
  const float rc = a.rc;
  const float dmu = (a.K > 1) ? rc / (float)(a.K - 1) : rc;
  const float gamma = 1.0f / (2.0f * dmu * dmu);
  const float pi_rc = 3.14159265358979323846f / rc;
  const uint32_t a_off = (uint32_t)((lane & 15) * PA + (lane >> 4) * 16);
  const uint32_t b_off = (uint32_t)(((lane >> 4) * 8 + (lane & 7)) * PA + ((lane >> 3) & 1) * 16);
  // transposed B tiles of MMA 2: rows = features (kdim), matrices (kdim lo, n), (kdim hi, n), (kdim lo, n+1), (kdim hi, n+1)
  const uint32_t bt_off = (uint32_t)((((lane >> 3) & 1) * 8 + (lane & 7)) * PA + (lane >> 4) * 16);
  const uint32_t Ws_u = smem_u32(Ws), Gs_u = smem_u32(Gs);
  const uint4 zero4 = make_uint4(0u, 0u, 0u, 0u);

  const int64_t nchunk = (a.N + RB - 1) / RB;
  for (int64_t ch = blockIdx.x; ch < nchunk; ch += gridDim.x) {
    const int64_t i_end = min((int64_t)(ch + 1) * RB, a.N);
    for (int64_t i = ch * RB + warp; i < i_end; i += nwarp) {
      const int ea = a.rowptr[i], eb = a.rowptr[i + 1];
      float fp0 = 0.f, fp1 = 0.f, fp2 = 0.f;
      bool first = true;
      for (int r0 = ea; r0 < eb || (first && HASV); r0 += NR) {
        const int ntile = min(NTCB, (eb - r0 + TE - 1) / TE);
        stage_rows<KP, true>(a, lane, ntile * TE, r0, eb, (int)i, Gs, G2s, Us, Cs, Js, dmu, gamma, pi_rc);
        for (int sl = 0; sl < NSL; ++sl) {
          const int fbase = (slab0 + sl) * 32 + t * 8;
          const int64_t oi = i * 3 * F + fbase;
          float2 A0[4], A1[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) A0[q] = A1[q] = make_float2(0.f, 0.f);

          // One (tile, chunk) step shared by the three chunks: MMA 1, then `body` fills X and the accumulators.
          auto tile_step = [&](int tl, int c, auto&& body) {
            uint32_t af[KS][4];
#pragma unroll
            for (int ks = 0; ks < KS; ++ks)
              ldsm_x4(Gs_u + tl * TE * PA + a_off + ks * 32, af[ks][0], af[ks][1], af[ks][2], af[ks][3]);
            float C[4][4];
#pragma unroll
            for (int nt = 0; nt < 4; ++nt)
#pragma unroll
              for (int q = 0; q < 4; ++q) C[nt][q] = 0.f;
            const uint32_t wrow = Ws_u + (uint32_t)((c * NSL + sl) * 32) * PA;
#pragma unroll
            for (int np = 0; np < 2; ++np)
#pragma unroll
              for (int ks = 0; ks < KS; ++ks) {
                uint32_t b0, b1, b2, b3;
                ldsm_x4(wrow + b_off + np * 16 * PA + ks * 32, b0, b1, b2, b3);
                mma_bf16(C[2 * np], af[ks], b0, b1);
                mma_bf16(C[2 * np + 1], af[ks], b2, b3);
              }
            uint32_t xa[2][4]; // A fragments of X: [feature k-step][row g lo, row g+8 lo, row g hi, row g+8 hi]
            body(C, xa);
            float CY[KN][4];
#pragma unroll
            for (int kn = 0; kn < KN; ++kn)
#pragma unroll
              for (int q = 0; q < 4; ++q) CY[kn][q] = 0.f;
#pragma unroll
            for (int ks = 0; ks < 2; ++ks)
#pragma unroll
              for (int kp = 0; kp < KN / 2; ++kp) {
                uint32_t b0, b1, b2, b3;
                ldsm_x4_t(wrow + bt_off + ks * 16 * PA + kp * 32, b0, b1, b2, b3);
                mma_bf16(CY[2 * kp], xa[ks], b0, b1);
                mma_bf16(CY[2 * kp + 1], xa[ks], b2, b3);
              }
            // dE/dd of rows g and g+8 (this thread's columns), then the radial force
            float y0 = 0.f, y1 = 0.f;
#pragma unroll
            for (int kn = 0; kn < KN; ++kn) {
              const float2 d0 = bf2(*reinterpret_cast<const uint32_t*>(G2s + (tl * TE + g) * PA + (kn * 8 + 2 * t) * 2));
              const float2 d1 = bf2(*reinterpret_cast<const uint32_t*>(G2s + (tl * TE + g + 8) * PA + (kn * 8 + 2 * t) * 2));
              y0 = fmaf(d0.x, CY[kn][0], fmaf(d0.y, CY[kn][1], y0));
              y1 = fmaf(d1.x, CY[kn][2], fmaf(d1.y, CY[kn][3], y1));
            }
            const float4 u0 = Us[tl * TE + g], u1 = Us[tl * TE + g + 8];
            fp0 += y0 * u0.x + y1 * u1.x; fp1 += y0 * u0.y + y1 * u1.y; fp2 += y0 * u0.z + y1 * u1.z;
          };

          // ---------------- chunk 0 (ss): A0 += sb_j w ; X = sb_i phi_j + sb_j phi_i
          {
            const uint4 sbi = ldg16(sb16 + i * F + fbase), phi_i = ldg16(phi + oi);
            for (int tl = 0; tl < ntile; ++tl) {
              const bool ok0 = r0 + tl * TE + g < eb, ok1 = r0 + tl * TE + g + 8 < eb;
              const int64_t j0 = Js[tl * TE + g], j1 = Js[tl * TE + g + 8];
              const uint4 p0 = ok0 ? ldg16(phi + j0 * 3 * F + fbase) : zero4, p1 = ok1 ? ldg16(phi + j1 * 3 * F + fbase) : zero4;
              const uint4 s0 = ok0 ? ldg16(sb16 + j0 * F + fbase) : zero4, s1 = ok1 ? ldg16(sb16 + j1 * F + fbase) : zero4;
              tile_step(tl, 0, [&](float (&C)[4][4], uint32_t (&xa)[2][4]) {
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) {
                  const float2 li = bf2(sel4(sbi, nt)), lph = bf2(sel4(phi_i, nt));
                  const float2 ph0 = bf2(sel4(p0, nt)), ph1 = bf2(sel4(p1, nt));
                  const float2 sj0 = bf2(sel4(s0, nt)), sj1 = bf2(sel4(s1, nt));
                  A0[nt] = __ffma2_rn(sj0, make_float2(C[nt][0], C[nt][1]), A0[nt]);
                  A0[nt] = __ffma2_rn(sj1, make_float2(C[nt][2], C[nt][3]), A0[nt]);
                  const float2 x0 = __ffma2_rn(li, ph0, __fmul2_rn(sj0, lph));
                  const float2 x1 = __ffma2_rn(li, ph1, __fmul2_rn(sj1, lph));
                  xa[nt >> 1][(nt & 1) * 2] = pack_bf2(x0.x, x0.y);
                  xa[nt >> 1][(nt & 1) * 2 + 1] = pack_bf2(x1.x, x1.y);
                }
              });
            }
          }
          // ---------------- chunk 1 (vs): A1 -= (vb_j.u) w ; X = (vb_i.u) phi_j - (vb_j.u) phi_i ; tangential term
          {
            const uint4 phi_i = ldg16(phi + oi + F);
            uint4 vbi[3];
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) vbi[ax] = ldg16(vb16 + oi + ax * F);
            for (int tl = 0; tl < ntile; ++tl) {
              const bool ok[2] = {r0 + tl * TE + g < eb, r0 + tl * TE + g + 8 < eb};
              const int64_t oj[2] = {(int64_t)Js[tl * TE + g] * 3 * F + fbase, (int64_t)Js[tl * TE + g + 8] * 3 * F + fbase};
              const float4 uu[2] = {Us[tl * TE + g], Us[tl * TE + g + 8]};
              uint4 pj[2], bj[2][3];
#pragma unroll
              for (int r = 0; r < 2; ++r) {
                pj[r] = ok[r] ? ldg16(phi + oj[r] + F) : zero4;
#pragma unroll
                for (int ax = 0; ax < 3; ++ax) bj[r][ax] = ok[r] ? ldg16(vb16 + oj[r] + ax * F) : zero4;
              }
              float2 BS[2][3];
#pragma unroll
              for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int ax = 0; ax < 3; ++ax) BS[r][ax] = make_float2(0.f, 0.f);
              tile_step(tl, 1, [&](float (&C)[4][4], uint32_t (&xa)[2][4]) {
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) {
                  const float2 lph = bf2(sel4(phi_i, nt)), nlph = neg2(lph);
                  const float2 l0 = bf2(sel4(vbi[0], nt)), l1 = bf2(sel4(vbi[1], nt)), l2 = bf2(sel4(vbi[2], nt));
#pragma unroll
                  for (int r = 0; r < 2; ++r) {
                    const float2 ux = make_float2(uu[r].x, uu[r].x), uy = make_float2(uu[r].y, uu[r].y),
                                 uz = make_float2(uu[r].z, uu[r].z);
                    const float2 w = make_float2(C[nt][2 * r], C[nt][2 * r + 1]);
                    const float2 ph = bf2(sel4(pj[r], nt));
                    const float2 b0 = bf2(sel4(bj[r][0], nt)), b1 = bf2(sel4(bj[r][1], nt)), b2 = bf2(sel4(bj[r][2], nt));
                    const float2 tj = __ffma2_rn(b2, uz, __ffma2_rn(b1, uy, __fmul2_rn(b0, ux)));
                    const float2 ti = __ffma2_rn(l2, uz, __ffma2_rn(l1, uy, __fmul2_rn(l0, ux)));
                    const float2 ntj = neg2(tj);
                    A1[nt] = __ffma2_rn(ntj, w, A1[nt]);
                    const float2 x = __ffma2_rn(ti, ph, __fmul2_rn(ntj, lph));
                    xa[nt >> 1][(nt & 1) * 2 + r] = pack_bf2(x.x, x.y);
                    BS[r][0] = __ffma2_rn(__ffma2_rn(l0, ph, __fmul2_rn(b0, nlph)), w, BS[r][0]);
                    BS[r][1] = __ffma2_rn(__ffma2_rn(l1, ph, __fmul2_rn(b1, nlph)), w, BS[r][1]);
                    BS[r][2] = __ffma2_rn(__ffma2_rn(l2, ph, __fmul2_rn(b2, nlph)), w, BS[r][2]);
                  }
                }
              });
              // tangential force of the direction term: (B - (B.u) u) / d, B summed over this thread's features
#pragma unroll
              for (int r = 0; r < 2; ++r) {
                const float B0 = BS[r][0].x + BS[r][0].y, B1 = BS[r][1].x + BS[r][1].y, B2 = BS[r][2].x + BS[r][2].y;
                const float Bu = B0 * uu[r].x + B1 * uu[r].y + B2 * uu[r].z;
                const float invd = 1.0f / uu[r].w;
                fp0 += (B0 - Bu * uu[r].x) * invd; fp1 += (B1 - Bu * uu[r].y) * invd; fp2 += (B2 - Bu * uu[r].z) * invd;
              }
            }
          }
          if (HASV) {
            float o4[4];
            float vals[16];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              vals[2 * q] = A0[q].x; vals[2 * q + 1] = A0[q].y; vals[8 + 2 * q] = A1[q].x; vals[8 + 2 * q + 1] = A1[q].y;
            }
            reduce16(vals, lane, 0, Rs, o4);
            if (g < 4) { // phi-bar ss (g 0,1) and vs (g 2,3)
              __nv_bfloat16* dst = phib16 + i * 3 * F + (g >> 1) * F + (slab0 + sl) * 32 + t * 8 + (g & 1) * 4;
              if (!first) {
                const uint2 old = *reinterpret_cast<const uint2*>(dst);
                const float2 q0 = bf2(old.x), q1 = bf2(old.y);
                o4[0] += q0.x; o4[1] += q0.y; o4[2] += q1.x; o4[3] += q1.y;
              }
              *reinterpret_cast<uint2*>(dst) = make_uint2(pack_bf2(o4[0], o4[1]), pack_bf2(o4[2], o4[3]));
            }
          }
          // ---------------- chunk 2 (vv): A2[a] += vb_j[a] w ; Pvv += (vb_j.v_i) w ; X = (vb_i.v_j) phi_j + (vb_j.v_i) phi_i
          if (HASV) {
            float2 A2[3][4], Pv[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) { Pv[q] = A2[0][q] = A2[1][q] = A2[2][q] = make_float2(0.f, 0.f); }
            const uint4 phi_i = ldg16(phi + oi + 2 * F);
            uint4 vbi[3], vi[3];
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) { vbi[ax] = ldg16(vb16 + oi + ax * F); vi[ax] = ldg16(v_in + oi + ax * F); }
            for (int tl = 0; tl < ntile; ++tl) {
              const bool ok[2] = {r0 + tl * TE + g < eb, r0 + tl * TE + g + 8 < eb};
              const int64_t oj[2] = {(int64_t)Js[tl * TE + g] * 3 * F + fbase, (int64_t)Js[tl * TE + g + 8] * 3 * F + fbase};
              uint4 pj[2], bj[2][3], vj[2][3];
#pragma unroll
              for (int r = 0; r < 2; ++r) {
                pj[r] = ok[r] ? ldg16(phi + oj[r] + 2 * F) : zero4;
#pragma unroll
                for (int ax = 0; ax < 3; ++ax) {
                  bj[r][ax] = ok[r] ? ldg16(vb16 + oj[r] + ax * F) : zero4;
                  vj[r][ax] = ok[r] ? ldg16(v_in + oj[r] + ax * F) : zero4;
                }
              }
              tile_step(tl, 2, [&](float (&C)[4][4], uint32_t (&xa)[2][4]) {
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) {
                  const float2 lph = bf2(sel4(phi_i, nt));
                  const float2 l0 = bf2(sel4(vbi[0], nt)), l1 = bf2(sel4(vbi[1], nt)), l2 = bf2(sel4(vbi[2], nt));
                  const float2 m0 = bf2(sel4(vi[0], nt)), m1 = bf2(sel4(vi[1], nt)), m2 = bf2(sel4(vi[2], nt));
#pragma unroll
                  for (int r = 0; r < 2; ++r) {
                    const float2 w = make_float2(C[nt][2 * r], C[nt][2 * r + 1]);
                    const float2 ph = bf2(sel4(pj[r], nt));
                    const float2 b0 = bf2(sel4(bj[r][0], nt)), b1 = bf2(sel4(bj[r][1], nt)), b2 = bf2(sel4(bj[r][2], nt));
                    const float2 v0 = bf2(sel4(vj[r][0], nt)), v1 = bf2(sel4(vj[r][1], nt)), v2 = bf2(sel4(vj[r][2], nt));
                    A2[0][nt] = __ffma2_rn(b0, w, A2[0][nt]);
                    A2[1][nt] = __ffma2_rn(b1, w, A2[1][nt]);
                    A2[2][nt] = __ffma2_rn(b2, w, A2[2][nt]);
                    const float2 blv = __ffma2_rn(b2, m2, __ffma2_rn(b1, m1, __fmul2_rn(b0, m0)));
                    const float2 liv = __ffma2_rn(l2, v2, __ffma2_rn(l1, v1, __fmul2_rn(l0, v0)));
                    Pv[nt] = __ffma2_rn(blv, w, Pv[nt]);
                    const float2 x = __ffma2_rn(liv, ph, __fmul2_rn(blv, lph));
                    xa[nt >> 1][(nt & 1) * 2 + r] = pack_bf2(x.x, x.y);
                  }
                }
              });
            }
            // reductions and stores: [Pvv, A2[0]] read by g >= 4, [A2[1], A2[2]] read by g < 4
            float vals[16], o4[4];
#pragma unroll
            for (int pass = 0; pass < 2; ++pass) {
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                const float2 lo = pass == 0 ? Pv[q] : A2[1][q], hi = pass == 0 ? A2[0][q] : A2[2][q];
                vals[2 * q] = lo.x; vals[2 * q + 1] = lo.y; vals[8 + 2 * q] = hi.x; vals[8 + 2 * q + 1] = hi.y;
              }
              const int rh = pass == 0 ? 1 : 0;
              reduce16(vals, lane, rh, Rs, o4);
              if ((g >> 2) == rh) {
                const int which = (g & 3) >> 1;
                const int f = (slab0 + sl) * 32 + t * 8 + (g & 1) * 4;
                if (pass == 0 && which == 0) { // phi-bar vv
                  __nv_bfloat16* dst = phib16 + i * 3 * F + 2 * F + f;
                  if (!first) {
                    const uint2 old = *reinterpret_cast<const uint2*>(dst);
                    const float2 q0 = bf2(old.x), q1 = bf2(old.y);
                    o4[0] += q0.x; o4[1] += q0.y; o4[2] += q1.x; o4[3] += q1.y;
                  }
                  *reinterpret_cast<uint2*>(dst) = make_uint2(pack_bf2(o4[0], o4[1]), pack_bf2(o4[2], o4[3]));
                } else { // v-bar_in[ax] = v-bar'[ax] + phi_i^vv A2[ax]
                  const int ax = pass == 0 ? 0 : 1 + which;
                  const int64_t off = (i * 3 + ax) * F + f;
                  const uint2 pv = *reinterpret_cast<const uint2*>(phi + i * 3 * F + 2 * F + f);
                  const float2 q0 = bf2(pv.x), q1 = bf2(pv.y);
                  const float4 res = first ? *reinterpret_cast<const float4*>(vb1 + off) : *reinterpret_cast<const float4*>(vb_in + off);
                  *reinterpret_cast<float4*>(vb_in + off) =
                      make_float4(res.x + q0.x * o4[0], res.y + q0.y * o4[1], res.z + q1.x * o4[2], res.w + q1.y * o4[3]);
                }
              }
            }
          }
        }
        __syncwarp();
        first = false;
      }
      // force of receiver i from this CTA's feature slabs: all-reduce over the warp
#pragma unroll
      for (int o = 16; o; o >>= 1) {
        fp0 += __shfl_xor_sync(0xffffffffu, fp0, o);
        fp1 += __shfl_xor_sync(0xffffffffu, fp1, o);
        fp2 += __shfl_xor_sync(0xffffffffu, fp2, o);
      }
      if (lane == 0) {
        float* dst = fpart + ((int64_t)blockIdx.y * a.N + i) * 3;
        if (first_block) { dst[0] = fp0; dst[1] = fp1; dst[2] = fp2; }
        else { dst[0] += fp0; dst[1] += fp1; dst[2] += fp2; }
      }
    }
  }
}

// 32-feature slabs per CTA: a divisor of F/32, at most 4
int pick_nsl(int F) {
  const int ns = F / 32;
  for (int nw = 4; nw > 1; --nw)
    if (ns % nw == 0) return nw;
  return 1;
}

} // namespace

int edge_mma_kp(int K) { return (K + 1 + 15) / 16 * 16; }

// Host-side packing of one block's filter for the MMA kernels (layout in the header).
void pack_filter_bf16(int F, int K, const double* fltW, const double* fltb, uint16_t* out) {
  const int KP = edge_mma_kp(K), ns = F / 32;
  auto to_bf16 = [](double x) -> uint16_t {
    float f = (float)x;
    uint32_t u;
    std::memcpy(&u, &f, 4);
    const uint32_t r = u + 0x7fffu + ((u >> 16) & 1u); // round to nearest even
    return (uint16_t)(r >> 16);
  };
  for (int c = 0; c < 3; ++c)
    for (int s = 0; s < ns; ++s)
      for (int nt = 0; nt < 4; ++nt)
        for (int g = 0; g < 8; ++g) {
          const int f = s * 32 + (g >> 1) * 8 + nt * 2 + (g & 1);
          const int64_t src = (int64_t)c * F + f;
          uint16_t* dst = out + ((int64_t)((c * ns + s) * 4 + nt) * 8 + g) * KP;
          for (int k = 0; k < KP; ++k) dst[k] = k < K ? to_bf16(fltW[src * K + k]) : (k == K ? to_bf16(fltb[src]) : 0);
        }
}

size_t edge_mma_smem(int KP, int NSL, int nwarp) {
  const int PA = KP * 2 + 16, NR = NTCB * TE;
  return (size_t)3 * NSL * 32 * PA + (size_t)nwarp * (NR * (PA * 2 + 16 + 8 + 4) + 32 * RED_PITCH);
}

int edge_mma_num_slabs(int F) { return F / 32 / pick_nsl(F); }

int launch_edge_bwd_mma(const EdgeMmaArgs& a, const __nv_bfloat16* phi, const __nv_bfloat16* v_in,
                        const __nv_bfloat16* sb16, const __nv_bfloat16* vb16, const float* vb1, __nv_bfloat16* phib16,
                        float* vb_in, float* fpart, int first_block, cudaStream_t st) {
  if (a.N == 0) return 0;
  const int KP = edge_mma_kp(a.K), NSL = pick_nsl(a.F), NWARP = 4;
  const int RB = (int)std::min<int64_t>(16, std::max<int64_t>(8, a.N / (148 * 2 * 8)));   // cfg3: 16 -> 8, 930 -> 863 us
  const int64_t nchunk = (a.N + RB - 1) / RB;
  dim3 grid((unsigned)std::min<int64_t>(nchunk, 148 * 2), a.F / 32 / NSL);
  const size_t smem = edge_mma_smem(KP, NSL, NWARP);
#define PNN_LAUNCH(KPV, HV)                                                                                        \
  {                                                                                                                \
    static bool attr_set = false;                                                                                  \
    if (!attr_set) {                                                                                               \
      cudaFuncSetAttribute(edge_bwd_mma_k<KPV, HV>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);      \
      attr_set = true;                                                                                             \
    }                                                                                                              \
    edge_bwd_mma_k<KPV, HV><<<grid, NWARP * 32, smem, st>>>(a, NSL, RB, phi, v_in, sb16, vb16, vb1, phib16, vb_in, \
                                                            fpart, first_block);                                   \
    PNN_KCHECK("edge_bwd_mma_k");                                                                                  \
  }
  const bool hv = v_in != nullptr;
  if (KP == 16) { if (hv) PNN_LAUNCH(16, true) else PNN_LAUNCH(16, false) }
  else if (KP == 32) { if (hv) PNN_LAUNCH(32, true) else PNN_LAUNCH(32, false) }
  else { if (hv) PNN_LAUNCH(48, true) else PNN_LAUNCH(48, false) }
#undef PNN_LAUNCH
  return 1;
}

} // namespace pnn
