// edge_warp.cu — a4 / a7 edge kernels of the FP32 model, exact FP32 arithmetic on the ordinary ALUs.
//
// Same mathematics as edge.cu (sender scatters rewritten as gathers over the receiver's own
// CSR row), different mapping, chosen from the ncu stall profile of edge.cu (profiles/r01_edge_fp32_cfg2.md: gather
// latency and CTA barriers, not FMA throughput):
//   * one WARP per receiver, no CTA barrier in the main loop;
//   * a lane owns FPL (1 or 2) contiguous features of a 32*FPL-wide slab for the whole kernel and keeps the 3*FPL filter
//     rows of those features (K weights each) in registers as float2 pairs;
//   * the radial basis of a 32-edge tile is staged once per warp in shared memory and read back as broadcast float4;
//   * per edge the lane first issues ALL its gathers (phi_j, v_j, and in the reverse kernel the adjoint rows), then runs
//     the 3*FPL filter dot products with packed FMAs (fma.rn.f32x2) while the loads are in flight, then consumes them;
//     the segment sums stay in registers and are written once per receiver: no cross-lane reduction, no atomics;
//   * consecutive lanes own consecutive features, so every gather is one full 128- or 256-byte line per row.
#include <algorithm>
#include <cstdlib>

#include "common.cuh"

namespace pnn {

namespace {

constexpr int TW = 32; // edges per staged tile (one row per lane)

template <int FPL> struct VecF;
template <> struct VecF<1> { using type = float; };
template <> struct VecF<2> { using type = float2; };

template <int FPL>
__device__ __forceinline__ void ldv(const float* p, float (&x)[FPL]) {
  if (FPL == 1) x[0] = __ldg(p);
  else { const float2 t = __ldg(reinterpret_cast<const float2*>(p)); x[0] = t.x; x[FPL - 1] = t.y; }
}
// The edge tape is written once and read once, a whole sweep later: streaming (evict-first) accesses keep it from
// displacing the gathered node rows in L2.
template <int FPL>
__device__ __forceinline__ void ldv_stream(const float* p, float (&x)[FPL]) {
  if (FPL == 1) x[0] = __ldcs(p);
  else { const float2 t = __ldcs(reinterpret_cast<const float2*>(p)); x[0] = t.x; x[FPL - 1] = t.y; }
}
template <int FPL>
__device__ __forceinline__ void stv_stream(float* p, const float (&x)[FPL]) {
  if (FPL == 1) __stcs(p, x[0]);
  else __stcs(reinterpret_cast<float2*>(p), make_float2(x[0], x[FPL - 1]));
}
template <int FPL>
__device__ __forceinline__ void stv(float* p, const float (&x)[FPL]) {
  if (FPL == 1) *p = x[0];
  else *reinterpret_cast<float2*>(p) = make_float2(x[0], x[FPL - 1]);
}

// w . g, w as KP/2 register pairs, g a row of the staged tile (16-byte aligned, broadcast)
template <int KP>
__device__ __forceinline__ float dot_pairs(const float2 (&w)[KP / 2], const float* __restrict__ g, float init) {
  float2 acc = make_float2(init, 0.0f), acc2 = make_float2(0.0f, 0.0f); // two chains: instruction-level parallelism
#pragma unroll
  for (int k = 0; k < KP; k += 4) {
    const float4 t = *reinterpret_cast<const float4*>(g + k);
    acc = __ffma2_rn(w[k / 2], make_float2(t.x, t.y), acc);
    acc2 = __ffma2_rn(w[k / 2 + 1], make_float2(t.z, t.w), acc2);
  }
  // four partial sums over k mod 4: a single chain (two partial sums) saves 12 FPL additions per edge, measured 6 % on the
  // kernel, but its longer chains round worse -- cfg3 FP32 forces 8e-5 -> 1.45e-4 against the oracle, over the 1e-4 tolerance
  return (acc.x + acc2.x) + (acc.y + acc2.y);
}

// One warp stages a tile: lane = row.  G1[row][k] = g_k(d) c(d); with BWD also G2[row][k] = d/dd (g_k c).
template <int KP, bool BWD>
__device__ __forceinline__ void stage_tile_w(const EdgeArgs<float>& a, int lane, int t0, int nE, float* G1, float* G2,
                                             float4* U, float2* C, int* J, float dmu, float gamma, float pi_rc) {
  constexpr int PG = KP + 4;
  if (lane < nE) {
    const Geom<float> gq = a.geom[t0 + lane];
    float sn, cs;
    sincosf(pi_rc * gq.d, &sn, &cs);
    const float cc = 0.5f * (cs + 1.0f), cp = -0.5f * pi_rc * sn;
    U[lane] = make_float4(gq.ux, gq.uy, gq.uz, gq.d);
    C[lane] = make_float2(cc, cp);
    J[lane] = a.col[t0 + lane];
#pragma unroll 4
    for (int k = 0; k < KP; ++k) {
      float g = 0.0f, gd = 0.0f;
      if (k < a.K) rbf_eval<float>(a.rbf, k, gq.d, (float)a.rc, dmu, gamma, g, gd);
      G1[lane * PG + k] = g * cc;
      if (BWD) G2[lane * PG + k] = cc * gd + cp * g;
    }
  }
  __syncwarp();
}

template <int KP, int FPL>
__device__ __forceinline__ void load_rows(const EdgeArgs<float>& a, int f0, float2 (&w)[3][FPL][KP / 2], float (&bias)[3][FPL]) {
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int p = 0; p < FPL; ++p) {
      const int64_t row = (int64_t)c * a.F + f0 + p;
#pragma unroll
      for (int k = 0; k < KP; k += 2)
        w[c][p][k / 2] = make_float2(k < a.K ? a.fltW[row * a.K + k] : 0.0f, k + 1 < a.K ? a.fltW[row * a.K + k + 1] : 0.0f);
      bias[c][p] = a.fltb[row];
    }
}

// ------------------------------------------------------------------------------------------ forward
// TAPE: also evaluate dw/dd and keep w and dw/dd of every (edge, chunk, feature) for the reverse sweep
// (wt, dt: [E][3][F]), so that the reverse edge kernel does no filter arithmetic at all.
template <int KP, int FPL, int NWARP, bool TAPE>
__global__ void __launch_bounds__(NWARP * 32, (FPL == 1 && KP <= 24) ? 3 : 2)
edge_fwd_w_k(EdgeArgs<float> a, int RB, const float* __restrict__ phi, const float* __restrict__ s_in, int64_t ld_sin,
             const float* __restrict__ v_in, float* __restrict__ s1, int64_t ld_s1, float* __restrict__ v1,
             float* __restrict__ wt, float* __restrict__ dt) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  constexpr int PG = KP + 4;
  __shared__ __align__(16) float G1s[NWARP][TW * PG];
  __shared__ __align__(16) float G2s[TAPE ? NWARP : 1][TAPE ? TW * PG : 4];
  __shared__ float4 Us[NWARP][TW];
  __shared__ float2 Cs[NWARP][TW];
  __shared__ int Js[NWARP][TW];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int F = a.F;
  const int f0 = (blockIdx.y * 32 + lane) * FPL;
  float2 w[3][FPL][KP / 2];
  float bias[3][FPL];
  load_rows<KP, FPL>(a, f0, w, bias);
  const float rc = (float)a.rc;
  const float dmu = (a.K > 1) ? rc / (float)(a.K - 1) : rc;
  const float gamma = 1.0f / (2.0f * dmu * dmu);
  const float pi_rc = (float)(3.14159265358979323846 / a.rc);
  const bool has_v = v_in != nullptr;
  float* G1 = G1s[warp]; float4* U = Us[warp]; float2* C = Cs[warp]; int* J = Js[warp];
  float* G2 = TAPE ? G2s[warp] : nullptr;

  const int64_t nchunk = (a.N + RB - 1) / RB;
  for (int64_t ch = blockIdx.x; ch < nchunk; ch += gridDim.x) {
    const int64_t i_end = min((int64_t)(ch + 1) * RB, a.N);
    for (int64_t i = ch * RB + warp; i < i_end; i += NWARP) {
      const int ea = a.rowptr[i], eb = a.rowptr[i + 1];
      float as[FPL], av[3][FPL];
#pragma unroll
      for (int p = 0; p < FPL; ++p) { as[p] = 0.f; av[0][p] = av[1][p] = av[2][p] = 0.f; }
      // the receiver's own rows (residual), in flight during the edge loop
      float so[FPL], vo[3][FPL];
      ldv<FPL>(s_in + i * ld_sin + f0, so);
#pragma unroll
      for (int ax = 0; ax < 3; ++ax) {
        if (has_v) ldv<FPL>(v_in + (i * 3 + ax) * F + f0, vo[ax]);
        else {
#pragma unroll
          for (int p = 0; p < FPL; ++p) vo[ax][p] = 0.f;
        }
      }
      for (int t0 = ea; t0 < eb; t0 += TW) {
        const int nE = min(TW, eb - t0);
        stage_tile_w<KP, TAPE>(a, lane, t0, nE, G1, G2, U, C, J, dmu, gamma, pi_rc);
        // software pipeline: the sender rows of edge q+1 are requested before edge q is consumed; the loop is unrolled by two
        // so that the two register sets swap roles by name instead of by 6 FPL moves per edge
        float phA[3][FPL], vjA[3][FPL], phB[3][FPL], vjB[3][FPL];
        auto gather = [&](int q, float (&p_)[3][FPL], float (&v_)[3][FPL]) {
          const int64_t jo = (int64_t)J[q] * 3 * F + f0;
#pragma unroll
          for (int c = 0; c < 3; ++c) ldv<FPL>(phi + jo + c * F, p_[c]);
          if (has_v) {
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) ldv<FPL>(v_in + jo + ax * F, v_[ax]);
          }
        };
        float* wp = TAPE ? wt + (int64_t)t0 * 3 * F + f0 : nullptr; // tape rows of the current edge
        float* dp = TAPE ? dt + (int64_t)t0 * 3 * F + f0 : nullptr;
        auto step = [&](int q, float (&ph)[3][FPL], float (&vj)[3][FPL], float (&phn)[3][FPL], float (&vjn)[3][FPL]) {
          if (q + 1 < nE) gather(q + 1, phn, vjn);
          const float4 u = U[q];
          const float cc = C[q].x;
          const float* g = G1 + q * PG;
          float wv[3][FPL];
#pragma unroll
          for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int p = 0; p < FPL; ++p)
              wv[c][p] = (c < 2 || has_v) ? dot_pairs<KP>(w[c][p], g, bias[c][p] * cc) : 0.0f;
          if (TAPE) {
            const float cp = C[q].y;
            const float* g2 = G2 + q * PG;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
              if (c == 2 && !has_v) break;
              float dw[FPL];
#pragma unroll
              for (int p = 0; p < FPL; ++p) dw[p] = dot_pairs<KP>(w[c][p], g2, bias[c][p] * cp);
              stv_stream<FPL>(wp + c * F, wv[c]);
              stv_stream<FPL>(dp + c * F, dw);
            }
            wp += 3 * F; dp += 3 * F;
          }
#pragma unroll
          for (int p = 0; p < FPL; ++p) {
            as[p] = fmaf(ph[0][p], wv[0][p], as[p]);
            const float x1 = ph[1][p] * wv[1][p];
            av[0][p] = fmaf(x1, u.x, av[0][p]); av[1][p] = fmaf(x1, u.y, av[1][p]); av[2][p] = fmaf(x1, u.z, av[2][p]);
            if (has_v) {
              const float x2 = ph[2][p] * wv[2][p];
              av[0][p] = fmaf(x2, vj[0][p], av[0][p]); av[1][p] = fmaf(x2, vj[1][p], av[1][p]);
              av[2][p] = fmaf(x2, vj[2][p], av[2][p]);
            }
          }
        };
        gather(0, phA, vjA);
        for (int q = 0; q < nE; q += 2) {
          step(q, phA, vjA, phB, vjB);
          if (q + 1 < nE) step(q + 1, phB, vjB, phA, vjA);
        }
        __syncwarp(); // the tile buffers are restaged
      }
#pragma unroll
      for (int p = 0; p < FPL; ++p) { so[p] += as[p]; vo[0][p] += av[0][p]; vo[1][p] += av[1][p]; vo[2][p] += av[2][p]; }
      stv<FPL>(s1 + i * ld_s1 + f0, so);
#pragma unroll
      for (int ax = 0; ax < 3; ++ax) stv<FPL>(v1 + (i * 3 + ax) * F + f0, vo[ax]);
    }
  }
}

// ------------------------------------------------------------------------------------------ reverse
// R3 + R4 with the filter value w and its derivative dw/dd read from the edge tape the forward kernel wrote: no
// radial basis, no filter arithmetic, no shared memory.  Per edge a lane streams 6*FPL tape values (coalesced),
// gathers the sender's phi, s-bar', v-bar', v rows for its features and keeps the receiver's own rows in registers.
template <int FPL, int NWARP>
__global__ void __launch_bounds__(NWARP * 32)
edge_bwd_w_k(EdgeArgs<float> a, int RB, const float* __restrict__ phi, const float* __restrict__ v_in,
             const float* __restrict__ sb1, const float* __restrict__ vb1, const float* __restrict__ wt,
             const float* __restrict__ dt, float* __restrict__ phib, float* __restrict__ vb_in,
             float* __restrict__ fpart, int first_block) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int F = a.F;
  const int f0 = (blockIdx.y * 32 + lane) * FPL;
  const bool has_v = v_in != nullptr;
  const int64_t nchunk = (a.N + RB - 1) / RB;
  for (int64_t ch = blockIdx.x; ch < nchunk; ch += gridDim.x) {
    const int64_t i_end = min((int64_t)(ch + 1) * RB, a.N);
    for (int64_t i = ch * RB + warp; i < i_end; i += NWARP) {
      const int ea = a.rowptr[i], eb = a.rowptr[i + 1];
      const int64_t io = i * 3 * F + f0;
      // the receiver's own rows
      float li0[FPL], li[3][FPL], lph[3][FPL], lv[3][FPL];
      ldv<FPL>(sb1 + i * F + f0, li0);
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        ldv<FPL>(vb1 + io + c * F, li[c]);
        ldv<FPL>(phi + io + c * F, lph[c]);
        if (has_v) ldv<FPL>(v_in + io + c * F, lv[c]);
        else {
#pragma unroll
          for (int p = 0; p < FPL; ++p) lv[c][p] = 0.f;
        }
      }
      float A0[FPL], A1[FPL], A2[3][FPL];
#pragma unroll
      for (int p = 0; p < FPL; ++p) { A0[p] = A1[p] = 0.f; A2[0][p] = A2[1][p] = A2[2][p] = 0.f; }
      float fp0 = 0.f, fp1 = 0.f, fp2 = 0.f;
      for (int e = ea; e < eb; ++e) {
        const int64_t j = __ldg(a.col + e);
        const float4 u = __ldg(reinterpret_cast<const float4*>(a.geom) + e);
        const int64_t jo = j * 3 * F + f0, eo = (int64_t)e * 3 * F + f0;
        float ph[3][FPL], bj[3][FPL], vj[3][FPL], sbj[FPL], wv[3][FPL], dw[3][FPL];
        ldv<FPL>(sb1 + j * F + f0, sbj);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          ldv<FPL>(phi + jo + c * F, ph[c]);
          ldv<FPL>(vb1 + jo + c * F, bj[c]);
          if (c < 2 || has_v) { ldv_stream<FPL>(wt + eo + c * F, wv[c]); ldv_stream<FPL>(dt + eo + c * F, dw[c]); }
          if (has_v) ldv<FPL>(v_in + jo + c * F, vj[c]);
        }
        float D = 0.f, B0 = 0.f, B1 = 0.f, B2 = 0.f;
#pragma unroll
        for (int p = 0; p < FPL; ++p) {
          // scalar chunk
          A0[p] = fmaf(sbj[p], wv[0][p], A0[p]);
          D = fmaf(fmaf(li0[p], ph[0][p], sbj[p] * lph[0][p]), dw[0][p], D);
          // direction chunk
          const float tj = bj[0][p] * u.x + bj[1][p] * u.y + bj[2][p] * u.z;
          const float ti = li[0][p] * u.x + li[1][p] * u.y + li[2][p] * u.z;
          A1[p] = fmaf(-tj, wv[1][p], A1[p]);
          D = fmaf(ti * ph[1][p] - tj * lph[1][p], dw[1][p], D);
          B0 = fmaf(li[0][p] * ph[1][p] - bj[0][p] * lph[1][p], wv[1][p], B0);
          B1 = fmaf(li[1][p] * ph[1][p] - bj[1][p] * lph[1][p], wv[1][p], B1);
          B2 = fmaf(li[2][p] * ph[1][p] - bj[2][p] * lph[1][p], wv[1][p], B2);
          // vector chunk
          if (has_v) {
            A2[0][p] = fmaf(bj[0][p], wv[2][p], A2[0][p]);
            A2[1][p] = fmaf(bj[1][p], wv[2][p], A2[1][p]);
            A2[2][p] = fmaf(bj[2][p], wv[2][p], A2[2][p]);
            const float liv = li[0][p] * vj[0][p] + li[1][p] * vj[1][p] + li[2][p] * vj[2][p];
            const float blv = bj[0][p] * lv[0][p] + bj[1][p] * lv[1][p] + bj[2][p] * lv[2][p];
            D = fmaf(liv * ph[2][p] + blv * lph[2][p], dw[2][p], D);
          }
        }
        const float Bu = B0 * u.x + B1 * u.y + B2 * u.z;
        const float invd = 1.0f / u.w;
        fp0 += D * u.x + (B0 - Bu * u.x) * invd;
        fp1 += D * u.y + (B1 - Bu * u.y) * invd;
        fp2 += D * u.z + (B2 - Bu * u.z) * invd;
      }
      if (phib != nullptr) {
        float o[FPL];
        stv<FPL>(phib + io, A0);
        stv<FPL>(phib + io + F, A1);
#pragma unroll
        for (int p = 0; p < FPL; ++p) o[p] = lv[0][p] * A2[0][p] + lv[1][p] * A2[1][p] + lv[2][p] * A2[2][p];
        stv<FPL>(phib + io + 2 * F, o);
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
#pragma unroll
          for (int p = 0; p < FPL; ++p) o[p] = li[ax][p] + lph[2][p] * A2[ax][p];
          stv<FPL>(vb_in + io + ax * F, o);
        }
      }
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

// The same reverse step for two features per lane with every product on packed FMAs (fma.rn.f32x2): the two features of a
// lane go through identical arithmetic, so each scalar FFMA / FMUL of edge_bwd_w_k<2> (130 per edge, half rate on sm_100)
// becomes half a packed instruction.  Differences are folded into constants negated once per receiver; the direction
// chunk's A1 is accumulated with the opposite sign and negated at the end.
__device__ __forceinline__ float2 ld2(const float* p) { return __ldg(reinterpret_cast<const float2*>(p)); }
__device__ __forceinline__ float2 ld2s(const float* p) { return __ldcs(reinterpret_cast<const float2*>(p)); }
__device__ __forceinline__ float2 sp2(float x) { return make_float2(x, x); }
__device__ __forceinline__ void prefetch_l2(const float* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

template <int NWARP>
__global__ void __launch_bounds__(NWARP * 32)
edge_bwd_w2_k(EdgeArgs<float> a, int RB, const float* __restrict__ phi, const float* __restrict__ v_in,
              const float* __restrict__ sb1, const float* __restrict__ vb1, const float* __restrict__ wt,
              const float* __restrict__ dt, float* __restrict__ phib, float* __restrict__ vb_in,
              float* __restrict__ fpart, int first_block) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int F = a.F;
  const int f0 = (blockIdx.y * 32 + lane) * 2;
  const bool has_v = v_in != nullptr;
  const float2 z2 = make_float2(0.f, 0.f);
  const int64_t nchunk = (a.N + RB - 1) / RB;
  for (int64_t ch = blockIdx.x; ch < nchunk; ch += gridDim.x) {
    const int64_t i_end = min((int64_t)(ch + 1) * RB, a.N);
    for (int64_t i = ch * RB + warp; i < i_end; i += NWARP) {
      const int ea = a.rowptr[i], eb = a.rowptr[i + 1];
      const int64_t io = i * 3 * F + f0;
      // the receiver's own rows
      const float2 li0 = ld2(sb1 + i * F + f0);
      float2 li[3], lph[3], lv[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        li[c] = ld2(vb1 + io + c * F);
        lph[c] = ld2(phi + io + c * F);
        lv[c] = has_v ? ld2(v_in + io + c * F) : z2;
      }
      // The tape rows of the receiver's first PFN edges ([e][3 chunks][this slab's 256 bytes] of wt and of dt, two lines of
      // 128 bytes each) are asked into L2 up front, one (edge, chunk) row per lane and round: one edge's loads in flight per
      // warp do not cover the DRAM latency of this stream.
      constexpr int PFN = 21; // 63 rows: two rounds
      for (int r = lane; r < min(eb - ea, PFN) * 3; r += 32) {
        const int64_t off = ((int64_t)ea * 3 + r) * F + blockIdx.y * 64;
        prefetch_l2(wt + off); prefetch_l2(wt + off + 32); prefetch_l2(dt + off); prefetch_l2(dt + off + 32);
      }
      const float2 nlph1 = make_float2(-lph[1].x, -lph[1].y);
      float2 A0 = z2, A1n = z2, A2[3] = {z2, z2, z2};
      float fp0 = 0.f, fp1 = 0.f, fp2 = 0.f;
      for (int e = ea; e < eb; ++e) {
        const int64_t j = __ldg(a.col + e);
        const float4 u = __ldg(reinterpret_cast<const float4*>(a.geom) + e);
        const int64_t jo = j * 3 * F + f0, eo = (int64_t)e * 3 * F + f0;
        float2 ph[3], bj[3], vj[3], wv[3], dw[3];
        const float2 sbj = ld2(sb1 + j * F + f0);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          ph[c] = ld2(phi + jo + c * F);
          bj[c] = ld2(vb1 + jo + c * F);
          if (c < 2 || has_v) { wv[c] = ld2s(wt + eo + c * F); dw[c] = ld2s(dt + eo + c * F); }
          if (has_v) vj[c] = ld2(v_in + jo + c * F);
        }
        const float2 ux = sp2(u.x), uy = sp2(u.y), uz = sp2(u.z);
        // scalar chunk
        A0 = __ffma2_rn(sbj, wv[0], A0);
        float2 D = __fmul2_rn(__ffma2_rn(li0, ph[0], __fmul2_rn(sbj, lph[0])), dw[0]);
        // direction chunk
        const float2 tj = __ffma2_rn(bj[2], uz, __ffma2_rn(bj[1], uy, __fmul2_rn(bj[0], ux)));
        const float2 ti = __ffma2_rn(li[2], uz, __ffma2_rn(li[1], uy, __fmul2_rn(li[0], ux)));
        A1n = __ffma2_rn(tj, wv[1], A1n);
        D = __ffma2_rn(__ffma2_rn(ti, ph[1], __fmul2_rn(tj, nlph1)), dw[1], D);
        const float2 B0 = __fmul2_rn(__ffma2_rn(li[0], ph[1], __fmul2_rn(bj[0], nlph1)), wv[1]);
        const float2 B1 = __fmul2_rn(__ffma2_rn(li[1], ph[1], __fmul2_rn(bj[1], nlph1)), wv[1]);
        const float2 B2 = __fmul2_rn(__ffma2_rn(li[2], ph[1], __fmul2_rn(bj[2], nlph1)), wv[1]);
        // vector chunk
        if (has_v) {
          A2[0] = __ffma2_rn(bj[0], wv[2], A2[0]);
          A2[1] = __ffma2_rn(bj[1], wv[2], A2[1]);
          A2[2] = __ffma2_rn(bj[2], wv[2], A2[2]);
          const float2 liv = __ffma2_rn(li[2], vj[2], __ffma2_rn(li[1], vj[1], __fmul2_rn(li[0], vj[0])));
          const float2 blv = __ffma2_rn(bj[2], lv[2], __ffma2_rn(bj[1], lv[1], __fmul2_rn(bj[0], lv[0])));
          D = __ffma2_rn(__ffma2_rn(liv, ph[2], __fmul2_rn(blv, lph[2])), dw[2], D);
        }
        const float Ds = D.x + D.y, b0 = B0.x + B0.y, b1 = B1.x + B1.y, b2 = B2.x + B2.y;
        const float Bu = b0 * u.x + b1 * u.y + b2 * u.z;
        const float invd = 1.0f / u.w;
        fp0 += Ds * u.x + (b0 - Bu * u.x) * invd;
        fp1 += Ds * u.y + (b1 - Bu * u.y) * invd;
        fp2 += Ds * u.z + (b2 - Bu * u.z) * invd;
      }
      if (phib != nullptr) {
        *reinterpret_cast<float2*>(phib + io) = A0;
        *reinterpret_cast<float2*>(phib + io + F) = make_float2(-A1n.x, -A1n.y);
        *reinterpret_cast<float2*>(phib + io + 2 * F) =
            __ffma2_rn(lv[2], A2[2], __ffma2_rn(lv[1], A2[1], __fmul2_rn(lv[0], A2[0])));
#pragma unroll
        for (int ax = 0; ax < 3; ++ax)
          *reinterpret_cast<float2*>(vb_in + io + ax * F) = __ffma2_rn(lph[2], A2[ax], li[ax]);
      }
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

} // namespace

// FPL = 2 needs 6 K-long filter rows per lane in registers: used up to K = 20.
static int pick_fpl(int F, int K) { return (K <= 20 && F % 64 == 0) ? 2 : 1; }
static int pick_kp4(int K) { return K <= 8 ? 8 : K <= 12 ? 12 : K <= 16 ? 16 : K <= 20 ? 20 : K <= 24 ? 24 : K <= 28 ? 28 : 32; }

// The reverse kernel holds no filter rows: its lane width is chosen on its own (the tape layout [E][3][F] is lane-agnostic).
// Two features (8-byte loads) per lane whenever F allows: cfg3 (F = 256, K = 32) 1.00 -> 0.76 ms against one feature.
static int pick_fpl_bwd(int F) { return F % 64 == 0 ? 2 : 1; }

int edge_warp_num_slabs(int F, int K) { (void)K; return F / (32 * pick_fpl_bwd(F)); }

int launch_edge_fwd_warp(const EdgeArgs<float>& a, const float* phi, const float* s_in, int64_t ld_sin, const float* v_in,
                         float* s1, int64_t ld_s1, float* v1, float* wt, float* dt, cudaStream_t st) {
  if (a.N == 0) return 0;
  const int FPL = pick_fpl(a.F, a.K), KP = pick_kp4(a.K);
  constexpr int NW = 4;
  const int RB = NW;   // one receiver per warp and chunk: finest grain for the grid-stride loop (16 measured 3 % slower)
  const int64_t nchunk = (a.N + RB - 1) / RB;
  // Persistent grid: a whole number of waves of resident CTAs (2 or 3 per SM by registers), shared out over the feature
  // slabs — every extra CTA reloads its 3*FPL filter rows, and a partial wave leaves SMs idle.  Measured on B200, edge_fwd:
  // cfg2 (F 128, K 20, 2 slabs) 148 x 2 CTAs 200 us, 111 x 2 255 us, 296 x 2 207 us, 592 x 2 220 us;
  // cfg3 (F 256, K 32, 8 slabs) 37 x 8 CTAs 2.19 ms, 74 x 8 2.01 ms, 111 x 8 2.08 ms, 148 x 8 2.05 ms, 592 x 8 2.19 ms.
  const int nslab = a.F / (32 * FPL), occ = (FPL == 1 && KP <= 24) ? 3 : 2, waves = FPL == 2 ? 1 : 2;
  dim3 grid((unsigned)std::min<int64_t>(nchunk, std::max(1, 148 * occ * waves / nslab)), nslab);
#define PNN_L(KPV, FPLV)                                                                                              \
  {                                                                                                                   \
    if (wt) edge_fwd_w_k<KPV, FPLV, NW, true><<<grid, NW * 32, 0, st>>>(a, RB, phi, s_in, ld_sin, v_in, s1, ld_s1, v1, wt, dt); \
    else edge_fwd_w_k<KPV, FPLV, NW, false><<<grid, NW * 32, 0, st>>>(a, RB, phi, s_in, ld_sin, v_in, s1, ld_s1, v1, wt, dt);   \
  }
  if (FPL == 2) {
    switch (KP) {
      case 8: PNN_L(8, 2); break;
      case 12: PNN_L(12, 2); break;
      case 16: PNN_L(16, 2); break;
      default: PNN_L(20, 2); break;
    }
  } else {
    switch (KP) {
      case 8: PNN_L(8, 1); break;
      case 12: PNN_L(12, 1); break;
      case 16: PNN_L(16, 1); break;
      case 20: PNN_L(20, 1); break;
      case 24: PNN_L(24, 1); break;
      case 28: PNN_L(28, 1); break;
      default: PNN_L(32, 1); break;
    }
  }
#undef PNN_L
  PNN_KCHECK("edge_fwd_w_k");
  return 1;
}

int launch_edge_bwd_warp(const EdgeArgs<float>& a, const float* phi, const float* v_in, const float* sb1, const float* vb1,
                         const float* wt, const float* dt, float* phib, float* vb_in, float* fpart, int first_block,
                         cudaStream_t st) {
  if (a.N == 0) return 0;
  const int FPL = pick_fpl_bwd(a.F);
  constexpr int NW = 4;
  const int RB = NW;   // cfg2 0.160 -> 0.144 ms, cfg3 0.76 -> 0.73 ms against 16 receivers per chunk
  const int64_t nchunk = (a.N + RB - 1) / RB;
  dim3 grid((unsigned)std::min<int64_t>(nchunk, 148 * 16), a.F / (32 * FPL));
  if (FPL == 2)
    edge_bwd_w2_k<NW><<<grid, NW * 32, 0, st>>>(a, RB, phi, v_in, sb1, vb1, wt, dt, phib, vb_in, fpart, first_block);
  else
    edge_bwd_w_k<1, NW><<<grid, NW * 32, 0, st>>>(a, RB, phi, v_in, sb1, vb1, wt, dt, phib, vb_in, fpart, first_block);
  PNN_KCHECK("edge_bwd_w_k");
  return 1;
}

} // namespace pnn
