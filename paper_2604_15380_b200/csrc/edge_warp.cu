// edge_warp.cu — a4 / a7 edge kernels of the FP32 model, exact FP32 arithmetic on the ordinary ALUs.
//
// Same mathematics as edge.cu (sender scatters rewritten as gathers over the receiver's own
// CSR row), different mapping, chosen from the ncu stall profile of edge.cu (profiles/r01_edge_bwd_cfg2_fp32.md: gather
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
      const float dd = gq.d - (float)k * dmu;
      const float g = (k < a.K) ? expf(-gamma * dd * dd) : 0.0f;
      G1[lane * PG + k] = g * cc;
      if (BWD) G2[lane * PG + k] = (cc * (-2.0f * gamma * dd) + cp) * g;
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
template <int KP, int FPL, int NWARP>
__global__ void __launch_bounds__(NWARP * 32, FPL == 1 ? 3 : 2)
edge_fwd_w_k(EdgeArgs<float> a, int RB, const float* __restrict__ phi, const float* __restrict__ s_in, int64_t ld_sin,
             const float* __restrict__ v_in, float* __restrict__ s1, int64_t ld_s1, float* __restrict__ v1) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  constexpr int PG = KP + 4;
  __shared__ __align__(16) float G1s[NWARP][TW * PG];
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
        stage_tile_w<KP, false>(a, lane, t0, nE, G1, nullptr, U, C, J, dmu, gamma, pi_rc);
        // software pipeline: the sender rows of edge q+1 are requested before edge q is consumed
        float ph[3][FPL], vj[3][FPL], phn[3][FPL], vjn[3][FPL];
        auto gather = [&](int q, float (&p_)[3][FPL], float (&v_)[3][FPL]) {
          const int64_t jo = (int64_t)J[q] * 3 * F + f0;
#pragma unroll
          for (int c = 0; c < 3; ++c) ldv<FPL>(phi + jo + c * F, p_[c]);
          if (has_v) {
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) ldv<FPL>(v_in + jo + ax * F, v_[ax]);
          }
        };
        gather(0, phn, vjn);
        for (int q = 0; q < nE; ++q) {
#pragma unroll
          for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int p = 0; p < FPL; ++p) { ph[c][p] = phn[c][p]; vj[c][p] = vjn[c][p]; }
          if (q + 1 < nE) gather(q + 1, phn, vjn);
          const float4 u = U[q];
          const float cc = C[q].x;
          const float* g = G1 + q * PG;
#pragma unroll
          for (int p = 0; p < FPL; ++p) {
            const float w0 = dot_pairs<KP>(w[0][p], g, bias[0][p] * cc);
            const float w1 = dot_pairs<KP>(w[1][p], g, bias[1][p] * cc);
            as[p] = fmaf(ph[0][p], w0, as[p]);
            const float x1 = ph[1][p] * w1;
            av[0][p] = fmaf(x1, u.x, av[0][p]); av[1][p] = fmaf(x1, u.y, av[1][p]); av[2][p] = fmaf(x1, u.z, av[2][p]);
            if (has_v) {
              const float w2 = dot_pairs<KP>(w[2][p], g, bias[2][p] * cc);
              const float x2 = ph[2][p] * w2;
              av[0][p] = fmaf(x2, vj[0][p], av[0][p]); av[1][p] = fmaf(x2, vj[1][p], av[1][p]);
              av[2][p] = fmaf(x2, vj[2][p], av[2][p]);
            }
          }
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

} // namespace

// FPL = 2 needs 6 K-long filter rows per lane in registers: used up to K = 20.
static int pick_fpl(int F, int K) { return (K <= 20 && F % 64 == 0) ? 2 : 1; }
static int pick_kp4(int K) { return K <= 8 ? 8 : K <= 12 ? 12 : K <= 16 ? 16 : K <= 20 ? 20 : K <= 24 ? 24 : K <= 28 ? 28 : 32; }

int edge_warp_num_slabs(int F, int K) { return F / (32 * pick_fpl(F, K)); }

int launch_edge_fwd_warp(const EdgeArgs<float>& a, const float* phi, const float* s_in, int64_t ld_sin, const float* v_in,
                         float* s1, int64_t ld_s1, float* v1, cudaStream_t st) {
  if (a.N == 0) return 0;
  const int FPL = pick_fpl(a.F, a.K), KP = pick_kp4(a.K);
  constexpr int NW = 4;
  const int RB = 16;
  const int64_t nchunk = (a.N + RB - 1) / RB;
  dim3 grid((unsigned)std::min<int64_t>(nchunk, 148 * 4), a.F / (32 * FPL));
#define PNN_L(KPV, FPLV) edge_fwd_w_k<KPV, FPLV, NW><<<grid, NW * 32, 0, st>>>(a, RB, phi, s_in, ld_sin, v_in, s1, ld_s1, v1)
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

} // namespace pnn
