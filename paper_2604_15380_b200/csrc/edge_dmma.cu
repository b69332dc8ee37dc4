// edge_dmma.cu — FP64 edge/message kernels with the filter contraction on the FP64 tensor cores (DMMA, mma.sync m8n8k4).
//
// Same arithmetic as edge.cu (SURVEY.md §8(c) B3 forward, R3 / R4 reverse; no atomics, sender scatters as gathers over the
// node's own row), other mapping.  In edge.cu a thread owns one filter row and spends K DFMAs and K/2 broadcast shared loads
// per edge on w_e = flt_W g(d_e) c(d_e): issue slots and the shared-memory pipe bind at 23 % of the FP64 pipe (cfg5).  Here
// the contraction of a tile of 8 edges x 8 features x 4 radial functions is ONE warp instruction (512 flop, same FP64 rate
// as 8 DFMA warp instructions: measured 37.1 TFLOP/s for either on B200):
//   D[edge][feature] (8 x 8) += A[edge][k] (8 x 4, the staged radial basis x cutoff) . B[k][feature] (4 x 8, filter rows)
// with the filter fragments resident in registers for the CTA's lifetime (K/4 x blocks doubles per lane, as many as a thread
// of edge.cu holds) and A read from shared memory once per warp and k-step.  D arrives as (edge row = lane / 4, two
// features per lane): each lane multiplies by its gathered sender payload, keeps the receiver's partial sums for its row in
// registers and the eight rows meet by three shuffles when the receiver ends.
//
// CTA = 12 warps on one 64-feature slab and RB consecutive receivers: warps 0-3 the scalar chunk (ss) of 16 features each,
// warps 4-11 the two vector chunks (vs, vv) of 8 features each, so that v' = v + sum (x^vs u + x^vv v_j) is finished in one
// warp.  A pass = the next <= 64 edges of ONE receiver in tiles of 8 (rows past the end carry cutoff 0, i.e. weight 0, and
// gather a valid row).  Used by the FP64 model whenever F is a multiple of 64.
#include <algorithm>
#include <type_traits>

#include "common.cuh"

namespace pnn {

namespace {

constexpr int DT = 8;        // edges per tile (M of the DMMA)
constexpr int DPASS = 64;    // edges per pass
constexpr int DFS = 64;      // features per CTA
constexpr int DTHR = 384;
constexpr int GPAD = 4;      // doubles of padding per staged row: rows 8 banks apart, A-fragment loads conflict-free

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__device__ __forceinline__ double2 ldg2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }

// 16-byte asynchronous global -> shared copies (LDGSTS): the gathers of the next tile land in the warp's shared-memory slots
// while the tensor cores work on the current one, without holding registers
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const uint32_t s_ = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s_), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
constexpr int GSLOTS = 8; // gather slots (16 bytes per lane each) per tile and warp, reverse kernel
constexpr int FSLOTS = 5; // ... forward kernel

// --------------------------------------------------------------------------------------------------- forward
// Staged pass (double-buffered): G = radial basis WITHOUT the cutoff (the epilogue multiplies by c(d): w = c (D + b)), so
// that staging G needs d only and runs in the same phase as staging u, c, j — one CTA barrier per pass.
template <int KS> // k-steps of 4 radial functions (K <= 4 KS)
__global__ void __launch_bounds__(DTHR)
edge_fwd_dmma_k(EdgeArgs<double> a, int RB, const double* __restrict__ phi, const double* __restrict__ s_in, int64_t ld_sin,
                const double* __restrict__ v_in, const double* __restrict__ v_res, double* __restrict__ s1, int64_t ld_s1,
                double* __restrict__ v1) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  constexpr int KP = 4 * KS, LD = KP + GPAD;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double (*const Gs)[DPASS * LD] = reinterpret_cast<double (*)[DPASS * LD]>(smem_raw);                 // [2] radial basis (no cutoff)
  double (*const Us)[DPASS * 4] = reinterpret_cast<double (*)[DPASS * 4]>(smem_raw + sizeof(double) * 2 * DPASS * LD); // [2] ux uy uz c(d)
  int (*const Js)[DPASS] = reinterpret_cast<int (*)[DPASS]>(smem_raw + sizeof(double) * 2 * DPASS * (LD + 4));       // [2]
  double2* const GS = reinterpret_cast<double2*>(smem_raw + sizeof(double) * 2 * DPASS * (LD + 4) + sizeof(int) * 2 * DPASS); // gathers
  const int F = a.F, K = a.K;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int row = lane >> 2, cp = lane & 3;
  const bool ss = warp < 4;
  const int f0 = blockIdx.y * DFS + (ss ? 16 * warp : 8 * (warp - 4)); // first feature of the warp
  // filter fragments: B[k][n] of block (x, ks): lane holds filter row (chunk, f0 + 8 x' + lane / 4), column 4 ks + lane % 4
  double wf[2][KS], bias[2][2];
#pragma unroll
  for (int x = 0; x < 2; ++x) {
    const int frow = ss ? (f0 + 8 * x + row) : ((1 + x) * F + f0 + row);
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      const int k = 4 * ks + cp;
      wf[x][ks] = (k < K) ? a.fltW[(int64_t)frow * K + k] : 0.0;
    }
    const int brow = ss ? (f0 + 8 * x + 2 * cp) : ((1 + x) * F + f0 + 2 * cp); // bias of the lane's two OUTPUT features
    bias[x][0] = a.fltb[brow]; bias[x][1] = a.fltb[brow + 1];
  }
  const double rc = a.rc;
  const double dmu = (K > 1) ? rc / (double)(K - 1) : rc;
  const double gamma = 1.0 / (2.0 * dmu * dmu);
  const double pi_rc = 3.14159265358979323846 / a.rc;
  const bool has_v = v_in != nullptr;
  const int64_t nwork = (a.N + RB - 1) / RB;

  auto stage = [&](int bsel, int p0, int nE) {
    const int nT = (nE + DT - 1) / DT;
    if (tid < nT * DT) {
      const int e = p0 + min(tid, nE - 1); // rows past the end: a valid sender, cutoff 0
      const Geom<double> gq = a.geom[e];
      double sn, cs;
      sincos(pi_rc * gq.d, &sn, &cs);
      Us[bsel][tid * 4 + 0] = gq.ux; Us[bsel][tid * 4 + 1] = gq.uy; Us[bsel][tid * 4 + 2] = gq.uz;
      Us[bsel][tid * 4 + 3] = (tid < nE) ? 0.5 * (cs + 1.0) : 0.0;
      Js[bsel][tid] = a.col[e];
    }
    for (int q = tid; q < nT * DT * KP; q += DTHR) {
      const int e = q / KP, k = q - e * KP;
      double g = 0.0, gd = 0.0;
      if (k < K && e < nE) rbf_eval<double>(a.rbf, k, a.geom[p0 + e].d, rc, dmu, gamma, g, gd);
      Gs[bsel][e * LD + k] = g;
    }
  };
  // writes the receiver's row: residual + sums (lanes of row 0 hold the sums after the shuffles)
  auto write_row = [&](int64_t i, const double (&acc)[3][2][2]) {
    if (row != 0) return;
    if (ss) {
#pragma unroll
      for (int x = 0; x < 2; ++x) {
        const int f = f0 + 8 * x + 2 * cp;
        const double2 r = *reinterpret_cast<const double2*>(s_in + i * ld_sin + f);
        *reinterpret_cast<double2*>(s1 + i * ld_s1 + f) = make_double2(r.x + acc[0][x][0], r.y + acc[0][x][1]);
      }
    } else {
      const int f = f0 + 2 * cp;
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        double2 r = make_double2(0.0, 0.0);
        if (v_res) r = *reinterpret_cast<const double2*>(v_res + (i * 3 + q) * F + f);
        *reinterpret_cast<double2*>(v1 + (i * 3 + q) * F + f) = make_double2(r.x + acc[q][0][0], r.y + acc[q][0][1]);
      }
    }
  };

  for (int64_t wk = blockIdx.x; wk < nwork; wk += gridDim.x) {
    const int64_t i1 = min(wk * RB + RB, a.N);
    double acc[3][2][2]; // ss warps: acc[0][x][h]; vector warps: acc[component][0][h]
    auto zero_acc = [&]() {
#pragma unroll
      for (int q = 0; q < 3; ++q)
#pragma unroll
        for (int x = 0; x < 2; ++x) { acc[q][x][0] = 0.0; acc[q][x][1] = 0.0; }
    };
    zero_acc();
    const double zero3[3][2][2] = {};
    // the pass sequence of this work item: (receiver i, first edge p0, end of row eb); receivers without edges are
    // written on the way
    int64_t i = wk * RB;
    int p0 = 0, eb = 0;
    auto find_pass = [&](int64_t ii, int& p0_, int& eb_) { // first receiver >= ii with edges; rows without edges = residual
      while (ii < i1) {
        const int ea_ = __ldg(a.rowptr + ii), e1_ = __ldg(a.rowptr + ii + 1);
        if (e1_ > ea_) { p0_ = ea_; eb_ = e1_; break; }
        write_row(ii, zero3);
        ++ii;
      }
      return ii;
    };
    i = find_pass(i, p0, eb);
    int cur = 0;
    __syncthreads(); // the buffers of the previous work item have been consumed
    if (i < i1) stage(0, p0, min(DPASS, eb - p0));
    __syncthreads();
    while (i < i1) {
      const int nE = min(DPASS, eb - p0), nT = (nE + DT - 1) / DT;
      const bool last = p0 + DPASS >= eb;
      // the next pass, staged into the other buffer while this one is consumed
      int64_t ni = i;
      int np0 = p0 + DPASS, neb = eb;
      const int64_t this_i = i;
      // Gathers of tile t + 1 travel as asynchronous copies into the warp's shared-memory slots and its DMMAs are issued
      // in the same basic block as the epilogue of tile t (independent instruction streams the scheduler can interleave:
      // the tensor pipe is then fed while the FP64 ALUs finish the previous tile).
      auto consume = [&](auto ss_c, auto hv_c) {
      constexpr bool SS_ = decltype(ss_c)::value, HV_ = decltype(hv_c)::value;
      double2* const gsw = GS + (warp * 2 * FSLOTS) * 32 + lane;
      auto issue = [&](int t) {
        const int64_t j = Js[cur][t * DT + row];
        const double* pj = phi + j * 3 * F + f0 + 2 * cp;
        double2* dst = gsw + (t & 1) * FSLOTS * 32;
        if (SS_) { cp_async16(dst, pj); cp_async16(dst + 32, pj + 8); }
        else {
          cp_async16(dst, pj + F);
          if (HV_) {
            cp_async16(dst + 32, pj + 2 * F);
            const double* vp = v_in + j * 3 * F + f0 + 2 * cp;
            cp_async16(dst + 64, vp); cp_async16(dst + 96, vp + F); cp_async16(dst + 128, vp + 2 * F);
          }
        }
        cp_async_commit();
      };
      auto mma = [&](int t, double (&d)[2][2]) {
        const double* Ar = &Gs[cur][(t * DT + row) * LD + cp];
        d[0][0] = d[0][1] = d[1][0] = d[1][1] = 0.0;
        if (SS_ || HV_) {
#pragma unroll
          for (int ks = 0; ks < KS; ++ks) {
            const double av = Ar[4 * ks];
            dmma884(d[0][0], d[0][1], av, wf[0][ks]);
            dmma884(d[1][0], d[1][1], av, wf[1][ks]);
          }
        } else {
#pragma unroll
          for (int ks = 0; ks < KS; ++ks) dmma884(d[0][0], d[0][1], Ar[4 * ks], wf[0][ks]);
        }
      };
      auto epi = [&](int t, const double (&d)[2][2]) {
        const int slot = t * DT + row;
        const double4 uc = *reinterpret_cast<const double4*>(&Us[cur][slot * 4]); // ux uy uz c
        const double2* src = gsw + (t & 1) * FSLOTS * 32;
        const double w00 = uc.w * (d[0][0] + bias[0][0]), w01 = uc.w * (d[0][1] + bias[0][1]);
        const double w10 = uc.w * (d[1][0] + bias[1][0]), w11 = uc.w * (d[1][1] + bias[1][1]);
        const double2 pa = src[0];
        if (SS_) {
          const double2 pb = src[32];
          acc[0][0][0] = fma(pa.x, w00, acc[0][0][0]); acc[0][0][1] = fma(pa.y, w01, acc[0][0][1]);
          acc[0][1][0] = fma(pb.x, w10, acc[0][1][0]); acc[0][1][1] = fma(pb.y, w11, acc[0][1][1]);
        } else {
          const double xs0 = pa.x * w00, xs1 = pa.y * w01;
          acc[0][0][0] = fma(xs0, uc.x, acc[0][0][0]); acc[0][0][1] = fma(xs1, uc.x, acc[0][0][1]);
          acc[1][0][0] = fma(xs0, uc.y, acc[1][0][0]); acc[1][0][1] = fma(xs1, uc.y, acc[1][0][1]);
          acc[2][0][0] = fma(xs0, uc.z, acc[2][0][0]); acc[2][0][1] = fma(xs1, uc.z, acc[2][0][1]);
          if (HV_) {
            const double2 pb = src[32], v0 = src[64], v1_ = src[96], v2 = src[128];
            const double xv0 = pb.x * w10, xv1 = pb.y * w11;
            acc[0][0][0] = fma(xv0, v0.x, acc[0][0][0]);  acc[0][0][1] = fma(xv1, v0.y, acc[0][0][1]);
            acc[1][0][0] = fma(xv0, v1_.x, acc[1][0][0]); acc[1][0][1] = fma(xv1, v1_.y, acc[1][0][1]);
            acc[2][0][0] = fma(xv0, v2.x, acc[2][0][0]);  acc[2][0][1] = fma(xv1, v2.y, acc[2][0][1]);
          }
        }
      };
      issue(0);
      // stage the next pass into the other buffer behind the first tile's gathers
      if (last) ni = find_pass(i + 1, np0, neb);
      if (ni < i1) stage(cur ^ 1, np0, min(DPASS, neb - np0));
      double dA[2][2], dB[2][2];
      mma(0, dA);
      for (int t = 0;;) { // DMMAs of tile t + 1 and epilogue of tile t in ONE basic block (two register sets, unrolled by two)
        if (t + 1 >= nT) { cp_async_wait<0>(); epi(t, dA); break; }
        issue(t + 1); cp_async_wait<1>(); mma(t + 1, dB); epi(t, dA);
        ++t;
        if (t + 1 >= nT) { cp_async_wait<0>(); epi(t, dB); break; }
        issue(t + 1); cp_async_wait<1>(); mma(t + 1, dA); epi(t, dB);
        ++t;
      }
      };
      if (ss) consume(std::true_type(), std::true_type());
      else if (has_v) consume(std::false_type(), std::true_type());
      else consume(std::false_type(), std::false_type());
      if (last) { // the eight edge rows of the warp meet; lanes 0-3 (row 0) write the receiver's row
#pragma unroll
        for (int q = 0; q < 3; ++q)
#pragma unroll
          for (int x = 0; x < 2; ++x)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              if ((ss && q > 0) || (!ss && x > 0)) continue;
              double tt = acc[q][x][h];
              tt += __shfl_xor_sync(0xffffffffu, tt, 4);
              tt += __shfl_xor_sync(0xffffffffu, tt, 8);
              tt += __shfl_xor_sync(0xffffffffu, tt, 16);
              acc[q][x][h] = tt;
            }
        write_row(this_i, acc);
        zero_acc();
      }
      i = ni; p0 = np0; eb = neb;
      cur ^= 1;
      __syncthreads();
    }
  }
}

// --------------------------------------------------------------------------------------------------- reverse
// R3 + R4 in gather form (edge.cu has the derivation): for node i and each of its CSR edges (i <- j), with the filter value
// w = c (D1 + b) and its derivative dw/dd = c D2 + c' (D1 + b), D1 = flt_W g, D2 = flt_W g' from the tensor cores (two staged
// tiles: g and g').  Same warp roles and pass structure as the forward kernel.  Per lane and tile the force terms of its
// features are summed BEFORE they are multiplied by the edge's direction (they share it).  Force partials of the 12 warps
// meet in shared memory (FW, double-buffered by receiver parity) and are added by three threads after the pass barrier.
template <int KS>
__global__ void __launch_bounds__(DTHR)
edge_bwd_dmma_k(EdgeArgs<double> a, int RB, const double* __restrict__ phi, const double* __restrict__ v_in,
                const double* __restrict__ sb1, const double* __restrict__ vb1, double* __restrict__ phib,
                double* __restrict__ vb_in, double* __restrict__ fpart, int first_block) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  constexpr int KP = 4 * KS, LD = KP + GPAD;
  constexpr int BUF_D = 2 * DPASS * LD + DPASS * 4 + DPASS * 2; // doubles per buffer: G1 | G2 | U | V
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* const sm = reinterpret_cast<double*>(smem_raw);
  double* const FW = sm + 2 * BUF_D;                               // [2][12][3]
  int* const Jb = reinterpret_cast<int*>(FW + 2 * 12 * 3);         // [2][DPASS]
  double2* const GS = reinterpret_cast<double2*>(Jb + 2 * DPASS);  // [12 warps][2 stages][GSLOTS][32 lanes]
  auto G1 = [&](int b) { return sm + b * BUF_D; };
  auto G2 = [&](int b) { return sm + b * BUF_D + DPASS * LD; };
  auto Ub = [&](int b) { return sm + b * BUF_D + 2 * DPASS * LD; };              // ux uy uz c
  auto Vb = [&](int b) { return sm + b * BUF_D + 2 * DPASS * LD + DPASS * 4; };  // c' 1/d
  const int F = a.F, K = a.K;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int row = lane >> 2, cp = lane & 3;
  const bool ss = warp < 4;
  const int f0 = blockIdx.y * DFS + (ss ? 16 * warp : 8 * (warp - 4));
  double wf[2][KS], bias[2][2];
#pragma unroll
  for (int x = 0; x < 2; ++x) {
    const int frow = ss ? (f0 + 8 * x + row) : ((1 + x) * F + f0 + row);
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      const int k = 4 * ks + cp;
      wf[x][ks] = (k < K) ? a.fltW[(int64_t)frow * K + k] : 0.0;
    }
    const int brow = ss ? (f0 + 8 * x + 2 * cp) : ((1 + x) * F + f0 + 2 * cp);
    bias[x][0] = a.fltb[brow]; bias[x][1] = a.fltb[brow + 1];
  }
  const double rc = a.rc;
  const double dmu = (K > 1) ? rc / (double)(K - 1) : rc;
  const double gamma = 1.0 / (2.0 * dmu * dmu);
  const double pi_rc = 3.14159265358979323846 / a.rc;
  const bool has_v = v_in != nullptr, has_out = phib != nullptr;
  const int64_t nwork = (a.N + RB - 1) / RB;
  const int fo = ss ? f0 + 2 * cp : f0 + 2 * cp; // the lane's first feature (ss: block x adds 8)

  auto stage = [&](int b, int p0, int nE) {
    const int nT = (nE + DT - 1) / DT;
    if (tid < nT * DT) {
      const int e = p0 + min(tid, nE - 1);
      const Geom<double> gq = a.geom[e];
      double sn, cs;
      sincos(pi_rc * gq.d, &sn, &cs);
      const bool ok = tid < nE;
      double* u = Ub(b) + tid * 4;
      u[0] = gq.ux; u[1] = gq.uy; u[2] = gq.uz; u[3] = ok ? 0.5 * (cs + 1.0) : 0.0;
      Vb(b)[tid * 2 + 0] = ok ? -0.5 * pi_rc * sn : 0.0;
      Vb(b)[tid * 2 + 1] = 1.0 / gq.d;
      Jb[b * DPASS + tid] = a.col[e];
    }
    for (int q = tid; q < nT * DT * KP; q += DTHR) {
      const int e = q / KP, k = q - e * KP;
      double g = 0.0, gd = 0.0;
      if (k < K && e < nE) rbf_eval<double>(a.rbf, k, a.geom[p0 + e].d, rc, dmu, gamma, g, gd);
      G1(b)[e * LD + k] = g;
      G2(b)[e * LD + k] = gd;
    }
  };

  int fpar = 0; // FW buffer of the receiver being accumulated
  for (int64_t wk = blockIdx.x; wk < nwork; wk += gridDim.x) {
    const int64_t i1 = min(wk * RB + RB, a.N);
    // the lane's view of the receiver's own rows: ss: own[x][h] = sb1_i, ownp[x][h] = phi_i^ss; vector: li[a][h] = vb1_i,
    // lv[a][h] = v_i, ownp[0][h] = phi_i^vs, ownp[1][h] = phi_i^vv
    double li[3][2], lv[3][2], ownp[2][2];
    double acc[4][2], fp[3]; // ss: acc[x][h]; vector: acc[0][h] = vs, acc[1 + a][h] = vv
    auto zero_acc = [&]() {
#pragma unroll
      for (int q = 0; q < 4; ++q) { acc[q][0] = 0.0; acc[q][1] = 0.0; }
      fp[0] = fp[1] = fp[2] = 0.0;
    };
    auto load_own = [&](int64_t i) {
      if (ss) {
#pragma unroll
        for (int x = 0; x < 2; ++x) {
          const double2 sv = ldg2(sb1 + i * F + fo + 8 * x), pv = ldg2(phi + i * 3 * F + fo + 8 * x);
          li[x][0] = sv.x; li[x][1] = sv.y; ownp[x][0] = pv.x; ownp[x][1] = pv.y;
        }
      } else {
        const double2 p1 = ldg2(phi + i * 3 * F + F + fo), p2 = ldg2(phi + i * 3 * F + 2 * F + fo);
        ownp[0][0] = p1.x; ownp[0][1] = p1.y; ownp[1][0] = p2.x; ownp[1][1] = p2.y;
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          const double2 b = ldg2(vb1 + (i * 3 + q) * F + fo);
          li[q][0] = b.x; li[q][1] = b.y;
          double2 v = make_double2(0.0, 0.0);
          if (has_v) v = ldg2(v_in + (i * 3 + q) * F + fo);
          lv[q][0] = v.x; lv[q][1] = v.y;
        }
      }
    };
    // node adjoints of receiver i from the sums in acc (lanes of row 0 after the shuffles); own rows must be loaded
    auto write_out = [&](int64_t i) {
      if (!has_out || row != 0) return;
      if (ss) {
#pragma unroll
        for (int x = 0; x < 2; ++x)
          *reinterpret_cast<double2*>(phib + i * 3 * F + fo + 8 * x) = make_double2(acc[x][0], acc[x][1]);
      } else {
        *reinterpret_cast<double2*>(phib + i * 3 * F + F + fo) = make_double2(acc[0][0], acc[0][1]);
        double2 pv = make_double2(0.0, 0.0);
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          pv.x = fma(lv[q][0], acc[1 + q][0], pv.x); pv.y = fma(lv[q][1], acc[1 + q][1], pv.y);
          *reinterpret_cast<double2*>(vb_in + (i * 3 + q) * F + fo) =
              make_double2(fma(ownp[1][0], acc[1 + q][0], li[q][0]), fma(ownp[1][1], acc[1 + q][1], li[q][1]));
        }
        *reinterpret_cast<double2*>(phib + i * 3 * F + 2 * F + fo) = pv;
      }
    };
    auto write_force = [&](int64_t i, int par, bool zero) { // three threads add the warp partials of a finished receiver
      if (tid < 3) {
        double s_ = 0.0;
        if (!zero)
          for (int w = 0; w < 12; ++w) s_ += FW[(par * 12 + w) * 3 + tid];
        double* dst = fpart + ((int64_t)blockIdx.y * a.N + i) * 3 + tid;
        *dst = first_block ? s_ : (*dst + s_);
      }
    };
    zero_acc();
    int64_t i = wk * RB;
    int p0 = 0, eb = 0;
    auto find_pass = [&](int64_t ii, int& p0_, int& eb_) { // first receiver >= ii with edges; others get their plain rows
      while (ii < i1) {
        const int ea_ = __ldg(a.rowptr + ii), e1_ = __ldg(a.rowptr + ii + 1);
        if (e1_ > ea_) { p0_ = ea_; eb_ = e1_; break; }
        if (has_out && row == 0) {
          const double2 z = make_double2(0.0, 0.0);
          if (ss) {
            *reinterpret_cast<double2*>(phib + ii * 3 * F + fo) = z;
            *reinterpret_cast<double2*>(phib + ii * 3 * F + fo + 8) = z;
          } else {
            *reinterpret_cast<double2*>(phib + ii * 3 * F + F + fo) = z;
            *reinterpret_cast<double2*>(phib + ii * 3 * F + 2 * F + fo) = z;
            for (int q = 0; q < 3; ++q)
              *reinterpret_cast<double2*>(vb_in + (ii * 3 + q) * F + fo) = ldg2(vb1 + (ii * 3 + q) * F + fo);
          }
        }
        write_force(ii, 0, true);
        ++ii;
      }
      return ii;
    };
    i = find_pass(i, p0, eb);
    int cur = 0;
    __syncthreads();
    if (i < i1) { stage(0, p0, min(DPASS, eb - p0)); load_own(i); }
    __syncthreads();
    while (i < i1) {
      const int nE = min(DPASS, eb - p0), nT = (nE + DT - 1) / DT;
      const bool last = p0 + DPASS >= eb;
      int64_t ni = i;
      int np0 = p0 + DPASS, neb = eb;
      const int64_t this_i = i;
      const double* g1 = G1(cur); const double* g2 = G2(cur); const double* ub = Ub(cur); const double* vb = Vb(cur);
      const int* jb = Jb + cur * DPASS;
      double2* const gsw = GS + (warp * 2 * GSLOTS) * 32 + lane; // this lane's slots: [stage][slot] at stride 32
      auto issue = [&](int t) { // asynchronous gathers of tile t into stage t & 1
        const int64_t j = jb[t * DT + row];
        double2* dst = gsw + (t & 1) * GSLOTS * 32;
        if (ss) {
          cp_async16(dst, phi + j * 3 * F + fo);      cp_async16(dst + 32, phi + j * 3 * F + fo + 8);
          cp_async16(dst + 64, sb1 + j * F + fo);     cp_async16(dst + 96, sb1 + j * F + fo + 8);
        } else {
          cp_async16(dst, phi + j * 3 * F + F + fo);  cp_async16(dst + 32, phi + j * 3 * F + 2 * F + fo);
#pragma unroll
          for (int q = 0; q < 3; ++q) cp_async16(dst + (2 + q) * 32, vb1 + (j * 3 + q) * F + fo);
          if (has_v) {
#pragma unroll
            for (int q = 0; q < 3; ++q) cp_async16(dst + (5 + q) * 32, v_in + (j * 3 + q) * F + fo);
          }
        }
        cp_async_commit();
      };
      issue(0);
      // stage the next pass into the other buffer behind the first tile's gathers
      if (last) ni = find_pass(i + 1, np0, neb);
      if (ni < i1) stage(cur ^ 1, np0, min(DPASS, neb - np0));
      for (int t = 0; t < nT; ++t) {
        const int slot = t * DT + row;
        if (t + 1 < nT) { issue(t + 1); cp_async_wait<1>(); } else cp_async_wait<0>();
        const double2* src = gsw + (t & 1) * GSLOTS * 32;
        double2 gq[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) gq[q] = ((ss && q >= 4) || (!ss && !has_v && q >= 5)) ? make_double2(0.0, 0.0) : src[q * 32];
        const double4 uc = *reinterpret_cast<const double4*>(ub + slot * 4);
        const double2 cd = *reinterpret_cast<const double2*>(vb + slot * 2); // c', 1/d
        double d1[2][2] = {}, d2[2][2] = {};
        const double* A1 = g1 + slot * LD + cp;
        const double* A2 = g2 + slot * LD + cp;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
          const double a1 = A1[4 * ks], a2 = A2[4 * ks];
          dmma884(d1[0][0], d1[0][1], a1, wf[0][ks]);
          dmma884(d2[0][0], d2[0][1], a2, wf[0][ks]);
          dmma884(d1[1][0], d1[1][1], a1, wf[1][ks]);
          dmma884(d2[1][0], d2[1][1], a2, wf[1][ks]);
        }
        double wv[2][2], dw[2][2];
#pragma unroll
        for (int x = 0; x < 2; ++x)
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const double base = d1[x][h] + bias[x][h];
            wv[x][h] = uc.w * base;
            dw[x][h] = fma(uc.w, d2[x][h], cd.x * base);
          }
        if (ss) {
          double dps = 0.0;
#pragma unroll
          for (int x = 0; x < 2; ++x) {
            const double ph[2] = {gq[x].x, gq[x].y}, sj[2] = {gq[2 + x].x, gq[2 + x].y};
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              acc[x][h] = fma(sj[h], wv[x][h], acc[x][h]);
              dps = fma(fma(li[x][h], ph[h], sj[h] * ownp[x][h]), dw[x][h], dps);
            }
          }
          fp[0] = fma(dps, uc.x, fp[0]); fp[1] = fma(dps, uc.y, fp[1]); fp[2] = fma(dps, uc.z, fp[2]);
        } else {
          double dps = 0.0, bs[3] = {0.0, 0.0, 0.0};
          const double u[3] = {uc.x, uc.y, uc.z};
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const double p1 = h ? gq[0].y : gq[0].x, p2 = h ? gq[1].y : gq[1].x;
            double b[3], vj[3];
#pragma unroll
            for (int q = 0; q < 3; ++q) { b[q] = h ? gq[2 + q].y : gq[2 + q].x; vj[q] = has_v ? (h ? gq[5 + q].y : gq[5 + q].x) : 0.0; }
            const double tj = fma(b[0], u[0], fma(b[1], u[1], b[2] * u[2]));
            const double ti = fma(li[0][h], u[0], fma(li[1][h], u[1], li[2][h] * u[2]));
            acc[0][h] = fma(-tj, wv[0][h], acc[0][h]);
            dps = fma(fma(ti, p1, -tj * ownp[0][h]), dw[0][h], dps);
#pragma unroll
            for (int q = 0; q < 3; ++q) {
              bs[q] = fma(fma(li[q][h], p1, -b[q] * ownp[0][h]), wv[0][h], bs[q]);
              acc[1 + q][h] = fma(b[q], wv[1][h], acc[1 + q][h]);
            }
            if (has_v) {
              const double lvj = fma(li[0][h], vj[0], fma(li[1][h], vj[1], li[2][h] * vj[2]));
              const double blv = fma(b[0], lv[0][h], fma(b[1], lv[1][h], b[2] * lv[2][h]));
              dps = fma(fma(lvj, p2, blv * ownp[1][h]), dw[1][h], dps);
            }
          }
          const double bu = fma(bs[0], u[0], fma(bs[1], u[1], bs[2] * u[2]));
#pragma unroll
          for (int q = 0; q < 3; ++q) fp[q] += fma(dps, u[q], (bs[q] - bu * u[q]) * cd.y);
        }
      }
      if (last) {
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            if (ss && q > 1) continue;
            double tt = acc[q][h];
            tt += __shfl_xor_sync(0xffffffffu, tt, 4);
            tt += __shfl_xor_sync(0xffffffffu, tt, 8);
            tt += __shfl_xor_sync(0xffffffffu, tt, 16);
            acc[q][h] = tt;
          }
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          double tt = fp[q];
#pragma unroll
          for (int o = 16; o; o >>= 1) tt += __shfl_xor_sync(0xffffffffu, tt, o);
          if (lane == 0) FW[(fpar * 12 + warp) * 3 + q] = tt;
        }
        write_out(this_i);
        zero_acc();
        if (ni < i1) load_own(ni);
      }
      i = ni; p0 = np0; eb = neb;
      cur ^= 1;
      __syncthreads();
      if (last) { write_force(this_i, fpar, false); fpar ^= 1; }
    }
  }
}

} // namespace

bool edge_dmma_supported(int F, int K) { return F % DFS == 0 && K <= 32; }

int launch_edge_fwd_dmma(const EdgeArgs<double>& a, const double* phi, const double* s_in, int64_t ld_sin, const double* v_in,
                         const double* v_res, double* s1, int64_t ld_s1, double* v1, cudaStream_t st) {
  if (a.N == 0) return 0;
  const int RB = 16;
  const int64_t nwork = (a.N + RB - 1) / RB;
  dim3 grid((unsigned)std::min<int64_t>(nwork, 148), a.F / DFS); // one CTA per SM and slab at a time; swept: 148 x 1..8 within 1 %
  const int KS = (a.K + 3) / 4;
  const size_t smem = sizeof(double) * 2 * DPASS * (4 * KS + GPAD + 4) + sizeof(int) * 2 * DPASS + (size_t)12 * 2 * FSLOTS * 32 * 16;
#define PNN_LAUNCH_DF(KSV)                                                                                              \
  {                                                                                                                     \
    static bool attr_set = false;                                                                                       \
    if (!attr_set) {                                                                                                    \
      cudaFuncSetAttribute(edge_fwd_dmma_k<KSV>, cudaFuncAttributeMaxDynamicSharedMemorySize, 128 * 1024);              \
      attr_set = true;                                                                                                  \
    }                                                                                                                   \
    edge_fwd_dmma_k<KSV><<<grid, DTHR, smem, st>>>(a, RB, phi, s_in, ld_sin, v_in, v_res, s1, ld_s1, v1);               \
  }
  switch (KS) {
    case 1: PNN_LAUNCH_DF(1) break;
    case 2: PNN_LAUNCH_DF(2) break;
    case 3: PNN_LAUNCH_DF(3) break;
    case 4: PNN_LAUNCH_DF(4) break;
    case 5: PNN_LAUNCH_DF(5) break;
    case 6: PNN_LAUNCH_DF(6) break;
    case 7: PNN_LAUNCH_DF(7) break;
    default: PNN_LAUNCH_DF(8) break;
  }
#undef PNN_LAUNCH_DF
  PNN_KCHECK("edge_fwd_dmma_k");
  return 1;
}

int launch_edge_bwd_dmma(const EdgeArgs<double>& a, const double* phi, const double* v_in, const double* sb1,
                         const double* vb1, double* phib, double* vb_in, double* fpart, int first_block, cudaStream_t st) {
  if (a.N == 0) return 0;
  const int RB = 16;
  const int64_t nwork = (a.N + RB - 1) / RB;
  dim3 grid((unsigned)std::min<int64_t>(nwork, 148), a.F / DFS); // one CTA per SM and slab at a time; swept: 148 x 1..8 within 1 %
  const int KS = (a.K + 3) / 4, LD = 4 * KS + GPAD;
  const size_t smem = sizeof(double) * (2 * (2 * DPASS * LD + DPASS * 6) + 2 * 12 * 3) + sizeof(int) * 2 * DPASS +
                      (size_t)12 * 2 * GSLOTS * 32 * 16;
#define PNN_LAUNCH_DB(KSV)                                                                                              \
  {                                                                                                                     \
    static bool attr_set = false;                                                                                       \
    if (!attr_set) {                                                                                                    \
      cudaFuncSetAttribute(edge_bwd_dmma_k<KSV>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);              \
      attr_set = true;                                                                                                  \
    }                                                                                                                   \
    edge_bwd_dmma_k<KSV><<<grid, DTHR, smem, st>>>(a, RB, phi, v_in, sb1, vb1, phib, vb_in, fpart, first_block);        \
  }
  switch (KS) {
    case 1: PNN_LAUNCH_DB(1) break;
    case 2: PNN_LAUNCH_DB(2) break;
    case 3: PNN_LAUNCH_DB(3) break;
    case 4: PNN_LAUNCH_DB(4) break;
    case 5: PNN_LAUNCH_DB(5) break;
    case 6: PNN_LAUNCH_DB(6) break;
    case 7: PNN_LAUNCH_DB(7) break;
    default: PNN_LAUNCH_DB(8) break;
  }
#undef PNN_LAUNCH_DB
  PNN_KCHECK("edge_bwd_dmma_k");
  return 1;
}

int edge_dmma_num_slabs(int F) { return F / DFS; }

} // namespace pnn
