// edge_scatter.cu — reverse message step (R3 + R4 of SURVEY.md §8(c)) for ASYMMETRIC edge sets, i.e. graphs built with the
// paper's max-neighbour cap (PAPER.md:231 "Max neighbors 20", :269 "64"; pnn_config.max_neighbors > 0).
//
// The fast reverse kernels (edge.cu, edge_warp.cu, edge_tc_bwd.cu) rewrite every scatter to the sender as a gather over
// the node's own CSR row, which needs (i <- j) in the graph whenever (j <- i) is.  A cap breaks that, so this kernel does
// R3 / R4 literally, per directed edge e = (i <- j), with atomic adds to the sender's rows:
//   x-bar^ss = s-bar'_i ;  x-bar^vs = sum_a v-bar'_i[a] u_e[a] ;  x-bar^vv = sum_a v-bar'_i[a] v_j[a]
//   phi-bar_j^c += x-bar^c w_e^c ;  v-bar_j[a] += v-bar'_i[a] phi_j^vv w_e^vv
//   dE/dd_e = sum_{c,f} x-bar^c phi_j^c dw_e^c/dd ;  u-bar_e[a] = sum_f v-bar'_i[a] phi_j^vs w_e^vs
//   G_e = dE/dd_e u_e + (u-bar_e - (u-bar_e . u_e) u_e) / d_e ;  force_i += G_e ;  force_j -= G_e
// One warp per receiver, lanes stride over the features; the filter value and derivative come from the FP32 edge tape of the
// forward kernel when there is one, else they are recomputed from the radial basis (K + 1 terms per feature and chunk).  It is the plain path: correctness for the paper's own graph setting, not a tuned kernel.
#include <algorithm>

#include "common.cuh"

namespace pnn {

namespace {

template <typename T, typename PT> __device__ __forceinline__ T ldx(const PT* p) { return (T)(*p); }
template <> __device__ __forceinline__ float ldx<float, __nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }

template <typename T> __device__ __forceinline__ void sincos_t(T x, T* s, T* c);
template <> __device__ __forceinline__ void sincos_t<float>(float x, float* s, float* c) { sincosf(x, s, c); }
template <> __device__ __forceinline__ void sincos_t<double>(double x, double* s, double* c) { sincos(x, s, c); }

template <typename T, typename PT>
__global__ void __launch_bounds__(128)
edge_bwd_scatter_k(EdgeArgs<T> a, const PT* __restrict__ phi, const PT* __restrict__ v_in, const T* __restrict__ sb1,
                   const T* __restrict__ vb1, T* phib, T* vb_in, T* fslab, const T* __restrict__ wt,
                   const T* __restrict__ dt) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  __shared__ T Gs[4][2][36]; // per warp: g_k c (k < K), c at k = K; and their d/dd
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int F = a.F, K = a.K;
  const T rc = (T)a.rc;
  const T dmu = (K > 1) ? rc / (T)(K - 1) : rc;
  const T gamma = T(1) / (T(2) * dmu * dmu);
  const T pi_rc = (T)(3.14159265358979323846 / a.rc);
  const bool has_v = v_in != nullptr, has_out = phib != nullptr;
  for (int64_t i = (int64_t)blockIdx.x * 4 + warp; i < a.N; i += (int64_t)gridDim.x * 4) {
    T fi0 = T(0), fi1 = T(0), fi2 = T(0);
    for (int e = a.rowptr[i]; e < a.rowptr[i + 1]; ++e) {
      const Geom<T> gq = a.geom[e];
      const int64_t j = a.col[e];
      T sn, cs;
      sincos_t<T>(pi_rc * gq.d, &sn, &cs);
      const T cc = T(0.5) * (cs + T(1)), cp = -T(0.5) * pi_rc * sn;
      __syncwarp();
      if (!wt)
      for (int k = lane; k <= K; k += 32) {
        T g = T(1), gd = T(0);
        if (k < K) rbf_eval<T>(a.rbf, k, gq.d, rc, dmu, gamma, g, gd);
        Gs[warp][0][k] = (k < K) ? g * cc : cc;            // column K multiplies flt_b
        Gs[warp][1][k] = (k < K) ? cc * gd + cp * g : cp;
      }
      __syncwarp();
      T dEdd = T(0), ub0 = T(0), ub1 = T(0), ub2 = T(0);
      for (int f = lane; f < F; f += 32) {
        T w[3], dw[3];
        if (wt) { // FP32 edge tape written by the forward kernel: w and dw/dd of this edge ([E][3][F]; vv only when v != 0)
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            const bool on = c < 2 || has_v;
            w[c] = on ? wt[(int64_t)e * 3 * F + c * F + f] : T(0);
            dw[c] = on ? dt[(int64_t)e * 3 * F + c * F + f] : T(0);
          }
        } else
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const T* row = a.fltW + ((int64_t)c * F + f) * K;
          T s = a.fltb[c * F + f] * Gs[warp][0][K], sd = a.fltb[c * F + f] * Gs[warp][1][K];
          for (int k = 0; k < K; ++k) { s = fma(row[k], Gs[warp][0][k], s); sd = fma(row[k], Gs[warp][1][k], sd); }
          w[c] = s; dw[c] = sd;
        }
        const T p0 = ldx<T, PT>(phi + j * 3 * F + f), p1 = ldx<T, PT>(phi + j * 3 * F + F + f),
                p2 = ldx<T, PT>(phi + j * 3 * F + 2 * F + f);
        const T sbi = sb1[i * F + f];
        const T l0 = vb1[(i * 3 + 0) * F + f], l1 = vb1[(i * 3 + 1) * F + f], l2 = vb1[(i * 3 + 2) * F + f];
        T vj0 = T(0), vj1 = T(0), vj2 = T(0);
        if (has_v) {
          vj0 = ldx<T, PT>(v_in + (j * 3 + 0) * F + f); vj1 = ldx<T, PT>(v_in + (j * 3 + 1) * F + f);
          vj2 = ldx<T, PT>(v_in + (j * 3 + 2) * F + f);
        }
        const T xss = sbi, xvs = l0 * gq.ux + l1 * gq.uy + l2 * gq.uz, xvv = l0 * vj0 + l1 * vj1 + l2 * vj2;
        if (has_out) {
          atomicAdd(phib + j * 3 * F + f, xss * w[0]);
          atomicAdd(phib + j * 3 * F + F + f, xvs * w[1]);
          atomicAdd(phib + j * 3 * F + 2 * F + f, xvv * w[2]);
          const T pw = p2 * w[2];
          atomicAdd(vb_in + (j * 3 + 0) * F + f, l0 * pw);
          atomicAdd(vb_in + (j * 3 + 1) * F + f, l1 * pw);
          atomicAdd(vb_in + (j * 3 + 2) * F + f, l2 * pw);
        }
        dEdd += xss * p0 * dw[0] + xvs * p1 * dw[1] + xvv * p2 * dw[2];
        const T q = p1 * w[1];
        ub0 = fma(l0, q, ub0); ub1 = fma(l1, q, ub1); ub2 = fma(l2, q, ub2);
      }
#pragma unroll
      for (int o = 16; o; o >>= 1) {
        dEdd += __shfl_xor_sync(0xffffffffu, dEdd, o);
        ub0 += __shfl_xor_sync(0xffffffffu, ub0, o);
        ub1 += __shfl_xor_sync(0xffffffffu, ub1, o);
        ub2 += __shfl_xor_sync(0xffffffffu, ub2, o);
      }
      const T uu = ub0 * gq.ux + ub1 * gq.uy + ub2 * gq.uz, invd = T(1) / gq.d;
      const T G0 = dEdd * gq.ux + (ub0 - uu * gq.ux) * invd, G1 = dEdd * gq.uy + (ub1 - uu * gq.uy) * invd,
              G2 = dEdd * gq.uz + (ub2 - uu * gq.uz) * invd;
      fi0 += G0; fi1 += G1; fi2 += G2;
      if (lane == 0) { // the sender's share: force_j -= G_e
        atomicAdd(fslab + j * 3 + 0, -G0); atomicAdd(fslab + j * 3 + 1, -G1); atomicAdd(fslab + j * 3 + 2, -G2);
      }
    }
    if (lane == 0) { atomicAdd(fslab + i * 3 + 0, fi0); atomicAdd(fslab + i * 3 + 1, fi1); atomicAdd(fslab + i * 3 + 2, fi2); }
  }
}

} // namespace

// phib [N,3F] and vb_in [N,3F] (both may be NULL together: first block, forces only) are overwritten: phib = scatter sums,
// vb_in = vb1 + scatter sums.  fslab [N,3]: force slab, zeroed here when first_block, otherwise accumulated into.
template <typename T, typename PT>
int launch_edge_bwd_scatter(const EdgeArgs<T>& a, const PT* phi, const PT* v_in, const T* sb1, const T* vb1, T* phib,
                            T* vb_in, T* fslab, int first_block, cudaStream_t st, const T* wt, const T* dt) {
  if (a.N == 0) return 0;
  if (phib) {
    cudaMemsetAsync(phib, 0, sizeof(T) * a.N * 3 * a.F, st);
    cudaMemcpyAsync(vb_in, vb1, sizeof(T) * a.N * 3 * a.F, cudaMemcpyDeviceToDevice, st);
  }
  if (first_block) cudaMemsetAsync(fslab, 0, sizeof(T) * a.N * 3, st);
  const unsigned grid = (unsigned)std::min<int64_t>((a.N + 3) / 4, 148 * 16);
  edge_bwd_scatter_k<T, PT><<<grid, 128, 0, st>>>(a, phi, v_in, sb1, vb1, phib, vb_in, fslab, wt, dt);
  PNN_KCHECK("edge_bwd_scatter_k");
  return 1;
}

template int launch_edge_bwd_scatter<float, float>(const EdgeArgs<float>&, const float*, const float*, const float*,
                                                   const float*, float*, float*, float*, int, cudaStream_t, const float*,
                                                   const float*);
template int launch_edge_bwd_scatter<double, double>(const EdgeArgs<double>&, const double*, const double*, const double*,
                                                     const double*, double*, double*, double*, int, cudaStream_t,
                                                     const double*, const double*);
template int launch_edge_bwd_scatter<float, __nv_bfloat16>(const EdgeArgs<float>&, const __nv_bfloat16*,
                                                           const __nv_bfloat16*, const float*, const float*, float*, float*,
                                                           float*, int, cudaStream_t, const float*, const float*);

} // namespace pnn
