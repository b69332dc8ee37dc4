// schnet.cu — the edge-side kernels of the second backbone (SchNet, one of the
// six backbones of the paper's architecture search; reading Q31), on the same CSR graph, geometry, radial basis and
// cutoff as the PaiNN path.  Per block:
//   W_e = (F2 silu(F1 g(d_e) + f1) + f2) c(d_e) ,  m_i = sum_{e = (i <- j)} (A x_j) o W_e ,  x_i += B2 silu(B1 m_i + b1) + b2
// The filter-generating network and all node layers are GEMMs of the library (launch_gemm: E rows for the filter, N rows for
// the nodes; FP64 on the tensor cores); this file has the radial-basis rows, the continuous-filter convolution and its adjoint.
// Reverse sweep (forces): the energy depends on a pair distance through both directed edges of the pair and the filter depends
// on d only, so with S_e = m-bar_i o x1_j + m-bar_j o x1_i (gathers from the receiver's side, no scatter) and the filter's
// derivative dW_e/dd = c dF/dd + c' F (dF/dd by forward-mode through the same two GEMMs: (g' F1^T) o silu' then F2^T):
//   dE/dd_pair = <S_e, dW_e/dd> ,  force_i = sum_{e = (i <- j)} dE/dd_pair u_e ,  x1-bar_i = sum_e W_e o m-bar_j   (edge-set symmetry)
// One warp per receiver, lanes over the features, segment sums in registers, no atomics.  Plain kernels: the second backbone
// is here for coverage of the paper's model space on the same boundary, not tuned.
#include <algorithm>

#include "common.cuh"

namespace pnn {

namespace {

template <typename T> __device__ __forceinline__ void sincos_t(T x, T* s, T* c);
template <> __device__ __forceinline__ void sincos_t<float>(float x, float* s, float* c) { sincosf(x, s, c); }
template <> __device__ __forceinline__ void sincos_t<double>(double x, double* s, double* c) { sincos(x, s, c); }

// G[e][k] = g_k(d_e), Gd[e][k] = dg_k/dd (k < K; zero in the padding columns K..KP-1); Gd may be NULL
template <typename T>
__global__ void __launch_bounds__(256)
sch_rbf_k(int64_t N, int K, int KP, int rbf, double rc_, const int32_t* __restrict__ rowptr, const Geom<T>* __restrict__ geom,
          T* __restrict__ G, T* __restrict__ Gd, const int* __restrict__ d_ovf) {
  if (*d_ovf & ERRF_EDGE_OVERFLOW) return;
  const int64_t E = rowptr[N];
  const T rc = (T)rc_;
  const T dmu = (K > 1) ? rc / (T)(K - 1) : rc;
  const T gamma = T(1) / (T(2) * dmu * dmu);
  for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < E * KP; q += (int64_t)gridDim.x * blockDim.x) {
    const int64_t e = q / KP;
    const int k = (int)(q - e * KP);
    T g = T(0), gd = T(0);
    if (k < K) rbf_eval<T>(rbf, k, geom[e].d, rc, dmu, gamma, g, gd);
    G[q] = g;
    if (Gd) Gd[q] = gd;
  }
}

template <typename T, int NF> // NF = F / 32 features per lane
__global__ void __launch_bounds__(128)
sch_conv_fwd_k(int64_t N, double rc_, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
               const Geom<T>* __restrict__ geom, const T* __restrict__ Wf, const T* __restrict__ x1, T* __restrict__ m,
               const int* __restrict__ d_ovf) {
  if (*d_ovf & ERRF_EDGE_OVERFLOW) return;
  constexpr int F = 32 * NF;
  const int lane = threadIdx.x & 31;
  const T pi_rc = (T)(3.14159265358979323846 / rc_);
  for (int64_t i = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5); i < N; i += (int64_t)gridDim.x * 4) {
    T acc[NF];
#pragma unroll
    for (int q = 0; q < NF; ++q) acc[q] = T(0);
    for (int e = rowptr[i]; e < rowptr[i + 1]; ++e) {
      const int64_t j = col[e];
      T sn, cs;
      sincos_t<T>(pi_rc * geom[e].d, &sn, &cs);
      const T c = T(0.5) * (cs + T(1));
#pragma unroll
      for (int q = 0; q < NF; ++q)
        acc[q] = fma(c * Wf[(int64_t)e * F + lane + 32 * q], x1[j * F + lane + 32 * q], acc[q]);
    }
#pragma unroll
    for (int q = 0; q < NF; ++q) m[i * F + lane + 32 * q] = acc[q];
  }
}

template <typename T, int NF>
__global__ void __launch_bounds__(128)
sch_conv_bwd_k(int64_t N, double rc_, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
               const Geom<T>* __restrict__ geom, const T* __restrict__ Wf, const T* __restrict__ dWf,
               const T* __restrict__ x1, const T* __restrict__ mb, T* __restrict__ x1b, T* __restrict__ forces,
               int first_block, const int* __restrict__ d_ovf) {
  if (*d_ovf & ERRF_EDGE_OVERFLOW) return;
  constexpr int F = 32 * NF;
  const int lane = threadIdx.x & 31;
  const T pi_rc = (T)(3.14159265358979323846 / rc_);
  for (int64_t i = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5); i < N; i += (int64_t)gridDim.x * 4) {
    T acc[NF], mi[NF], xi[NF];
#pragma unroll
    for (int q = 0; q < NF; ++q) { acc[q] = T(0); mi[q] = mb[i * F + lane + 32 * q]; xi[q] = x1[i * F + lane + 32 * q]; }
    T f0 = T(0), f1 = T(0), f2 = T(0);
    for (int e = rowptr[i]; e < rowptr[i + 1]; ++e) {
      const int64_t j = col[e];
      const Geom<T> gq = geom[e];
      T sn, cs;
      sincos_t<T>(pi_rc * gq.d, &sn, &cs);
      const T c = T(0.5) * (cs + T(1)), cd = -T(0.5) * pi_rc * sn;
      T D = T(0);
#pragma unroll
      for (int q = 0; q < NF; ++q) {
        const int f = lane + 32 * q;
        const T w = Wf[(int64_t)e * F + f], dw = dWf[(int64_t)e * F + f];
        const T mj = mb[j * F + f], xj = x1[j * F + f];
        acc[q] = fma(c * w, mj, acc[q]);
        D = fma(fma(mi[q], xj, mj * xi[q]), fma(c, dw, cd * w), D);
      }
#pragma unroll
      for (int o = 16; o; o >>= 1) D += __shfl_xor_sync(0xffffffffu, D, o);
      f0 = fma(D, gq.ux, f0); f1 = fma(D, gq.uy, f1); f2 = fma(D, gq.uz, f2);
    }
    if (x1b) {
#pragma unroll
      for (int q = 0; q < NF; ++q) x1b[i * F + lane + 32 * q] = acc[q];
    }
    if (lane == 0) {
      T* dst = forces + i * 3;
      if (first_block) { dst[0] = f0; dst[1] = f1; dst[2] = f2; }
      else { dst[0] += f0; dst[1] += f1; dst[2] += f2; }
    }
  }
}

} // namespace

template <typename T>
int launch_sch_rbf(int64_t N, int64_t maxE, int K, int KP, int rbf, double rc, const int32_t* rowptr, const void* geom, T* G,
                   T* Gd, const int* d_ovf, cudaStream_t st) {
  if (N == 0 || maxE == 0) return 0;
  const unsigned grid = (unsigned)std::min<int64_t>((maxE * KP + 255) / 256, 148 * 16);
  sch_rbf_k<T><<<grid, 256, 0, st>>>(N, K, KP, rbf, rc, rowptr, (const Geom<T>*)geom, G, Gd, d_ovf);
  PNN_KCHECK("sch_rbf_k");
  return 1;
}

#define PNN_SCH_DISPATCH(KERNEL, ...)                                                                           \
  switch (F / 32) {                                                                                             \
    case 1: KERNEL<T, 1><<<grid, 128, 0, st>>>(__VA_ARGS__); break;                                             \
    case 2: KERNEL<T, 2><<<grid, 128, 0, st>>>(__VA_ARGS__); break;                                             \
    case 3: KERNEL<T, 3><<<grid, 128, 0, st>>>(__VA_ARGS__); break;                                             \
    case 4: KERNEL<T, 4><<<grid, 128, 0, st>>>(__VA_ARGS__); break;                                             \
    case 5: KERNEL<T, 5><<<grid, 128, 0, st>>>(__VA_ARGS__); break;                                             \
    case 6: KERNEL<T, 6><<<grid, 128, 0, st>>>(__VA_ARGS__); break;                                             \
    case 7: KERNEL<T, 7><<<grid, 128, 0, st>>>(__VA_ARGS__); break;                                             \
    default: KERNEL<T, 8><<<grid, 128, 0, st>>>(__VA_ARGS__); break;                                            \
  }

template <typename T>
int launch_sch_conv_fwd(int64_t N, int F, double rc, const int32_t* rowptr, const int32_t* col, const void* geom, const T* Wf,
                        const T* x1, T* m, const int* d_ovf, cudaStream_t st) {
  if (N == 0) return 0;
  const unsigned grid = (unsigned)std::min<int64_t>((N + 3) / 4, 148 * 16);
  PNN_SCH_DISPATCH(sch_conv_fwd_k, N, rc, rowptr, col, (const Geom<T>*)geom, Wf, x1, m, d_ovf)
  PNN_KCHECK("sch_conv_fwd_k");
  return 1;
}

template <typename T>
int launch_sch_conv_bwd(int64_t N, int F, double rc, const int32_t* rowptr, const int32_t* col, const void* geom, const T* Wf,
                        const T* dWf, const T* x1, const T* mb, T* x1b, T* forces, int first_block, const int* d_ovf,
                        cudaStream_t st) {
  if (N == 0) return 0;
  const unsigned grid = (unsigned)std::min<int64_t>((N + 3) / 4, 148 * 16);
  PNN_SCH_DISPATCH(sch_conv_bwd_k, N, rc, rowptr, col, (const Geom<T>*)geom, Wf, dWf, x1, mb, x1b, forces, first_block, d_ovf)
  PNN_KCHECK("sch_conv_bwd_k");
  return 1;
}
#undef PNN_SCH_DISPATCH

#define PNN_INST_SCH(T)                                                                                                       \
  template int launch_sch_rbf<T>(int64_t, int64_t, int, int, int, double, const int32_t*, const void*, T*, T*, const int*,    \
                                 cudaStream_t);                                                                               \
  template int launch_sch_conv_fwd<T>(int64_t, int, double, const int32_t*, const int32_t*, const void*, const T*, const T*,  \
                                      T*, const int*, cudaStream_t);                                                          \
  template int launch_sch_conv_bwd<T>(int64_t, int, double, const int32_t*, const int32_t*, const void*, const T*, const T*,  \
                                      const T*, const T*, T*, T*, int, const int*, cudaStream_t);
PNN_INST_SCH(float)
PNN_INST_SCH(double)
#undef PNN_INST_SCH

} // namespace pnn
