// branch.cu — composition-conditioned branch weights (reading Q28): per structure
// the element fractions c (histogram of Z over the structure's atoms), a small MLP with SiLU hidden layers, and a softmax
// over the heads.  24.5 k parameters: the whole router lives in L2 / L1; one CTA evaluates SPB structures so that every
// weight it reads is used SPB times, thread o owns output unit o of the current layer (weights stored input-major on the
// device, so a warp reads 32 consecutive outputs of one input row).
#include <algorithm>

#include "common.cuh"

namespace pnn {

namespace {
constexpr int BR_MAXW = 256;   // widest layer (include/pnn.h)
constexpr int BR_SPB = 4;      // structures per CTA
constexpr int BR_THREADS = 128;

template <typename T>
__global__ void __launch_bounds__(BR_THREADS) branch_mlp_k(int S, BranchMlpDims dm, const int32_t* __restrict__ Z,
                                                           const int32_t* __restrict__ sptr,
                                                           const T* __restrict__ params, T* __restrict__ out,
                                                           int* __restrict__ d_err) {
  __shared__ T xa[BR_SPB][BR_MAXW];
  __shared__ T xb[BR_SPB][BR_MAXW];
  __shared__ int cnt[BR_SPB][BR_MAXW];
  const int tid = threadIdx.x;
  const int g0 = blockIdx.x * BR_SPB;
  const int W0 = dm.width[0];

  for (int i = tid; i < BR_SPB * BR_MAXW; i += BR_THREADS) (&cnt[0][0])[i] = 0;
  __syncthreads();
  bool bad = false;
  for (int s = 0; s < BR_SPB; ++s) {
    const int g = g0 + s;
    if (g >= S) break;
    const int a0 = sptr[g], a1 = sptr[g + 1];
    for (int a = a0 + tid; a < a1; a += BR_THREADS) {
      const int z = Z[a];
      if (z < 1 || z > W0) { bad = true; continue; }
      atomicAdd(&cnt[s][z - 1], 1);
    }
  }
  if (bad) atomicOr(d_err, ERRF_BAD_Z);
  __syncthreads();
  for (int s = 0; s < BR_SPB; ++s) {
    const int g = g0 + s;
    const int n = g < S ? sptr[g + 1] - sptr[g] : 0;
    for (int i = tid; i < W0; i += BR_THREADS) xa[s][i] = n > 0 ? T(cnt[s][i]) / T(n) : T(0);
  }
  __syncthreads();

  T(*xin)[BR_MAXW] = xa;
  T(*xout)[BR_MAXW] = xb;
  for (int l = 0; l < dm.n_layers; ++l) {
    const int n_in = dm.width[l], n_out = dm.width[l + 1];
    const T* __restrict__ Wt = params + dm.off_w[l];      // [n_in][n_out]
    const T* __restrict__ bl = params + dm.off_b[l];
    const bool last = l + 1 == dm.n_layers;
    for (int o = tid; o < n_out; o += BR_THREADS) {
      T acc[BR_SPB];
#pragma unroll
      for (int s = 0; s < BR_SPB; ++s) acc[s] = bl[o];
      for (int i = 0; i < n_in; ++i) {
        const T w = Wt[(size_t)i * n_out + o];
#pragma unroll
        for (int s = 0; s < BR_SPB; ++s) acc[s] = fma(w, xin[s][i], acc[s]);
      }
#pragma unroll
      for (int s = 0; s < BR_SPB; ++s) xout[s][o] = last ? acc[s] : silu_f<T>(acc[s]);
    }
    __syncthreads();
    T(*t)[BR_MAXW] = xin; xin = xout; xout = t;
  }

  // softmax over the heads (xin holds the logits): one thread per structure, H <= 256 terms
  const int H = dm.width[dm.n_layers];
  if (tid < BR_SPB && g0 + tid < S) {
    const T* lg = xin[tid];
    T mx = lg[0];
    for (int h = 1; h < H; ++h) mx = lg[h] > mx ? lg[h] : mx;
    T sum = T(0);
    for (int h = 0; h < H; ++h) sum += exp(lg[h] - mx);
    T* o = out + (size_t)(g0 + tid) * H;
    for (int h = 0; h < H; ++h) o[h] = exp(lg[h] - mx) / sum;
  }
}
} // namespace

template <typename T>
int launch_branch_mlp(int64_t S, const BranchMlpDims& dm, const int32_t* Z, const int32_t* sptr, const T* params,
                      T* out, int* d_err, cudaStream_t st) {
  if (S <= 0) return 0;
  branch_mlp_k<T><<<(unsigned)((S + BR_SPB - 1) / BR_SPB), BR_THREADS, 0, st>>>((int)S, dm, Z, sptr, params, out, d_err);
  PNN_KCHECK("branch_mlp_k");
  return 1;
}
template int launch_branch_mlp<float>(int64_t, const BranchMlpDims&, const int32_t*, const int32_t*, const float*,
                                      float*, int*, cudaStream_t);
template int launch_branch_mlp<double>(int64_t, const BranchMlpDims&, const int32_t*, const int32_t*, const double*,
                                       double*, int*, cudaStream_t);

} // namespace pnn

// ---- plain-ALU peak ("FP32-ALU and FP64 peaks are nominal and must be measured on the box by a small
// FMA micro-benchmark"): independent FMA chains in registers, nothing else in the loop.  FP32 uses the packed
// fma.rn.f32x2 the kernels use (two FMAs per issued instruction).
namespace pnn {
namespace {
constexpr int PK_CHAINS = 8, PK_ITERS = 4096;

__global__ void __launch_bounds__(256) peak_f32_k(float2* out, float2 a, float2 b) {
  float2 acc[PK_CHAINS];
#pragma unroll
  for (int c = 0; c < PK_CHAINS; ++c) acc[c] = make_float2(threadIdx.x * 1e-3f + c, blockIdx.x * 1e-3f - c);
  for (int it = 0; it < PK_ITERS; ++it) {
#pragma unroll
    for (int c = 0; c < PK_CHAINS; ++c) acc[c] = __ffma2_rn(acc[c], a, b);
  }
  float2 s = make_float2(0.f, 0.f);
#pragma unroll
  for (int c = 0; c < PK_CHAINS; ++c) { s.x += acc[c].x; s.y += acc[c].y; }
  if (s.x == 123.456f) out[0] = s;   // keeps the chains alive; never true for these inputs
}

__global__ void __launch_bounds__(256) peak_f64_k(double* out, double a, double b) {
  double acc[PK_CHAINS];
#pragma unroll
  for (int c = 0; c < PK_CHAINS; ++c) acc[c] = threadIdx.x * 1e-3 + c;
  for (int it = 0; it < PK_ITERS; ++it) {
#pragma unroll
    for (int c = 0; c < PK_CHAINS; ++c) acc[c] = fma(acc[c], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int c = 0; c < PK_CHAINS; ++c) s += acc[c];
  if (s == 123.456) out[0] = s;
}
} // namespace

// TFLOP/s of the FMA pipe, best of `reps` launches timed with CUDA events on `st`.  Synchronises.  Returns < 0 on error.
double measure_alu_peak(bool fp64, void* scratch, cudaStream_t st) {
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0;
  const int grid = 148 * 8, block = 256, reps = 5;
  double best = 0.0;
  for (int r = 0; r < reps + 1; ++r) {
    cudaEventRecord(e0, st);
    if (fp64) peak_f64_k<<<grid, block, 0, st>>>((double*)scratch, 0.999999, 1e-7);
    else peak_f32_k<<<grid, block, 0, st>>>((float2*)scratch, make_float2(0.999999f, 0.999998f), make_float2(1e-7f, 2e-7f));
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flop = (double)grid * block * PK_ITERS * PK_CHAINS * (fp64 ? 2.0 : 4.0);
    if (r > 0 && ms > 0.f) best = std::max(best, flop / (ms * 1e-3) * 1e-12);   // launch 0 is the warm-up
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return best;
}
// L2 read bandwidth: every CTA streams the whole buffer (32 MB, a quarter of the 126 MB L2; after the warm-up pass it is
// L2-resident and far larger than L1) in 512-byte rows per warp, the access shape of the edge kernels' gathers.
__global__ void __launch_bounds__(256) peak_l2_k(const float4* __restrict__ buf, int64_t n4, int passes, float* out) {
  float acc = 0.f;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int p = 0; p < passes; ++p) {
    // start offset differs per CTA and pass so that the CTAs do not walk the buffer in lockstep
    int64_t i = ((int64_t)blockIdx.x * 7919 + p * 104729) % n4;
    i = (i / 32) * 32 + threadIdx.x % 32 + (int64_t)(threadIdx.x / 32) * 32;
    for (int64_t k = 0; k < n4; k += stride) {
      int64_t j = i + k;
      if (j >= n4) j -= n4;
      const float4 v = __ldcg(buf + j);
      acc += v.x + v.y + v.z + v.w;
    }
  }
  if (acc == 12345.678f) out[0] = acc; // never true for the zero-filled buffer: keeps the loads alive
}

double measure_l2_peak(void* buf, int64_t bytes, cudaStream_t st) {
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0;
  const int grid = 148 * 4, block = 256, passes = 8, reps = 5;
  const int64_t n4 = bytes / 16;
  double best = 0.0;
  for (int r = 0; r < reps + 1; ++r) {
    cudaEventRecord(e0, st);
    peak_l2_k<<<grid, block, 0, st>>>((const float4*)buf, n4, passes, (float*)buf);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    // per pass the grid reads ceil(n4 / stride) * stride vectors
    const int64_t stride = (int64_t)grid * block;
    const double moved = (double)((n4 + stride - 1) / stride) * stride * 16.0 * passes;
    if (r > 0 && ms > 0.f) best = std::max(best, moved / (ms * 1e-3) * 1e-9);   // launch 0 is the warm-up; GB/s
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return best;
}
} // namespace pnn
