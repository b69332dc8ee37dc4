// pool_head.cu — the paper's graph-level output heads ("Output heads 16 (graph-level)", "Head architecture
// 2 shared layers (dim 50) + 2 branch layers (dim 776)"; reading Q29):
//   x_g = mean_{i in g} s_i                                  (mean pooling of the final scalar features)
//   y1 = silu(P1 x_g + p1) ; y2 = silu(P2 y1 + p2)           (shared trunk, width d1)
//   z1 = silu(B1_h y2 + q1_h) ; z2 = silu(B2_h z1 + q2_h)    (branch of the structure's head h, width d2)
//   E_g = w3_h . z2 + q3_h
// and its adjoint for forces: x-bar_g = P1^T (P2^T (B1_h^T (B2_h^T (w3_h . silu'(.)) . silu'(.)) . silu'(.)) . silu'(.)),
// s-bar_i = x-bar_{g(i)} / n_g.
//
// The branch layers are the cost (d2 x d2 weights per head, one matrix-vector product per structure), so structures are
// counting-sorted by head first and a CTA takes G structures (16 in FP32, 8 in FP64) of ONE head: every weight read from L2 is
// used G times.  A layer is a thread-per-output matrix-vector product over weights stored [in][out] (coalesced), the G input
// vectors broadcast from shared memory; the adjoint is the same routine over the original [out][in] weights.
// Forward and adjoint run back to back in the same CTA with the pre-activations in shared memory: no tape, one launch.
#include <algorithm>

#include "common.cuh"

namespace pnn {

namespace {

constexpr int POOL_THREADS = 256;
constexpr int POOL_RT = 2;      // outputs per thread of pooled_head_k (register tile POOL_RT x G)
constexpr int POOL_U = 16;      // weight loads in flight per thread
constexpr int POOL_MAXT = 512;  // threads of pooled_head_k: one per POOL_RT output features of the widest layer
constexpr int POOL_MAXH = 1024;

// x[g][f] = mean_i s[i][f]; one CTA per structure (grid-stride), threads over (atom slice, feature)
template <typename T>
__global__ void __launch_bounds__(POOL_THREADS)
pool_mean_k(int64_t S, int F, const int32_t* __restrict__ sptr, const T* __restrict__ s, T* __restrict__ x) {
  __shared__ T part[POOL_THREADS];
  const int f = threadIdx.x % F, a0 = threadIdx.x / F, na = POOL_THREADS / F; // F in {32..256}, multiple of 32
  for (int64_t g = blockIdx.x; g < S; g += gridDim.x) {
    const int i0 = sptr[g], i1 = sptr[g + 1];
    T acc = T(0);
    if (a0 < na)
      for (int i = i0 + a0; i < i1; i += na) acc += s[(int64_t)i * F + f];
    part[threadIdx.x] = acc;
    __syncthreads();
    if (threadIdx.x < F) {
      T t = T(0);
      for (int a = 0; a < na; ++a) t += part[a * F + f];
      x[g * F + f] = (i1 > i0) ? t / (T)(i1 - i0) : T(0);
    }
    __syncthreads();
  }
}

// Counting sort of the structures by head (one CTA): perm[] lists the structures head by head, tiles[] = (head, first
// position in perm, count <= G) for every CTA of pooled_head_k, *ntiles their number.  Structures with a head index out
// of range raise ERRF_BAD_HEAD and are left out (their energy stays 0).
__global__ void __launch_bounds__(1024)
head_sort_k(int64_t S, int H, int G, const int32_t* __restrict__ head, int32_t* __restrict__ perm, int4* __restrict__ tiles,
            int32_t* __restrict__ ntiles, int* __restrict__ d_err) {
  __shared__ int cnt[POOL_MAXH], start[POOL_MAXH], tstart[POOL_MAXH], cur[POOL_MAXH];
  for (int h = threadIdx.x; h < H; h += blockDim.x) { cnt[h] = 0; cur[h] = 0; }
  __syncthreads();
  for (int64_t g = threadIdx.x; g < S; g += blockDim.x) {
    const int h = head[g];
    if (h < 0 || h >= H) atomicOr(d_err, ERRF_BAD_HEAD);
    else atomicAdd(&cnt[h], 1);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int a = 0, t = 0;
    for (int h = 0; h < H; ++h) { start[h] = a; tstart[h] = t; a += cnt[h]; t += (cnt[h] + G - 1) / G; }
    *ntiles = t;
  }
  __syncthreads();
  for (int64_t g = threadIdx.x; g < S; g += blockDim.x) {
    const int h = head[g];
    if (h >= 0 && h < H) perm[start[h] + atomicAdd(&cur[h], 1)] = (int32_t)g;
  }
  for (int h = threadIdx.x; h < H; h += blockDim.x)
    for (int t = 0, c = cnt[h]; c > 0; ++t, c -= G) tiles[tstart[h] + t] = make_int4(h, start[h] + t * G, min(c, G), 0);
}

template <typename T> __device__ __forceinline__ T silu_f(T x) { return x / (T(1) + exp(-x)); }
template <typename T> __device__ __forceinline__ T dsilu_f(T x) {
  const T sg = T(1) / (T(1) + exp(-x));
  return sg * (T(1) + x * (T(1) - sg));
}

template <typename T> struct alignas(16) Vec16 { T v[16 / sizeof(T)]; };
template <typename T, int RT> struct alignas(RT * sizeof(T) >= 16 ? 16 : RT * sizeof(T)) VecR { T v[RT]; };

template <typename T, int G, int RT, int U>
struct MatTile {
  static constexpr int VW = 16 / sizeof(T);
  T acc[RT][G];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int i = 0; i < RT; ++i)
#pragma unroll
      for (int j = 0; j < G; ++j) acc[i][j] = T(0);
  }
  // acc += sum_{c in [c0, c1)} M[c][r0 .. r0+4) (x) v[c][0..G); the weight loads of the next U rows are in flight while
  // the FMAs of the current U rows issue
  __device__ __forceinline__ void run(int r0, int n_r, int c0, int c1, const T* __restrict__ M, const T* v) {
    const bool vec = (n_r % RT) == 0;
    const T* col = M + r0;
    auto load_w = [&](int c, VecR<T, RT>& w) {
      if (vec) { w = *reinterpret_cast<const VecR<T, RT>*>(col + (int64_t)c * n_r); }
      else {
#pragma unroll
        for (int i = 0; i < RT; ++i) w.v[i] = (r0 + i < n_r) ? __ldg(col + (int64_t)c * n_r + i) : T(0);
      }
    };
    auto fmas = [&](const VecR<T, RT>& w, int c) {
      const Vec16<T>* vc = reinterpret_cast<const Vec16<T>*>(v + c * G);
#pragma unroll
      for (int q = 0; q < G / VW; ++q) {
        const Vec16<T> x = vc[q];
#pragma unroll
        for (int i = 0; i < RT; ++i)
#pragma unroll
          for (int e = 0; e < VW; ++e) acc[i][q * VW + e] = fma(w.v[i], x.v[e], acc[i][q * VW + e]);
      }
    };
    int c = c0;
    for (; c + U <= c1; c += U) { // U weight loads in flight per thread, then their FMAs
      VecR<T, RT> w[U];
#pragma unroll
      for (int u = 0; u < U; ++u) load_w(c + u, w[u]);
#pragma unroll
      for (int u = 0; u < U; ++u) fmas(w[u], c + u);
    }
    for (; c < c1; ++c) {
      VecR<T, RT> w;
      load_w(c, w);
      fmas(w, c);
    }
  }
};

// out[r][g] = sum_c M[c][r] v[c][g] for the CTA's G structures, then epi(r, g, value).  A thread owns RT = POOL_RT consecutive
// outputs r for all G structures (an RT x G register tile): per c one 16-byte (float) weight load, coalesced over r, and
// G values of v broadcast from shared memory for RT * G FMAs (a thread per output would spend G broadcast loads on G FMAs
// and is bound by the shared-memory return path).  Narrow layers (all outputs inside one warp) split the sum over c
// between the warps and add the partial tiles in warp order through `scratch` (deterministic).
// Serves the forward layers with the transposed weights (M = W^T [in][out]) and the adjoint with the original ones
// (M = W [out][in]).  M must be 16-byte aligned; rows are loaded as vectors when n_r is a multiple of RT.
template <typename T, int G, typename Epi>
__device__ __forceinline__ void matvec(int n_r, int n_c, const T* __restrict__ M, const T* v, T* scratch, int scratch_elems,
                                       Epi epi) {
  constexpr int RT = POOL_RT;
  const int nw = blockDim.x >> 5, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  MatTile<T, G, RT, POOL_U> t;
  if (n_r <= 32 * RT && n_c >= 64 && nw * n_r * G <= scratch_elems) { // split over c
    const int per = (n_c + nw - 1) / nw, c0 = warp * per, c1 = min(n_c, c0 + per), r0 = lane * RT;
    if (r0 < n_r) {
      t.zero();
      t.run(r0, n_r, c0, c1, M, v);
#pragma unroll
      for (int i = 0; i < RT; ++i)
        if (r0 + i < n_r) {
#pragma unroll
          for (int j = 0; j < G; ++j) scratch[(warp * n_r + r0 + i) * G + j] = t.acc[i][j];
        }
    }
    __syncthreads();
    for (int e = threadIdx.x; e < n_r * G; e += blockDim.x) {
      T sum = T(0);
      for (int w = 0; w < nw; ++w) sum += scratch[w * n_r * G + e];
      epi(e / G, e % G, sum);
    }
    return;
  }
  for (int r0 = threadIdx.x * RT; r0 < n_r; r0 += blockDim.x * RT) {
    t.zero();
    t.run(r0, n_r, 0, n_c, M, v);
#pragma unroll
    for (int i = 0; i < RT; ++i)
      if (r0 + i < n_r) {
#pragma unroll
        for (int j = 0; j < G; ++j) epi(r0 + i, j, t.acc[i][j]);
      }
  }
}

// One CTA per tile of <= G structures of one head.  Shared memory ([feature][G], the G structures of a feature side by
// side): PRE1 [d1] | PRE2 [d1] | PRE3 [d2] | PRE4 [d2] | A [dm] | B [dm], dm = max(F, d1, d2); A and B ping-pong as the
// input and output of consecutive layers, forward and reverse.
template <typename T, int G>
__global__ void __launch_bounds__(POOL_MAXT)
pooled_head_k(int F, int d1, int d2, const T* __restrict__ Wt, PoolHeadW pw, const int32_t* __restrict__ perm,
              const int4* __restrict__ tiles, const int32_t* __restrict__ ntiles, const T* __restrict__ x,
              T* __restrict__ energy, T* __restrict__ xbar) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  if ((int)blockIdx.x >= *ntiles) return;
  const int4 tl = tiles[blockIdx.x];
  const int h = tl.x, p0 = tl.y, cnt = tl.z;
  const int dm = max(F, max(d1, d2));
  T* PRE1 = reinterpret_cast<T*>(smem_raw);
  T* PRE2 = PRE1 + d1 * G; T* PRE3 = PRE2 + d1 * G; T* PRE4 = PRE3 + d2 * G; T* A = PRE4 + d2 * G; T* B = A + dm * G;
  const T* B1 = Wt + pw.br + (int64_t)h * pw.br_stride;
  const T* q1 = B1 + pw.oq1; const T* B2 = B1 + pw.oB2; const T* q2 = B1 + pw.oq2; const T* w3 = B1 + pw.ow3;
  const T* q3 = B1 + pw.oq3; const T* B1t = B1 + pw.oB1t; const T* B2t = B1 + pw.oB2t;
  for (int t = threadIdx.x; t < F * G; t += blockDim.x) { // padding slots repeat the last structure (results not written)
    const int f = t / G, g = t - f * G;
    B[t] = x[(int64_t)perm[p0 + min(g, cnt - 1)] * F + f];
  }
  __syncthreads();
  // split: PRE3 | PRE4 are free (not yet written / already consumed) and may hold the partial tiles of a narrow layer
  auto fwd = [&](int n_out, int n_in, const T* Mt, const T* bias, const T* in, T* pre, T* out, bool split) {
    matvec<T, G>(n_out, n_in, Mt, in, PRE3, split ? 2 * d2 * G : 0, [&](int o, int g, T acc) {
      const T p = acc + bias[o];
      pre[o * G + g] = p; out[o * G + g] = silu_f<T>(p);
    });
    __syncthreads();
  };
  fwd(d1, F, Wt + pw.P1t, Wt + pw.p1, B, PRE1, A, true);
  fwd(d1, d1, Wt + pw.P2t, Wt + pw.p2, A, PRE2, B, true);
  fwd(d2, d1, B1t, q1, B, PRE3, A, false);
  fwd(d2, d2, B2t, q2, A, PRE4, B, false);
  { // E_g = w3 . z2 + q3: a warp per structure
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int g = warp; g < cnt; g += blockDim.x / 32) {
      T a = T(0);
      for (int o = lane; o < d2; o += 32) a = fma(w3[o], B[o * G + g], a);
#pragma unroll
      for (int m = 16; m; m >>= 1) a += __shfl_xor_sync(0xffffffffu, a, m);
      if (lane == 0) energy[perm[p0 + g]] = a + q3[0];
    }
  }
  if (!xbar) return;
  for (int t = threadIdx.x; t < G * d2; t += blockDim.x) A[t] = w3[t / G] * dsilu_f<T>(PRE4[t]); // z2-bar (pre-activation)
  __syncthreads();
  auto bwd = [&](int n_out, int n_in, const T* M, const T* gb, const T* dpre, T* out, bool split) {
    matvec<T, G>(n_in, n_out, M, gb, PRE3, split ? 2 * d2 * G : 0, [&](int i, int g, T acc) {
      out[i * G + g] = dpre ? acc * dsilu_f<T>(dpre[i * G + g]) : acc;
    });
    __syncthreads();
  };
  bwd(d2, d2, B2, A, PRE3, B, false);                      // z1-bar
  bwd(d2, d1, B1, B, PRE2, A, true);                       // y2-bar
  bwd(d1, d1, Wt + pw.P2, A, PRE1, B, true);               // y1-bar
  bwd(d1, F, Wt + pw.P1, B, (const T*)nullptr, A, true);   // x-bar
  for (int t = threadIdx.x; t < F * G; t += blockDim.x) {
    const int f = t / G, g = t - f * G;
    if (g < cnt) xbar[(int64_t)perm[p0 + g] * F + f] = A[t];
  }
}

// s-bar_i = x-bar_{g(i)} / n_g
template <typename T>
__global__ void __launch_bounds__(256)
pool_bcast_k(int64_t n, int F, const int32_t* __restrict__ a2s, const int32_t* __restrict__ sptr, const T* __restrict__ xbar,
             T* __restrict__ sb) {
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = t / F;
    const int f = (int)(t - i * F), g = a2s[i];
    sb[t] = xbar[(int64_t)g * F + f] / (T)(sptr[g + 1] - sptr[g]);
  }
}

template <typename T> constexpr int pool_group() { return sizeof(T) == 8 ? 8 : 16; }

} // namespace

int64_t pool_head_scratch_bytes(int64_t maxS, int F, int H, size_t elem) {
  const int64_t G = elem == 8 ? 8 : 16;
  return 2 * ((maxS * F * (int64_t)elem + 255) / 256 * 256) + (maxS * 4 + 255) / 256 * 256 +
         (((maxS + G - 1) / G + H) * 16 + 255) / 256 * 256 + 256;
}

bool pool_head_supported(int F, int d1, int d2, int H, size_t elem) {
  if (d1 < 1 || d2 < 1 || d1 > 4096 || d2 > 4096 || H > POOL_MAXH) return false;
  const int64_t G = elem == 8 ? 8 : 16, dm = std::max(F, std::max(d1, d2));
  return G * (2 * d1 + 2 * d2 + 2 * dm) * (int64_t)elem <= 227 * 1024;
}

// energy [S] and, when sb != NULL, s-bar [N][F] of the pooled head.  scratch: pool_head_scratch_bytes().  Returns the
// number of launches, -1 when the shapes are not supported.
template <typename T>
int launch_pool_head(int64_t N, int64_t S, int F, int H, int d1, int d2, const T* s, const int32_t* a2s,
                     const int32_t* sptr, const int32_t* head, const T* W, const PoolHeadW& pw, void* scratch, T* energy,
                     T* sb, int* d_err, cudaStream_t st) {
  if (S == 0) return 0;
  if (!pool_head_supported(F, d1, d2, H, sizeof(T))) return -1;
  constexpr int G = pool_group<T>();
  char* p = (char*)scratch;
  auto carve = [&](int64_t b) { char* q = p; p += (b + 255) / 256 * 256; return q; };
  T* x = (T*)carve(S * F * (int64_t)sizeof(T));
  T* xbar = (T*)carve(S * F * (int64_t)sizeof(T));
  int32_t* perm = (int32_t*)carve(S * 4);
  const int64_t max_tiles = (S + G - 1) / G + H;
  int4* tiles = (int4*)carve(max_tiles * 16);
  int32_t* ntiles = (int32_t*)carve(4);
  cudaMemsetAsync(energy, 0, sizeof(T) * S, st);
  pool_mean_k<T><<<(unsigned)std::min<int64_t>(S, 148 * 8), POOL_THREADS, 0, st>>>(S, F, sptr, s, x);
  PNN_KCHECK("pool_mean_k");
  head_sort_k<<<1, 1024, 0, st>>>(S, H, G, head, perm, tiles, ntiles, d_err);
  PNN_KCHECK("head_sort_k");
  const int dm = std::max(F, std::max(d1, d2));
  const size_t smem = (size_t)G * (2 * d1 + 2 * d2 + 2 * dm) * sizeof(T);
  const int nq = (dm + POOL_RT - 1) / POOL_RT; // a thread per POOL_RT outputs
  const int rounds = (nq + POOL_MAXT - 1) / POOL_MAXT;
  const int nthr = std::max(64, ((nq + rounds - 1) / rounds + 31) / 32 * 32);
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(pooled_head_k<T, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    attr_set = true;
  }
  pooled_head_k<T, G><<<(unsigned)max_tiles, nthr, smem, st>>>(F, d1, d2, W, pw, perm, tiles, ntiles, x, energy,
                                                                       sb ? xbar : nullptr);
  PNN_KCHECK("pooled_head_k");
  int nl = 3;
  if (sb && N > 0) {
    const int64_t n = N * F;
    pool_bcast_k<T><<<(unsigned)std::min<int64_t>((n + 255) / 256, 148 * 16), 256, 0, st>>>(n, F, a2s, sptr, xbar, sb);
    PNN_KCHECK("pool_bcast_k");
    ++nl;
  }
  return nl;
}

template int launch_pool_head<float>(int64_t, int64_t, int, int, int, int, const float*, const int32_t*, const int32_t*,
                                     const int32_t*, const float*, const PoolHeadW&, void*, float*, float*, int*,
                                     cudaStream_t);
template int launch_pool_head<double>(int64_t, int64_t, int, int, int, int, const double*, const int32_t*, const int32_t*,
                                      const int32_t*, const double*, const PoolHeadW&, void*, double*, double*, int*,
                                      cudaStream_t);

} // namespace pnn
