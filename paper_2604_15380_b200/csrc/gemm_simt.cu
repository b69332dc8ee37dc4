// gemm_simt.cu — FP32 / FP64 dense node contractions (a3, a5 and their adjoints) on the ordinary ALUs.
//
//   C[M,N] = epi( A[M,K] * B[K,N] ),  all row-major, K a multiple of 16, N a multiple of 4.
//
// tcgen05 has no true-FP32 kind (SURVEY.md §7 hard part 2), so the FP32 model runs its Linear layers here: a
// register-blocked, shared-memory tiled FFMA kernel with a double-buffered global->register->shared pipeline.  The FP64
// model uses the FP64 tensor-core kernel of gemm_dmma.cu whenever the shape allows and the DFMA instance of this kernel
// otherwise (N not a multiple of 64); the BF16 model uses gemm_tc.cu (tcgen05 + TMA + TMEM).
// Epilogues fuse what follows each Linear in SURVEY.md §8(c): bias, SiLU (+ store of the pre-activation for the
// reverse sweep), multiplication by silu'(stored pre-activation), and accumulation into C (residual adjoints).
#include <type_traits>

#include "common.cuh"

namespace pnn {

namespace {

template <typename T> struct V4;
template <> struct V4<float> { using type = float4; };
template <> struct V4<double> { using type = double4; };

// acc[i][j] += a[i] b[j].  FP32: packed fma.rn.f32x2 on column pairs (two FMAs per issued instruction; the plain
// three-register FFMA issues at half rate on sm_100, B300_MICROARCH.md "Pipe rates").
template <typename T, int TM, int TN>
__device__ __forceinline__ void mac_tile(const T (&a)[TM], const T (&b)[TN], T (&acc)[TM][TN]) {
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
}
template <int TM, int TN>
__device__ __forceinline__ void mac_tile_f2(const float (&a)[TM], const float (&b)[TN], float (&acc)[TM][TN]) {
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    const float2 ai = make_float2(a[i], a[i]);
#pragma unroll
    for (int j = 0; j < TN; j += 2) {
      const float2 r = __ffma2_rn(ai, make_float2(b[j], b[j + 1]), make_float2(acc[i][j], acc[i][j + 1]));
      acc[i][j] = r.x; acc[i][j + 1] = r.y;
    }
  }
}
template <> __device__ __forceinline__ void mac_tile<float, 4, 4>(const float (&a)[4], const float (&b)[4], float (&acc)[4][4]) { mac_tile_f2<4, 4>(a, b, acc); }
template <> __device__ __forceinline__ void mac_tile<float, 8, 8>(const float (&a)[8], const float (&b)[8], float (&acc)[8][8]) { mac_tile_f2<8, 8>(a, b, acc); }

template <typename T, int BM, int BN, int TM, int TN, int BK, int MINB = 0>
__global__ void __launch_bounds__((BM / TM) * (BN / TN), MINB)
gemm_k(int64_t M, int N, int K, const T* __restrict__ A, int64_t lda, const T* __restrict__ B, int64_t ldb,
       T* __restrict__ C, int64_t ldc, GemmEpi<T> epi) {
  constexpr int NT = (BM / TM) * (BN / TN);
  constexpr int PAD = 4;
  using V = typename V4<T>::type;
  static_assert(TM % 4 == 0 && TN % 4 == 0, "micro tile in units of 4");
  constexpr int A_V = BM * BK / 4, B_V = BK * BN / 4;   // vectors per tile
  constexpr int A_LD = (A_V + NT - 1) / NT;             // vector loads per thread (the last one guarded if ragged)
  constexpr int B_LD = (B_V + NT - 1) / NT;

  __shared__ __align__(32) T As[2][BK][BM + PAD]; // transposed A tile
  __shared__ __align__(32) T Bs[2][BK][BN + PAD];

  const int tid = threadIdx.x;
  const int tx = tid % (BN / TN), ty = tid / (BN / TN);
  const int64_t m0 = (int64_t)blockIdx.x * BM;
  const int n0 = blockIdx.y * BN;

  T acc[TM][TN];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) acc[i][j] = T(0);

  V ra[A_LD], rb[B_LD];
  auto gload = [&](int k0) {
#pragma unroll
    for (int q = 0; q < A_LD; ++q) {
      const int v = tid + q * NT;          // vector index in the BM x (BK/4) tile
      const int r = v / (BK / 4), kq = v % (BK / 4);
      const int64_t m = m0 + r;
      if (A_V % NT != 0 && v >= A_V) continue;
      if (m < M) ra[q] = *reinterpret_cast<const V*>(A + m * lda + k0 + kq * 4);
      else ra[q] = V{T(0), T(0), T(0), T(0)};
    }
#pragma unroll
    for (int q = 0; q < B_LD; ++q) {
      const int v = tid + q * NT;          // vector index in the BK x (BN/4) tile
      const int r = v / (BN / 4), nq = v % (BN / 4);
      const int n = n0 + nq * 4;
      if (B_V % NT != 0 && v >= B_V) continue;
      if (n < N) rb[q] = *reinterpret_cast<const V*>(B + (int64_t)(k0 + r) * ldb + n);
      else rb[q] = V{T(0), T(0), T(0), T(0)};
    }
  };
  auto sstore = [&](int buf) {
#pragma unroll
    for (int q = 0; q < A_LD; ++q) {
      const int v = tid + q * NT;
      const int r = v / (BK / 4), kq = v % (BK / 4);
      if (A_V % NT != 0 && v >= A_V) continue;
      As[buf][kq * 4 + 0][r] = ra[q].x; As[buf][kq * 4 + 1][r] = ra[q].y;
      As[buf][kq * 4 + 2][r] = ra[q].z; As[buf][kq * 4 + 3][r] = ra[q].w;
    }
#pragma unroll
    for (int q = 0; q < B_LD; ++q) {
      const int v = tid + q * NT;
      const int r = v / (BN / 4), nq = v % (BN / 4);
      if (B_V % NT != 0 && v >= B_V) continue;
      *reinterpret_cast<V*>(&Bs[buf][r][nq * 4]) = rb[q];
    }
  };

  // micro-tile ownership: TM/4 groups of 4 rows spaced BM/(TM/4) apart, same for columns (conflict-free LDS.128)
  constexpr int GM = TM / 4, GN = TN / 4;
  constexpr int SM_ = BM / GM, SN_ = BN / GN;

  gload(0);
  sstore(0);
  __syncthreads();
  const int nk = K / BK;
  for (int kt = 0; kt < nk; ++kt) {
    const int buf = kt & 1;
    if (kt + 1 < nk) gload((kt + 1) * BK);
#pragma unroll 8 // not 16: the fully unrolled k-block (about 800 instructions) ran 16 % of its issue cycles short of
                 // instructions (ncu: stall_no_instruction 0.46 per issue); halves measured: cfg2 gemm_3N 61.1 -> 58.0 us,
                 // cfg3 split-K 67.6 -> 65.0 us
    for (int k = 0; k < BK; ++k) {
      T a[TM], b[TN];
#pragma unroll
      for (int gi = 0; gi < GM; ++gi) {
        const V t = *reinterpret_cast<const V*>(&As[buf][k][gi * SM_ + ty * 4]);
        a[gi * 4 + 0] = t.x; a[gi * 4 + 1] = t.y; a[gi * 4 + 2] = t.z; a[gi * 4 + 3] = t.w;
      }
#pragma unroll
      for (int gj = 0; gj < GN; ++gj) {
        const V t = *reinterpret_cast<const V*>(&Bs[buf][k][gj * SN_ + tx * 4]);
        b[gj * 4 + 0] = t.x; b[gj * 4 + 1] = t.y; b[gj * 4 + 2] = t.z; b[gj * 4 + 3] = t.w;
      }
      mac_tile<T, TM, TN>(a, b, acc);
    }
    if (kt + 1 < nk) {
      sstore(buf ^ 1);
      __syncthreads();
    }
  }

  // epilogue
#pragma unroll
  for (int gi = 0; gi < GM; ++gi)
#pragma unroll
    for (int ii = 0; ii < 4; ++ii) {
      const int64_t m = m0 + gi * SM_ + ty * 4 + ii;
      if (m >= M) continue;
#pragma unroll
      for (int gj = 0; gj < GN; ++gj) {
        const int n = n0 + gj * SN_ + tx * 4;
        if (n >= N) continue;
        T r[4];
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) r[jj] = acc[gi * 4 + ii][gj * 4 + jj];
        if (epi.bias) {
          const V bv = *reinterpret_cast<const V*>(epi.bias + n);
          r[0] += bv.x; r[1] += bv.y; r[2] += bv.z; r[3] += bv.w;
        }
        if (epi.act == ACT_SILU) {
          if (epi.pre) *reinterpret_cast<V*>(epi.pre + m * epi.ldpre + n) = V{r[0], r[1], r[2], r[3]};
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) r[jj] = silu_f<T>(r[jj]);
        } else if (epi.act == ACT_MUL_DSILU) {
          const V xv = *reinterpret_cast<const V*>(epi.aux + m * epi.ldaux + n);
          r[0] *= dsilu_f<T>(xv.x); r[1] *= dsilu_f<T>(xv.y); r[2] *= dsilu_f<T>(xv.z); r[3] *= dsilu_f<T>(xv.w);
        }
        V* cp = reinterpret_cast<V*>(C + m * ldc + n);
        if (epi.accumulate) {
          const V cv = *cp;
          r[0] += cv.x; r[1] += cv.y; r[2] += cv.z; r[3] += cv.w;
        }
        *cp = V{r[0], r[1], r[2], r[3]};
      }
    }
}

// ------------------------------------------------------------------------------------------ split-K over a CTA pair (FP32)
// The 64 x 128 tile with 8 x 8 values per thread reaches about twice the rate of the 4 x 4 tiles (one LDS.128 per 8 packed
// FMAs instead of per 4), but the small GEMMs of a molecular batch (10,354 x 128) make only 162 such tiles for 148 SMs.
// Here a CLUSTER of two CTAs shares one tile: CTA r contracts k in [r K/2, (r+1) K/2), then each CTA keeps the 32 rows of the
// tile that its threads hold in micro-tile group r, adds the partner's partial sums of those rows — read from the partner's
// shared memory over DSMEM — and runs the epilogue on them: 324 CTAs of 128 threads, three per SM, one wave.  The order of
// the sum is fixed (k-halves in rank order), so results are deterministic.
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cluster_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ float4 ld_peer4(uint32_t local_addr, uint32_t peer_rank) {
  uint32_t ra;
  float4 v;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(local_addr), "r"(peer_rank));
  asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(ra) : "memory");
  return v;
}

__global__ void __launch_bounds__(128, 3)
gemm_sk_k(int64_t M, int N, int K, const float* __restrict__ A, int64_t lda, const float* __restrict__ B, int64_t ldb,
          float* __restrict__ C, int64_t ldc, GemmEpi<float> epi) {
  constexpr int BM = 64, BN = 128, BK = 16, TM = 8, TN = 8, NT = 128, PAD = 4;
  constexpr int A_LD = BM * BK / 4 / NT, B_LD = BK * BN / 4 / NT; // 2 and 4 vector loads per thread and k-block
  // one buffer: the double-buffered tiles of the main loop, then the 16 KB exchange area of the split-K reduction
  __shared__ __align__(16) float smem[2 * BK * (BM + PAD) + 2 * BK * (BN + PAD)];
  float (*As)[BK][BM + PAD] = reinterpret_cast<float (*)[BK][BM + PAD]>(smem);
  float (*Bs)[BK][BN + PAD] = reinterpret_cast<float (*)[BK][BN + PAD]>(smem + 2 * BK * (BM + PAD));
  static_assert(2 * BK * (BM + PAD) + 2 * BK * (BN + PAD) >= NT * 32, "exchange area");
  const int tid = threadIdx.x;
  const int tx = tid % (BN / TN), ty = tid / (BN / TN);
  const int64_t m0 = (int64_t)blockIdx.x * BM;
  const int n0 = blockIdx.y * BN;
  const uint32_t rank = blockIdx.z; // rank in the cluster (1, 1, 2)
  const int kb0 = (int)rank * (K / 2), kb1 = kb0 + K / 2;

  float acc[TM][TN];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) acc[i][j] = 0.0f;
  float4 ra[A_LD], rb[B_LD];
  auto gload = [&](int k0) {
#pragma unroll
    for (int q = 0; q < A_LD; ++q) {
      const int v = tid + q * NT, r = v / (BK / 4), kq = v % (BK / 4);
      const int64_t m = m0 + r;
      ra[q] = (m < M) ? *reinterpret_cast<const float4*>(A + m * lda + k0 + kq * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll
    for (int q = 0; q < B_LD; ++q) {
      const int v = tid + q * NT, r = v / (BN / 4), nq = v % (BN / 4);
      rb[q] = *reinterpret_cast<const float4*>(B + (int64_t)(k0 + r) * ldb + n0 + nq * 4);
    }
  };
  auto sstore = [&](int buf) {
#pragma unroll
    for (int q = 0; q < A_LD; ++q) {
      const int v = tid + q * NT, r = v / (BK / 4), kq = v % (BK / 4);
      As[buf][kq * 4 + 0][r] = ra[q].x; As[buf][kq * 4 + 1][r] = ra[q].y;
      As[buf][kq * 4 + 2][r] = ra[q].z; As[buf][kq * 4 + 3][r] = ra[q].w;
    }
#pragma unroll
    for (int q = 0; q < B_LD; ++q) {
      const int v = tid + q * NT, r = v / (BN / 4), nq = v % (BN / 4);
      *reinterpret_cast<float4*>(&Bs[buf][r][nq * 4]) = rb[q];
    }
  };
  gload(kb0);
  sstore(0);
  __syncthreads();
  const int nk = (kb1 - kb0) / BK;
  for (int kt = 0; kt < nk; ++kt) {
    const int buf = kt & 1;
    if (kt + 1 < nk) gload(kb0 + (kt + 1) * BK);
#pragma unroll 8
    for (int k = 0; k < BK; ++k) {
      float a[TM], b[TN];
#pragma unroll
      for (int gi = 0; gi < 2; ++gi) {
        const float4 t = *reinterpret_cast<const float4*>(&As[buf][k][gi * 32 + ty * 4]);
        a[gi * 4 + 0] = t.x; a[gi * 4 + 1] = t.y; a[gi * 4 + 2] = t.z; a[gi * 4 + 3] = t.w;
      }
#pragma unroll
      for (int gj = 0; gj < 2; ++gj) {
        const float4 t = *reinterpret_cast<const float4*>(&Bs[buf][k][gj * 64 + tx * 4]);
        b[gj * 4 + 0] = t.x; b[gj * 4 + 1] = t.y; b[gj * 4 + 2] = t.z; b[gj * 4 + 3] = t.w;
      }
      mac_tile<float, TM, TN>(a, b, acc);
    }
    if (kt + 1 < nk) {
      sstore(buf ^ 1);
      __syncthreads();
    }
  }
  // exchange: a thread hands the partner the 4 x 8 sums of the micro-tile group the partner keeps (group 1 - rank) through
  // its own shared memory ([value][thread]: conflict-free), and fetches the partner's sums of its own group over DSMEM
  __syncthreads(); // the tiles are dead
  float r[4][8];
  auto exchange = [&](auto keep_c) { // compile-time group indices: acc stays in registers
    constexpr int keep = decltype(keep_c)::value, give = 1 - keep;
#pragma unroll
    for (int ii = 0; ii < 4; ++ii)
#pragma unroll
      for (int j4 = 0; j4 < 2; ++j4)
        *reinterpret_cast<float4*>(&smem[((ii * 2 + j4) * NT + tid) * 4]) =
            make_float4(acc[give * 4 + ii][j4 * 4 + 0], acc[give * 4 + ii][j4 * 4 + 1], acc[give * 4 + ii][j4 * 4 + 2],
                        acc[give * 4 + ii][j4 * 4 + 3]);
    cluster_sync();
#pragma unroll
    for (int ii = 0; ii < 4; ++ii)
#pragma unroll
      for (int j4 = 0; j4 < 2; ++j4) {
        const float4 p = ld_peer4(smem_addr(&smem[((ii * 2 + j4) * NT + tid) * 4]), (uint32_t)give);
        // rank 0 holds the first k-half: the sum is always (first half) + (second half)
        const float* mine = &acc[keep * 4 + ii][j4 * 4];
        r[ii][j4 * 4 + 0] = keep == 0 ? mine[0] + p.x : p.x + mine[0];
        r[ii][j4 * 4 + 1] = keep == 0 ? mine[1] + p.y : p.y + mine[1];
        r[ii][j4 * 4 + 2] = keep == 0 ? mine[2] + p.z : p.z + mine[2];
        r[ii][j4 * 4 + 3] = keep == 0 ? mine[3] + p.w : p.w + mine[3];
      }
  };
  if (rank == 0) exchange(std::integral_constant<int, 0>()); else exchange(std::integral_constant<int, 1>());
  const int keep = (int)rank;
  cluster_sync(); // the partner has read my shared memory: it may be released
  // epilogue on the kept rows (as gemm_k)
#pragma unroll
  for (int ii = 0; ii < 4; ++ii) {
    const int64_t m = m0 + keep * 32 + ty * 4 + ii;
    if (m >= M) continue;
#pragma unroll
    for (int gj = 0; gj < 2; ++gj) {
      const int n = n0 + gj * 64 + tx * 4;
      float x[4] = {r[ii][gj * 4 + 0], r[ii][gj * 4 + 1], r[ii][gj * 4 + 2], r[ii][gj * 4 + 3]};
      if (epi.bias) {
        const float4 bv = *reinterpret_cast<const float4*>(epi.bias + n);
        x[0] += bv.x; x[1] += bv.y; x[2] += bv.z; x[3] += bv.w;
      }
      if (epi.act == ACT_SILU) {
        if (epi.pre) *reinterpret_cast<float4*>(epi.pre + m * epi.ldpre + n) = make_float4(x[0], x[1], x[2], x[3]);
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) x[jj] = silu_f<float>(x[jj]);
      } else if (epi.act == ACT_MUL_DSILU) {
        const float4 xv = *reinterpret_cast<const float4*>(epi.aux + m * epi.ldaux + n);
        x[0] *= dsilu_f<float>(xv.x); x[1] *= dsilu_f<float>(xv.y); x[2] *= dsilu_f<float>(xv.z); x[3] *= dsilu_f<float>(xv.w);
      }
      float4* cp = reinterpret_cast<float4*>(C + m * ldc + n);
      if (epi.accumulate) {
        const float4 cv = *cp;
        x[0] += cv.x; x[1] += cv.y; x[2] += cv.z; x[3] += cv.w;
      }
      *cp = make_float4(x[0], x[1], x[2], x[3]);
    }
  }
}

} // namespace

template <typename T>
int launch_gemm(int64_t M, int N, int K, const T* A, int64_t lda, const T* B, int64_t ldb, T* C, int64_t ldc,
                const GemmEpi<T>& epi, cudaStream_t st) {
  if (M <= 0) return 0;
  if constexpr (sizeof(T) == 4) {
    // FP32: 64x128 tiles, 128 threads, 8x8 per thread (4 LDS.128 per 32 packed FMAs; 154 registers -> 3 CTAs per SM)
    // once there are two CTAs per SM; below that 64x64 tiles with 4x4 per thread (four times the warps, but two
    // LDS.128 per 8 packed FMAs: the shared-memory pipe binds it at ~28 TFLOP/s against ~50 for the 8x8 tile;
    // B200 measurements in DESIGN.md section 10).
    const int64_t wide_tiles = ((M + 63) / 64) * ((N + 127) / 128);
    if (N >= 128 && wide_tiles >= 2 * 148) {
      dim3 grid((unsigned)((M + 63) / 64), (unsigned)((N + 127) / 128));
      gemm_k<T, 64, 128, 8, 8, 16, 3><<<grid, 128, 0, st>>>(M, N, K, A, lda, B, ldb, C, ldc, epi); PNN_KCHECK("gemm_k");
    } else if (N % 128 == 0 && K % 32 == 0 && K >= 256 && 2 * wide_tiles >= 148 * 3 && 2 * wide_tiles <= 148 * 4) {
      // too few wide tiles for the SMs, but twice as many fill them (three CTAs of 128 threads per SM): two CTAs (a cluster)
      // per tile, each contracting half of K (gemm_sk_k).  Measured: cfg3 FP32 (8,192 x 256 outputs, 512 CTAs) 78 -> 70 us per
      // launch; cfg2 (10,354 x 128: 324 CTAs, 2.2 per SM) 31 -> 33 us, hence the lower bound
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)((M + 63) / 64), (unsigned)(N / 128), 2);
      cfg.blockDim = dim3(128);
      cfg.stream = st;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = 1; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 2;
      cfg.attrs = at; cfg.numAttrs = 1;
      cudaLaunchKernelEx(&cfg, gemm_sk_k, M, N, K, (const float*)A, lda, (const float*)B, ldb, (float*)C, ldc, epi);
      PNN_KCHECK("gemm_sk_k");
    } else {
      // The small GEMMs are one wave of co-resident CTAs, so their time follows the LARGEST number of CTAs on one SM
      // (measured, 64x64 tiles, K = 384: 2 per SM 30.8 us, 3 per SM 41.0 us, 4 per SM 45.1 us).  10,354 rows make 324
      // CTAs of 64 rows (three on 28 SMs) but 288 of 72 rows (two everywhere): take 72-row tiles when that pays.
      auto cost = [&](int bm) {
        const int64_t ctas = ((M + bm - 1) / bm) * ((N + 63) / 64), per_sm = (ctas + 147) / 148;
        const double f = per_sm <= 1 ? 0.8 : per_sm == 2 ? 1.0 : per_sm == 3 ? 1.33 : per_sm == 4 ? 1.46 : 0.37 * per_sm;
        return bm * f;
      };
      if (cost(72) < 0.97 * cost(64)) {
        dim3 grid((unsigned)((M + 71) / 72), (unsigned)((N + 63) / 64));
        gemm_k<T, 72, 64, 4, 4, 16><<<grid, 288, 0, st>>>(M, N, K, A, lda, B, ldb, C, ldc, epi); PNN_KCHECK("gemm_k");
      } else {
        dim3 grid((unsigned)((M + 63) / 64), (unsigned)((N + 63) / 64));
        gemm_k<T, 64, 64, 4, 4, 16><<<grid, 256, 0, st>>>(M, N, K, A, lda, B, ldb, C, ldc, epi); PNN_KCHECK("gemm_k");
      }
    }
  } else {
    // FP64: the tensor-core kernel (gemm_dmma.cu) whenever the shape allows; the ALU kernel takes the rest (N < 64, ...)
    if (gemm_dmma_supported(M, N, K)) return launch_gemm_dmma(M, N, K, A, lda, B, ldb, C, ldc, epi, st);
    // FP64: 128x128 tiles (8x8 per thread) for large problems, 64x64 (4x4) below ~2 waves of big tiles.
    const int64_t big_tiles = ((M + 127) / 128) * ((N + 127) / 128);
    if (big_tiles >= 2 * 148 && N >= 128) {
      dim3 grid((unsigned)((M + 127) / 128), (unsigned)((N + 127) / 128));
      gemm_k<T, 128, 128, 8, 8, 8><<<grid, 256, 0, st>>>(M, N, K, A, lda, B, ldb, C, ldc, epi); PNN_KCHECK("gemm_k");
    } else {
      dim3 grid((unsigned)((M + 63) / 64), (unsigned)((N + 63) / 64));
      gemm_k<T, 64, 64, 4, 4, 16><<<grid, 256, 0, st>>>(M, N, K, A, lda, B, ldb, C, ldc, epi); PNN_KCHECK("gemm_k");
    }
  }
  return 1;
}

template int launch_gemm<float>(int64_t, int, int, const float*, int64_t, const float*, int64_t, float*, int64_t,
                                const GemmEpi<float>&, cudaStream_t);
template int launch_gemm<double>(int64_t, int, int, const double*, int64_t, const double*, int64_t, double*, int64_t,
                                 const GemmEpi<double>&, cudaStream_t);

} // namespace pnn
