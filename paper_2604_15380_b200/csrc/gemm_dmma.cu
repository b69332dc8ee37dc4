// gemm_dmma.cu — FP64 dense node contractions (a3, a5 and their adjoints) on the FP64 tensor cores.
//
//   C[M,N] = epi( A[M,K] * B[K,N] ),  all row-major, K a multiple of 16, N a multiple of 64 (gemm_simt.cu takes the rest).
//
// tcgen05 has no FP64 kind (SURVEY.md §7 hard part 2); the FP64 tensor-core instruction of sm_100 is the warp-level
// mma.sync.m8n8k4 (DMMA): 512 flop per warp instruction at the same peak rate as eight DFMA warp instructions (measured
// 37.1 TFLOP/s for either), i.e. one eighth of the issue slots and no broadcast shared-memory loads per FMA, which is what
// held gemm_k<double> at 41-44 % of the FP64 peak.  CTA tile 128 x 64, eight warps of 32 x 32 (4 x 4 DMMA tiles, 32
// accumulators per lane), BK = 16 per stage, three stages filled by 16-byte asynchronous copies (rows past M zero-filled).
// Shared-memory strides are chosen so that every fragment load is the minimum two wavefronts: A rows 20 doubles apart, B rows
// 72 doubles apart.  Epilogues as gemm_simt.cu: bias, SiLU (+ pre-activation store), multiplication by silu'(aux), C +=.
#include "common.cuh"

namespace pnn {

namespace {

constexpr int BM = 128, BN = 64, BK = 16, NSTAGE = 3, NT = 256;
constexpr int LDA_S = BK + 4, LDB_S = BN + 8;
constexpr int STAGE_D = BM * LDA_S + BK * LDB_S; // doubles per stage

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16_zfill(void* smem_dst, const void* gsrc, bool valid) {
  const uint32_t s_ = (uint32_t)__cvta_generic_to_shared(smem_dst);
  const int n = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s_), "l"(gsrc), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__global__ void __launch_bounds__(NT, 2)
gemm_dmma_k(int64_t M, int N, int K, const double* __restrict__ A, int64_t lda, const double* __restrict__ B, int64_t ldb,
            double* __restrict__ C, int64_t ldc, GemmEpi<double> epi) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* const sm = reinterpret_cast<double*>(smem_raw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1; // 4 x 2 warps of 32 x 32
  const int row = lane >> 2, cp = lane & 3;
  const int64_t m0 = (int64_t)blockIdx.x * BM;
  const int n0 = blockIdx.y * BN;

  auto load_stage = [&](int st, int k0) {
    double* As = sm + st * STAGE_D;
    double* Bs = As + BM * LDA_S;
#pragma unroll
    for (int q = 0; q < (BM * BK / 2) / NT; ++q) { // A tile: BM rows x BK doubles, 16 bytes per copy
      const int v = tid + q * NT, r = v / (BK / 2), kq = v % (BK / 2);
      const int64_t m = m0 + r;
      const bool ok = m < M;
      cp_async16_zfill(As + r * LDA_S + kq * 2, A + (ok ? m : 0) * lda + k0 + kq * 2, ok);
    }
#pragma unroll
    for (int q = 0; q < (BK * BN / 2) / NT; ++q) { // B tile: BK rows x BN doubles
      const int v = tid + q * NT, r = v / (BN / 2), nq = v % (BN / 2);
      cp_async16_zfill(Bs + r * LDB_S + nq * 2, B + (int64_t)(k0 + r) * ldb + n0 + nq * 2, true);
    }
  };

  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

  const int nk = K / BK;
#pragma unroll
  for (int s = 0; s < NSTAGE - 1; ++s) {
    if (s < nk) load_stage(s, s * BK);
    cp_async_commit();
  }
  for (int kt = 0; kt < nk; ++kt) {
    cp_async_wait<NSTAGE - 2>(); // stage kt has landed (for this thread's copies)
    __syncthreads();             // ... for everyone's; and everyone has finished reading stage kt - 1
    if (kt + NSTAGE - 1 < nk) load_stage((kt + NSTAGE - 1) % NSTAGE, (kt + NSTAGE - 1) * BK);
    cp_async_commit();
    const double* As = sm + (kt % NSTAGE) * STAGE_D + (wm * 32 + row) * LDA_S + cp;
    const double* Bs = sm + (kt % NSTAGE) * STAGE_D + BM * LDA_S + cp * LDB_S + wn * 32 + row;
#pragma unroll
    for (int ks = 0; ks < BK / 4; ++ks) {
      double a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[i * 8 * LDA_S + ks * 4];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[ks * 4 * LDB_S + j * 8];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
  }

  // epilogue: lane holds rows wm*32 + i*8 + row, columns wn*32 + j*8 + 2 cp + {0, 1}
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t m = m0 + wm * 32 + i * 8 + row;
    if (m >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + wn * 32 + j * 8 + 2 * cp;
      double r0 = acc[i][j][0], r1 = acc[i][j][1];
      if (epi.bias) {
        const double2 bv = *reinterpret_cast<const double2*>(epi.bias + n);
        r0 += bv.x; r1 += bv.y;
      }
      if (epi.act == ACT_SILU) {
        if (epi.pre) *reinterpret_cast<double2*>(epi.pre + m * epi.ldpre + n) = make_double2(r0, r1);
        r0 = silu_f<double>(r0); r1 = silu_f<double>(r1);
      } else if (epi.act == ACT_MUL_DSILU) {
        const double2 xv = *reinterpret_cast<const double2*>(epi.aux + m * epi.ldaux + n);
        r0 *= dsilu_f<double>(xv.x); r1 *= dsilu_f<double>(xv.y);
      }
      double2* cptr = reinterpret_cast<double2*>(C + m * ldc + n);
      if (epi.accumulate) {
        const double2 cv = *cptr;
        r0 += cv.x; r1 += cv.y;
      }
      *cptr = make_double2(r0, r1);
    }
  }
}

} // namespace

bool gemm_dmma_supported(int64_t M, int N, int K) { return M > 0 && N % BN == 0 && K % BK == 0; }

int launch_gemm_dmma(int64_t M, int N, int K, const double* A, int64_t lda, const double* B, int64_t ldb, double* C,
                     int64_t ldc, const GemmEpi<double>& epi, cudaStream_t st) {
  if (M <= 0) return 0;
  constexpr size_t smem = sizeof(double) * NSTAGE * STAGE_D;
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(gemm_dmma_k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr_set = true;
  }
  dim3 grid((unsigned)((M + BM - 1) / BM), (unsigned)(N / BN));
  gemm_dmma_k<<<grid, NT, smem, st>>>(M, N, K, A, lda, B, ldb, C, ldc, epi);
  PNN_KCHECK("gemm_dmma_k");
  return 1;
}

} // namespace pnn
