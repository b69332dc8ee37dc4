// gemm_tc.cuh — BF16 tensor-core (tcgen05 + TMA + TMEM) GEMM of the BF16 model: declarations.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace pnn {

// C[M,N] = epi( A[M,K] * Wt[N,K]^T ), A and Wt BF16 row-major (both K-major), FP32 accumulation in TMEM.
// Epilogue order: + bias[n]; ACT_SILU stores the pre-activation to `pre` then applies SiLU; ACT_MUL_DSILU multiplies
// by silu'(aux[m][n]); `accumulate` adds the previous C.  Result goes to C (FP32, may be null) and / or Cb (BF16, may
// be null).  K and N are multiples of 32; lda is the row stride of A in elements (multiple of 8).
struct TcEpi {
  const float* bias = nullptr;
  int act = 0;
  float* pre = nullptr;
  int64_t ldpre = 0;
  const float* aux = nullptr;
  int64_t ldaux = 0;
  int accumulate = 0;
  float* C = nullptr;
  int64_t ldc = 0;
  __nv_bfloat16* Cb = nullptr;
  int64_t ldcb = 0;
};

// Returns the number of kernels launched (0 or 1); < 0 when the TMA descriptor could not be encoded.
int launch_gemm_tc(int64_t M, int N, int K, const __nv_bfloat16* A, int64_t lda, const __nv_bfloat16* Wt, int64_t ldw,
                   const TcEpi& epi, cudaStream_t st);

// dst[i] = bf16(src[i])
int launch_f32_to_bf16(int64_t n, const float* src, __nv_bfloat16* dst, cudaStream_t st);

} // namespace pnn
