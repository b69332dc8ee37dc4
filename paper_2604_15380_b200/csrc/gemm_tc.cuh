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
  // Multi-head readout mode (launch_readout_tc): column tile = one head.  Rows whose structure has another head are
  // skipped; for the others eatom[m] = sum_n w2[n] silu(x[m][n] + bias[n]) + b2[head], opre[m][n - n0] = x + bias.
  int readout = 0;
  const int32_t* a2s = nullptr;
  const int32_t* head = nullptr;
  const float* w2 = nullptr;
  const float* b2 = nullptr;
  float* eatom = nullptr;
  float* opre = nullptr;
  int H = 0;
  int* d_err = nullptr;
  const unsigned long long* head_mask = nullptr; // [row tiles of 128]: bit h = some row of the tile uses head h
};

// Returns the number of kernels launched (0 or 1); < 0 when the TMA descriptor could not be encoded.
int launch_gemm_tc(int64_t M, int N, int K, const __nv_bfloat16* A, int64_t lda, const __nv_bfloat16* Wt, int64_t ldw,
                   const TcEpi& epi, cudaStream_t st);

// a6 on the tensor cores: eatom[i] = w2^h . silu(W1^h s_i + b1^h) + b2^h with h = head[a2s[i]] as ONE GEMM against the
// stacked first layers of all heads, W1all [H*Fh][F] (BF16): a column tile is exactly one head (Fh in {32, 64, 128}); a
// persistent CTA walks row tiles and, per row tile, only the heads that occur in it; the epilogue keeps the rows of its head.  bias = b1 of all heads [H*Fh], w2 [H*Fh], b2 [H].  opre (FP32 [N][Fh], pre-activation for R1) may be NULL.
// Returns kernels launched, or -1 if the shape is not supported (readout_tc_supported) or a TMA descriptor could not be
// encoded (an error for the caller).
bool readout_tc_supported(int F, int H);
// head_mask: scratch of ceil(N / 128) 64-bit words (which heads occur in each 128-row tile; written by a small kernel
// first, so that only the (row tile, head) pairs that exist are computed).  H <= 64.
int launch_readout_tc(int64_t N, int F, int H, const __nv_bfloat16* s16, const __nv_bfloat16* W1all, const float* b1,
                      const float* w2, const float* b2, const int32_t* a2s, const int32_t* head, float* opre,
                      float* eatom, int* d_err, unsigned long long* head_mask, cudaStream_t st);

// dst[i] = bf16(src[i])
int launch_f32_to_bf16(int64_t n, const float* src, __nv_bfloat16* dst, cudaStream_t st);

} // namespace pnn
