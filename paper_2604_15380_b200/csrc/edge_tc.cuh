// edge_tc.cuh — edge kernels of the BF16 model with the filter contraction on the tcgen05 tensor cores (edge_tc.cu forward,
// edge_tc_bwd.cu reverse).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"

namespace pnn {

struct EdgeMmaArgs {
  int64_t N;
  int F, K;
  int rbf = 0; // 0 Gaussian, 1 Bessel
  float rc;
  const int32_t* rowptr;
  const int32_t* col;
  const Geom<float>* geom;
  const int* d_err;
};

int edge_mma_kp(int K); // columns of the MMA operands: K radial functions + 1 (flt_b), padded to a multiple of 16

// edge_tc.cu — forward message step on tcgen05 (features on the TMEM lanes, 16 consecutive CSR edges per MMA tile).
// fltT: one block's filter packed by pack_filter_tc (edge_tc_filter_elems(K) BF16 elements).
int64_t edge_tc_filter_elems(int K);
void pack_filter_tc(int F, int K, const double* fltW, const double* fltb, uint16_t* out);
int launch_edge_fwd_tc(const EdgeMmaArgs& a, const __nv_bfloat16* fltT, const __nv_bfloat16* phi, const float* s_in,
                       int64_t ld_sin, const __nv_bfloat16* v_in, const float* v_res, float* s1, int64_t ld_s1, float* v1,
                       const EdgeMirror& mir, cudaStream_t st);

// edge_tc_bwd.cu — reverse message step on tcgen05 (same arguments as launch_edge_bwd_mma plus the filter image fltT);
// adds the block's force contribution into fpart [edge_tc_bwd_num_slabs()][N][3].
int launch_edge_bwd_tc(const EdgeMmaArgs& a, const __nv_bfloat16* fltT, const __nv_bfloat16* phi, const __nv_bfloat16* v_in,
                       const __nv_bfloat16* sb16, const __nv_bfloat16* vb16, const float* vb1, __nv_bfloat16* phib16,
                       float* vb_in, float* fpart, int first_block, cudaStream_t st);
int edge_tc_bwd_num_slabs();

} // namespace pnn
