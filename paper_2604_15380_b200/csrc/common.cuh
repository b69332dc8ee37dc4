// common.cuh — shared declarations of the CUDA library (internal; the public boundary is include/pnn.h).
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace pnn {

// Records the first failed kernel launch (checked with cudaPeekAtLastError after every launch); pnn_api.cu
// turns it into PNN_ERR_CUDA.
void note_launch(const char* where);
#define PNN_KCHECK(name) ::pnn::note_launch(name)

// device-side error flags (workspace->d_err)
enum : int { ERRF_EDGE_OVERFLOW = 1, ERRF_BAD_Z = 2, ERRF_BAD_HEAD = 4, ERRF_STALE_GRAPH = 8 };

// Per-edge geometry in model precision: unit vector receiver->sender image and distance.
template <typename T>
struct __align__(sizeof(T) * 4) Geom {
  T ux, uy, uz, d;
};

// Per-structure cell-grid descriptor written by the graph builder.
struct GridDesc {
  double C[9];      // lattice rows (identity when not periodic)
  double Ci[9];     // inverse
  double fmin[3];   // fractional origin of the binning box (0 on periodic axes)
  double fscale[3]; // cells per unit of fractional coordinate on each axis
  int32_t dim[3];   // cells per axis
  int32_t per[3];   // axis is periodic
  int32_t periodic; // any axis periodic
  int32_t ncell;    // dim[0]*dim[1]*dim[2]
};

template <typename T>
__device__ __forceinline__ T silu_f(T x) {
  return x / (T(1) + exp(-x));
}
template <>
__device__ __forceinline__ float silu_f<float>(float x) {
  return x / (1.0f + expf(-x));
}
// silu'(x) = sg (1 + x (1 - sg)), sg = 1/(1+e^-x)
template <typename T>
__device__ __forceinline__ T dsilu_f(T x) {
  const T sg = T(1) / (T(1) + exp(-x));
  return sg * (T(1) + x * (T(1) - sg));
}
template <>
__device__ __forceinline__ float dsilu_f<float>(float x) {
  const float sg = 1.0f / (1.0f + expf(-x));
  return sg * (1.0f + x * (1.0f - sg));
}

// Radial basis function k of type `rbf` at distance d and its derivative (SURVEY.md §8(c) B3 / reading Q2):
//   rbf 0  Gaussian  g_k = exp(-gamma (d - k dmu)^2),  dmu = r_c / (K - 1), gamma = 1 / (2 dmu^2)
//   rbf 1  Bessel    b_n = sqrt(2 / r_c) sin(n pi d / r_c) / d,  n = k + 1   (the paper's lead model)
template <typename T>
__device__ __forceinline__ void rbf_eval(int rbf, int k, T d, T rc, T dmu, T gamma, T& g, T& gd) {
  if (rbf == 1) {
    const T wn = T(k + 1) * T(3.14159265358979323846) / rc, A = sqrt(T(2) / rc);
    T sn, cs;
    sincos(wn * d, &sn, &cs);
    g = A * sn / d;
    gd = A * wn * cs / d - g / d;
  } else {
    const T dd = d - T(k) * dmu;
    g = exp(-gamma * dd * dd);
    gd = -T(2) * gamma * dd * g;
  }
}
template <>
__device__ __forceinline__ void rbf_eval<float>(int rbf, int k, float d, float rc, float dmu, float gamma, float& g, float& gd) {
  if (rbf == 1) {
    const float wn = (float)(k + 1) * 3.14159265358979323846f / rc, A = sqrtf(2.0f / rc);
    float sn, cs;
    sincosf(wn * d, &sn, &cs);
    g = A * sn / d;
    gd = A * wn * cs / d - g / d;
  } else {
    const float dd = d - (float)k * dmu;
    g = expf(-gamma * dd * dd);
    gd = -2.0f * gamma * dd * g;
  }
}

// ---------------------------------------------------------------------------------------------
// launch wrappers (one per kernel family); every wrapper returns the number of kernels launched
// ---------------------------------------------------------------------------------------------

// graph.cu
struct GraphBuffers {
  int32_t* a2s;        // [N] atom -> structure
  GridDesc* desc;      // [S]
  int32_t* ncell;      // [S+1] cells per structure, then exclusive scan in cell_off
  int32_t* cell_off;   // [S+1]
  int32_t* cid;        // [N] global cell of atom
  int32_t* cell_cnt;   // [N+S+1]
  int32_t* cell_start; // [N+S+2]
  int32_t* cell_fill;  // [N+S+1]
  int32_t* sorted;     // [N] atoms ordered by (structure, cell, index)
  int32_t* deg;        // [N+1]
  int32_t* rowptr;     // [N+1]
  int32_t* col;        // [Emax]
  int8_t* shift;       // [Emax,3]
  void* geom;          // [Emax] Geom<T>
  int32_t* scan_tmp;   // scratch for the scans
  int64_t max_edges;
  int* d_err;   // sticky flags (ERRF_*), cleared by pnn_check_async_errors
  int* d_ovf;   // ERRF_EDGE_OVERFLOW or 0 for the CURRENT graph: rewritten by every build, tested by the edge kernels
  unsigned long long* d_poschk; // [2]: checksum of the positions the graph was built from / scratch for pnn_eval's check
  // max-neighbour cap (pnn_config.max_neighbors > 0 only; NULL otherwise): scratch of the compaction pass
  int32_t* cap_col = nullptr;   // [Emax]
  int8_t* cap_shift = nullptr;  // [Emax,3]
  void* cap_geom = nullptr;     // [Emax] Geom<T>
  uint8_t* cap_keep = nullptr;  // [Emax]
  int32_t* cap_deg = nullptr;   // [N+1]
  int32_t* cap_rowptr = nullptr; // [N+1]
};
// Flags ERRF_STALE_GRAPH when the checksum of pos differs from the one recorded by the last launch_graph_build.
int launch_pos_check(const GraphBuffers& g, int64_t N, const double* pos, cudaStream_t st);
int launch_graph_build(const GraphBuffers& g, int64_t N, int64_t S, const double* pos, const int32_t* struct_ptr,
                       const double* cell, const uint8_t* pbc, double rc, int prec, int all_images, int max_neighbors,
                       cudaStream_t st);

// gemm_simt.cu :  C[M,N] (ldc) = epi( A[M,K] (lda) * B[K,N] (ldb) )
enum : int { ACT_NONE = 0, ACT_SILU = 1, ACT_MUL_DSILU = 2 };
template <typename T>
struct GemmEpi {
  const T* bias = nullptr; // [N] added before the activation
  int act = ACT_NONE;
  T* pre = nullptr;        // ACT_SILU: also store the pre-activation here (ld = ldpre)
  int64_t ldpre = 0;
  const T* aux = nullptr;  // ACT_MUL_DSILU: result *= silu'(aux[m][n]) (ld = ldaux)
  int64_t ldaux = 0;
  int accumulate = 0;      // C += result
};
template <typename T>
int launch_gemm(int64_t M, int N, int K, const T* A, int64_t lda, const T* B, int64_t ldb, T* C, int64_t ldc,
                const GemmEpi<T>& epi, cudaStream_t st);

// gemm_dmma.cu: the FP64 contraction on the FP64 tensor cores (N a multiple of 64, K of 16)
bool gemm_dmma_supported(int64_t M, int N, int K);
int launch_gemm_dmma(int64_t M, int N, int K, const double* A, int64_t lda, const double* B, int64_t ldb, double* C,
                     int64_t ldc, const GemmEpi<double>& epi, cudaStream_t st);

// edge.cu
template <typename T>
struct EdgeArgs {
  int64_t N;
  int F, K;
  int rbf = 0; // 0 Gaussian, 1 Bessel (rbf_eval)
  double rc;
  const int32_t* rowptr;
  const int32_t* col;
  const Geom<T>* geom;
  const T* fltW; // [3F][K]
  const T* fltb; // [3F]
  const int* d_err;
};
// optional BF16 copies of the forward outputs (BF16 model: operands of the next GEMMs)
struct EdgeMirror {
  __nv_bfloat16* s1 = nullptr;
  int64_t ld_s1 = 0;
  __nv_bfloat16* v1 = nullptr;
};
// forward message step (B3b): s1 = s_in + sum, v1 = v_res + sum.  s_in/s1 have leading dimensions.  phi and v_in
// are the gathered sender payloads (type PT = T, or BF16 in the BF16 model); v_res is the receiver's own row of v.
template <typename T, typename PT>
int launch_edge_fwd(const EdgeArgs<T>& a, const PT* phi, const T* s_in, int64_t ld_sin, const PT* v_in,
                    const T* v_res, T* s1, int64_t ld_s1, T* v1, const EdgeMirror& mir, cudaStream_t st);
// reverse message step (R3 + R4 partial): from sb1 [N,F], vb1 [N,3F] and the forward phi, v_in produce
// phib [N,3F], vb_in [N,3F] and add this block's force contribution into fpart [nslab][N][3].
// (phib16 != null: phib is written there in BF16 instead of to phib.)
template <typename T, typename PT>
int launch_edge_bwd(const EdgeArgs<T>& a, const PT* phi, const PT* v_in, const T* sb1, const T* vb1, T* phib,
                    T* vb_in, T* fpart, int first_block, __nv_bfloat16* phib16, cudaStream_t st);
int edge_num_slabs(int F);
// edge_scatter.cu — the reverse message step in scatter form (atomic adds) for asymmetric edge sets (max-neighbour cap)
template <typename T, typename PT>
int launch_edge_bwd_scatter(const EdgeArgs<T>& a, const PT* phi, const PT* v_in, const T* sb1, const T* vb1, T* phib,
                            T* vb_in, T* fslab, int first_block, cudaStream_t st, const T* wt = nullptr,
                            const T* dt = nullptr); // wt, dt: the FP32 edge tape (w, dw/dd [E][3][F]) or NULL = recompute

// edge_warp.cu — the FP32 model's edge kernels (warp per receiver, filter rows in registers, no CTA barriers)
// wt, dt (both or neither): edge tape [E][3][F] that receives the filter value w and dw/dd of every edge; the reverse
// kernel reads them back instead of recomputing the filter.
int launch_edge_fwd_warp(const EdgeArgs<float>& a, const float* phi, const float* s_in, int64_t ld_sin, const float* v_in,
                         float* s1, int64_t ld_s1, float* v1, float* wt, float* dt, cudaStream_t st);
int launch_edge_bwd_warp(const EdgeArgs<float>& a, const float* phi, const float* v_in, const float* sb1, const float* vb1,
                         const float* wt, const float* dt, float* phib, float* vb_in, float* fpart, int first_block,
                         cudaStream_t st);
int edge_warp_num_slabs(int F, int K);

// node.cu
// (the trailing BF16 pointers are optional copies / replacements of an output for the BF16 model's GEMM operands)
template <typename T>
int launch_embed(int64_t N, int F, int Zmax, const int32_t* Z, const T* emb, T* s, int* d_err, cudaStream_t st,
                 __nv_bfloat16* s16 = nullptr);
// s[i][f] += sum_q globW[f][q] glob[a2s[i]][q] (global attributes: charge, spin; reading Q30); s16: BF16 copy rewritten
template <typename T>
int launch_embed_globals(int64_t N, int F, int G, const int32_t* a2s, const double* glob, const T* globW, T* s,
                         __nv_bfloat16* s16, cudaStream_t st);
// edge_dmma.cu: FP64 edge kernels with the filter contraction on the FP64 tensor cores (F a multiple of 64)
bool edge_dmma_supported(int F, int K);
int launch_edge_fwd_dmma(const EdgeArgs<double>& a, const double* phi, const double* s_in, int64_t ld_sin, const double* v_in,
                         const double* v_res, double* s1, int64_t ld_s1, double* v1, cudaStream_t st);
int launch_edge_bwd_dmma(const EdgeArgs<double>& a, const double* phi, const double* v_in, const double* sb1,
                         const double* vb1, double* phib, double* vb_in, double* fpart, int first_block, cudaStream_t st);
int edge_dmma_num_slabs(int F);
// schnet.cu: edge-side kernels of the second backbone (continuous-filter convolution; reading Q31)
template <typename T>
int launch_sch_rbf(int64_t N, int64_t maxE, int K, int KP, int rbf, double rc, const int32_t* rowptr, const void* geom, T* G,
                   T* Gd, const int* d_ovf, cudaStream_t st);
template <typename T>
int launch_sch_conv_fwd(int64_t N, int F, double rc, const int32_t* rowptr, const int32_t* col, const void* geom, const T* Wf,
                        const T* x1, T* m, const int* d_ovf, cudaStream_t st);
template <typename T>
int launch_sch_conv_bwd(int64_t N, int F, double rc, const int32_t* rowptr, const int32_t* col, const void* geom, const T* Wf,
                        const T* dWf, const T* x1, const T* mb, T* x1b, T* forces, int first_block, const int* d_ovf,
                        cudaStream_t st);
// pool_head.cu: the paper's graph-level heads (mean pooling -> shared layers -> per-head branch layers; reading Q29)
// element offsets in the device weight buffer (every array starts on a multiple of 4 elements: 16-byte loads): shared
// layers P1 [d1][F], p1, P2 [d1][d1], p2 and the transposes P1t [F][d1], P2t [d1][d1]; per head, at br + h * br_stride:
// B1 [d2][d1] at 0, q1, B2 [d2][d2], q2, w3, q3, B1t [d1][d2], B2t [d2][d2] at the o* offsets
struct PoolHeadW {
  int64_t P1, p1, P2, p2, P1t, P2t, br, br_stride;
  int64_t oq1, oB2, oq2, ow3, oq3, oB1t, oB2t;
};
int64_t pool_head_scratch_bytes(int64_t maxS, int F, int H, size_t elem);
bool pool_head_supported(int F, int d1, int d2, int H, size_t elem);
template <typename T>
int launch_pool_head(int64_t N, int64_t S, int F, int H, int d1, int d2, const T* s, const int32_t* a2s,
                     const int32_t* sptr, const int32_t* head, const T* W, const PoolHeadW& pw, void* scratch, T* energy,
                     T* sb, int* d_err, cudaStream_t st);
// IT: storage type of P | Q and of the gate values a (= T, or BF16 in the BF16 model)
template <typename T, typename IT>
int launch_norm(int64_t N, int F, const IT* PQ, T* sn, T eps, cudaStream_t st, __nv_bfloat16* sn16 = nullptr);
template <typename T, typename IT>
int launch_update(int64_t N, int F, const T* sn, const T* v1, const IT* PQ, const IT* a, T* s_out, T* v_out,
                  cudaStream_t st, __nv_bfloat16* s16 = nullptr, __nv_bfloat16* v16 = nullptr);
template <typename T, typename IT>
int launch_update_bwd1(int64_t N, int F, const T* sb, const T* vb, const IT* a, const IT* PQ, T* ab, T* PQb,
                       cudaStream_t st, __nv_bfloat16* ab16 = nullptr);
template <typename T, typename IT>
int launch_update_bwd2(int64_t N, int F, const T* zb, const IT* PQ, T eps, T* sb, T* PQb, cudaStream_t st,
                       __nv_bfloat16* PQb16 = nullptr, __nv_bfloat16* sb16 = nullptr);
// readout (B5 / R1).  W1t: [H][F][F/2] (transposed), W1: [H][F/2][F], b1 [H][F/2], w2 [H][F/2], b2 [H].
template <typename T>
int launch_readout(int64_t N, int64_t S, int F, int H, const T* s, const int32_t* a2s, const int32_t* head,
                   const int32_t* struct_ptr, const T* W1t, const T* b1, const T* w2, const T* b2, T* opre, T* eatom,
                   T* energy, int* d_err, cudaStream_t st);
// blended multi-head readout: hw [S][H] branch weights, heads with hw < thr skipped; opre_all [N][H][F/2]
template <typename T>
int launch_readout_blend(int64_t N, int64_t S, int F, int H, const T* s, const int32_t* a2s, const T* hw, T thr,
                         const int32_t* struct_ptr, const T* W1t, const T* b1, const T* w2, const T* b2, T* opre_all,
                         T* eatom, T* energy, cudaStream_t st);
template <typename T>
int launch_readout_blend_bwd(int64_t N, int F, int H, const T* opre_all, const int32_t* a2s, const T* hw, T thr,
                             const T* W1, const T* w2, T* sb, cudaStream_t st);
template <typename T>
int launch_struct_sum(int64_t S, const int32_t* struct_ptr, const T* eatom, T* energy, cudaStream_t st);
template <typename T>
int launch_readout_bwd(int64_t N, int F, int H, const T* opre, const int32_t* a2s, const int32_t* head, const T* W1,
                       const T* w2, T* sb, cudaStream_t st);
template <typename T>
int launch_force_assemble(int64_t N, int nslab, const T* fpart, T* forces, cudaStream_t st);

// ---- branch.cu: composition -> softmax branch weights -------------------------------
// Device parameter layout: per layer Wt [in][out] (input-major, i.e. the transpose of the C ABI's [out][in]) at off_w[l],
// then b [out] at off_b[l].
struct BranchMlpDims {
  int n_layers;
  int width[9];
  int off_w[8], off_b[8];
};
template <typename T>
int launch_branch_mlp(int64_t S, const BranchMlpDims& dm, const int32_t* Z, const int32_t* sptr, const T* params,
                      T* out, int* d_err, cudaStream_t st);
double measure_alu_peak(bool fp64, void* scratch, cudaStream_t st);   // TFLOP/s of the FMA pipe (packed FP32 / FP64)
double measure_l2_peak(void* buf, int64_t bytes, cudaStream_t st);      // GB/s of L2-resident reads (512-byte rows per warp)

} // namespace pnn
