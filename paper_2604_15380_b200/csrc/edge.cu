// edge.cu — a4 fused edge/message kernel and the edge part of a7 (analytic adjoint), FP32 / FP64.
//
// Forward: per edge e = (i <- j): g_k(d) = exp(-gamma (d - mu_k)^2), c(d) = (cos(pi d/r_c)+1)/2,
// w_e = (flt_W g + flt_b) c,  x_e = phi_j o w_e,  s'_i = s_i + sum x^ss,  v'_i = v_i + sum (x^vs u_e + x^vv o v_j).
// Reverse (R3, R4): the scatters to the sender are rewritten as gathers over the node's own receiver segment,
// valid because the edge set is symmetric, d and hence w_e are equal on (i<-j) and (j<-i) and u flips sign
// (note under R4).  No atomics anywhere; rows are summed in CSR order.
//
// Thread mapping: a CTA owns RB consecutive receivers (one contiguous CSR edge range) and one slab of FS <= 128
// features.  Thread (c, f) owns filter row c*F + f (c = ss / vs / vv chunk): its K filter weights live in
// registers for the CTA's lifetime, the per-edge radial basis (times cutoff) is staged once per 32-edge tile in
// shared memory and read as broadcast vectors, the sender rows phi_j / v_j (and their adjoints) are gathered with
// fully coalesced loads (consecutive threads = consecutive features), and each thread keeps its running segment
// sum in registers until the receiver changes.  Per-receiver partials meet in shared memory and are written out
// coalesced once per work item.
#include <algorithm>

#include "common.cuh"

namespace pnn {

namespace {

constexpr int ET = 32; // edges per staged tile

template <typename T> __device__ __forceinline__ T t_exp(T x);
template <> __device__ __forceinline__ float t_exp<float>(float x) { return expf(x); }
template <> __device__ __forceinline__ double t_exp<double>(double x) { return exp(x); }
template <typename T> __device__ __forceinline__ void t_sincos(T x, T* s, T* c);
template <> __device__ __forceinline__ void t_sincos<float>(float x, float* s, float* c) { sincosf(x, s, c); }
template <> __device__ __forceinline__ void t_sincos<double>(double x, double* s, double* c) { sincos(x, s, c); }

// gathered payloads (phi_j, v_j) may be stored narrower than the arithmetic type (BF16 model, reading Q19)
template <typename T, typename PT> __device__ __forceinline__ T ldp(const PT* p) { return (T)(*p); }
template <> __device__ __forceinline__ float ldp<float, __nv_bfloat16>(const __nv_bfloat16* p) {
  return __bfloat162float(*p);
}

template <typename T, int KP>
__device__ __forceinline__ void load_filter_row(const EdgeArgs<T>& a, int row, T (&w)[KP], T& bias) {
#pragma unroll
  for (int k = 0; k < KP; ++k) w[k] = (k < a.K) ? a.fltW[(int64_t)row * a.K + k] : T(0);
  bias = a.fltb[row];
}

// w . g with g read from shared memory as 16-byte broadcast vectors (KP is a multiple of 4, rows 16-byte aligned)
template <int KP>
__device__ __forceinline__ float dotK(const float (&w)[KP], const float* __restrict__ g) {
  float acc = 0.0f;
#pragma unroll
  for (int k = 0; k < KP; k += 4) {
    const float4 t = *reinterpret_cast<const float4*>(g + k);
    acc = fmaf(w[k], t.x, acc); acc = fmaf(w[k + 1], t.y, acc);
    acc = fmaf(w[k + 2], t.z, acc); acc = fmaf(w[k + 3], t.w, acc);
  }
  return acc;
}
template <int KP>
__device__ __forceinline__ double dotK(const double (&w)[KP], const double* __restrict__ g) {
  // four independent chains: a single DFMA chain of KP links is bound by the FP64 pipe's latency, not its rate
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
#pragma unroll
  for (int k = 0; k < KP; k += 4) {
    const double2 t = *reinterpret_cast<const double2*>(g + k);
    const double2 u = *reinterpret_cast<const double2*>(g + k + 2);
    a0 = fma(w[k], t.x, a0); a1 = fma(w[k + 1], t.y, a1);
    a2 = fma(w[k + 2], u.x, a2); a3 = fma(w[k + 3], u.y, a3);
  }
  return (a0 + a1) + (a2 + a3);
}

// ------------------------------------------------------------------------------------------ forward
template <typename T, int KP, typename PT>
__global__ void __launch_bounds__(384)
edge_fwd_k(EdgeArgs<T> a, int FS, int RB, const PT* __restrict__ phi, const T* __restrict__ s_in, int64_t ld_sin,
           const PT* __restrict__ v_in, const T* __restrict__ v_res, T* __restrict__ s1, int64_t ld_s1,
           T* __restrict__ v1, EdgeMirror mir) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* G = reinterpret_cast<T*>(smem_raw);            // [ET][KP]
  T* Cc = G + ET * KP;                              // [ET]
  T* U = Cc + ET;                                   // [ET][4]  ux uy uz d
  T* Acc = U + ET * 4;                              // [RB][7][FS]
  int* J = reinterpret_cast<int*>(Acc + (size_t)RB * 7 * FS); // [ET]
  int* RP = J + ET;                                 // [RB+1]

  const int F = a.F, K = a.K;
  const int nthr = blockDim.x, tid = threadIdx.x;
  const int c = tid / FS, fl = tid % FS;
  const int f = blockIdx.y * FS + fl;
  T w[KP], bias;
  load_filter_row<T, KP>(a, c * F + f, w, bias);
  const T rc = (T)a.rc;
  const T dmu = (K > 1) ? rc / (T)(K - 1) : rc;
  const T gamma = T(1) / (T(2) * dmu * dmu);
  const T pi_rc = (T)(3.14159265358979323846 / a.rc);
  const int64_t nwork = (a.N + RB - 1) / RB;

  for (int64_t wk = blockIdx.x; wk < nwork; wk += gridDim.x) {
    const int64_t i0 = wk * RB;
    const int nrecv = (int)min((int64_t)RB, a.N - i0);
    __syncthreads(); // previous work item fully written out
    if (tid <= nrecv) RP[tid] = a.rowptr[i0 + tid];
    __syncthreads();
    const int ea = RP[0], eb = RP[nrecv];
    int r = 0, rend = RP[1];
    T acc0 = T(0), acc1 = T(0), acc2 = T(0);
    auto flush = [&]() {
      if (c == 0) Acc[(r * 7 + 0) * FS + fl] = acc0;
      else {
        const int base = (c == 1) ? 1 : 4;
        Acc[(r * 7 + base + 0) * FS + fl] = acc0;
        Acc[(r * 7 + base + 1) * FS + fl] = acc1;
        Acc[(r * 7 + base + 2) * FS + fl] = acc2;
      }
      acc0 = acc1 = acc2 = T(0);
    };
    for (int t0 = ea; t0 < eb; t0 += ET) {
      const int nE = min(ET, eb - t0);
      __syncthreads();
      for (int q = tid; q < nE; q += nthr) {
        const Geom<T> gq = a.geom[t0 + q];
        U[q * 4 + 0] = gq.ux; U[q * 4 + 1] = gq.uy; U[q * 4 + 2] = gq.uz; U[q * 4 + 3] = gq.d;
        T sn, cs;
        t_sincos<T>(pi_rc * gq.d, &sn, &cs);
        Cc[q] = T(0.5) * (cs + T(1));
        J[q] = a.col[t0 + q];
      }
      __syncthreads();
      for (int q = tid; q < nE * KP; q += nthr) {
        const int e = q / KP, k = q % KP;
        T g = T(0), gd = T(0);
        if (k < K) rbf_eval<T>(a.rbf, k, U[e * 4 + 3], rc, dmu, gamma, g, gd);
        G[q] = g * Cc[e];
      }
      __syncthreads();
      for (int q = 0; q < nE; ++q) {
        const int e = t0 + q;
        while (e >= rend) { flush(); ++r; rend = RP[r + 1]; }
        const int64_t j = J[q];
        const T wv = fma(bias, Cc[q], dotK<KP>(w, G + q * KP));
        if (c == 0) {
          acc0 = fma(ldp<T, PT>(phi + j * 3 * F + f), wv, acc0);
        } else if (c == 1) {
          const T x = ldp<T, PT>(phi + j * 3 * F + F + f) * wv;
          acc0 = fma(x, U[q * 4 + 0], acc0);
          acc1 = fma(x, U[q * 4 + 1], acc1);
          acc2 = fma(x, U[q * 4 + 2], acc2);
        } else if (v_in != nullptr) {
          const T x = ldp<T, PT>(phi + j * 3 * F + 2 * F + f) * wv;
          acc0 = fma(x, ldp<T, PT>(v_in + (j * 3 + 0) * F + f), acc0);
          acc1 = fma(x, ldp<T, PT>(v_in + (j * 3 + 1) * F + f), acc1);
          acc2 = fma(x, ldp<T, PT>(v_in + (j * 3 + 2) * F + f), acc2);
        }
      }
    }
    while (r < nrecv) { flush(); ++r; }
    __syncthreads();
    // coalesced write-out: item (r, comp, fl), comp 0 = s, 1..3 = v_a
    for (int idx = tid; idx < nrecv * 4 * FS; idx += nthr) {
      const int rr = idx / (4 * FS), rem = idx % (4 * FS);
      const int comp = rem / FS, ff = rem % FS;
      const int64_t i = i0 + rr;
      const int fo = blockIdx.y * FS + ff;
      if (comp == 0) {
        const T r = s_in[i * ld_sin + fo] + Acc[(rr * 7 + 0) * FS + ff];
        s1[i * ld_s1 + fo] = r;
        if (mir.s1) mir.s1[i * mir.ld_s1 + fo] = __float2bfloat16_rn((float)r);
      } else {
        const T vin = v_res ? v_res[(i * 3 + (comp - 1)) * F + fo] : T(0);
        const T r = vin + Acc[(rr * 7 + comp) * FS + ff] + Acc[(rr * 7 + 3 + comp) * FS + ff];
        v1[(i * 3 + (comp - 1)) * F + fo] = r;
        if (mir.v1) mir.v1[(i * 3 + (comp - 1)) * F + fo] = __float2bfloat16_rn((float)r);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------ reverse
template <typename T, int KP, typename PT>
__global__ void __launch_bounds__(384)
edge_bwd_k(EdgeArgs<T> a, int FS, int RB, const PT* __restrict__ phi, const PT* __restrict__ v_in,
           const T* __restrict__ sb1, const T* __restrict__ vb1, T* __restrict__ phib, T* __restrict__ vb_in,
           T* __restrict__ fpart, int first_block, __nv_bfloat16* __restrict__ phib16) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* G1 = reinterpret_cast<T*>(smem_raw);           // [ET][KP]  g_k c
  T* G2 = G1 + ET * KP;                             // [ET][KP]  c g'_k + c' g_k
  T* Cc = G2 + ET * KP;                             // [ET]      c
  T* Cp = Cc + ET;                                  // [ET]      c'
  T* U = Cp + ET;                                   // [ET][4]   ux uy uz d
  T* Acc = U + ET * 4;                              // [RB][5][FS]
  T* FW = Acc + (size_t)RB * 5 * FS;                // [RB][12][3]
  int* J = reinterpret_cast<int*>(FW + RB * 12 * 3);
  int* RP = J + ET;

  const int F = a.F, K = a.K;
  const int nthr = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = (nthr + 31) >> 5;
  const int c = tid / FS, fl = tid % FS;
  const int f = blockIdx.y * FS + fl;
  T w[KP], bias;
  load_filter_row<T, KP>(a, c * F + f, w, bias);
  const T rc = (T)a.rc;
  const T dmu = (K > 1) ? rc / (T)(K - 1) : rc;
  const T gamma = T(1) / (T(2) * dmu * dmu);
  const T pi_rc = (T)(3.14159265358979323846 / a.rc);
  const int64_t nwork = (a.N + RB - 1) / RB;
  const bool has_v = (v_in != nullptr);

  for (int64_t wk = blockIdx.x; wk < nwork; wk += gridDim.x) {
    const int64_t i0 = wk * RB;
    const int nrecv = (int)min((int64_t)RB, a.N - i0);
    __syncthreads();
    if (tid <= nrecv) RP[tid] = a.rowptr[i0 + tid];
    __syncthreads();
    const int ea = RP[0], eb = RP[nrecv];
    int r = 0, rend = RP[1];
    // this thread's view of the receiver's own rows
    T li0 = T(0), li1 = T(0), li2 = T(0), lv0 = T(0), lv1 = T(0), lv2 = T(0), lph = T(0);
    auto load_local = [&]() {
      const int64_t i = i0 + r;
      lph = ldp<T, PT>(phi + i * 3 * F + c * F + f);
      if (c == 0) li0 = sb1[i * F + f];
      else {
        li0 = vb1[(i * 3 + 0) * F + f]; li1 = vb1[(i * 3 + 1) * F + f]; li2 = vb1[(i * 3 + 2) * F + f];
        if (c == 2 && has_v) {
          lv0 = ldp<T, PT>(v_in + (i * 3 + 0) * F + f); lv1 = ldp<T, PT>(v_in + (i * 3 + 1) * F + f);
          lv2 = ldp<T, PT>(v_in + (i * 3 + 2) * F + f);
        }
      }
    };
    T acc0 = T(0), acc1 = T(0), acc2 = T(0), fp0 = T(0), fp1 = T(0), fp2 = T(0);
    auto flush = [&]() {
      if (c < 2) Acc[(r * 5 + c) * FS + fl] = acc0;
      else {
        Acc[(r * 5 + 2) * FS + fl] = acc0; Acc[(r * 5 + 3) * FS + fl] = acc1; Acc[(r * 5 + 4) * FS + fl] = acc2;
      }
      for (int o = 16; o; o >>= 1) {
        fp0 += __shfl_xor_sync(0xffffffffu, fp0, o);
        fp1 += __shfl_xor_sync(0xffffffffu, fp1, o);
        fp2 += __shfl_xor_sync(0xffffffffu, fp2, o);
      }
      if (lane == 0) {
        FW[(r * 12 + warp) * 3 + 0] = fp0; FW[(r * 12 + warp) * 3 + 1] = fp1; FW[(r * 12 + warp) * 3 + 2] = fp2;
      }
      acc0 = acc1 = acc2 = fp0 = fp1 = fp2 = T(0);
    };
    if (nrecv > 0) load_local();
    for (int t0 = ea; t0 < eb; t0 += ET) {
      const int nE = min(ET, eb - t0);
      __syncthreads();
      for (int q = tid; q < nE; q += nthr) {
        const Geom<T> gq = a.geom[t0 + q];
        U[q * 4 + 0] = gq.ux; U[q * 4 + 1] = gq.uy; U[q * 4 + 2] = gq.uz; U[q * 4 + 3] = gq.d;
        T sn, cs;
        t_sincos<T>(pi_rc * gq.d, &sn, &cs);
        Cc[q] = T(0.5) * (cs + T(1));
        Cp[q] = -T(0.5) * pi_rc * sn;
        J[q] = a.col[t0 + q];
      }
      __syncthreads();
      for (int q = tid; q < nE * KP; q += nthr) {
        const int e = q / KP, k = q % KP;
        T g = T(0), gd = T(0);
        if (k < K) rbf_eval<T>(a.rbf, k, U[e * 4 + 3], rc, dmu, gamma, g, gd);
        G1[q] = g * Cc[e];
        G2[q] = Cc[e] * gd + Cp[e] * g;
      }
      __syncthreads();
      for (int q = 0; q < nE; ++q) {
        const int e = t0 + q;
        while (e >= rend) { flush(); ++r; rend = RP[r + 1]; load_local(); }
        const int64_t j = J[q];
        const T wv = fma(bias, Cc[q], dotK<KP>(w, G1 + q * KP));
        const T dw = fma(bias, Cp[q], dotK<KP>(w, G2 + q * KP));
        const T ux = U[q * 4 + 0], uy = U[q * 4 + 1], uz = U[q * 4 + 2];
        const T phj = ldp<T, PT>(phi + j * 3 * F + c * F + f);
        if (c == 0) {
          const T sbj = sb1[j * F + f];
          acc0 = fma(sbj, wv, acc0);
          const T Dp = (li0 * phj + sbj * lph) * dw;
          fp0 = fma(Dp, ux, fp0); fp1 = fma(Dp, uy, fp1); fp2 = fma(Dp, uz, fp2);
        } else {
          const T b0 = vb1[(j * 3 + 0) * F + f], b1 = vb1[(j * 3 + 1) * F + f], b2 = vb1[(j * 3 + 2) * F + f];
          if (c == 1) {
            const T tj = b0 * ux + b1 * uy + b2 * uz;
            const T ti = li0 * ux + li1 * uy + li2 * uz;
            acc0 = fma(-tj, wv, acc0);
            const T Dp = (ti * phj - tj * lph) * dw;
            const T B0 = (li0 * phj - b0 * lph) * wv, B1 = (li1 * phj - b1 * lph) * wv,
                    B2 = (li2 * phj - b2 * lph) * wv;
            const T Bu = B0 * ux + B1 * uy + B2 * uz;
            const T invd = T(1) / U[q * 4 + 3];
            fp0 += Dp * ux + (B0 - Bu * ux) * invd;
            fp1 += Dp * uy + (B1 - Bu * uy) * invd;
            fp2 += Dp * uz + (B2 - Bu * uz) * invd;
          } else {
            acc0 = fma(b0, wv, acc0); acc1 = fma(b1, wv, acc1); acc2 = fma(b2, wv, acc2);
            if (has_v) {
              const T vj0 = ldp<T, PT>(v_in + (j * 3 + 0) * F + f), vj1 = ldp<T, PT>(v_in + (j * 3 + 1) * F + f),
                      vj2 = ldp<T, PT>(v_in + (j * 3 + 2) * F + f);
              const T Dp = ((li0 * vj0 + li1 * vj1 + li2 * vj2) * phj + (b0 * lv0 + b1 * lv1 + b2 * lv2) * lph) * dw;
              fp0 = fma(Dp, ux, fp0); fp1 = fma(Dp, uy, fp1); fp2 = fma(Dp, uz, fp2);
            }
          }
        }
      }
    }
    while (r < nrecv) { flush(); ++r; if (r < nrecv) load_local(); }
    __syncthreads();
    // forces: sum the warp partials of each receiver
    for (int idx = tid; idx < nrecv * 3; idx += nthr) {
      const int rr = idx / 3, ax = idx % 3;
      T s = T(0);
      for (int ww = 0; ww < nwarp; ++ww) s += FW[(rr * 12 + ww) * 3 + ax];
      T* dst = fpart + ((int64_t)blockIdx.y * a.N + i0 + rr) * 3 + ax;
      *dst = first_block ? s : (*dst + s);
    }
    if (phib != nullptr || phib16 != nullptr) {
      // node adjoints: item (r, comp, fl): comp 0,1 phib ss/vs; 2 phib vv; 3..5 vb_in[a]
      for (int idx = tid; idx < nrecv * 6 * FS; idx += nthr) {
        const int rr = idx / (6 * FS), rem = idx % (6 * FS);
        const int comp = rem / FS, ff = rem % FS;
        const int64_t i = i0 + rr;
        const int fo = blockIdx.y * FS + ff;
        const T* A = Acc + (size_t)(rr * 5) * FS;
        if (comp < 3) {
          T s = T(0);
          if (comp < 2) s = A[comp * FS + ff];
          else if (has_v)
            s = ldp<T, PT>(v_in + (i * 3 + 0) * F + fo) * A[2 * FS + ff] +
                ldp<T, PT>(v_in + (i * 3 + 1) * F + fo) * A[3 * FS + ff] +
                ldp<T, PT>(v_in + (i * 3 + 2) * F + fo) * A[4 * FS + ff];
          if (phib16) phib16[i * 3 * F + comp * F + fo] = __float2bfloat16_rn((float)s);
          else phib[i * 3 * F + comp * F + fo] = s;
        } else {
          const int ax = comp - 3;
          vb_in[(i * 3 + ax) * F + fo] =
              vb1[(i * 3 + ax) * F + fo] + ldp<T, PT>(phi + i * 3 * F + 2 * F + fo) * A[(2 + ax) * FS + ff];
        }
      }
    }
  }
}

int pick_kp(int K) { return K <= 8 ? 8 : K <= 16 ? 16 : K <= 20 ? 20 : K <= 24 ? 24 : 32; }

template <typename T>
int pick_rb() { return sizeof(T) == 8 ? 4 : 8; }

} // namespace

int edge_num_slabs(int F) { return (F + 127) / 128; }

template <typename T, typename PT>
int launch_edge_fwd(const EdgeArgs<T>& a, const PT* phi, const T* s_in, int64_t ld_sin, const PT* v_in,
                    const T* v_res, T* s1, int64_t ld_s1, T* v1, const EdgeMirror& mir, cudaStream_t st) {
  if (a.N == 0) return 0;
  const int nslab = edge_num_slabs(a.F), FS = a.F / nslab, RB = pick_rb<T>(), KP = pick_kp(a.K);
  const int64_t nwork = (a.N + RB - 1) / RB;
  dim3 grid((unsigned)std::min<int64_t>(nwork, 148 * 4), nslab);   // whole waves: cfg5 148*6 525 ms, 148*4 495 ms
  const size_t smem = sizeof(T) * (ET * KP + ET + ET * 4 + (size_t)RB * 7 * FS) + sizeof(int) * (ET + RB + 1);
#define PNN_LAUNCH_FWD(KPV)                                                                                   \
  {                                                                                                           \
    static bool attr_set = false;                                                                             \
    if (!attr_set) {                                                                                          \
      cudaFuncSetAttribute(edge_fwd_k<T, KPV, PT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);   \
      attr_set = true;                                                                                        \
    }                                                                                                         \
    edge_fwd_k<T, KPV, PT><<<grid, 3 * FS, smem, st>>>(a, FS, RB, phi, s_in, ld_sin, v_in, v_res, s1, ld_s1,  \
                                                       v1, mir); PNN_KCHECK("edge_fwd_k");                    \
  }
  switch (KP) {
    case 8: PNN_LAUNCH_FWD(8) break;
    case 16: PNN_LAUNCH_FWD(16) break;
    case 20: PNN_LAUNCH_FWD(20) break;
    case 24: PNN_LAUNCH_FWD(24) break;
    default: PNN_LAUNCH_FWD(32) break;
  }
#undef PNN_LAUNCH_FWD
  return 1;
}

template <typename T, typename PT>
int launch_edge_bwd(const EdgeArgs<T>& a, const PT* phi, const PT* v_in, const T* sb1, const T* vb1, T* phib,
                    T* vb_in, T* fpart, int first_block, __nv_bfloat16* phib16, cudaStream_t st) {
  if (a.N == 0) return 0;
  const int nslab = edge_num_slabs(a.F), FS = a.F / nslab, RB = pick_rb<T>(), KP = pick_kp(a.K);
  const int64_t nwork = (a.N + RB - 1) / RB;
  dim3 grid((unsigned)std::min<int64_t>(nwork, 148 * 4), nslab);   // whole waves: cfg5 148*6 525 ms, 148*4 495 ms
  const size_t smem = sizeof(T) * (2 * ET * KP + 2 * ET + ET * 4 + (size_t)RB * 5 * FS + RB * 12 * 3) +
                      sizeof(int) * (ET + RB + 1);
#define PNN_LAUNCH_BWD(KPV)                                                                                   \
  {                                                                                                           \
    static bool attr_set = false;                                                                             \
    if (!attr_set) {                                                                                          \
      cudaFuncSetAttribute(edge_bwd_k<T, KPV, PT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);   \
      attr_set = true;                                                                                        \
    }                                                                                                         \
    edge_bwd_k<T, KPV, PT><<<grid, 3 * FS, smem, st>>>(a, FS, RB, phi, v_in, sb1, vb1, phib, vb_in, fpart,     \
                                                       first_block, phib16); PNN_KCHECK("edge_bwd_k");        \
  }
  switch (KP) {
    case 8: PNN_LAUNCH_BWD(8) break;
    case 16: PNN_LAUNCH_BWD(16) break;
    case 20: PNN_LAUNCH_BWD(20) break;
    case 24: PNN_LAUNCH_BWD(24) break;
    default: PNN_LAUNCH_BWD(32) break;
  }
#undef PNN_LAUNCH_BWD
  return 1;
}

#define PNN_INST_EDGE(T, PT)                                                                                        \
  template int launch_edge_fwd<T, PT>(const EdgeArgs<T>&, const PT*, const T*, int64_t, const PT*, const T*, T*,    \
                                      int64_t, T*, const EdgeMirror&, cudaStream_t);                               \
  template int launch_edge_bwd<T, PT>(const EdgeArgs<T>&, const PT*, const PT*, const T*, const T*, T*, T*, T*,    \
                                      int, __nv_bfloat16*, cudaStream_t);
PNN_INST_EDGE(float, float)
PNN_INST_EDGE(double, double)
#undef PNN_INST_EDGE

} // namespace pnn
