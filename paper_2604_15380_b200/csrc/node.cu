// node.cu — per-atom element-wise pieces of the path, FP32 / FP64:
//   a2 embedding (B2), the non-GEMM parts of the update block a5 (B4: n = sqrt(sum_a Q_a^2 + eps), gated
//   scalar-vector products) and of its adjoint (R2), a6 multi-head readout + per-structure segmented sum (B5)
//   and its adjoint (R1), and the final force assembly (R4).  Formulas: SURVEY.md §8(c).
// All are streaming kernels: one thread per (atom, feature), consecutive threads on consecutive features.
#include <type_traits>

#include "common.cuh"

namespace pnn {

namespace {

constexpr int RT = 16; // atoms per readout tile

// P | Q and the gate values a may be stored narrower than the arithmetic type (BF16 model: tensor-core GEMM outputs)
template <typename T, typename IT> __device__ __forceinline__ T ldi(const IT* p) { return (T)(*p); }
template <> __device__ __forceinline__ float ldi<float, __nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }

template <typename T>
__global__ void __launch_bounds__(256) embed_k(int64_t N, int F, int Zmax, const int32_t* __restrict__ Z,
                                               const T* __restrict__ emb, T* __restrict__ s, int* d_err,
                                               __nv_bfloat16* __restrict__ s16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * F) return;
  const int64_t i = idx / F;
  const int f = (int)(idx % F);
  int z = Z[i];
  if (z < 1 || z > Zmax) {
    if (f == 0) atomicOr(d_err, ERRF_BAD_Z);
    z = 1;
  }
  const T e = emb[(int64_t)z * F + f];
  s[idx] = e;
  if (s16) s16[idx] = __float2bfloat16_rn((float)e);
}

template <typename T>
__global__ void __launch_bounds__(256) embed_globals_k(int64_t N, int F, int G, const int32_t* __restrict__ a2s,
                                                       const double* __restrict__ glob, const T* __restrict__ globW,
                                                       T* __restrict__ s, __nv_bfloat16* __restrict__ s16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * F) return;
  const int64_t i = idx / F;
  const int f = (int)(idx % F);
  const double* gq = glob + (int64_t)a2s[i] * G;
  T acc = s[idx];
  for (int q = 0; q < G; ++q) acc += globW[(int64_t)f * G + q] * (T)gq[q];
  s[idx] = acc;
  if (s16) s16[idx] = __float2bfloat16_rn((float)acc);
}

// FP32: four features per thread (16-byte loads / stores, 8-byte BF16 copy)
__global__ void __launch_bounds__(256) embed4_k(int64_t N, int F4, int Zmax, const int32_t* __restrict__ Z,
                                                const float4* __restrict__ emb, float4* __restrict__ s, int* d_err,
                                                uint2* __restrict__ s16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * F4) return;
  const int64_t i = idx / F4;
  const int q = (int)(idx - i * F4);
  int z = Z[i];
  if (z < 1 || z > Zmax) {
    if (q == 0) atomicOr(d_err, ERRF_BAD_Z);
    z = 1;
  }
  const float4 e = __ldg(emb + (int64_t)z * F4 + q);
  s[idx] = e;
  if (s16) {
    __nv_bfloat162 lo = __floats2bfloat162_rn(e.x, e.y), hi = __floats2bfloat162_rn(e.z, e.w);
    s16[idx] = make_uint2(*reinterpret_cast<uint32_t*>(&lo), *reinterpret_cast<uint32_t*>(&hi));
  }
}

// PQ [N][3][2F] (P | Q)  ->  sn[:, F:2F] = sqrt(sum_a Q_a^2 + eps)          (B4)
template <typename T, typename IT>
__global__ void __launch_bounds__(256) norm_k(int64_t N, int F, const IT* __restrict__ PQ, T* __restrict__ sn, T eps,
                                              __nv_bfloat16* __restrict__ sn16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * F) return;
  const int64_t i = idx / F;
  const int f = (int)(idx % F);
  const T q0 = ldi<T, IT>(PQ + (i * 3 + 0) * 2 * F + F + f), q1 = ldi<T, IT>(PQ + (i * 3 + 1) * 2 * F + F + f),
          q2 = ldi<T, IT>(PQ + (i * 3 + 2) * 2 * F + F + f);
  const T n = sqrt(q0 * q0 + q1 * q1 + q2 * q2 + eps);
  if (sn16) sn16[i * 2 * F + F + f] = __float2bfloat16_rn((float)n);
  else sn[i * 2 * F + F + f] = n;
}

// s'' = s' + a_sv <P,Q> + a_ss ;  v'' = v' + a_vv P                          (B4)
template <typename T, typename IT>
__global__ void __launch_bounds__(256) update_k(int64_t N, int F, const T* __restrict__ sn, const T* __restrict__ v1,
                                                const IT* __restrict__ PQ, const IT* __restrict__ a,
                                                T* __restrict__ s_out, T* __restrict__ v_out,
                                                __nv_bfloat16* __restrict__ s16, __nv_bfloat16* __restrict__ v16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * F) return;
  const int64_t i = idx / F;
  const int f = (int)(idx % F);
  const T avv = ldi<T, IT>(a + i * 3 * F + f), asv = ldi<T, IT>(a + i * 3 * F + F + f),
          ass = ldi<T, IT>(a + i * 3 * F + 2 * F + f);
  T dot = T(0);
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    const T p = ldi<T, IT>(PQ + (i * 3 + ax) * 2 * F + f), q = ldi<T, IT>(PQ + (i * 3 + ax) * 2 * F + F + f);
    dot = fma(p, q, dot);
    if (v_out) {
      const T r = fma(avv, p, v1[(i * 3 + ax) * F + f]);
      v_out[(i * 3 + ax) * F + f] = r;
      if (v16) v16[(i * 3 + ax) * F + f] = __float2bfloat16_rn((float)r);
    }
  }
  const T r = sn[i * 2 * F + f] + asv * dot + ass;
  s_out[idx] = r;
  if (s16) s16[idx] = __float2bfloat16_rn((float)r);
}

// ---- FP32-arithmetic versions of norm_k / update_k with 4 features per thread (16-byte FP32 and 8-byte BF16 accesses):
// these kernels are pure HBM streams, so the access width decides the achieved bandwidth.
template <typename IT> struct Ld4;
template <> struct Ld4<float> {
  static __device__ __forceinline__ float4 ld(const float* p) { return *reinterpret_cast<const float4*>(p); }
};
template <> struct Ld4<__nv_bfloat16> {
  static __device__ __forceinline__ float4 ld(const __nv_bfloat16* p) {
    const uint2 r = *reinterpret_cast<const uint2*>(p);
    return make_float4(__uint_as_float(r.x << 16), __uint_as_float(r.x & 0xffff0000u), __uint_as_float(r.y << 16),
                       __uint_as_float(r.y & 0xffff0000u));
  }
};
__device__ __forceinline__ void st4_bf16(__nv_bfloat16* p, float4 v) {
  const __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), b = __floats2bfloat162_rn(v.z, v.w);
  *reinterpret_cast<uint2*>(p) = make_uint2(*reinterpret_cast<const uint32_t*>(&a), *reinterpret_cast<const uint32_t*>(&b));
}

template <typename IT>
__global__ void __launch_bounds__(256) norm4_k(int64_t N, int F, const IT* __restrict__ PQ, float* __restrict__ sn, float eps,
                                               __nv_bfloat16* __restrict__ sn16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int F4 = F / 4;
  if (idx >= N * F4) return;
  const int64_t i = idx / F4;
  const int f = (int)(idx % F4) * 4;
  const float4 q0 = Ld4<IT>::ld(PQ + (i * 3 + 0) * 2 * F + F + f), q1 = Ld4<IT>::ld(PQ + (i * 3 + 1) * 2 * F + F + f),
               q2 = Ld4<IT>::ld(PQ + (i * 3 + 2) * 2 * F + F + f);
  const float4 n = make_float4(sqrtf(q0.x * q0.x + q1.x * q1.x + q2.x * q2.x + eps), sqrtf(q0.y * q0.y + q1.y * q1.y + q2.y * q2.y + eps),
                               sqrtf(q0.z * q0.z + q1.z * q1.z + q2.z * q2.z + eps), sqrtf(q0.w * q0.w + q1.w * q1.w + q2.w * q2.w + eps));
  if (sn16) st4_bf16(sn16 + i * 2 * F + F + f, n);
  else *reinterpret_cast<float4*>(sn + i * 2 * F + F + f) = n;
}

template <typename IT>
__global__ void __launch_bounds__(256) update4_k(int64_t N, int F, const float* __restrict__ sn, const float* __restrict__ v1,
                                                 const IT* __restrict__ PQ, const IT* __restrict__ a,
                                                 float* __restrict__ s_out, float* __restrict__ v_out,
                                                 __nv_bfloat16* __restrict__ s16, __nv_bfloat16* __restrict__ v16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int F4 = F / 4;
  if (idx >= N * F4) return;
  const int64_t i = idx / F4;
  const int f = (int)(idx % F4) * 4;
  const float4 avv = Ld4<IT>::ld(a + i * 3 * F + f), asv = Ld4<IT>::ld(a + i * 3 * F + F + f),
               ass = Ld4<IT>::ld(a + i * 3 * F + 2 * F + f);
  float4 dot = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    const float4 p = Ld4<IT>::ld(PQ + (i * 3 + ax) * 2 * F + f), q = Ld4<IT>::ld(PQ + (i * 3 + ax) * 2 * F + F + f);
    dot.x = fmaf(p.x, q.x, dot.x); dot.y = fmaf(p.y, q.y, dot.y); dot.z = fmaf(p.z, q.z, dot.z); dot.w = fmaf(p.w, q.w, dot.w);
    if (v_out) {
      const float4 v = *reinterpret_cast<const float4*>(v1 + (i * 3 + ax) * F + f);
      const float4 r = make_float4(fmaf(avv.x, p.x, v.x), fmaf(avv.y, p.y, v.y), fmaf(avv.z, p.z, v.z), fmaf(avv.w, p.w, v.w));
      *reinterpret_cast<float4*>(v_out + (i * 3 + ax) * F + f) = r;
      if (v16) st4_bf16(v16 + (i * 3 + ax) * F + f, r);
    }
  }
  const float4 s1 = *reinterpret_cast<const float4*>(sn + i * 2 * F + f);
  const float4 r = make_float4(s1.x + asv.x * dot.x + ass.x, s1.y + asv.y * dot.y + ass.y, s1.z + asv.z * dot.z + ass.z,
                               s1.w + asv.w * dot.w + ass.w);
  *reinterpret_cast<float4*>(s_out + idx * 4) = r;
  if (s16) st4_bf16(s16 + idx * 4, r);
}

// R2, first half: a-bar [N,3F] and the direct parts of P-bar, Q-bar [N][3][2F]
template <typename T, typename IT>
__global__ void __launch_bounds__(256) update_bwd1_k(int64_t N, int F, const T* __restrict__ sb,
                                                     const T* __restrict__ vb, const IT* __restrict__ a,
                                                     const IT* __restrict__ PQ, T* __restrict__ ab,
                                                     T* __restrict__ PQb, __nv_bfloat16* __restrict__ ab16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * F) return;
  const int64_t i = idx / F;
  const int f = (int)(idx % F);
  const T sbf = sb[idx];
  const T avv = ldi<T, IT>(a + i * 3 * F + f), asv = ldi<T, IT>(a + i * 3 * F + F + f);
  T p[3], q[3], vbf[3];
  T dot = T(0), avvb = T(0);
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    p[ax] = ldi<T, IT>(PQ + (i * 3 + ax) * 2 * F + f);
    q[ax] = ldi<T, IT>(PQ + (i * 3 + ax) * 2 * F + F + f);
    vbf[ax] = vb ? vb[(i * 3 + ax) * F + f] : T(0);
    dot = fma(p[ax], q[ax], dot);
    avvb = fma(vbf[ax], p[ax], avvb);
  }
  if (ab16) {
    ab16[i * 3 * F + f] = __float2bfloat16_rn((float)avvb);
    ab16[i * 3 * F + F + f] = __float2bfloat16_rn((float)(sbf * dot));
    ab16[i * 3 * F + 2 * F + f] = __float2bfloat16_rn((float)sbf);
  } else {
    ab[i * 3 * F + f] = avvb;
    ab[i * 3 * F + F + f] = sbf * dot;
    ab[i * 3 * F + 2 * F + f] = sbf;
  }
  const T dotb = sbf * asv;
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    PQb[(i * 3 + ax) * 2 * F + f] = vbf[ax] * avv + dotb * q[ax];
    PQb[(i * 3 + ax) * 2 * F + F + f] = dotb * p[ax];
  }
}

// R2, second half: s-bar' = s-bar'' + z-bar[0:F];  Q-bar += n-bar Q / n
template <typename T, typename IT>
__global__ void __launch_bounds__(256) update_bwd2_k(int64_t N, int F, const T* __restrict__ zb,
                                                     const IT* __restrict__ PQ, T eps, T* __restrict__ sb,
                                                     T* __restrict__ PQb, __nv_bfloat16* __restrict__ PQb16,
                                                     __nv_bfloat16* __restrict__ sb16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * F) return;
  const int64_t i = idx / F;
  const int f = (int)(idx % F);
  const T sbn = sb[idx] + zb[i * 2 * F + f];
  sb[idx] = sbn;
  if (sb16) sb16[idx] = __float2bfloat16_rn((float)sbn);
  const T nb = zb[i * 2 * F + F + f];
  const T q0 = ldi<T, IT>(PQ + (i * 3 + 0) * 2 * F + F + f), q1 = ldi<T, IT>(PQ + (i * 3 + 1) * 2 * F + F + f),
          q2 = ldi<T, IT>(PQ + (i * 3 + 2) * 2 * F + F + f);
  const T r = nb / sqrt(q0 * q0 + q1 * q1 + q2 * q2 + eps);
  const T qq[3] = {q0, q1, q2};
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    const int64_t o = (i * 3 + ax) * 2 * F + f;
    const T qb = PQb[o + F] + r * qq[ax];
    if (PQb16) {
      PQb16[o] = __float2bfloat16_rn((float)PQb[o]);
      PQb16[o + F] = __float2bfloat16_rn((float)qb);
    } else {
      PQb[o + F] = qb;
    }
  }
}

// ---- 4 features per thread versions of the two kernels above (FP32 arithmetic; same formulas)
__device__ __forceinline__ float4 f4mul(float4 a, float4 b) { return make_float4(a.x * b.x, a.y * b.y, a.z * b.z, a.w * b.w); }
__device__ __forceinline__ float4 f4fma(float4 a, float4 b, float4 c) {
  return make_float4(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y), fmaf(a.z, b.z, c.z), fmaf(a.w, b.w, c.w));
}
template <typename IT>
__global__ void __launch_bounds__(256) update_bwd1_4_k(int64_t N, int F, const float* __restrict__ sb,
                                                       const float* __restrict__ vb, const IT* __restrict__ a,
                                                       const IT* __restrict__ PQ, float* __restrict__ ab,
                                                       float* __restrict__ PQb, __nv_bfloat16* __restrict__ ab16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int F4 = F / 4;
  if (idx >= N * F4) return;
  const int64_t i = idx / F4;
  const int f = (int)(idx % F4) * 4;
  const float4 sbf = *reinterpret_cast<const float4*>(sb + i * F + f);
  const float4 avv = Ld4<IT>::ld(a + i * 3 * F + f), asv = Ld4<IT>::ld(a + i * 3 * F + F + f);
  float4 p[3], q[3], vbf[3];
  float4 dot = make_float4(0.f, 0.f, 0.f, 0.f), avvb = dot;
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    p[ax] = Ld4<IT>::ld(PQ + (i * 3 + ax) * 2 * F + f);
    q[ax] = Ld4<IT>::ld(PQ + (i * 3 + ax) * 2 * F + F + f);
    vbf[ax] = vb ? *reinterpret_cast<const float4*>(vb + (i * 3 + ax) * F + f) : make_float4(0.f, 0.f, 0.f, 0.f);
    dot = f4fma(p[ax], q[ax], dot);
    avvb = f4fma(vbf[ax], p[ax], avvb);
  }
  const float4 sd = f4mul(sbf, dot);
  if (ab16) {
    st4_bf16(ab16 + i * 3 * F + f, avvb); st4_bf16(ab16 + i * 3 * F + F + f, sd); st4_bf16(ab16 + i * 3 * F + 2 * F + f, sbf);
  } else {
    *reinterpret_cast<float4*>(ab + i * 3 * F + f) = avvb;
    *reinterpret_cast<float4*>(ab + i * 3 * F + F + f) = sd;
    *reinterpret_cast<float4*>(ab + i * 3 * F + 2 * F + f) = sbf;
  }
  const float4 dotb = f4mul(sbf, asv);
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    *reinterpret_cast<float4*>(PQb + (i * 3 + ax) * 2 * F + f) = f4fma(dotb, q[ax], f4mul(vbf[ax], avv));
    *reinterpret_cast<float4*>(PQb + (i * 3 + ax) * 2 * F + F + f) = f4mul(dotb, p[ax]);
  }
}

template <typename IT>
__global__ void __launch_bounds__(256) update_bwd2_4_k(int64_t N, int F, const float* __restrict__ zb,
                                                       const IT* __restrict__ PQ, float eps, float* __restrict__ sb,
                                                       float* __restrict__ PQb, __nv_bfloat16* __restrict__ PQb16,
                                                       __nv_bfloat16* __restrict__ sb16) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int F4 = F / 4;
  if (idx >= N * F4) return;
  const int64_t i = idx / F4;
  const int f = (int)(idx % F4) * 4;
  const float4 s0 = *reinterpret_cast<const float4*>(sb + i * F + f), z0 = *reinterpret_cast<const float4*>(zb + i * 2 * F + f);
  const float4 sbn = make_float4(s0.x + z0.x, s0.y + z0.y, s0.z + z0.z, s0.w + z0.w);
  *reinterpret_cast<float4*>(sb + i * F + f) = sbn;
  if (sb16) st4_bf16(sb16 + i * F + f, sbn);
  const float4 nb = *reinterpret_cast<const float4*>(zb + i * 2 * F + F + f);
  float4 q[3];
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) q[ax] = Ld4<IT>::ld(PQ + (i * 3 + ax) * 2 * F + F + f);
  const float4 r = make_float4(nb.x / sqrtf(q[0].x * q[0].x + q[1].x * q[1].x + q[2].x * q[2].x + eps),
                               nb.y / sqrtf(q[0].y * q[0].y + q[1].y * q[1].y + q[2].y * q[2].y + eps),
                               nb.z / sqrtf(q[0].z * q[0].z + q[1].z * q[1].z + q[2].z * q[2].z + eps),
                               nb.w / sqrtf(q[0].w * q[0].w + q[1].w * q[1].w + q[2].w * q[2].w + eps));
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    const int64_t o = (i * 3 + ax) * 2 * F + f;
    const float4 qb = f4fma(r, q[ax], *reinterpret_cast<const float4*>(PQb + o + F));
    if (PQb16) {
      st4_bf16(PQb16 + o, *reinterpret_cast<const float4*>(PQb + o));
      st4_bf16(PQb16 + o + F, qb);
    } else {
      *reinterpret_cast<float4*>(PQb + o + F) = qb;
    }
  }
}

// ------------------------------------------------------------------------------------------ readout
// One CTA per tile of RT consecutive atoms.  Atoms of a structure are contiguous and share a head, so the tile
// splits into a few runs of equal head; each run is a small [run x F] x [F x F/2] product with the head's W1.
template <typename T>
__global__ void __launch_bounds__(128) readout_k(int64_t N, int F, int H, const T* __restrict__ s,
                                                 const int32_t* __restrict__ a2s, const int32_t* __restrict__ head,
                                                 const T* __restrict__ W1t, const T* __restrict__ b1,
                                                 const T* __restrict__ w2, const T* __restrict__ b2,
                                                 T* __restrict__ opre, T* __restrict__ eatom, int* d_err) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* S = reinterpret_cast<T*>(smem_raw);      // [RT][F]
  T* Eo = S + RT * F;                         // [RT][Fh]
  __shared__ int Hs[RT];
  const int Fh = F / 2;
  const int64_t i0 = (int64_t)blockIdx.x * RT;
  const int nt = (int)min((int64_t)RT, N - i0);
  for (int q = threadIdx.x; q < nt * F; q += blockDim.x) S[q] = s[i0 * F + q];
  if (threadIdx.x < nt) {
    int h = head[a2s[i0 + threadIdx.x]];
    if (h < 0 || h >= H) { atomicOr(d_err, ERRF_BAD_HEAD); h = 0; }
    Hs[threadIdx.x] = h;
  }
  __syncthreads();
  for (int o = threadIdx.x; o < Fh; o += blockDim.x) {
    int r0 = 0;
    while (r0 < nt) {
      const int h = Hs[r0];
      int r1 = r0 + 1;
      while (r1 < nt && Hs[r1] == h) ++r1;
      T acc[RT];
#pragma unroll
      for (int r = 0; r < RT; ++r) acc[r] = T(0);
      const T* Wp = W1t + (int64_t)h * F * Fh + o;
      for (int k = 0; k < F; ++k) {
        const T wv = Wp[(int64_t)k * Fh];
#pragma unroll
        for (int r = 0; r < RT; ++r)
          if (r0 + r < r1) acc[r] = fma(wv, S[(r0 + r) * F + k], acc[r]);
      }
      const T bb = b1[h * Fh + o], ww = w2[h * Fh + o];
#pragma unroll
      for (int r = 0; r < RT; ++r)
        if (r0 + r < r1) {
          const T pre = acc[r] + bb;
          if (opre) opre[(i0 + r0 + r) * Fh + o] = pre;
          Eo[(r0 + r) * Fh + o] = ww * silu_f<T>(pre);
        }
      r0 = r1;
    }
  }
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int r = warp; r < nt; r += 4) {
    T e = T(0);
    for (int o = lane; o < Fh; o += 32) e += Eo[r * Fh + o];
    for (int sft = 16; sft; sft >>= 1) e += __shfl_xor_sync(0xffffffffu, e, sft);
    if (lane == 0) eatom[i0 + r] = e + b2[Hs[r]];
  }
}

// ---- readout, second version: all threads busy.  A CTA takes RT = 16 atoms; thread (og, rg) owns 4 consecutive hidden
// units (og) of rows rg and rg + 8.  Per input feature k it reads its head's 4 weights as one vector (coalesced over og,
// L1-resident across the 8 row groups) and the two activations from shared memory: 8 FMAs per 3 loads (readout_k: 16
// per 17), and no thread idles when F/2 < blockDim.  Each row uses the first layer of its own head, so a tile may mix
// heads freely.  blockDim = 8 * Fh / 4.
template <typename T> struct Vec4;
template <> struct Vec4<float> {
  static __device__ __forceinline__ void ld(const float* p, float (&x)[4]) {
    const float4 v = *reinterpret_cast<const float4*>(p); x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
  }
};
template <> struct Vec4<double> {
  static __device__ __forceinline__ void ld(const double* p, double (&x)[4]) {
    const double2 a = *reinterpret_cast<const double2*>(p), b = *reinterpret_cast<const double2*>(p + 2);
    x[0] = a.x; x[1] = a.y; x[2] = b.x; x[3] = b.y;
  }
};

template <typename T>
__global__ void __launch_bounds__(256) readout2_k(int64_t N, int F, int H, const T* __restrict__ s,
                                                  const int32_t* __restrict__ a2s, const int32_t* __restrict__ head,
                                                  const T* __restrict__ W1t, const T* __restrict__ b1,
                                                  const T* __restrict__ w2, const T* __restrict__ b2,
                                                  T* __restrict__ opre, T* __restrict__ eatom, int* d_err) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int Fh = F / 2, NOG = Fh / 4;
  T* S = reinterpret_cast<T*>(smem_raw);  // [RT][F]
  T* Ep = S + RT * F;                     // [RT][NOG] partial energies
  __shared__ int Hs[RT];
  const int64_t i0 = (int64_t)blockIdx.x * RT;
  const int nt = (int)min((int64_t)RT, N - i0);
  for (int q = threadIdx.x; q < RT * F; q += blockDim.x) S[q] = (q < nt * F) ? s[i0 * F + q] : T(0);
  if (threadIdx.x < RT) {
    int h = 0;
    if (threadIdx.x < nt) {
      h = head[a2s[i0 + threadIdx.x]];
      if (h < 0 || h >= H) { atomicOr(d_err, ERRF_BAD_HEAD); h = 0; }
    }
    Hs[threadIdx.x] = h;
  }
  __syncthreads();
  const int og = threadIdx.x % NOG, rg = threadIdx.x / NOG; // rg in 0..7
  const int h0 = Hs[rg], h1 = Hs[rg + 8];
  const T* W0 = W1t + (int64_t)h0 * F * Fh + og * 4;
  const T* W1p = W1t + (int64_t)h1 * F * Fh + og * 4;
  T acc0[4] = {T(0), T(0), T(0), T(0)}, acc1[4] = {T(0), T(0), T(0), T(0)};
  if (__all_sync(0xffffffffu, h0 == h1)) {   // the usual case (rows 8 apart in one structure): one weight vector for both
#pragma unroll 4
    for (int k = 0; k < F; ++k) {
      T wa[4];
      Vec4<T>::ld(W0 + (int64_t)k * Fh, wa);
      const T x0 = S[rg * F + k], x1 = S[(rg + 8) * F + k];
#pragma unroll
      for (int j = 0; j < 4; ++j) { acc0[j] = fma(wa[j], x0, acc0[j]); acc1[j] = fma(wa[j], x1, acc1[j]); }
    }
  } else {
#pragma unroll 4
    for (int k = 0; k < F; ++k) {
      T wa[4], wb[4];
      Vec4<T>::ld(W0 + (int64_t)k * Fh, wa);
      Vec4<T>::ld(W1p + (int64_t)k * Fh, wb);
      const T x0 = S[rg * F + k], x1 = S[(rg + 8) * F + k];
#pragma unroll
      for (int j = 0; j < 4; ++j) { acc0[j] = fma(wa[j], x0, acc0[j]); acc1[j] = fma(wb[j], x1, acc1[j]); }
    }
  }
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int row = rg + 8 * r, h = r ? h1 : h0;
    T e = T(0);
    if (row < nt) {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int o = og * 4 + j;
        const T pre = (r ? acc1[j] : acc0[j]) + b1[h * Fh + o];
        if (opre) opre[(i0 + row) * Fh + o] = pre;
        e = fma(w2[h * Fh + o], silu_f<T>(pre), e);
      }
    }
    Ep[row * NOG + og] = e;
  }
  __syncthreads();
  if (threadIdx.x < nt) {
    T e = T(0);
    for (int q = 0; q < NOG; ++q) e += Ep[threadIdx.x * NOG + q];
    eatom[i0 + threadIdx.x] = e + b2[Hs[threadIdx.x]];
  }
}

// R1, second version: thread (kg, rg) owns 4 consecutive input features of rows rg and rg + 8.  blockDim = 8 * F / 4.
template <typename T>
__global__ void __launch_bounds__(512) readout_bwd2_k(int64_t N, int F, int H, const T* __restrict__ opre,
                                                      const int32_t* __restrict__ a2s, const int32_t* __restrict__ head,
                                                      const T* __restrict__ W1, const T* __restrict__ w2,
                                                      T* __restrict__ sb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int Fh = F / 2, NKG = F / 4;
  T* Pb = reinterpret_cast<T*>(smem_raw); // [RT][Fh]  p = w2 o silu'(pre)
  __shared__ int Hs[RT];
  const int64_t i0 = (int64_t)blockIdx.x * RT;
  const int nt = (int)min((int64_t)RT, N - i0);
  if (threadIdx.x < RT) {
    int h = 0;
    if (threadIdx.x < nt) { h = head[a2s[i0 + threadIdx.x]]; if (h < 0 || h >= H) h = 0; }
    Hs[threadIdx.x] = h;
  }
  __syncthreads();
  for (int q = threadIdx.x; q < RT * Fh; q += blockDim.x) {
    const int r = q / Fh, o = q % Fh;
    Pb[q] = (r < nt) ? w2[Hs[r] * Fh + o] * dsilu_f<T>(opre[(i0 + r) * Fh + o]) : T(0);
  }
  __syncthreads();
  const int kg = threadIdx.x % NKG, rg = threadIdx.x / NKG;
  const T* Wa = W1 + (int64_t)Hs[rg] * Fh * F + kg * 4;
  const T* Wb = W1 + (int64_t)Hs[rg + 8] * Fh * F + kg * 4;
  T acc0[4] = {T(0), T(0), T(0), T(0)}, acc1[4] = {T(0), T(0), T(0), T(0)};
  if (__all_sync(0xffffffffu, Hs[rg] == Hs[rg + 8])) {   // same head for both rows: one weight vector
#pragma unroll 4
    for (int o = 0; o < Fh; ++o) {
      T wa[4];
      Vec4<T>::ld(Wa + (int64_t)o * F, wa);
      const T p0 = Pb[rg * Fh + o], p1 = Pb[(rg + 8) * Fh + o];
#pragma unroll
      for (int j = 0; j < 4; ++j) { acc0[j] = fma(wa[j], p0, acc0[j]); acc1[j] = fma(wa[j], p1, acc1[j]); }
    }
  } else {
#pragma unroll 4
    for (int o = 0; o < Fh; ++o) {
      T wa[4], wb[4];
      Vec4<T>::ld(Wa + (int64_t)o * F, wa);
      Vec4<T>::ld(Wb + (int64_t)o * F, wb);
      const T p0 = Pb[rg * Fh + o], p1 = Pb[(rg + 8) * Fh + o];
#pragma unroll
      for (int j = 0; j < 4; ++j) { acc0[j] = fma(wa[j], p0, acc0[j]); acc1[j] = fma(wb[j], p1, acc1[j]); }
    }
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    if (rg < nt) sb[(i0 + rg) * F + kg * 4 + j] = acc0[j];
    if (rg + 8 < nt) sb[(i0 + rg + 8) * F + kg * 4 + j] = acc1[j];
  }
}

// ---- blended multi-head readout (Fig. 5): every atom is read out by
// ALL heads whose branch weight w[g,h] for its structure g is >= thr ("branch skipping"), eatom_i = sum_h w[g,h] eps_i^h.
// Same thread mapping as readout2_k; the two rows of a thread share the head inside the h loop, so one weight vector
// serves both.  opre_all [N][H][Fh] keeps the pre-activations of the evaluated heads for the reverse sweep.
template <typename T>
__global__ void __launch_bounds__(256) readout_blend_k(int64_t N, int F, int H, const T* __restrict__ s,
                                                       const int32_t* __restrict__ a2s, const T* __restrict__ hw, T thr,
                                                       const T* __restrict__ W1t, const T* __restrict__ b1,
                                                       const T* __restrict__ w2, const T* __restrict__ b2,
                                                       T* __restrict__ opre_all, T* __restrict__ eatom) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int Fh = F / 2, NOG = Fh / 4;
  T* S = reinterpret_cast<T*>(smem_raw);  // [RT][F]
  T* Ep = S + RT * F;                     // [RT][NOG]
  __shared__ int Gs[RT];
  const int64_t i0 = (int64_t)blockIdx.x * RT;
  const int nt = (int)min((int64_t)RT, N - i0);
  for (int q = threadIdx.x; q < RT * F; q += blockDim.x) S[q] = (q < nt * F) ? s[i0 * F + q] : T(0);
  if (threadIdx.x < RT) Gs[threadIdx.x] = threadIdx.x < nt ? a2s[i0 + threadIdx.x] : -1;
  __syncthreads();
  const int og = threadIdx.x % NOG, rg = threadIdx.x / NOG;
  const int g0 = Gs[rg], g1 = Gs[rg + 8];
  T e0 = T(0), e1 = T(0);
  for (int h = 0; h < H; ++h) {
    T w0 = g0 >= 0 ? hw[(int64_t)g0 * H + h] : T(0), w1 = g1 >= 0 ? hw[(int64_t)g1 * H + h] : T(0);
    if (w0 < thr) w0 = T(0);
    if (w1 < thr) w1 = T(0);
    if (w0 == T(0) && w1 == T(0)) continue;
    const T* Wp = W1t + (int64_t)h * F * Fh + og * 4;
    T acc0[4] = {T(0), T(0), T(0), T(0)}, acc1[4] = {T(0), T(0), T(0), T(0)};
#pragma unroll 4
    for (int k = 0; k < F; ++k) {
      T wa[4];
      Vec4<T>::ld(Wp + (int64_t)k * Fh, wa);
      const T x0 = S[rg * F + k], x1 = S[(rg + 8) * F + k];
#pragma unroll
      for (int j = 0; j < 4; ++j) { acc0[j] = fma(wa[j], x0, acc0[j]); acc1[j] = fma(wa[j], x1, acc1[j]); }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int o = og * 4 + j;
      const T bb = b1[h * Fh + o], ww = w2[h * Fh + o];
      const T p0 = acc0[j] + bb, p1 = acc1[j] + bb;
      if (w0 != T(0)) {
        if (opre_all) opre_all[((i0 + rg) * H + h) * Fh + o] = p0;
        e0 = fma(w0 * ww, silu_f<T>(p0), e0);
      }
      if (w1 != T(0)) {
        if (opre_all) opre_all[((i0 + rg + 8) * H + h) * Fh + o] = p1;
        e1 = fma(w1 * ww, silu_f<T>(p1), e1);
      }
    }
  }
  Ep[rg * NOG + og] = e0;
  Ep[(rg + 8) * NOG + og] = e1;
  __syncthreads();
  if (threadIdx.x < nt) {
    T e = T(0);
    for (int q = 0; q < NOG; ++q) e += Ep[threadIdx.x * NOG + q];
    const int g = Gs[threadIdx.x];
    for (int h = 0; h < H; ++h) {
      const T w = hw[(int64_t)g * H + h];
      if (!(w < thr)) e = fma(w, b2[h], e);
    }
    eatom[i0 + threadIdx.x] = e;
  }
}

// R1 of the blended readout: s-bar_i = sum_h w[g,h] out_W1^{hT} (out_w2^h o silu'(pre_i^h)) over the evaluated heads.
template <typename T>
__global__ void __launch_bounds__(512) readout_blend_bwd_k(int64_t N, int F, int H, const T* __restrict__ opre_all,
                                                           const int32_t* __restrict__ a2s, const T* __restrict__ hw,
                                                           T thr, const T* __restrict__ W1, const T* __restrict__ w2,
                                                           T* __restrict__ sb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int Fh = F / 2, NKG = F / 4;
  T* Pb = reinterpret_cast<T*>(smem_raw); // [RT][Fh]  w[g,h] w2 o silu'(pre) of the current head
  __shared__ int Gs[RT];
  const int64_t i0 = (int64_t)blockIdx.x * RT;
  const int nt = (int)min((int64_t)RT, N - i0);
  if (threadIdx.x < RT) Gs[threadIdx.x] = threadIdx.x < nt ? a2s[i0 + threadIdx.x] : -1;
  __syncthreads();
  const int kg = threadIdx.x % NKG, rg = threadIdx.x / NKG;
  T acc0[4] = {T(0), T(0), T(0), T(0)}, acc1[4] = {T(0), T(0), T(0), T(0)};
  for (int h = 0; h < H; ++h) {
    bool any = false; // tile-uniform: every thread scans the 16 rows
    for (int r = 0; r < nt; ++r) any = any || !(hw[(int64_t)Gs[r] * H + h] < thr);
    if (!any) continue;
    __syncthreads();
    for (int q = threadIdx.x; q < RT * Fh; q += blockDim.x) {
      const int r = q / Fh, o = q % Fh;
      T p = T(0);
      if (r < nt) {
        const T w = hw[(int64_t)Gs[r] * H + h];
        if (!(w < thr)) p = w * w2[h * Fh + o] * dsilu_f<T>(opre_all[((i0 + r) * H + h) * Fh + o]);
      }
      Pb[q] = p;
    }
    __syncthreads();
    const T* Wp = W1 + (int64_t)h * Fh * F + kg * 4;
#pragma unroll 4
    for (int o = 0; o < Fh; ++o) {
      T wa[4];
      Vec4<T>::ld(Wp + (int64_t)o * F, wa);
      const T p0 = Pb[rg * Fh + o], p1 = Pb[(rg + 8) * Fh + o];
#pragma unroll
      for (int j = 0; j < 4; ++j) { acc0[j] = fma(wa[j], p0, acc0[j]); acc1[j] = fma(wa[j], p1, acc1[j]); }
    }
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    if (rg < nt) sb[(i0 + rg) * F + kg * 4 + j] = acc0[j];
    if (rg + 8 < nt) sb[(i0 + rg + 8) * F + kg * 4 + j] = acc1[j];
  }
}

// E_g = sum of the structure's atom energies (segmented sum, fixed tree order)
template <typename T>
__global__ void __launch_bounds__(128) struct_sum_k(const int32_t* __restrict__ sptr, const T* __restrict__ eatom,
                                                    T* __restrict__ energy) {
  const int g = blockIdx.x;
  const int a0 = sptr[g], a1 = sptr[g + 1];
  T e = T(0);
  for (int i = a0 + threadIdx.x; i < a1; i += 128) e += eatom[i];
  for (int sft = 16; sft; sft >>= 1) e += __shfl_xor_sync(0xffffffffu, e, sft);
  __shared__ T ws[4];
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = e;
  __syncthreads();
  if (threadIdx.x == 0) energy[g] = (ws[0] + ws[1]) + (ws[2] + ws[3]);
}

// R1: s-bar_i = out_W1^T (out_w2 o silu'(pre_i))
template <typename T>
__global__ void __launch_bounds__(256) readout_bwd_k(int64_t N, int F, int H, const T* __restrict__ opre,
                                                     const int32_t* __restrict__ a2s,
                                                     const int32_t* __restrict__ head, const T* __restrict__ W1,
                                                     const T* __restrict__ w2, T* __restrict__ sb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* Pb = reinterpret_cast<T*>(smem_raw); // [RT][Fh]
  __shared__ int Hs[RT];
  const int Fh = F / 2;
  const int64_t i0 = (int64_t)blockIdx.x * RT;
  const int nt = (int)min((int64_t)RT, N - i0);
  if (threadIdx.x < nt) {
    int h = head[a2s[i0 + threadIdx.x]];
    if (h < 0 || h >= H) h = 0;
    Hs[threadIdx.x] = h;
  }
  __syncthreads();
  for (int q = threadIdx.x; q < nt * Fh; q += blockDim.x) {
    const int r = q / Fh, o = q % Fh;
    Pb[q] = w2[Hs[r] * Fh + o] * dsilu_f<T>(opre[(i0 + r) * Fh + o]);
  }
  __syncthreads();
  for (int k = threadIdx.x; k < F; k += blockDim.x) {
    int r0 = 0;
    while (r0 < nt) {
      const int h = Hs[r0];
      int r1 = r0 + 1;
      while (r1 < nt && Hs[r1] == h) ++r1;
      T acc[RT];
#pragma unroll
      for (int r = 0; r < RT; ++r) acc[r] = T(0);
      const T* Wp = W1 + (int64_t)h * Fh * F + k;
      for (int o = 0; o < Fh; ++o) {
        const T wv = Wp[(int64_t)o * F];
#pragma unroll
        for (int r = 0; r < RT; ++r)
          if (r0 + r < r1) acc[r] = fma(wv, Pb[(r0 + r) * Fh + o], acc[r]);
      }
#pragma unroll
      for (int r = 0; r < RT; ++r)
        if (r0 + r < r1) sb[(i0 + r0 + r) * F + k] = acc[r];
      r0 = r1;
    }
  }
}

template <typename T>
__global__ void __launch_bounds__(256) force_assemble_k(int64_t n3, int nslab, const T* __restrict__ fpart,
                                                        T* __restrict__ forces) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n3) return;
  T s = T(0);
  for (int b = 0; b < nslab; ++b) s += fpart[(int64_t)b * n3 + idx];
  forces[idx] = s;
}

inline unsigned nblk(int64_t n, int b) { return (unsigned)((n + b - 1) / b); }

} // namespace

template <typename T>
int launch_embed_globals(int64_t N, int F, int G, const int32_t* a2s, const double* glob, const T* globW, T* s,
                         __nv_bfloat16* s16, cudaStream_t st) {
  if (N == 0) return 0;
  embed_globals_k<T><<<nblk(N * F, 256), 256, 0, st>>>(N, F, G, a2s, glob, globW, s, s16);
  PNN_KCHECK("embed_globals_k");
  return 1;
}

template <typename T>
int launch_embed(int64_t N, int F, int Zmax, const int32_t* Z, const T* emb, T* s, int* d_err, cudaStream_t st,
                 __nv_bfloat16* s16) {
  if (N == 0) return 0;
  if constexpr (std::is_same<T, float>::value) {
    embed4_k<<<nblk(N * (F / 4), 256), 256, 0, st>>>(N, F / 4, Zmax, Z, reinterpret_cast<const float4*>(emb),
                                                     reinterpret_cast<float4*>(s), d_err, reinterpret_cast<uint2*>(s16));
    PNN_KCHECK("embed4_k");
    return 1;
  }
  embed_k<T><<<nblk(N * F, 256), 256, 0, st>>>(N, F, Zmax, Z, emb, s, d_err, s16); PNN_KCHECK("embed_k");
  return 1;
}
template <typename T, typename IT>
int launch_norm(int64_t N, int F, const IT* PQ, T* sn, T eps, cudaStream_t st, __nv_bfloat16* sn16) {
  if (N == 0) return 0;
  if constexpr (std::is_same<T, float>::value) {
    norm4_k<IT><<<nblk(N * (F / 4), 256), 256, 0, st>>>(N, F, PQ, sn, eps, sn16); PNN_KCHECK("norm4_k");
    return 1;
  }
  norm_k<T, IT><<<nblk(N * F, 256), 256, 0, st>>>(N, F, PQ, sn, eps, sn16); PNN_KCHECK("norm_k");
  return 1;
}
template <typename T, typename IT>
int launch_update(int64_t N, int F, const T* sn, const T* v1, const IT* PQ, const IT* a, T* s_out, T* v_out,
                  cudaStream_t st, __nv_bfloat16* s16, __nv_bfloat16* v16) {
  if (N == 0) return 0;
  if constexpr (std::is_same<T, float>::value) {
    update4_k<IT><<<nblk(N * (F / 4), 256), 256, 0, st>>>(N, F, sn, v1, PQ, a, s_out, v_out, s16, v16); PNN_KCHECK("update4_k");
    return 1;
  }
  update_k<T, IT><<<nblk(N * F, 256), 256, 0, st>>>(N, F, sn, v1, PQ, a, s_out, v_out, s16, v16); PNN_KCHECK("update_k");
  return 1;
}
template <typename T, typename IT>
int launch_update_bwd1(int64_t N, int F, const T* sb, const T* vb, const IT* a, const IT* PQ, T* ab, T* PQb,
                       cudaStream_t st, __nv_bfloat16* ab16) {
  if (N == 0) return 0;
  if constexpr (std::is_same<T, float>::value) {
    update_bwd1_4_k<IT><<<nblk(N * (F / 4), 256), 256, 0, st>>>(N, F, sb, vb, a, PQ, ab, PQb, ab16); PNN_KCHECK("update_bwd1_4_k");
    return 1;
  }
  update_bwd1_k<T, IT><<<nblk(N * F, 256), 256, 0, st>>>(N, F, sb, vb, a, PQ, ab, PQb, ab16); PNN_KCHECK("update_bwd1_k");
  return 1;
}
template <typename T, typename IT>
int launch_update_bwd2(int64_t N, int F, const T* zb, const IT* PQ, T eps, T* sb, T* PQb, cudaStream_t st,
                       __nv_bfloat16* PQb16, __nv_bfloat16* sb16) {
  if (N == 0) return 0;
  if constexpr (std::is_same<T, float>::value) {
    update_bwd2_4_k<IT><<<nblk(N * (F / 4), 256), 256, 0, st>>>(N, F, zb, PQ, eps, sb, PQb, PQb16, sb16); PNN_KCHECK("update_bwd2_4_k");
    return 1;
  }
  update_bwd2_k<T, IT><<<nblk(N * F, 256), 256, 0, st>>>(N, F, zb, PQ, eps, sb, PQb, PQb16, sb16); PNN_KCHECK("update_bwd2_k");
  return 1;
}
template <typename T>
int launch_readout(int64_t N, int64_t S, int F, int H, const T* s, const int32_t* a2s, const int32_t* head,
                   const int32_t* struct_ptr, const T* W1t, const T* b1, const T* w2, const T* b2, T* opre, T* eatom,
                   T* energy, int* d_err, cudaStream_t st) {
  int nl = 0;
  if (N > 0) {
    const size_t smem = sizeof(T) * (RT * F + RT * (F / 2));
    static bool attr_set = false;
    if (!attr_set) {
      cudaFuncSetAttribute(readout_k<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
      attr_set = true;
    }
    if (F % 8 == 0 && F <= 256) {
      const size_t smem2 = sizeof(T) * (RT * F + RT * (F / 8));
      static bool attr2 = false;
      if (!attr2) { cudaFuncSetAttribute(readout2_k<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024); attr2 = true; }
      readout2_k<T><<<nblk(N, RT), 8 * (F / 8), smem2, st>>>(N, F, H, s, a2s, head, W1t, b1, w2, b2, opre, eatom, d_err); PNN_KCHECK("readout2_k");
    } else {
      readout_k<T><<<nblk(N, RT), 128, smem, st>>>(N, F, H, s, a2s, head, W1t, b1, w2, b2, opre, eatom, d_err); PNN_KCHECK("readout_k");
    }
    ++nl;
  }
  if (S > 0) {
    struct_sum_k<T><<<(unsigned)S, 128, 0, st>>>(struct_ptr, eatom, energy); PNN_KCHECK("struct_sum_k");
    ++nl;
  }
  return nl;
}
template <typename T>
int launch_readout_blend(int64_t N, int64_t S, int F, int H, const T* s, const int32_t* a2s, const T* hw, T thr,
                         const int32_t* struct_ptr, const T* W1t, const T* b1, const T* w2, const T* b2, T* opre_all,
                         T* eatom, T* energy, cudaStream_t st) {
  int nl = 0;
  if (N > 0) {
    const size_t smem = sizeof(T) * (RT * F + RT * (F / 8));
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(readout_blend_k<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024); attr = true; }
    readout_blend_k<T><<<nblk(N, RT), 8 * (F / 8), smem, st>>>(N, F, H, s, a2s, hw, thr, W1t, b1, w2, b2, opre_all, eatom);
    PNN_KCHECK("readout_blend_k");
    ++nl;
  }
  if (S > 0) {
    struct_sum_k<T><<<(unsigned)S, 128, 0, st>>>(struct_ptr, eatom, energy); PNN_KCHECK("struct_sum_k");
    ++nl;
  }
  return nl;
}
template <typename T>
int launch_readout_blend_bwd(int64_t N, int F, int H, const T* opre_all, const int32_t* a2s, const T* hw, T thr,
                             const T* W1, const T* w2, T* sb, cudaStream_t st) {
  if (N == 0) return 0;
  const size_t smem = sizeof(T) * (RT * (F / 2));
  readout_blend_bwd_k<T><<<nblk(N, RT), 8 * (F / 4), smem, st>>>(N, F, H, opre_all, a2s, hw, thr, W1, w2, sb);
  PNN_KCHECK("readout_blend_bwd_k");
  return 1;
}
template <typename T>
int launch_struct_sum(int64_t S, const int32_t* struct_ptr, const T* eatom, T* energy, cudaStream_t st) {
  if (S <= 0) return 0;
  struct_sum_k<T><<<(unsigned)S, 128, 0, st>>>(struct_ptr, eatom, energy); PNN_KCHECK("struct_sum_k");
  return 1;
}
template <typename T>
int launch_readout_bwd(int64_t N, int F, int H, const T* opre, const int32_t* a2s, const int32_t* head, const T* W1,
                       const T* w2, T* sb, cudaStream_t st) {
  if (N == 0) return 0;
  const size_t smem = sizeof(T) * (RT * (F / 2));
  if (F % 8 == 0 && F <= 256) {
    readout_bwd2_k<T><<<nblk(N, RT), 8 * (F / 4), smem, st>>>(N, F, H, opre, a2s, head, W1, w2, sb); PNN_KCHECK("readout_bwd2_k");
    return 1;
  }
  readout_bwd_k<T><<<nblk(N, RT), F < 256 ? (F < 64 ? 64 : F) : 256, smem, st>>>(N, F, H, opre, a2s, head, W1, w2, sb); PNN_KCHECK("readout_bwd_k");
  return 1;
}
template <typename T>
int launch_force_assemble(int64_t N, int nslab, const T* fpart, T* forces, cudaStream_t st) {
  if (N == 0) return 0;
  force_assemble_k<T><<<nblk(N * 3, 256), 256, 0, st>>>(N * 3, nslab, fpart, forces); PNN_KCHECK("force_assemble_k");
  return 1;
}

#define PNN_INST(T)                                                                                                  \
  template int launch_embed<T>(int64_t, int, int, const int32_t*, const T*, T*, int*, cudaStream_t,                  \
                               __nv_bfloat16*);                                                                      \
  template int launch_readout<T>(int64_t, int64_t, int, int, const T*, const int32_t*, const int32_t*,               \
                                 const int32_t*, const T*, const T*, const T*, const T*, T*, T*, T*, int*,           \
                                 cudaStream_t);                                                                      \
  template int launch_struct_sum<T>(int64_t, const int32_t*, const T*, T*, cudaStream_t);                            \
  template int launch_readout_blend<T>(int64_t, int64_t, int, int, const T*, const int32_t*, const T*, T,            \
                                       const int32_t*, const T*, const T*, const T*, const T*, T*, T*, T*,           \
                                       cudaStream_t);                                                                \
  template int launch_readout_blend_bwd<T>(int64_t, int, int, const T*, const int32_t*, const T*, T, const T*,       \
                                           const T*, T*, cudaStream_t);                                              \
  template int launch_readout_bwd<T>(int64_t, int, int, const T*, const int32_t*, const int32_t*, const T*,          \
                                     const T*, T*, cudaStream_t);                                                    \
  template int launch_force_assemble<T>(int64_t, int, const T*, T*, cudaStream_t);                                  \
  template int launch_embed_globals<T>(int64_t, int, int, const int32_t*, const double*, const T*, T*,              \
                                       __nv_bfloat16*, cudaStream_t);
#define PNN_INST2(T, IT)                                                                                             \
  template int launch_norm<T, IT>(int64_t, int, const IT*, T*, T, cudaStream_t, __nv_bfloat16*);                     \
  template int launch_update<T, IT>(int64_t, int, const T*, const T*, const IT*, const IT*, T*, T*, cudaStream_t,    \
                                    __nv_bfloat16*, __nv_bfloat16*);                                                 \
  template int launch_update_bwd1<T, IT>(int64_t, int, const T*, const T*, const IT*, const IT*, T*, T*,             \
                                         cudaStream_t, __nv_bfloat16*);                                              \
  template int launch_update_bwd2<T, IT>(int64_t, int, const T*, const IT*, T, T*, T*, cudaStream_t, __nv_bfloat16*, \
                                         __nv_bfloat16*);
PNN_INST(float)
PNN_INST(double)
PNN_INST2(float, float)
PNN_INST2(double, double)
PNN_INST2(float, __nv_bfloat16)
#undef PNN_INST
#undef PNN_INST2

} // namespace pnn
