// edge_mma.cu — a4 / a7 edge kernels of the BF16 model: the filter contraction runs on the tensor cores.
//
// Forward: per edge e = (i <- j): w_e = (flt_W g(d_e) + flt_b) c(d_e), x_e = phi_j o w_e,
// s'_i = s_i + sum x^ss, v'_i = v_i + sum (x^vs u_e + x^vv o v_j).
//
// The filter is a small-K GEMM [edges x K] . [K x 3F] (SURVEY.md §7 hard part 3).  Here a 16-edge tile of ONE receiver
// is the M dimension of mma.sync.m16n8k16 (BF16 operands, FP32 accumulation): A = radial basis times cutoff, rounded
// to BF16, with the cutoff itself as an extra column so that flt_b rides along as an extra weight row; B = filter
// weights.  A warp owns a 32-feature slab of all three chunks.  The MMA columns are permuted (on the host, when the
// model is created) so that thread (g, t) of the accumulator fragment owns the 8 CONTIGUOUS features t*8 .. t*8+7 of
// the slab: the gathered sender rows phi_j / v_j (BF16) are then read with one 16-byte load per row and chunk, straight
// into the fragment layout, and multiplied in registers with packed FP32 FMAs (fma.rn.f32x2).  Rows g and g+8 of a
// tile belong to the same receiver, so every thread keeps a running FP32 sum; the 8 row groups meet once per receiver
// in a 3-stage shuffle reduce-scatter after which lane (g, t) holds component g>>1 (s, v_x, v_y, v_z) of 4 contiguous
// features and does the residual add and the coalesced FP32 + BF16 stores.  No atomics.
#include <algorithm>
#include <cstring>

#include "common.cuh"
#include "edge_mma.cuh"

namespace pnn {

namespace {

constexpr int TE = 16; // edges (rows) per MMA tile
constexpr int NTC = 2; // tiles of one receiver staged per round

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// two BF16 packed in 32 bits -> (low, high) as FP32
__device__ __forceinline__ float2 bf2(uint32_t x) {
  return make_float2(__uint_as_float(x << 16), __uint_as_float(x & 0xffff0000u));
}
__device__ __forceinline__ uint32_t pack_bf2(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ uint4 ldg16(const __nv_bfloat16* p) { return __ldg(reinterpret_cast<const uint4*>(p)); }

// Sum the 32 per-thread partials over the 8 row groups of the fragment layout (lanes t, t+4, ..., t+28) through a
// per-warp shared-memory buffer of 32 x RED_PITCH bytes, 16 values at a time.
// In: acc[a], a = comp*8 + fi.  Out: lane (g, t) holds a = g*4 .. g*4+3, i.e. comp = g>>1, fi = (g&1)*4 + q.
constexpr int RED_PITCH = 80; // 16 floats + 16 bytes: conflict-free 16-byte accesses
__device__ __forceinline__ void reduce_scatter32(const float (&acc)[32], int lane, unsigned char* red, float (&out)[4]) {
  const int g = lane >> 2, t = lane & 3;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
#pragma unroll
    for (int q = 0; q < 4; ++q)
      *reinterpret_cast<float4*>(red + lane * RED_PITCH + q * 16) =
          make_float4(acc[16 * h + 4 * q], acc[16 * h + 4 * q + 1], acc[16 * h + 4 * q + 2], acc[16 * h + 4 * q + 3]);
    __syncwarp();
    if ((g >> 2) == h) {
      float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int gg = 0; gg < 8; ++gg) {
        const float4 x = *reinterpret_cast<const float4*>(red + (gg * 4 + t) * RED_PITCH + (g & 3) * 16);
        s.x += x.x; s.y += x.y; s.z += x.z; s.w += x.w;
      }
      out[0] = s.x; out[1] = s.y; out[2] = s.z; out[3] = s.w;
    }
    __syncwarp();
  }
}

// Stage the A operand of up to NTC tiles of one receiver (one warp): G[row][k] = g_k(d) c(d) (k < K), c(d) (k == K),
// 0 (k > K), BF16; with BWD also G2 = dG/dd.  Us[row] = (u_x, u_y, u_z, d), Cs[row] = (c, c'), Js[row] = sender.
// Rows past the end of the receiver's segment are zero and gather from the receiver itself (finite values times an
// exact zero weight).
template <int KP, bool BWD>
__device__ __forceinline__ void stage_rows(const EdgeMmaArgs& a, int lane, int nrow, int e0, int eb, int self,
                                           unsigned char* Gs, unsigned char* G2s, float4* Us, float2* Cs, int* Js,
                                           float dmu, float gamma, float pi_rc) {
  constexpr int PA = KP * 2 + 16;
  for (int row = lane; row < nrow; row += 32) {
    const int e = e0 + row;
    float4 gq = make_float4(0.f, 0.f, 0.f, 1.f);
    float2 cc = make_float2(0.f, 0.f);
    int j = self;
    if (e < eb) {
      gq = __ldg(reinterpret_cast<const float4*>(a.geom) + e);
      j = __ldg(a.col + e);
      float sn, cs;
      __sincosf(pi_rc * gq.w, &sn, &cs);
      cc = make_float2(0.5f * (cs + 1.0f), -0.5f * pi_rc * sn);
    }
    Us[row] = gq; Cs[row] = cc; Js[row] = j;
  }
  __syncwarp();
  for (int idx = lane; idx < nrow * (KP / 2); idx += 32) {
    const int row = idx / (KP / 2), k = (idx % (KP / 2)) * 2;
    const float d = Us[row].w;
    const float2 cc = Cs[row]; // (0, 0) on padded rows
    const float d0 = d - (float)k * dmu, d1 = d0 - dmu;
    const float r0 = (k < a.K) ? __expf(-gamma * d0 * d0) : 0.f;
    const float r1 = (k + 1 < a.K) ? __expf(-gamma * d1 * d1) : 0.f;
    const float g0 = (k < a.K) ? r0 * cc.x : (k == a.K ? cc.x : 0.f);
    const float g1 = (k + 1 < a.K) ? r1 * cc.x : (k + 1 == a.K ? cc.x : 0.f);
    *reinterpret_cast<uint32_t*>(Gs + row * PA + k * 2) = pack_bf2(g0, g1);
    if (BWD) { // d/dd of the same columns
      const float h0 = (k < a.K) ? r0 * (cc.y - 2.0f * gamma * d0 * cc.x) : (k == a.K ? cc.y : 0.f);
      const float h1 = (k + 1 < a.K) ? r1 * (cc.y - 2.0f * gamma * d1 * cc.x) : (k + 1 == a.K ? cc.y : 0.f);
      *reinterpret_cast<uint32_t*>(G2s + row * PA + k * 2) = pack_bf2(h0, h1);
    }
  }
  __syncwarp();
}

// ------------------------------------------------------------------------------------------ forward
// One warp per receiver (warps of a CTA take neighbouring receivers, so the gathered rows of a structure stay in
// L1): the warp stages the A operand of up to NTC tiles once and then walks the CTA's NSL 32-feature slabs.
// Receivers with more than NTC tiles are processed in rounds; a later round adds to the output of the previous one.
template <int KP, bool HASV>
__global__ void __launch_bounds__(256, 2)
edge_fwd_mma_k(EdgeMmaArgs a, int NSL, int RB, const __nv_bfloat16* __restrict__ phi, const float* s_in,
               int64_t ld_sin, const __nv_bfloat16* __restrict__ v_in, const float* v_res, float* s1, int64_t ld_s1,
               float* v1, EdgeMirror mir) {
  if (*a.d_err & ERRF_EDGE_OVERFLOW) return;
  constexpr int PA = KP * 2 + 16; // padded row pitch (bytes): conflict-free ldmatrix
  constexpr int KS = KP / 16;
  constexpr int NR = NTC * TE;    // staged rows per round
  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
  unsigned char* Ws = smem;                                                     // [3][NSL][32 rows][PA]
  unsigned char* Gs = Ws + (size_t)3 * NSL * 32 * PA + (size_t)warp * NR * PA;  // per warp [NR][PA]
  float4* Us = reinterpret_cast<float4*>(Ws + (size_t)3 * NSL * 32 * PA + (size_t)nwarp * NR * PA) + warp * NR;
  float2* Cs = reinterpret_cast<float2*>(reinterpret_cast<float4*>(Ws + (size_t)3 * NSL * 32 * PA +
                                                                   (size_t)nwarp * NR * PA) + nwarp * NR) + warp * NR;
  int* Js = reinterpret_cast<int*>(reinterpret_cast<float2*>(reinterpret_cast<float4*>(
                Ws + (size_t)3 * NSL * 32 * PA + (size_t)nwarp * NR * PA) + nwarp * NR) + nwarp * NR) + warp * NR;

  unsigned char* Rs = reinterpret_cast<unsigned char*>(
      reinterpret_cast<int*>(reinterpret_cast<float2*>(reinterpret_cast<float4*>(
          Ws + (size_t)3 * NSL * 32 * PA + (size_t)nwarp * NR * PA) + nwarp * NR) + nwarp * NR) + nwarp * NR) +
      (size_t)warp * 32 * RED_PITCH;                                            // per warp [32][RED_PITCH]

  const int F = a.F;
  const int g = lane >> 2, t = lane & 3;
  const int slab0 = blockIdx.y * NSL; // first 32-feature slab of this CTA
  // filter weights of this CTA's slabs -> shared memory (packed rows are KP*2 bytes; smem rows are padded)
  {
    const int nslab_tot = F / 32;
    constexpr int V = KP * 2 / 16; // 16-byte vectors per row
    for (int idx = tid; idx < 3 * NSL * 32 * V; idx += nthr) {
      const int v = idx % V, r = idx / V; // r = (c*NSL + w)*32 + row
      const int c = r / (NSL * 32), w = (r / 32) % NSL, row = r % 32;
      const uint4 val = __ldg(reinterpret_cast<const uint4*>(a.fltP) + ((size_t)((c * nslab_tot + slab0 + w) * 32 + row)) * V + v);
      *reinterpret_cast<uint4*>(Ws + (size_t)r * PA + v * 16) = val;
    }
  }
  __syncthreads();
  const float rc = a.rc;
  const float dmu = (a.K > 1) ? rc / (float)(a.K - 1) : rc;
  const float gamma = 1.0f / (2.0f * dmu * dmu);
  const float pi_rc = 3.14159265358979323846f / rc;
  // ldmatrix lane addressing: A tile (rows = lane&15, k half = lane>>4), B tiles (row = lane&7, k half = (lane>>3)&1,
  // n-tile of the pair = lane>>4)
  const uint32_t a_off = (uint32_t)((lane & 15) * PA + (lane >> 4) * 16);
  const uint32_t b_off = (uint32_t)(((lane >> 4) * 8 + (lane & 7)) * PA + ((lane >> 3) & 1) * 16);
  const uint32_t Ws_u = smem_u32(Ws), Gs_u = smem_u32(Gs);

  const int64_t nchunk = (a.N + RB - 1) / RB;
  for (int64_t ch = blockIdx.x; ch < nchunk; ch += gridDim.x) {
    const int64_t i_end = min((int64_t)(ch + 1) * RB, a.N);
    for (int64_t i = ch * RB + warp; i < i_end; i += nwarp) {
      const int ea = a.rowptr[i], eb = a.rowptr[i + 1];
      // The warp's next receiver: pull its geometry, sender indices and own rows towards L2 now, so that the DRAM
      // latency of these streaming reads overlaps the work on the current receiver.
      if (i + nwarp < i_end) {
        const int64_t in = i + nwarp;
        const int en = __ldg(a.rowptr + in);
        if (lane < 4) prefetch_l2(a.geom + en + lane * 8);
        else if (lane == 4) prefetch_l2(a.col + en);
        else if (lane < 5 + NSL) prefetch_l2(s_in + in * ld_sin + (slab0 + lane - 5) * 32);
        else if (HASV && lane < 5 + 4 * NSL) {
          const int q = lane - 5 - NSL;
          prefetch_l2(v_res + (in * 3 + q / NSL) * F + (slab0 + q % NSL) * 32);
        }
      }
      bool first = true;
      for (int r0 = ea; first || r0 < eb; r0 += NR) {
        const int ntile = min(NTC, (eb - r0 + TE - 1) / TE);
        stage_rows<KP, false>(a, lane, ntile * TE, r0, eb, (int)i, Gs, nullptr, Us, Cs, Js, dmu, gamma, pi_rc);
        for (int sl = 0; sl < NSL; ++sl) {
          const int fbase = (slab0 + sl) * 32 + t * 8; // first of this thread's 8 contiguous features
          float2 acc[16]; // [comp: s, v_x, v_y, v_z][n-tile]: the thread's 8 features as 4 pairs
#pragma unroll
          for (int q = 0; q < 16; ++q) acc[q] = make_float2(0.f, 0.f);
          // the receiver's own row (residual input) is fetched now and used after the reduction
          const int comp = g >> 1;
          const int f = (slab0 + sl) * 32 + t * 8 + (g & 1) * 4;
          const int64_t voff = (i * 3 + (comp - 1)) * F + f;
          float4 own = make_float4(0.f, 0.f, 0.f, 0.f);
          if (comp == 0) own = first ? *reinterpret_cast<const float4*>(s_in + i * ld_sin + f)
                                     : *reinterpret_cast<const float4*>(s1 + i * ld_s1 + f);
          else if (!first) own = *reinterpret_cast<const float4*>(v1 + voff);
          else if (HASV) own = *reinterpret_cast<const float4*>(v_res + voff);
          for (int tl = 0; tl < ntile; ++tl) {
            uint32_t af[KS][4];
#pragma unroll
            for (int ks = 0; ks < KS; ++ks)
              ldsm_x4(Gs_u + tl * TE * PA + a_off + ks * 32, af[ks][0], af[ks][1], af[ks][2], af[ks][3]);
            // rows past the segment end have zero weights; their gathers are skipped (payload = 0)
            const bool ok0 = r0 + tl * TE + g < eb, ok1 = r0 + tl * TE + g + 8 < eb;
            const int64_t o0 = (int64_t)Js[tl * TE + g] * 3 * F + fbase, o1 = (int64_t)Js[tl * TE + g + 8] * 3 * F + fbase;
            const float4 u0 = Us[tl * TE + g], u1 = Us[tl * TE + g + 8];
            const uint4 zero4 = make_uint4(0u, 0u, 0u, 0u);
            // all gathers of the tile are issued before the first MMA (one memory latency per tile and slab)
            uint4 pp0[3], pp1[3], va0[3], va1[3];
#pragma unroll
            for (int c = 0; c < (HASV ? 3 : 2); ++c) {
              pp0[c] = ok0 ? ldg16(phi + o0 + c * F) : zero4;
              pp1[c] = ok1 ? ldg16(phi + o1 + c * F) : zero4;
            }
            if (HASV) {
#pragma unroll
              for (int ax = 0; ax < 3; ++ax) {
                va0[ax] = ok0 ? ldg16(v_in + o0 + ax * F) : zero4;
                va1[ax] = ok1 ? ldg16(v_in + o1 + ax * F) : zero4;
              }
            }
#pragma unroll
            for (int c = 0; c < (HASV ? 3 : 2); ++c) {
              const uint4 p0 = pp0[c], p1 = pp1[c];
              float C[4][4];
#pragma unroll
              for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                for (int q = 0; q < 4; ++q) C[nt][q] = 0.f;
              const uint32_t wbase = Ws_u + (uint32_t)((c * NSL + sl) * 32) * PA + b_off;
#pragma unroll
              for (int np = 0; np < 2; ++np)
#pragma unroll
                for (int ks = 0; ks < KS; ++ks) {
                  uint32_t b0, b1, b2, b3;
                  ldsm_x4(wbase + np * 16 * PA + ks * 32, b0, b1, b2, b3);
                  mma_bf16(C[2 * np], af[ks], b0, b1);
                  mma_bf16(C[2 * np + 1], af[ks], b2, b3);
                }
              const uint32_t pw0[4] = {p0.x, p0.y, p0.z, p0.w}, pw1[4] = {p1.x, p1.y, p1.z, p1.w};
#pragma unroll
              for (int nt = 0; nt < 4; ++nt) {
                const float2 ph0 = bf2(pw0[nt]), ph1 = bf2(pw1[nt]);
                const float2 w0 = make_float2(C[nt][0], C[nt][1]), w1 = make_float2(C[nt][2], C[nt][3]);
                if (c == 0) {
                  acc[nt] = __ffma2_rn(ph0, w0, acc[nt]);
                  acc[nt] = __ffma2_rn(ph1, w1, acc[nt]);
                } else {
                  const float2 x0 = __fmul2_rn(ph0, w0), x1 = __fmul2_rn(ph1, w1);
#pragma unroll
                  for (int ax = 0; ax < 3; ++ax) {
                    float2 m0, m1;
                    if (c == 1) {
                      const float ua0 = ax == 0 ? u0.x : (ax == 1 ? u0.y : u0.z);
                      const float ua1 = ax == 0 ? u1.x : (ax == 1 ? u1.y : u1.z);
                      m0 = make_float2(ua0, ua0); m1 = make_float2(ua1, ua1);
                    } else {
                      const uint32_t q0 = nt == 0 ? va0[ax].x : nt == 1 ? va0[ax].y : nt == 2 ? va0[ax].z : va0[ax].w;
                      const uint32_t q1 = nt == 0 ? va1[ax].x : nt == 1 ? va1[ax].y : nt == 2 ? va1[ax].z : va1[ax].w;
                      m0 = bf2(q0); m1 = bf2(q1);
                    }
                    acc[4 * (1 + ax) + nt] = __ffma2_rn(x0, m0, acc[4 * (1 + ax) + nt]);
                    acc[4 * (1 + ax) + nt] = __ffma2_rn(x1, m1, acc[4 * (1 + ax) + nt]);
                  }
                }
              }
            }
          }
          // reduction over the 8 row groups, residual add, stores
          float accf[32], r4[4];
#pragma unroll
          for (int q = 0; q < 16; ++q) { accf[2 * q] = acc[q].x; accf[2 * q + 1] = acc[q].y; }
          reduce_scatter32(accf, lane, Rs, r4);
          const float4 o = make_float4(own.x + r4[0], own.y + r4[1], own.z + r4[2], own.w + r4[3]);
          if (comp == 0) {
            *reinterpret_cast<float4*>(s1 + i * ld_s1 + f) = o;
            if (mir.s1)
              *reinterpret_cast<uint2*>(mir.s1 + i * mir.ld_s1 + f) = make_uint2(pack_bf2(o.x, o.y), pack_bf2(o.z, o.w));
          } else {
            *reinterpret_cast<float4*>(v1 + voff) = o;
            if (mir.v1) *reinterpret_cast<uint2*>(mir.v1 + voff) = make_uint2(pack_bf2(o.x, o.y), pack_bf2(o.z, o.w));
          }
        }
        __syncwarp(); // the staging buffers are rewritten by the next round / receiver
        first = false;
      }
    }
  }
}

// 32-feature slabs per CTA: a divisor of F/32, at most 4
int pick_nsl(int F) {
  const int ns = F / 32;
  for (int nw = 4; nw > 1; --nw)
    if (ns % nw == 0) return nw;
  return 1;
}

} // namespace

int edge_mma_kp(int K) { return (K + 1 + 15) / 16 * 16; }

// Host-side packing of one block's filter for the MMA kernels (layout in the header).
void pack_filter_bf16(int F, int K, const double* fltW, const double* fltb, uint16_t* out) {
  const int KP = edge_mma_kp(K), ns = F / 32;
  auto to_bf16 = [](double x) -> uint16_t {
    float f = (float)x;
    uint32_t u;
    std::memcpy(&u, &f, 4);
    const uint32_t r = u + 0x7fffu + ((u >> 16) & 1u); // round to nearest even
    return (uint16_t)(r >> 16);
  };
  for (int c = 0; c < 3; ++c)
    for (int s = 0; s < ns; ++s)
      for (int nt = 0; nt < 4; ++nt)
        for (int g = 0; g < 8; ++g) {
          const int f = s * 32 + (g >> 1) * 8 + nt * 2 + (g & 1);
          const int64_t src = (int64_t)c * F + f;
          uint16_t* dst = out + ((int64_t)((c * ns + s) * 4 + nt) * 8 + g) * KP;
          for (int k = 0; k < KP; ++k) dst[k] = k < K ? to_bf16(fltW[src * K + k]) : (k == K ? to_bf16(fltb[src]) : 0);
        }
}

size_t edge_mma_smem(int KP, int NSL, int nwarp, bool bwd) {
  const int PA = KP * 2 + 16, NR = NTC * TE;
  return (size_t)3 * NSL * 32 * PA + (size_t)nwarp * (NR * (PA * (bwd ? 2 : 1) + 16 + 8 + 4) + 32 * RED_PITCH);
}

int launch_edge_fwd_mma(const EdgeMmaArgs& a, const __nv_bfloat16* phi, const float* s_in, int64_t ld_sin,
                        const __nv_bfloat16* v_in, const float* v_res, float* s1, int64_t ld_s1, float* v1,
                        const EdgeMirror& mir, cudaStream_t st) {
  if (a.N == 0) return 0;
  const int KP = edge_mma_kp(a.K), NSL = pick_nsl(a.F), NWARP = 8;
  const int RB = 32;
  const int64_t nchunk = (a.N + RB - 1) / RB;
  dim3 grid((unsigned)std::min<int64_t>(nchunk, 148 * 2), a.F / 32 / NSL);
  const size_t smem = edge_mma_smem(KP, NSL, NWARP, false);
#define PNN_LAUNCH(KPV, HV)                                                                                        \
  {                                                                                                                \
    static bool attr_set = false;                                                                                  \
    if (!attr_set) {                                                                                               \
      cudaFuncSetAttribute(edge_fwd_mma_k<KPV, HV>, cudaFuncAttributeMaxDynamicSharedMemorySize, 110 * 1024);      \
      attr_set = true;                                                                                             \
    }                                                                                                              \
    edge_fwd_mma_k<KPV, HV><<<grid, NWARP * 32, smem, st>>>(a, NSL, RB, phi, s_in, ld_sin, v_in, v_res, s1, ld_s1, \
                                                            v1, mir);                                              \
    PNN_KCHECK("edge_fwd_mma_k");                                                                                  \
  }
  const bool hv = v_in != nullptr;
  if (KP == 16) { if (hv) PNN_LAUNCH(16, true) else PNN_LAUNCH(16, false) }
  else if (KP == 32) { if (hv) PNN_LAUNCH(32, true) else PNN_LAUNCH(32, false) }
  else { if (hv) PNN_LAUNCH(48, true) else PNN_LAUNCH(48, false) }
#undef PNN_LAUNCH
  return 1;
}

} // namespace pnn
