// graph.cu — a1: cell-list radius graph with minimum-image PBC, emitted as receiver-sorted CSR.
//
// Definition followed ("Cutoff radius", PAPER.md:269 periodic boundary
// conditions): edge (i <- j) iff i != j, same structure, |x_j - x_i + shift.C|^2 < r_c^2 evaluated in FP64,
// with shift = -round(frac(x_j - x_i)) on periodic axes (one image per ordered pair).
//
// Design: every structure gets its own grid of cells at least r_c wide (GridDesc); a structure with <= BRUTE_N
// atoms, or narrower than 3 cells along a periodic axis, degenerates to one cell on that axis, i.e. the same
// code does the all-pairs search for small molecules and the 27-cell stencil for the 100,000-atom cell.
// One warp per receiver scans its candidate cells 32 atoms at a time; __ballot_sync compaction gives every
// accepted sender its slot, so rows come out in a deterministic order without atomics.  Two passes (count,
// exclusive scan, emit).  The emit pass also stores the per-edge unit vector and distance in model precision.
#include <algorithm>

#include "common.cuh"

namespace pnn {

namespace {

constexpr int BRUTE_N = 256;   // structures up to this size use a single cell (all-pairs)
constexpr int SCAN_ITEMS = 1024;

// ------------------------------------------------------------------------------------------ scans
__global__ void __launch_bounds__(256) scan_reduce_k(const int32_t* __restrict__ in, int64_t n, int32_t* bsum) {
  const int64_t base = (int64_t)blockIdx.x * SCAN_ITEMS;
  int s = 0;
  for (int q = threadIdx.x; q < SCAN_ITEMS; q += 256) {
    const int64_t idx = base + q;
    if (idx < n) s += in[idx];
  }
  __shared__ int ws[8];
  for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    int t = 0;
    for (int w = 0; w < 8; ++w) t += ws[w];
    bsum[blockIdx.x] = t;
  }
}

// single block: exclusive scan of bsum[0..nb) in place, bsum[nb] = total
__global__ void __launch_bounds__(1024) scan_bsums_k(int32_t* bsum, int nb) {
  __shared__ int ws[32];
  __shared__ int carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < nb; base += 1024) {
    const int idx = base + threadIdx.x;
    const int x = idx < nb ? bsum[idx] : 0;
    int incl = x;
    for (int o = 1; o < 32; o <<= 1) {
      const int y = __shfl_up_sync(0xffffffffu, incl, o);
      if ((threadIdx.x & 31) >= o) incl += y;
    }
    if ((threadIdx.x & 31) == 31) ws[threadIdx.x >> 5] = incl;
    __syncthreads();
    if (threadIdx.x < 32) {
      int v = ws[threadIdx.x], iv = v;
      for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, iv, o);
        if (threadIdx.x >= o) iv += y;
      }
      ws[threadIdx.x] = iv - v; // exclusive warp offsets
    }
    __syncthreads();
    const int carry = carry_s;
    const int excl = carry + ws[threadIdx.x >> 5] + incl - x;
    if (idx < nb) bsum[idx] = excl;
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = excl + x;
    __syncthreads();
  }
  if (threadIdx.x == 0) bsum[nb] = carry_s;
}

// out[i] = exclusive prefix of in over [0,n); out[n] = total.  256 threads x 4 consecutive items.
__global__ void __launch_bounds__(256) scan_apply_k(const int32_t* __restrict__ in, int64_t n,
                                                    const int32_t* __restrict__ bsum, int32_t* out) {
  const int64_t base = (int64_t)blockIdx.x * SCAN_ITEMS + threadIdx.x * 4;
  int x[4], tsum = 0;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    x[q] = (base + q < n) ? in[base + q] : 0;
    tsum += x[q];
  }
  int incl = tsum;
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(0xffffffffu, incl, o);
    if ((threadIdx.x & 31) >= o) incl += y;
  }
  __shared__ int ws[8];
  if ((threadIdx.x & 31) == 31) ws[threadIdx.x >> 5] = incl;
  __syncthreads();
  int woff = 0;
  for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) woff += ws[w];
  int run = bsum[blockIdx.x] + woff + incl - tsum;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (base + q < n) out[base + q] = run;
    run += x[q];
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 255) out[n] = bsum[gridDim.x];
}

// Small inputs (molecular batches: a few thousand cells / atoms): the whole scan in ONE block, 1024 threads x 4 items per
// round with a running carry — one launch instead of three latency-bound ones.  out[n] = total.
__global__ void __launch_bounds__(1024) scan_small_k(const int32_t* __restrict__ in, int n, int32_t* __restrict__ out) {
  __shared__ int ws[32];
  __shared__ int carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < n; base += 4096) {
    const int i0 = base + threadIdx.x * 4;
    int x[4], tsum = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      x[q] = (i0 + q < n) ? in[i0 + q] : 0;
      tsum += x[q];
    }
    int incl = tsum;
    for (int o = 1; o < 32; o <<= 1) {
      const int y = __shfl_up_sync(0xffffffffu, incl, o);
      if ((threadIdx.x & 31) >= o) incl += y;
    }
    if ((threadIdx.x & 31) == 31) ws[threadIdx.x >> 5] = incl;
    __syncthreads();
    if (threadIdx.x < 32) {
      int v = ws[threadIdx.x], iv = v;
      for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, iv, o);
        if (threadIdx.x >= o) iv += y;
      }
      ws[threadIdx.x] = iv - v; // exclusive warp offsets
    }
    __syncthreads();
    int run = carry_s + ws[threadIdx.x >> 5] + incl - tsum;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (i0 + q < n) out[i0 + q] = run;
      run += x[q];
    }
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = run;
    __syncthreads();
  }
  if (threadIdx.x == 0) out[n] = carry_s;
}

int exclusive_scan(const int32_t* in, int64_t n, int32_t* out, int32_t* tmp, cudaStream_t st) {
  if (n <= 16384) {
    scan_small_k<<<1, 1024, 0, st>>>(in, (int)n, out); PNN_KCHECK("scan_small_k");
    return 1;
  }
  const int nb = (int)((n + SCAN_ITEMS - 1) / SCAN_ITEMS);
  scan_reduce_k<<<nb, 256, 0, st>>>(in, n, tmp); PNN_KCHECK("scan_reduce_k");
  scan_bsums_k<<<1, 1024, 0, st>>>(tmp, nb); PNN_KCHECK("scan_bsums_k");
  scan_apply_k<<<nb, 256, 0, st>>>(in, n, tmp, out); PNN_KCHECK("scan_apply_k");
  return 3;
}

// ------------------------------------------------------------------------------------------ grid descriptors
__device__ void inverse3(const double* C, double* Ci) {
  const double a = C[0], b = C[1], c = C[2], d = C[3], e = C[4], f = C[5], g = C[6], h = C[7], i = C[8];
  const double det = a * (e * i - f * h) - b * (d * i - f * g) + c * (d * h - e * g);
  Ci[0] = (e * i - f * h) / det; Ci[1] = (c * h - b * i) / det; Ci[2] = (b * f - c * e) / det;
  Ci[3] = (f * g - d * i) / det; Ci[4] = (a * i - c * g) / det; Ci[5] = (c * d - a * f) / det;
  Ci[6] = (d * h - e * g) / det; Ci[7] = (b * g - a * h) / det; Ci[8] = (a * e - b * d) / det;
}

// One CTA per structure: atom->structure map, lattice, fractional bounding box, cell grid dimensions.
__global__ void __launch_bounds__(128) desc_k(int64_t S, const double* __restrict__ pos,
                                              const int32_t* __restrict__ sptr, const double* __restrict__ cell,
                                              const uint8_t* __restrict__ pbc, double rc, GridDesc* desc,
                                              int32_t* ncell, int32_t* a2s) {
  const int g = blockIdx.x;
  const int a0 = sptr[g], a1 = sptr[g + 1], n = a1 - a0;
  for (int i = a0 + threadIdx.x; i < a1; i += blockDim.x) a2s[i] = g;
  __shared__ GridDesc d;
  __shared__ double rmin[3][128], rmax[3][128];
  if (threadIdx.x == 0) {
    int per[3] = {0, 0, 0};
    if (cell && pbc)
      for (int a = 0; a < 3; ++a) per[a] = pbc[3 * g + a] ? 1 : 0;
    d.periodic = per[0] | per[1] | per[2];
    for (int q = 0; q < 9; ++q) d.C[q] = d.Ci[q] = (q % 4 == 0) ? 1.0 : 0.0;
    if (d.periodic) {
      for (int q = 0; q < 9; ++q) d.C[q] = cell[9 * (int64_t)g + q];
      inverse3(d.C, d.Ci);
    }
    for (int a = 0; a < 3; ++a) { d.per[a] = per[a]; d.dim[a] = 1; d.fmin[a] = 0.0; d.fscale[a] = 0.0; }
    d.ncell = 1;
  }
  __syncthreads();
  if (n > BRUTE_N) { // block-uniform
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int i = a0 + threadIdx.x; i < a1; i += blockDim.x) {
      const double x = pos[3 * (int64_t)i], y = pos[3 * (int64_t)i + 1], z = pos[3 * (int64_t)i + 2];
      for (int a = 0; a < 3; ++a) {
        const double f = x * d.Ci[0 + a] + y * d.Ci[3 + a] + z * d.Ci[6 + a];
        lo[a] = fmin(lo[a], f); hi[a] = fmax(hi[a], f);
      }
    }
    for (int a = 0; a < 3; ++a) { rmin[a][threadIdx.x] = lo[a]; rmax[a][threadIdx.x] = hi[a]; }
    __syncthreads();
    if (threadIdx.x == 0) {
      for (int a = 0; a < 3; ++a) {
        double l = rmin[a][0], h = rmax[a][0];
        for (int t = 1; t < 128; ++t) { l = fmin(l, rmin[a][t]); h = fmax(h, rmax[a][t]); }
        const double cn = sqrt(d.Ci[0 + a] * d.Ci[0 + a] + d.Ci[3 + a] * d.Ci[3 + a] + d.Ci[6 + a] * d.Ci[6 + a]);
        const double ext = d.per[a] ? 1.0 : (h - l);
        const double width = ext / cn; // distance between the bounding planes f_a = const
        int m = (int)fmin(floor(width / rc), 1024.0);
        if (d.per[a]) { if (m < 3) m = 1; } else { if (m < 1) m = 1; }
        d.dim[a] = m;
        d.fmin[a] = d.per[a] ? 0.0 : l;
        rmax[a][0] = ext; // keep for fscale below
      }
      // never more cells than atoms (the cell arrays are sized N + S)
      while ((int64_t)d.dim[0] * d.dim[1] * d.dim[2] > (int64_t)n) {
        int a = 0;
        if (d.dim[1] > d.dim[a]) a = 1;
        if (d.dim[2] > d.dim[a]) a = 2;
        int m = d.dim[a] / 2;
        if (d.per[a] && m < 3) m = 1;
        if (m < 1) m = 1;
        d.dim[a] = m;
      }
      for (int a = 0; a < 3; ++a) {
        const double ext = rmax[a][0];
        d.fscale[a] = (ext > 0.0) ? (double)d.dim[a] / ext : 0.0;
      }
      d.ncell = d.dim[0] * d.dim[1] * d.dim[2];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { desc[g] = d; ncell[g] = d.ncell; }
}

__device__ __forceinline__ int cell_coord(const GridDesc& d, int a, double f) {
  if (d.dim[a] == 1) return 0;
  double t;
  if (d.per[a]) t = (f - floor(f)) * d.fscale[a];
  else t = (f - d.fmin[a]) * d.fscale[a];
  int c = (int)t;
  if (c < 0) c = 0;
  if (c > d.dim[a] - 1) c = d.dim[a] - 1;
  return c;
}

__global__ void __launch_bounds__(256) bin_k(int64_t N, const double* __restrict__ pos,
                                             const int32_t* __restrict__ sptr, const int32_t* __restrict__ a2s,
                                             const GridDesc* __restrict__ desc, const int32_t* __restrict__ cell_off,
                                             int32_t* cid, int32_t* cell_cnt, int32_t* sorted) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int g = a2s[i];
  const GridDesc& d = desc[g];
  if (d.ncell == 1) {
    const int c = cell_off[g];
    cid[i] = c;
    sorted[i] = (int)i; // the single cell lists the structure's atoms in index order
    if (i == sptr[g]) cell_cnt[c] = sptr[g + 1] - sptr[g];
    return;
  }
  const double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
  int cc[3];
  for (int a = 0; a < 3; ++a) cc[a] = cell_coord(d, a, x * d.Ci[0 + a] + y * d.Ci[3 + a] + z * d.Ci[6 + a]);
  const int c = cell_off[g] + (cc[0] * d.dim[1] + cc[1]) * d.dim[2] + cc[2];
  cid[i] = c;
  atomicAdd(&cell_cnt[c], 1);
}

__global__ void __launch_bounds__(256) fill_k(int64_t N, const int32_t* __restrict__ a2s,
                                              const GridDesc* __restrict__ desc, const int32_t* __restrict__ cid,
                                              const int32_t* __restrict__ cell_start, int32_t* cell_fill,
                                              int32_t* sorted) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  if (desc[a2s[i]].ncell == 1) return;
  const int c = cid[i];
  sorted[cell_start[c] + atomicAdd(&cell_fill[c], 1)] = (int)i;
}

// One warp per cell: order the cell's atoms by index.  The lanes first test whether the run is already ordered (always so
// for single-cell structures, where one thread walking 40 dependent global loads used to take 24 us); only an unordered
// cell (~10 atoms, filled through atomics) falls back to lane 0's insertion sort.
__global__ void __launch_bounds__(256) sortcells_k(int64_t ncap, const int32_t* __restrict__ cell_start,
                                                   int32_t* sorted) {
  const int64_t c = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (c >= ncap) return;
  const int b = cell_start[c], e = cell_start[c + 1];
  bool ok = true;
  for (int p = b + 1 + lane; p < e; p += 32) ok = ok && (sorted[p - 1] <= sorted[p]);
  if (__all_sync(0xffffffffu, ok)) return;
  if (lane != 0) return;
  for (int p = b + 1; p < e; ++p) {
    const int v = sorted[p];
    int q = p - 1;
    while (q >= b && sorted[q] > v) { sorted[q + 1] = sorted[q]; --q; }
    sorted[q + 1] = v;
  }
}

// ------------------------------------------------------------------------------------------ neighbour passes
template <typename T, bool EMIT, bool ALLIMG>
__global__ void __launch_bounds__(256) neigh_k(int64_t N, const double* __restrict__ pos,
                                               const int32_t* __restrict__ a2s, const GridDesc* __restrict__ desc,
                                               const int32_t* __restrict__ cell_off, const int32_t* __restrict__ cid,
                                               const int32_t* __restrict__ cell_start,
                                               const int32_t* __restrict__ sorted, double rc2, int32_t* deg,
                                               const int32_t* __restrict__ rowptr, int32_t* col, int8_t* shift,
                                               Geom<T>* geom, int64_t max_edges) {
  constexpr int all_images = ALLIMG ? 1 : 0;
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; // one warp per receiver
  const int lane = threadIdx.x & 31;
  if (i >= N) return;
  const int g = a2s[i];
  const GridDesc& d = desc[g];
  const double xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
  const int periodic = d.periodic;
  double C[9], Ci[9];
  int per[3];
#pragma unroll
  for (int q = 0; q < 9; ++q) { C[q] = d.C[q]; Ci[q] = d.Ci[q]; }
#pragma unroll
  for (int a = 0; a < 3; ++a) per[a] = d.per[a];
  const int dx = d.dim[0], dy = d.dim[1], dz = d.dim[2];
  const int c0 = cell_off[g];
  int lc = cid[i] - c0;
  const int cz = lc % dz; lc /= dz;
  const int cy = lc % dy;
  const int cx = lc / dy;
  // all_images: on a periodic axis too narrow for a cell list (one cell), every image within the cutoff is an edge, the
  // atom's own images included; M[a] shifts are tried on either side of the nearest image.  On an axis with >= 3 cells
  // (each >= r_c wide) only the nearest image can be inside the cutoff.
  int M0 = 0, M1 = 0, M2 = 0;
  if (ALLIMG && periodic) {
    const double rc = sqrt(rc2);
    if (per[0] && dx == 1) M0 = (int)floor(rc * sqrt(Ci[0] * Ci[0] + Ci[3] * Ci[3] + Ci[6] * Ci[6])) + 1;
    if (per[1] && dy == 1) M1 = (int)floor(rc * sqrt(Ci[1] * Ci[1] + Ci[4] * Ci[4] + Ci[7] * Ci[7])) + 1;
    if (per[2] && dz == 1) M2 = (int)floor(rc * sqrt(Ci[2] * Ci[2] + Ci[5] * Ci[5] + Ci[8] * Ci[8])) + 1;
  }
  int base = 0;
  bool ok_row = true;
  if (EMIT) {
    base = rowptr[i];
    ok_row = (int64_t)rowptr[i + 1] <= max_edges;
  }
  int total = 0;
  for (int ox = (dx > 1 ? -1 : 0); ox <= (dx > 1 ? 1 : 0); ++ox) {
    int nx = cx + ox;
    if (nx < 0 || nx >= dx) { if (!per[0]) continue; nx = (nx + dx) % dx; }
    for (int oy = (dy > 1 ? -1 : 0); oy <= (dy > 1 ? 1 : 0); ++oy) {
      int ny = cy + oy;
      if (ny < 0 || ny >= dy) { if (!per[1]) continue; ny = (ny + dy) % dy; }
      for (int oz = (dz > 1 ? -1 : 0); oz <= (dz > 1 ? 1 : 0); ++oz) {
        int nz = cz + oz;
        if (nz < 0 || nz >= dz) { if (!per[2]) continue; nz = (nz + dz) % dz; }
        const int c = c0 + (nx * dy + ny) * dz + nz;
        const int pb = cell_start[c], pe = cell_start[c + 1];
        for (int p0 = pb; p0 < pe; p0 += 32) {
          const int p = p0 + lane;
          int j = -1, n0 = 0, n1 = 0, n2 = 0;
          double D0 = 0, D1 = 0, D2 = 0;
          const bool cand = p < pe;
          if (cand) {
            j = sorted[p];
            // same operation order as the definition (oracle B1): D, f = D.C^-1, n = round(f), r = D - n.C
            D0 = pos[3 * (int64_t)j] - xi; D1 = pos[3 * (int64_t)j + 1] - yi; D2 = pos[3 * (int64_t)j + 2] - zi;
            if (periodic) {
              if (per[0]) n0 = (int)round(D0 * Ci[0] + D1 * Ci[3] + D2 * Ci[6]);
              if (per[1]) n1 = (int)round(D0 * Ci[1] + D1 * Ci[4] + D2 * Ci[7]);
              if (per[2]) n2 = (int)round(D0 * Ci[2] + D1 * Ci[5] + D2 * Ci[8]);
            }
          }
          for (int e0 = -M0; e0 <= M0; ++e0)
            for (int e1 = -M1; e1 <= M1; ++e1)
              for (int e2 = -M2; e2 <= M2; ++e2) { // warp-uniform trip counts: one ballot per image
                bool hit = false;
                const int m0 = n0 + e0, m1 = n1 + e1, m2 = n2 + e2;
                double r0 = 0, r1 = 0, r2 = 0;
                if (cand && (j != (int)i || (all_images && (m0 | m1 | m2) != 0))) {
                  r0 = D0 + (-(m0 * C[0] + m1 * C[3] + m2 * C[6]));
                  r1 = D1 + (-(m0 * C[1] + m1 * C[4] + m2 * C[7]));
                  r2 = D2 + (-(m0 * C[2] + m1 * C[5] + m2 * C[8]));
                  hit = (r0 * r0 + r1 * r1 + r2 * r2) < rc2;
                }
                const unsigned m = __ballot_sync(0xffffffffu, hit);
                if (EMIT) {
                  if (hit && ok_row) {
                    const int64_t e = (int64_t)base + total + __popc(m & ((1u << lane) - 1u));
                    col[e] = j;
                    shift[3 * e] = (int8_t)(-m0); shift[3 * e + 1] = (int8_t)(-m1); shift[3 * e + 2] = (int8_t)(-m2);
                    const double dd = sqrt(r0 * r0 + r1 * r1 + r2 * r2);
                    Geom<T> q;
                    q.ux = (T)(r0 / dd); q.uy = (T)(r1 / dd); q.uz = (T)(r2 / dd); q.d = (T)dd;
                    geom[e] = q;
                  }
                }
                total += __popc(m);
              }
        }
      }
    }
  }
  if (!EMIT && lane == 0) deg[i] = total;
}

__global__ void check_edges_k(int64_t N, const int32_t* rowptr, int64_t max_edges, int* d_err, int* d_ovf) {
  const bool over = (int64_t)rowptr[N] > max_edges;
  *d_ovf = over ? ERRF_EDGE_OVERFLOW : 0; // per-graph word: only the next build resets it
  if (over) atomicOr(d_err, ERRF_EDGE_OVERFLOW);
}

// ---- max-neighbour cap (reading Q16): a receiver keeps its `cap` nearest senders, smallest
// FP64 squared distance first, ties by sender index, then by lattice shift.  One warp per receiver; the rank of an entry is
// the number of entries of its row with a smaller key (rows are a few dozen entries long).
__device__ __forceinline__ double cap_d2(const double* __restrict__ pos, const GridDesc& D, int64_t i, int j,
                                         const int8_t* __restrict__ sh) {
  double q = 0.0;
#pragma unroll
  for (int b = 0; b < 3; ++b) {
    const double sc = (double)sh[0] * D.C[0 + b] + (double)sh[1] * D.C[3 + b] + (double)sh[2] * D.C[6 + b];
    const double r = pos[3 * (int64_t)j + b] - pos[3 * i + b] + sc;
    q += r * r;
  }
  return q;
}
__global__ void __launch_bounds__(256) cap_mark_k(int64_t N, int cap, const double* __restrict__ pos,
                                                  const int32_t* __restrict__ a2s, const GridDesc* __restrict__ desc,
                                                  const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                                                  const int8_t* __restrict__ shift, uint8_t* __restrict__ keep,
                                                  int32_t* __restrict__ deg2, int64_t max_edges) {
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (i >= N || (int64_t)rowptr[N] > max_edges) return;
  const int ea = rowptr[i], eb = rowptr[i + 1], deg = eb - ea;
  if (lane == 0) deg2[i] = min(deg, cap);
  if (deg <= cap) {
    for (int e = ea + lane; e < eb; e += 32) keep[e] = 1;
    return;
  }
  const GridDesc& D = desc[a2s[i]];
  for (int e = ea + lane; e < eb; e += 32) {
    const double de = cap_d2(pos, D, i, col[e], shift + 3 * (int64_t)e);
    int rank = 0;
    for (int o = ea; o < eb; ++o) {
      if (o == e) continue;
      const double dv = cap_d2(pos, D, i, col[o], shift + 3 * (int64_t)o);
      bool less = dv < de;
      if (dv == de) {
        if (col[o] != col[e]) less = col[o] < col[e];
        else {
          less = false;
          for (int b = 0; b < 3; ++b)
            if (shift[3 * (int64_t)o + b] != shift[3 * (int64_t)e + b]) { less = shift[3 * (int64_t)o + b] < shift[3 * (int64_t)e + b]; break; }
        }
      }
      rank += less ? 1 : 0;
    }
    keep[e] = rank < cap ? 1 : 0;
  }
}
// ok[0] = 1 when the uncapped graph fitted (the compaction ran); the primary rowptr is replaced only then
__global__ void cap_finish_k(int64_t N, const int32_t* rowptr, const int32_t* rowptr2, int64_t max_edges, int32_t* ok) {
  *ok = ((int64_t)rowptr[N] <= max_edges) ? 1 : 0;
}
__global__ void __launch_bounds__(256) cap_rowptr_k(int64_t N, const int32_t* __restrict__ rowptr2, int32_t* rowptr,
                                                    const int32_t* ok) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i <= N && *ok) rowptr[i] = rowptr2[i];
}
template <typename T>
__global__ void __launch_bounds__(256) cap_compact_k(int64_t N, const int32_t* __restrict__ rowptr,
                                                     const int32_t* __restrict__ rowptr2, const uint8_t* __restrict__ keep,
                                                     const int32_t* __restrict__ col, const int8_t* __restrict__ shift,
                                                     const Geom<T>* __restrict__ geom, int32_t* __restrict__ col2,
                                                     int8_t* __restrict__ shift2, Geom<T>* __restrict__ geom2,
                                                     int64_t max_edges) {
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (i >= N || (int64_t)rowptr[N] > max_edges) return;
  const int ea = rowptr[i], eb = rowptr[i + 1];
  int out = rowptr2[i];
  for (int e0 = ea; e0 < eb; e0 += 32) { // stable: kept entries stay in their order
    const int e = e0 + lane;
    const bool k = e < eb && keep[e];
    const unsigned m = __ballot_sync(0xffffffffu, k);
    if (k) {
      const int o = out + __popc(m & ((1u << lane) - 1u));
      col2[o] = col[e];
      shift2[3 * (int64_t)o] = shift[3 * (int64_t)e]; shift2[3 * (int64_t)o + 1] = shift[3 * (int64_t)e + 1];
      shift2[3 * (int64_t)o + 2] = shift[3 * (int64_t)e + 2];
      geom2[o] = geom[e];
    }
    out += __popc(m);
  }
}

// Order-independent 64-bit checksum of the position array (xor of a mix of (index, bit pattern)).
__device__ __forceinline__ unsigned long long mix64(unsigned long long x) {
  x ^= x >> 33; x *= 0xff51afd7ed558ccdULL; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ULL; x ^= x >> 33;
  return x;
}
__global__ void __launch_bounds__(256) pos_hash_k(int64_t n, const double* __restrict__ pos, unsigned long long* out) {
  unsigned long long h = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    h ^= mix64((unsigned long long)__double_as_longlong(pos[i]) + 0x9e3779b97f4a7c15ULL * (unsigned long long)(i + 1));
#pragma unroll
  for (int o = 16; o; o >>= 1) h ^= __shfl_xor_sync(0xffffffffu, h, o);
  if ((threadIdx.x & 31) == 0 && h) atomicXor(out, h);
}
__global__ void pos_cmp_k(unsigned long long* chk, int* d_err) {
  if (chk[1] != chk[0]) atomicOr(d_err, ERRF_STALE_GRAPH);
  chk[1] = 0;
}

} // namespace

int launch_graph_build(const GraphBuffers& gb, int64_t N, int64_t S, const double* pos, const int32_t* sptr,
                       const double* cell, const uint8_t* pbc, double rc, int prec, int all_images, int max_neighbors,
                       cudaStream_t st) {
  int nl = 0;
  cudaMemsetAsync(gb.d_poschk, 0, 2 * sizeof(unsigned long long), st);
  if (N == 0 || S == 0) {
    cudaMemsetAsync(gb.rowptr, 0, sizeof(int32_t) * (N + 1), st);
    cudaMemsetAsync(gb.d_ovf, 0, sizeof(int), st);
    return 0;
  }
  pos_hash_k<<<(unsigned)std::min<int64_t>((3 * N + 255) / 256, 592), 256, 0, st>>>(3 * N, pos, gb.d_poschk);
  PNN_KCHECK("pos_hash_k"); ++nl;
  const int64_t ncap = N + S; // upper bound on the number of cells
  desc_k<<<(unsigned)S, 128, 0, st>>>(S, pos, sptr, cell, pbc, rc, gb.desc, gb.ncell, gb.a2s); PNN_KCHECK("desc_k"); ++nl;
  nl += exclusive_scan(gb.ncell, S, gb.cell_off, gb.scan_tmp, st);
  cudaMemsetAsync(gb.cell_cnt, 0, sizeof(int32_t) * (ncap + 1), st);
  cudaMemsetAsync(gb.cell_fill, 0, sizeof(int32_t) * (ncap + 1), st);
  const unsigned nbA = (unsigned)((N + 255) / 256);
  bin_k<<<nbA, 256, 0, st>>>(N, pos, sptr, gb.a2s, gb.desc, gb.cell_off, gb.cid, gb.cell_cnt, gb.sorted); PNN_KCHECK("bin_k"); ++nl;
  nl += exclusive_scan(gb.cell_cnt, ncap, gb.cell_start, gb.scan_tmp, st);
  fill_k<<<nbA, 256, 0, st>>>(N, gb.a2s, gb.desc, gb.cid, gb.cell_start, gb.cell_fill, gb.sorted); PNN_KCHECK("fill_k"); ++nl;
  sortcells_k<<<(unsigned)((ncap * 32 + 255) / 256), 256, 0, st>>>(ncap, gb.cell_start, gb.sorted); PNN_KCHECK("sortcells_k"); ++nl;
  const unsigned nbW = (unsigned)((N * 32 + 255) / 256);
  const double rc2 = rc * rc;
#define PNN_NEIGH(TT, EM, ...)                                                                          \
  {                                                                                                     \
    if (all_images) neigh_k<TT, EM, true><<<nbW, 256, 0, st>>>(__VA_ARGS__);                            \
    else neigh_k<TT, EM, false><<<nbW, 256, 0, st>>>(__VA_ARGS__);                                      \
    PNN_KCHECK("neigh_k");                                                                              \
  }
  PNN_NEIGH(float, false, N, pos, gb.a2s, gb.desc, gb.cell_off, gb.cid, gb.cell_start, gb.sorted, rc2, gb.deg, nullptr,
            nullptr, nullptr, (Geom<float>*)nullptr, gb.max_edges)
  ++nl;
  nl += exclusive_scan(gb.deg, N, gb.rowptr, gb.scan_tmp, st);
  check_edges_k<<<1, 1, 0, st>>>(N, gb.rowptr, gb.max_edges, gb.d_err, gb.d_ovf); PNN_KCHECK("check_edges_k"); ++nl;
  if (prec == 2) {
    PNN_NEIGH(double, true, N, pos, gb.a2s, gb.desc, gb.cell_off, gb.cid, gb.cell_start, gb.sorted, rc2, nullptr,
              gb.rowptr, gb.col, gb.shift, (Geom<double>*)gb.geom, gb.max_edges)
  } else {
    PNN_NEIGH(float, true, N, pos, gb.a2s, gb.desc, gb.cell_off, gb.cid, gb.cell_start, gb.sorted, rc2, nullptr,
              gb.rowptr, gb.col, gb.shift, (Geom<float>*)gb.geom, gb.max_edges)
  }
#undef PNN_NEIGH
  ++nl;
  if (max_neighbors > 0 && gb.cap_col) { // keep the nearest max_neighbors senders of every receiver (stable compaction)
    cap_mark_k<<<nbW, 256, 0, st>>>(N, max_neighbors, pos, gb.a2s, gb.desc, gb.rowptr, gb.col, gb.shift, gb.cap_keep,
                                    gb.cap_deg, gb.max_edges);
    PNN_KCHECK("cap_mark_k"); ++nl;
    nl += exclusive_scan(gb.cap_deg, N, gb.cap_rowptr, gb.scan_tmp, st);
    const size_t gs = prec == 2 ? sizeof(Geom<double>) : sizeof(Geom<float>);
    if (prec == 2)
      cap_compact_k<double><<<nbW, 256, 0, st>>>(N, gb.rowptr, gb.cap_rowptr, gb.cap_keep, gb.col, gb.shift,
                                                 (const Geom<double>*)gb.geom, gb.cap_col, gb.cap_shift,
                                                 (Geom<double>*)gb.cap_geom, gb.max_edges);
    else
      cap_compact_k<float><<<nbW, 256, 0, st>>>(N, gb.rowptr, gb.cap_rowptr, gb.cap_keep, gb.col, gb.shift,
                                                (const Geom<float>*)gb.geom, gb.cap_col, gb.cap_shift,
                                                (Geom<float>*)gb.cap_geom, gb.max_edges);
    PNN_KCHECK("cap_compact_k"); ++nl;
    // back into the primary arrays (an overflowing graph was left untouched and stays flagged)
    cap_finish_k<<<1, 1, 0, st>>>(N, gb.rowptr, gb.cap_rowptr, gb.max_edges, gb.cap_deg + N); PNN_KCHECK("cap_finish_k"); ++nl;
    cudaMemcpyAsync(gb.col, gb.cap_col, sizeof(int32_t) * gb.max_edges, cudaMemcpyDeviceToDevice, st);
    cudaMemcpyAsync(gb.shift, gb.cap_shift, 3 * gb.max_edges, cudaMemcpyDeviceToDevice, st);
    cudaMemcpyAsync(gb.geom, gb.cap_geom, gs * gb.max_edges, cudaMemcpyDeviceToDevice, st);
    cap_rowptr_k<<<(unsigned)((N + 1 + 255) / 256), 256, 0, st>>>(N, gb.cap_rowptr, gb.rowptr, gb.cap_deg + N);
    PNN_KCHECK("cap_rowptr_k"); ++nl;
  }
  return nl;
}

int launch_pos_check(const GraphBuffers& gb, int64_t N, const double* pos, cudaStream_t st) {
  if (N == 0) return 0;
  pos_hash_k<<<(unsigned)std::min<int64_t>((3 * N + 255) / 256, 592), 256, 0, st>>>(3 * N, pos, gb.d_poschk + 1);
  PNN_KCHECK("pos_hash_k");
  pos_cmp_k<<<1, 1, 0, st>>>(gb.d_poschk, gb.d_err);
  PNN_KCHECK("pos_cmp_k");
  return 2;
}

} // namespace pnn
