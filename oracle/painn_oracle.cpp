// oracle/painn_oracle.cpp
//
// TEST INFRASTRUCTURE ONLY.  A plain, slow, FP64 CPU implementation of the hot path
// (radius graph -> PaiNN forward -> per-head readout -> reverse sweep -> forces), written
// from the paper's statement of the problem, to be the parity oracle for the CUDA library.
// It shares no code, header, table or helper with paper_2604_15380_b200/; only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
//
// What it follows (the paper has no PaiNN equations):
//   PAPER.md:147, 499   backbone = PaiNN, ref [48] (Schuett, Unke, Gastegger, ICML 2021)
//   PAPER.md:242        "pairwise interaction structure with low-order scalar/vector updates"
//   PAPER.md:53         forces are energy gradients with respect to positions
//   PAPER.md:126, 232   shared trunk, 16 per-dataset output heads
//   PAPER.md:229-231    radial basis, cutoff radius;  PAPER.md:269 periodic boundary conditions
//   SURVEY.md §8(c)     steps B1..B5 (forward) and R1..R4 (reverse sweep), readings Q1..Q23
//
// Style: one loop nest per equation, in the order and notation of SURVEY.md §8(c); no
// blocking, no fusion, no BLAS.  `#pragma omp parallel for` is placed only on loops over
// atoms whose iterations write disjoint outputs (deterministic, race free).
//
// Parity pins (tests/test_oracle_*.py, -m "not gpu"): brute-force neighbour definitions on
// lattices with textbook shell counts, closed forms of the RBF/cutoff, rotation /
// translation / permutation invariance, equivariance of v, isolated-atom closed form,
// hand-expanded 2-atom F=1 model, finite differences, forward-mode dual numbers (the
// templated scalar below), sum F = 0, torque = 0.
// "parity unpinned": the paper's trained-model figures (|dE| 0.021 / 0.080 eV, Table XV) —
// the checkpoint and datasets are not available.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// ------------------------------------------------------------------ forward-mode dual numbers
struct Dual {
  double v, d;
  Dual() : v(0.0), d(0.0) {}
  Dual(double a) : v(a), d(0.0) {}
  Dual(double a, double b) : v(a), d(b) {}
};
inline Dual operator+(Dual a, Dual b) { return Dual(a.v + b.v, a.d + b.d); }
inline Dual operator-(Dual a, Dual b) { return Dual(a.v - b.v, a.d - b.d); }
inline Dual operator-(Dual a) { return Dual(-a.v, -a.d); }
inline Dual operator*(Dual a, Dual b) { return Dual(a.v * b.v, a.d * b.v + a.v * b.d); }
inline Dual operator/(Dual a, Dual b) { return Dual(a.v / b.v, (a.d * b.v - a.v * b.d) / (b.v * b.v)); }
inline Dual& operator+=(Dual& a, Dual b) { a = a + b; return a; }
inline Dual s_exp(Dual a) { double e = std::exp(a.v); return Dual(e, e * a.d); }
inline Dual s_sqrt(Dual a) { double r = std::sqrt(a.v); return Dual(r, a.d / (2.0 * r)); }
inline Dual s_cos(Dual a) { return Dual(std::cos(a.v), -std::sin(a.v) * a.d); }
inline Dual s_sin(Dual a) { return Dual(std::sin(a.v), std::cos(a.v) * a.d); }
inline double s_exp(double a) { return std::exp(a); }
inline double s_sqrt(double a) { return std::sqrt(a); }
inline double s_cos(double a) { return std::cos(a); }
inline double s_sin(double a) { return std::sin(a); }
inline double value_of(double a) { return a; }
inline double value_of(Dual a) { return a.v; }

// ------------------------------------------------------------------ model = views into the blob
struct Cfg { int F, T, K, H, Zmax; double rc, eps; int rbf; int images; int max_nb; int n_glob; int head_type, d1, d2; };  // rbf: 0 Gaussian, 1 Bessel; images: 0 minimum image, 1 all; max_nb: 0 = no cap; n_glob: global attributes per structure
struct Block {
  const double *msg_W1, *msg_b1, *msg_W2, *msg_b2, *flt_W, *flt_b;
  const double *upd_U, *upd_V, *upd_A1, *upd_c1, *upd_A2, *upd_c2;
};
struct Head { const double *W1, *b1, *w2, *b2; };
// Pooled graph-level head of the paper's lead model ("Output heads 16 (graph-level)", "2 shared layers
// (dim 50) + 2 branch layers (dim 776)"; reading Q29): x_g = mean_i s_i, two shared Linear+SiLU layers of width
// d1, then per head two Linear+SiLU layers of width d2 and a linear output.
struct PoolShared { const double *W1, *b1, *W2, *b2; };                 // [d1][F], [d1], [d1][d1], [d1]
struct PoolBranch { const double *W1, *b1, *W2, *b2, *w3, *b3; };       // [d2][d1], [d2], [d2][d2], [d2], [d2], [1]
struct Model {
  Cfg c; const double* emb; std::vector<Block> blk; std::vector<Head> head; const double* glob_W;
  PoolShared ps; std::vector<PoolBranch> pb;
};

// Blob order: SURVEY.md §8(b) "Weight blob"; matrices row-major [out][in], y = W x + b.
long parse_blob(const Cfg& c, const double* w, Model* m) {
  const long F = c.F, K = c.K;
  const double* p = w;
  auto take = [&](long n) { const double* q = p; p += n; return q; };
  if (m) { m->c = c; m->blk.resize(c.T); m->head.resize(c.H); }
  const double* emb = take((long)(c.Zmax + 1) * F);
  if (m) m->emb = emb;
  for (int t = 0; t < c.T; ++t) {
    Block b;
    b.msg_W1 = take(F * F);     b.msg_b1 = take(F);
    b.msg_W2 = take(3 * F * F); b.msg_b2 = take(3 * F);
    b.flt_W = take(3 * F * K);  b.flt_b = take(3 * F);
    b.upd_U = take(F * F);      b.upd_V = take(F * F);
    b.upd_A1 = take(F * 2 * F); b.upd_c1 = take(F);
    b.upd_A2 = take(3 * F * F); b.upd_c2 = take(3 * F);
    if (m) m->blk[t] = b;
  }
  if (c.head_type == 1) {
    const long d1 = c.d1, d2 = c.d2;
    PoolShared ps;
    ps.W1 = take(d1 * F); ps.b1 = take(d1); ps.W2 = take(d1 * d1); ps.b2 = take(d1);
    if (m) { m->ps = ps; m->pb.resize(c.H); }
    for (int h = 0; h < c.H; ++h) {
      PoolBranch b;
      b.W1 = take(d2 * d1); b.b1 = take(d2); b.W2 = take(d2 * d2); b.b2 = take(d2); b.w3 = take(d2); b.b3 = take(1);
      if (m) m->pb[h] = b;
    }
  } else
  for (int h = 0; h < c.H; ++h) {
    Head hd;
    hd.W1 = take((F / 2) * F); hd.b1 = take(F / 2); hd.w2 = take(F / 2); hd.b2 = take(1);
    if (m) m->head[h] = hd;
  }
  // global attributes ("global attributes such as charge and spin used as additional input features";
  // DESIGN.md reading Q30): glob_W [F][n_glob], appended to the blob when n_glob > 0
  const double* gw = take((long)F * c.n_glob);
  if (m) m->glob_W = gw;
  return (long)(p - w);
}

// ------------------------------------------------------------------ B1: neighbours, O(n^2) per structure
struct Edges {
  std::vector<int32_t> recv, send;      // e = (i <- j): receiver i, sender j
  std::vector<int8_t> shift;            // [E][3] integer lattice shift
  std::vector<double> shift_cart;       // [E][3] shift . C  (constant w.r.t. positions)
  std::vector<int32_t> rowptr;          // [N+1] receiver-sorted CSR
};

void inverse3(const double* C, double* Ci) {
  const double a = C[0], b = C[1], c = C[2], d = C[3], e = C[4], f = C[5], g = C[6], h = C[7], i = C[8];
  const double det = a * (e * i - f * h) - b * (d * i - f * g) + c * (d * h - e * g);
  Ci[0] = (e * i - f * h) / det; Ci[1] = (c * h - b * i) / det; Ci[2] = (b * f - c * e) / det;
  Ci[3] = (f * g - d * i) / det; Ci[4] = (a * i - c * g) / det; Ci[5] = (c * d - a * f) / det;
  Ci[6] = (d * h - e * g) / det; Ci[7] = (b * g - a * h) / det; Ci[8] = (a * e - b * d) / det;
}

// SURVEY §8(c) B1.  Rows of C are the lattice vectors; positions are row vectors.
// all_images = 0: one (minimum) image per ordered pair (reading Q13).  all_images = 1: the radius graph of the infinite
// periodic structure — every ordered pair (i, j), i == j included, and every integer lattice shift s with
// 0 < |x_j - x_i + s.C| < rc; needed when a cell is narrower than 2 rc.
// max_nb > 0: the paper's "Max neighbors" (Table V: 20; 64 with periodic boundary conditions;
// DESIGN.md reading Q16): every receiver keeps only its max_nb NEAREST senders inside the cutoff — smallest squared distance
// first, ties broken by the sender index, then by the lattice shift — so the edge set is no longer symmetric.
void cap_neighbours(int N, const double* pos, int max_nb, Edges* E);
void neighbours_all(int N, int S, const double* pos, const int32_t* sptr, const double* cell,
                    const uint8_t* pbc, double rc, Edges* E, int all_images);
void neighbours(int N, int S, const double* pos, const int32_t* sptr, const double* cell,
                const uint8_t* pbc, double rc, Edges* E, int all_images = 0, int max_nb = 0) {
  neighbours_all(N, S, pos, sptr, cell, pbc, rc, E, all_images);
  if (max_nb > 0) cap_neighbours(N, pos, max_nb, E);
}
void cap_neighbours(int N, const double* pos, int max_nb, Edges* E) {
  Edges out;
  out.rowptr.assign(N + 1, 0);
  for (int i = 0; i < N; ++i) {
    const int a = E->rowptr[i], b = E->rowptr[i + 1];
    std::vector<int> idx(b - a);
    std::vector<double> d2(b - a);
    for (int e = a; e < b; ++e) {
      idx[e - a] = e;
      double q = 0.0;
      for (int c = 0; c < 3; ++c) {
        const double r = pos[3 * E->send[e] + c] - pos[3 * i + c] + E->shift_cart[3 * e + c];
        q += r * r;
      }
      d2[e - a] = q;
    }
    // plain selection sort of the row by (d^2, sender, shift): the first max_nb entries are kept
    for (int x = 0; x < (int)idx.size(); ++x)
      for (int y = x + 1; y < (int)idx.size(); ++y) {
        const int ex = idx[x], ey = idx[y];
        bool less = d2[ey - a] < d2[ex - a];
        if (d2[ey - a] == d2[ex - a]) {
          if (E->send[ey] != E->send[ex]) less = E->send[ey] < E->send[ex];
          else
            for (int c = 0; c < 3; ++c)
              if (E->shift[3 * ey + c] != E->shift[3 * ex + c]) { less = E->shift[3 * ey + c] < E->shift[3 * ex + c]; break; }
        }
        if (less) { idx[x] = ey; idx[y] = ex; }
      }
    const int keep = std::min<int>(max_nb, (int)idx.size());
    std::vector<int> kept(idx.begin(), idx.begin() + keep);
    for (int x = 0; x < keep; ++x)          // back to the original (ascending sender) order within the row
      for (int y = x + 1; y < keep; ++y)
        if (kept[y] < kept[x]) { const int t = kept[x]; kept[x] = kept[y]; kept[y] = t; }
    for (int e : kept) {
      out.recv.push_back(i); out.send.push_back(E->send[e]);
      for (int c = 0; c < 3; ++c) { out.shift.push_back(E->shift[3 * e + c]); out.shift_cart.push_back(E->shift_cart[3 * e + c]); }
    }
    out.rowptr[i + 1] = out.rowptr[i] + keep;
  }
  *E = out;
}
void neighbours_all(int N, int S, const double* pos, const int32_t* sptr, const double* cell,
                    const uint8_t* pbc, double rc, Edges* E, int all_images) {
  E->rowptr.assign(N + 1, 0);
  for (int g = 0; g < S; ++g) {
    const bool periodic = cell && pbc && (pbc[3 * g] || pbc[3 * g + 1] || pbc[3 * g + 2]);
    double C[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1}, Ci[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
    if (periodic) { std::memcpy(C, cell + 9 * g, sizeof C); inverse3(C, Ci); }
    if (periodic && all_images) {
      int M[3] = {0, 0, 0};   // shifts tried around the nearest image: enough to cover rc on every periodic axis
      for (int a = 0; a < 3; ++a) {
        const double cn = std::sqrt(Ci[0 + a] * Ci[0 + a] + Ci[3 + a] * Ci[3 + a] + Ci[6 + a] * Ci[6 + a]);
        if (pbc[3 * g + a]) M[a] = (int)std::floor(rc * cn) + 1;   // 1/cn = distance between lattice planes of axis a
      }
      for (int i = sptr[g]; i < sptr[g + 1]; ++i)
        for (int j = sptr[g]; j < sptr[g + 1]; ++j) {
          const double D[3] = {pos[3 * j] - pos[3 * i], pos[3 * j + 1] - pos[3 * i + 1], pos[3 * j + 2] - pos[3 * i + 2]};
          int n0[3] = {0, 0, 0};
          for (int a = 0; a < 3; ++a)
            if (pbc[3 * g + a]) n0[a] = (int)std::round(D[0] * Ci[0 + a] + D[1] * Ci[3 + a] + D[2] * Ci[6 + a]);
          for (int s0 = -n0[0] - M[0]; s0 <= -n0[0] + M[0]; ++s0)      // ascending shift: the canonical edge order
            for (int s1 = -n0[1] - M[1]; s1 <= -n0[1] + M[1]; ++s1)
              for (int s2 = -n0[2] - M[2]; s2 <= -n0[2] + M[2]; ++s2) {
                if (j == i && s0 == 0 && s1 == 0 && s2 == 0) continue;
                const int sh[3] = {s0, s1, s2};
                double sc[3], r[3];
                for (int b = 0; b < 3; ++b) {
                  sc[b] = sh[0] * C[0 + b] + sh[1] * C[3 + b] + sh[2] * C[6 + b];
                  r[b] = D[b] + sc[b];
                }
                if (r[0] * r[0] + r[1] * r[1] + r[2] * r[2] < rc * rc) {
                  E->recv.push_back(i); E->send.push_back(j);
                  for (int b = 0; b < 3; ++b) { E->shift.push_back((int8_t)sh[b]); E->shift_cart.push_back(sc[b]); }
                  E->rowptr[i + 1]++;
                }
              }
        }
      continue;
    }
    for (int i = sptr[g]; i < sptr[g + 1]; ++i) {
      for (int j = sptr[g]; j < sptr[g + 1]; ++j) {
        if (j == i) continue;                                       // Q12: no self edge
        const double D[3] = {pos[3 * j] - pos[3 * i], pos[3 * j + 1] - pos[3 * i + 1], pos[3 * j + 2] - pos[3 * i + 2]};
        int n[3] = {0, 0, 0};
        if (periodic) {
          for (int a = 0; a < 3; ++a) {
            const double f = D[0] * Ci[0 + a] + D[1] * Ci[3 + a] + D[2] * Ci[6 + a];   // f = D . C^-1
            if (pbc[3 * g + a]) n[a] = (int)std::round(f);
          }
        }
        double sc[3], r[3];
        for (int b = 0; b < 3; ++b) {
          sc[b] = -(n[0] * C[0 + b] + n[1] * C[3 + b] + n[2] * C[6 + b]);               // shift . C, shift = -n
          r[b] = D[b] + sc[b];
        }
        if (r[0] * r[0] + r[1] * r[1] + r[2] * r[2] < rc * rc) {                       // strict, FP64 (Q3)
          E->recv.push_back(i); E->send.push_back(j);
          for (int b = 0; b < 3; ++b) { E->shift.push_back((int8_t)(-n[b])); E->shift_cart.push_back(sc[b]); }
          E->rowptr[i + 1]++;
        }
      }
    }
  }
  for (int i = 0; i < N; ++i) E->rowptr[i + 1] += E->rowptr[i];
}

// ------------------------------------------------------------------ elementary functions
template <class S> inline S silu(S x) { return x / (S(1.0) + s_exp(-x)); }            // x / (1 + e^-x)
inline double dsilu(double x) { const double sg = 1.0 / (1.0 + std::exp(-x)); return sg * (1.0 + x * (1.0 - sg)); }

// Gaussian radial basis (Q2): centres mu_k = k rc/(K-1), gamma = 1/(2 dmu^2), dmu = rc/(K-1).
// Bessel radial basis (the paper's lead model, "4 (Bessel)"; type 1): the zeroth-order spherical Bessel
// functions b_n(d) = sqrt(2/rc) sin(n pi d / rc) / d, n = k + 1 = 1..K, orthonormal on [0, rc] with weight d^2.
template <class S> inline S rbf(S d, int k, int K, double rc, int type = 0) {
  if (type == 1) return S(std::sqrt(2.0 / rc)) * s_sin(S((k + 1) * M_PI / rc) * d) / d;
  const double dmu = (K > 1) ? rc / (K - 1) : rc;
  const double gamma = 1.0 / (2.0 * dmu * dmu), mu = k * dmu;
  return s_exp(S(-gamma) * (d - S(mu)) * (d - S(mu)));
}
// cosine cutoff (Q3): c(d) = 1/2 (cos(pi d / rc) + 1)
template <class S> inline S fcut(S d, double rc) { return S(0.5) * (s_cos(S(M_PI / rc) * d) + S(1.0)); }

// ------------------------------------------------------------------ tape of one evaluation
template <class S> struct BlockTape {
  std::vector<S> s_in, v_in;       // block input s [N][F], v [N][3][F]
  std::vector<S> hpre, phi;        // msg_W1 s + b1 [N][F];  phi [N][3F]
  std::vector<S> s1, v1;           // s', v' after the message step
  std::vector<S> P, Q, n, dot;     // [N][3][F] x2, [N][F] x2
  std::vector<S> kpre, a;          // [N][F], [N][3F]
};
template <class S> struct Tape {
  std::vector<S> r, d, u;          // per edge: r [E][3], d [E], u [E][3]
  std::vector<BlockTape<S>> blk;
  std::vector<S> s_out, v_out;     // final features
  std::vector<S> opre;             // readout pre-activation [N][F/2]
  std::vector<S> eatom;            // per-atom energy
  std::vector<S> pool_pre;         // pooled head: pre-activations per structure [S][2 d1 + 2 d2]
};

// ------------------------------------------------------------------ forward (B2..B5)
template <class S>
void forward(const Model& m, int N, int nS, const int32_t* Z, const S* pos, const int32_t* sptr,
             const int32_t* head, const Edges& ed, Tape<S>& tp, S* energy, const double* glob = nullptr) {
  const int F = m.c.F, K = m.c.K, T = m.c.T;
  const double rc = m.c.rc;
  const long E = (long)ed.recv.size();

  // edge geometry: r_e = x_j - x_i + shift.C, d = |r|, u = r/d
  tp.r.assign(3 * E, S(0.0)); tp.d.assign(E, S(0.0)); tp.u.assign(3 * E, S(0.0));
#pragma omp parallel for schedule(static)
  for (long e = 0; e < E; ++e) {
    const int i = ed.recv[e], j = ed.send[e];
    S d2 = S(0.0);
    for (int b = 0; b < 3; ++b) {
      tp.r[3 * e + b] = pos[3 * j + b] - pos[3 * i + b] + S(ed.shift_cart[3 * e + b]);
      d2 += tp.r[3 * e + b] * tp.r[3 * e + b];
    }
    tp.d[e] = s_sqrt(d2);
    for (int b = 0; b < 3; ++b) tp.u[3 * e + b] = tp.r[3 * e + b] / tp.d[e];
  }

  // B2 embedding
  std::vector<S> s((long)N * F), v((long)N * 3 * F, S(0.0));
  for (int i = 0; i < N; ++i)
    for (int f = 0; f < F; ++f) s[(long)i * F + f] = S(m.emb[(long)Z[i] * F + f]);
  if (m.c.n_glob > 0 && glob) {   // s0_i += glob_W . (charge, spin, ...) of the atom's structure (reading Q30)
    for (int g = 0; g < nS; ++g)
      for (int i = sptr[g]; i < sptr[g + 1]; ++i)
        for (int f = 0; f < F; ++f)
          for (int q = 0; q < m.c.n_glob; ++q)
            s[(long)i * F + f] += S(m.glob_W[(long)f * m.c.n_glob + q] * glob[(long)g * m.c.n_glob + q]);
  }

  tp.blk.resize(T);
  for (int t = 0; t < T; ++t) {
    const Block& w = m.blk[t];
    BlockTape<S>& bt = tp.blk[t];
    bt.s_in = s; bt.v_in = v;
    bt.hpre.assign((long)N * F, S(0.0)); bt.phi.assign((long)N * 3 * F, S(0.0));
    // B3a  phi_j = msg_W2 silu(msg_W1 s_j + msg_b1) + msg_b2
#pragma omp parallel for schedule(static)
    for (int j = 0; j < N; ++j) {
      std::vector<S> h(F);
      for (int o = 0; o < F; ++o) {
        S acc = S(w.msg_b1[o]);
        for (int k = 0; k < F; ++k) acc += S(w.msg_W1[(long)o * F + k]) * s[(long)j * F + k];
        bt.hpre[(long)j * F + o] = acc;
        h[o] = silu(acc);
      }
      for (int o = 0; o < 3 * F; ++o) {
        S acc = S(w.msg_b2[o]);
        for (int k = 0; k < F; ++k) acc += S(w.msg_W2[(long)o * F + k]) * h[k];
        bt.phi[(long)j * 3 * F + o] = acc;
      }
    }
    // B3b  per receiver i, ascending sender (Q21): filter, message, segment sum, residual
    bt.s1 = s; bt.v1 = v;
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < N; ++i) {
      std::vector<S> g(K), wf(3 * F);
      for (int e = ed.rowptr[i]; e < ed.rowptr[i + 1]; ++e) {
        const int j = ed.send[e];
        const S d = tp.d[e];
        for (int k = 0; k < K; ++k) g[k] = rbf(d, k, K, rc, m.c.rbf);
        const S c = fcut(d, rc);
        for (int o = 0; o < 3 * F; ++o) {                     // w_e = (flt_W g + flt_b) c(d)
          S acc = S(w.flt_b[o]);
          for (int k = 0; k < K; ++k) acc += S(w.flt_W[(long)o * K + k]) * g[k];
          wf[o] = acc * c;
        }
        for (int f = 0; f < F; ++f) {
          const S xss = bt.phi[(long)j * 3 * F + f] * wf[f];
          const S xvs = bt.phi[(long)j * 3 * F + F + f] * wf[F + f];
          const S xvv = bt.phi[(long)j * 3 * F + 2 * F + f] * wf[2 * F + f];
          bt.s1[(long)i * F + f] += xss;
          for (int a = 0; a < 3; ++a)
            bt.v1[((long)i * 3 + a) * F + f] += xvs * tp.u[3 * e + a] + xvv * v[((long)j * 3 + a) * F + f];
        }
      }
    }
    // B4 update
    bt.P.assign((long)N * 3 * F, S(0.0)); bt.Q.assign((long)N * 3 * F, S(0.0));
    bt.n.assign((long)N * F, S(0.0)); bt.dot.assign((long)N * F, S(0.0));
    bt.kpre.assign((long)N * F, S(0.0)); bt.a.assign((long)N * 3 * F, S(0.0));
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
      for (int a = 0; a < 3; ++a)
        for (int o = 0; o < F; ++o) {
          S p = S(0.0), q = S(0.0);
          for (int k = 0; k < F; ++k) {
            p += S(w.upd_U[(long)o * F + k]) * bt.v1[((long)i * 3 + a) * F + k];
            q += S(w.upd_V[(long)o * F + k]) * bt.v1[((long)i * 3 + a) * F + k];
          }
          bt.P[((long)i * 3 + a) * F + o] = p; bt.Q[((long)i * 3 + a) * F + o] = q;
        }
      for (int f = 0; f < F; ++f) {
        S q2 = S(0.0), pq = S(0.0);
        for (int a = 0; a < 3; ++a) {
          q2 += bt.Q[((long)i * 3 + a) * F + f] * bt.Q[((long)i * 3 + a) * F + f];
          pq += bt.P[((long)i * 3 + a) * F + f] * bt.Q[((long)i * 3 + a) * F + f];
        }
        bt.n[(long)i * F + f] = s_sqrt(q2 + S(m.c.eps));
        bt.dot[(long)i * F + f] = pq;
      }
      std::vector<S> kk(F);
      for (int o = 0; o < F; ++o) {                            // k = silu(upd_A1 [s'; n] + upd_c1)
        S acc = S(w.upd_c1[o]);
        for (int k = 0; k < F; ++k) acc += S(w.upd_A1[(long)o * 2 * F + k]) * bt.s1[(long)i * F + k];
        for (int k = 0; k < F; ++k) acc += S(w.upd_A1[(long)o * 2 * F + F + k]) * bt.n[(long)i * F + k];
        bt.kpre[(long)i * F + o] = acc;
        kk[o] = silu(acc);
      }
      for (int o = 0; o < 3 * F; ++o) {                        // a = upd_A2 k + upd_c2 -> (a_vv, a_sv, a_ss)
        S acc = S(w.upd_c2[o]);
        for (int k = 0; k < F; ++k) acc += S(w.upd_A2[(long)o * F + k]) * kk[k];
        bt.a[(long)i * 3 * F + o] = acc;
      }
      for (int f = 0; f < F; ++f) {
        const S avv = bt.a[(long)i * 3 * F + f], asv = bt.a[(long)i * 3 * F + F + f], ass = bt.a[(long)i * 3 * F + 2 * F + f];
        s[(long)i * F + f] = bt.s1[(long)i * F + f] + asv * bt.dot[(long)i * F + f] + ass;
        for (int a = 0; a < 3; ++a)
          v[((long)i * 3 + a) * F + f] = bt.v1[((long)i * 3 + a) * F + f] + avv * bt.P[((long)i * 3 + a) * F + f];
      }
    }
  }
  tp.s_out = s; tp.v_out = v;

  if (m.c.head_type == 1) {   // pooled graph-level head (reading Q29)
    const int d1 = m.c.d1, d2 = m.c.d2, W = 2 * d1 + 2 * d2;
    tp.pool_pre.assign((long)nS * W, S(0.0)); tp.eatom.assign(N, S(0.0)); tp.opre.clear();
    for (int g = 0; g < nS; ++g) {
      const int n = sptr[g + 1] - sptr[g];
      std::vector<S> x(F, S(0.0)), y1(d1), y2(d1), z1(d2), z2(d2);
      for (int i = sptr[g]; i < sptr[g + 1]; ++i)
        for (int f = 0; f < F; ++f) x[f] += s[(long)i * F + f];
      if (n > 0) for (int f = 0; f < F; ++f) x[f] = x[f] / S((double)n);          // mean over the structure's atoms
      S* pre = tp.pool_pre.data() + (long)g * W;
      const PoolBranch& b = m.pb[head[g]];
      for (int o = 0; o < d1; ++o) { S a = S(m.ps.b1[o]); for (int k = 0; k < F; ++k) a += S(m.ps.W1[(long)o * F + k]) * x[k]; pre[o] = a; y1[o] = silu(a); }
      for (int o = 0; o < d1; ++o) { S a = S(m.ps.b2[o]); for (int k = 0; k < d1; ++k) a += S(m.ps.W2[(long)o * d1 + k]) * y1[k]; pre[d1 + o] = a; y2[o] = silu(a); }
      for (int o = 0; o < d2; ++o) { S a = S(b.b1[o]); for (int k = 0; k < d1; ++k) a += S(b.W1[(long)o * d1 + k]) * y2[k]; pre[2 * d1 + o] = a; z1[o] = silu(a); }
      for (int o = 0; o < d2; ++o) { S a = S(b.b2[o]); for (int k = 0; k < d2; ++k) a += S(b.W2[(long)o * d2 + k]) * z1[k]; pre[2 * d1 + d2 + o] = a; z2[o] = silu(a); }
      S Eg = S(b.b3[0]);
      for (int o = 0; o < d2; ++o) Eg += S(b.w3[o]) * z2[o];
      energy[g] = Eg;
    }
    return;
  }
  // B5 readout: eps_i = out_w2 . silu(out_W1 s_i + out_b1) + out_b2 with the structure's head; E_g = sum_i eps_i
  const int Fh = F / 2;
  tp.opre.assign((long)N * Fh, S(0.0)); tp.eatom.assign(N, S(0.0));
  std::vector<int> sof(N, 0);
  for (int g = 0; g < nS; ++g) for (int i = sptr[g]; i < sptr[g + 1]; ++i) sof[i] = g;
#pragma omp parallel for schedule(static)
  for (int i = 0; i < N; ++i) {
    const Head& hd = m.head[head[sof[i]]];
    S ei = S(hd.b2[0]);
    for (int o = 0; o < Fh; ++o) {
      S acc = S(hd.b1[o]);
      for (int k = 0; k < F; ++k) acc += S(hd.W1[(long)o * F + k]) * s[(long)i * F + k];
      tp.opre[(long)i * Fh + o] = acc;
      ei += S(hd.w2[o]) * silu(acc);
    }
    tp.eatom[i] = ei;
  }
  for (int g = 0; g < nS; ++g) {                              // ascending atom order (Q21)
    S Eg = S(0.0);
    for (int i = sptr[g]; i < sptr[g + 1]; ++i) Eg += tp.eatom[i];
    energy[g] = Eg;
  }
}

// ------------------------------------------------------------------ reverse sweep (R1..R4), FP64 only
void reverse(const Model& m, int N, int nS, const int32_t* sptr, const int32_t* head, const Edges& ed,
             const Tape<double>& tp, double* forces) {
  const int F = m.c.F, K = m.c.K, T = m.c.T, Fh = F / 2;
  const double rc = m.c.rc;
  const long E = (long)ed.recv.size();
  std::vector<double> sb((long)N * F, 0.0), vb((long)N * 3 * F, 0.0);    // s-bar, v-bar
  std::vector<double> dEdd(E, 0.0), ub(3 * E, 0.0);                      // dE/dd_e, u-bar_e

  // edges grouped by sender (a counting sort of the edge list), so that the R3 scatter
  // "v-bar_j += ..., phi-bar_j += ..." can run in parallel over senders j without races.
  std::vector<int32_t> sptr_e(N + 1, 0), by_sender(E);
  for (long e = 0; e < E; ++e) sptr_e[ed.send[e] + 1]++;
  for (int i = 0; i < N; ++i) sptr_e[i + 1] += sptr_e[i];
  { std::vector<int32_t> cur(sptr_e.begin(), sptr_e.end() - 1);
    for (long e = 0; e < E; ++e) by_sender[cur[ed.send[e]]++] = (int32_t)e; }

  // R1 readout: p-bar = out_w2 . silu'(pre) ; s-bar_i = out_W1^T p-bar ; v-bar_i = 0
  std::vector<int> sof(N, 0);
  for (int g = 0; g < nS; ++g) for (int i = sptr[g]; i < sptr[g + 1]; ++i) sof[i] = g;
  if (m.c.head_type == 1) {   // pooled head: back through the branch and shared layers to x-bar_g; s-bar_i = x-bar_g / n_g
    const int d1 = m.c.d1, d2 = m.c.d2, W = 2 * d1 + 2 * d2;
    for (int g = 0; g < nS; ++g) {
      const int n = sptr[g + 1] - sptr[g];
      if (n == 0) continue;
      const double* pre = tp.pool_pre.data() + (long)g * W;
      const PoolBranch& b = m.pb[head[g]];
      std::vector<double> z2b(d2), z1b(d2), y2b(d1), y1b(d1), xb(F);
      for (int o = 0; o < d2; ++o) z2b[o] = b.w3[o] * dsilu(pre[2 * d1 + d2 + o]);
      for (int k = 0; k < d2; ++k) { double a = 0.0; for (int o = 0; o < d2; ++o) a += b.W2[(long)o * d2 + k] * z2b[o]; z1b[k] = a * dsilu(pre[2 * d1 + k]); }
      for (int k = 0; k < d1; ++k) { double a = 0.0; for (int o = 0; o < d2; ++o) a += b.W1[(long)o * d1 + k] * z1b[o]; y2b[k] = a * dsilu(pre[d1 + k]); }
      for (int k = 0; k < d1; ++k) { double a = 0.0; for (int o = 0; o < d1; ++o) a += m.ps.W2[(long)o * d1 + k] * y2b[o]; y1b[k] = a * dsilu(pre[k]); }
      for (int k = 0; k < F; ++k) { double a = 0.0; for (int o = 0; o < d1; ++o) a += m.ps.W1[(long)o * F + k] * y1b[o]; xb[k] = a; }
      for (int i = sptr[g]; i < sptr[g + 1]; ++i)
        for (int k = 0; k < F; ++k) sb[(long)i * F + k] = xb[k] / (double)n;
    }
  } else {
#pragma omp parallel for schedule(static)
  for (int i = 0; i < N; ++i) {
    const Head& hd = m.head[head[sof[i]]];
    for (int o = 0; o < Fh; ++o) {
      const double pb = hd.w2[o] * dsilu(tp.opre[(long)i * Fh + o]);
      for (int k = 0; k < F; ++k) sb[(long)i * F + k] += hd.W1[(long)o * F + k] * pb;
    }
  }
  }

  for (int t = T - 1; t >= 0; --t) {
    const Block& w = m.blk[t];
    const BlockTape<double>& bt = tp.blk[t];
    // R2 update block: (sb, vb) are s-bar'', v-bar''  ->  overwritten with s-bar', v-bar'
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
      std::vector<double> ab(3 * F), dotb(F), Pb(3 * F), Qb(3 * F), kb(F), zb(2 * F);
      for (int f = 0; f < F; ++f) {
        const double sbf = sb[(long)i * F + f];
        const double avv = bt.a[(long)i * 3 * F + f], asv = bt.a[(long)i * 3 * F + F + f];
        double avvb = 0.0;
        for (int a = 0; a < 3; ++a) avvb += vb[((long)i * 3 + a) * F + f] * bt.P[((long)i * 3 + a) * F + f];
        ab[f] = avvb; ab[F + f] = sbf * bt.dot[(long)i * F + f]; ab[2 * F + f] = sbf;
        dotb[f] = sbf * asv;
        for (int a = 0; a < 3; ++a) {
          Pb[a * F + f] = vb[((long)i * 3 + a) * F + f] * avv + dotb[f] * bt.Q[((long)i * 3 + a) * F + f];
          Qb[a * F + f] = dotb[f] * bt.P[((long)i * 3 + a) * F + f];
        }
      }
      for (int k = 0; k < F; ++k) {                            // k-bar = upd_A2^T a-bar
        double acc = 0.0;
        for (int o = 0; o < 3 * F; ++o) acc += w.upd_A2[(long)o * F + k] * ab[o];
        kb[k] = acc * dsilu(bt.kpre[(long)i * F + k]);         // times silu'(pre_k)
      }
      for (int c = 0; c < 2 * F; ++c) {                        // z-bar = upd_A1^T (k-bar . silu')
        double acc = 0.0;
        for (int o = 0; o < F; ++o) acc += w.upd_A1[(long)o * 2 * F + c] * kb[o];
        zb[c] = acc;
      }
      for (int f = 0; f < F; ++f) {
        sb[(long)i * F + f] += zb[f];                          // s-bar' = s-bar'' + z-bar[0:F]
        const double nb = zb[F + f];
        for (int a = 0; a < 3; ++a) Qb[a * F + f] += nb * bt.Q[((long)i * 3 + a) * F + f] / bt.n[(long)i * F + f];
      }
      for (int a = 0; a < 3; ++a)
        for (int k = 0; k < F; ++k) {                          // v-bar' += U^T P-bar + V^T Q-bar
          double acc = 0.0;
          for (int o = 0; o < F; ++o)
            acc += w.upd_U[(long)o * F + k] * Pb[a * F + o] + w.upd_V[(long)o * F + k] * Qb[a * F + o];
          vb[((long)i * 3 + a) * F + k] += acc;
        }
    }
    // R3 message block.  (sb, vb) are s-bar', v-bar' of the receivers.  The residual passes
    // them through to the block input; the edge terms scatter to the SENDER j.
    std::vector<double> vb_in(vb), phib((long)N * 3 * F, 0.0);
#pragma omp parallel for schedule(dynamic, 16)
    for (int j = 0; j < N; ++j) {
      std::vector<double> g(K), gp(K), wf(3 * F), dwf(3 * F);
      for (int q = sptr_e[j]; q < sptr_e[j + 1]; ++q) {
        const long e = by_sender[q];
        const int i = ed.recv[e];
        const double d = tp.d[e];
        const double dmu = (K > 1) ? rc / (K - 1) : rc, gamma = 1.0 / (2.0 * dmu * dmu);
        for (int k = 0; k < K; ++k) {
          g[k] = rbf(d, k, K, rc, m.c.rbf);
          if (m.c.rbf == 1) {  // d/dd [A sin(n pi d/rc) / d] = A (n pi/rc) cos(n pi d/rc) / d - g / d
            const double wn = (k + 1) * M_PI / rc;
            gp[k] = std::sqrt(2.0 / rc) * wn * std::cos(wn * d) / d - g[k] / d;
          } else {
            gp[k] = -2.0 * gamma * (d - k * dmu) * g[k];
          }
        }
        const double c = fcut(d, rc), cp = -(M_PI / (2.0 * rc)) * std::sin(M_PI * d / rc);
        for (int o = 0; o < 3 * F; ++o) {
          double lin = w.flt_b[o], dlin = 0.0;
          for (int k = 0; k < K; ++k) { lin += w.flt_W[(long)o * K + k] * g[k]; dlin += w.flt_W[(long)o * K + k] * gp[k]; }
          wf[o] = lin * c;                                     // w_e
          dwf[o] = c * dlin + cp * lin;                        // dw_e/dd
        }
        double dE = 0.0, ube[3] = {0.0, 0.0, 0.0};
        for (int f = 0; f < F; ++f) {
          const double* ph = &bt.phi[(long)j * 3 * F];
          const double xb_ss = sb[(long)i * F + f];
          double xb_vs = 0.0, xb_vv = 0.0;
          for (int a = 0; a < 3; ++a) {
            xb_vs += vb[((long)i * 3 + a) * F + f] * tp.u[3 * e + a];
            xb_vv += vb[((long)i * 3 + a) * F + f] * bt.v_in[((long)j * 3 + a) * F + f];
          }
          const double x_vs = ph[F + f] * wf[F + f], x_vv = ph[2 * F + f] * wf[2 * F + f];
          for (int a = 0; a < 3; ++a) {
            vb_in[((long)j * 3 + a) * F + f] += vb[((long)i * 3 + a) * F + f] * x_vv;   // v-bar_j += v-bar'_i . x^vv
            ube[a] += vb[((long)i * 3 + a) * F + f] * x_vs;                             // u-bar_e
          }
          phib[(long)j * 3 * F + f] += xb_ss * wf[f];                                   // phi-bar_j += x-bar . w
          phib[(long)j * 3 * F + F + f] += xb_vs * wf[F + f];
          phib[(long)j * 3 * F + 2 * F + f] += xb_vv * wf[2 * F + f];
          dE += xb_ss * ph[f] * dwf[f] + xb_vs * ph[F + f] * dwf[F + f] + xb_vv * ph[2 * F + f] * dwf[2 * F + f];
        }
        dEdd[e] += dE;
        for (int a = 0; a < 3; ++a) ub[3 * e + a] += ube[a];
      }
    }
    vb.swap(vb_in);
#pragma omp parallel for schedule(static)
    for (int j = 0; j < N; ++j) {                              // h-bar = msg_W2^T phi-bar ; s-bar += msg_W1^T (h-bar . silu')
      std::vector<double> hb(F);
      for (int k = 0; k < F; ++k) {
        double acc = 0.0;
        for (int o = 0; o < 3 * F; ++o) acc += w.msg_W2[(long)o * F + k] * phib[(long)j * 3 * F + o];
        hb[k] = acc * dsilu(bt.hpre[(long)j * F + k]);
      }
      for (int k = 0; k < F; ++k) {
        double acc = 0.0;
        for (int o = 0; o < F; ++o) acc += w.msg_W1[(long)o * F + k] * hb[o];
        sb[(long)j * F + k] += acc;
      }
    }
  }
  // R4 geometry: G_e = dE/dd u + (u-bar - (u-bar.u) u)/d ; dE/dx_j += G_e ; dE/dx_i -= G_e ; F = -dE/dx
  std::vector<double> gx((long)N * 3, 0.0);
  for (long e = 0; e < E; ++e) {
    const int i = ed.recv[e], j = ed.send[e];
    const double* u = &tp.u[3 * e];
    const double ubu = ub[3 * e] * u[0] + ub[3 * e + 1] * u[1] + ub[3 * e + 2] * u[2];
    for (int a = 0; a < 3; ++a) {
      const double G = dEdd[e] * u[a] + (ub[3 * e + a] - ubu * u[a]) / tp.d[e];
      gx[(long)j * 3 + a] += G;
      gx[(long)i * 3 + a] -= G;
    }
  }
  for (long q = 0; q < (long)N * 3; ++q) forces[q] = -gx[q];
}

Cfg make_cfg(const int32_t* ic, const double* dc) {
  return Cfg{ic[0], ic[1], ic[2], ic[3], ic[4], dc[0], dc[1], ic[5], ic[6], ic[7], ic[8], ic[9], ic[10], ic[11]};
}

}  // namespace

// ================================================================== C interface (host pointers)
extern "C" {

// Number of scalars in the weight blob.
int64_t oracle_weights_count(const int32_t* icfg /*F,T,K,H,Zmax*/) {
  double dc[2] = {1.0, 0.0};
  return parse_blob(make_cfg(icfg, dc), nullptr, nullptr);
}

// B1 only.  Pass 1: call with recv == NULL to get the edge count.  Pass 2: fill arrays.
int64_t oracle_neighbours_images(int32_t N, int32_t S, const double* pos, const int32_t* sptr, const double* cell,
                                 const uint8_t* pbc, double rc, int32_t all_images, int32_t* rowptr, int32_t* recv,
                                 int32_t* send, int8_t* shift, double* rvec);
int64_t oracle_neighbours(int32_t N, int32_t S, const double* pos, const int32_t* sptr, const double* cell,
                          const uint8_t* pbc, double rc, int32_t* rowptr, int32_t* recv, int32_t* send,
                          int8_t* shift, double* rvec) {
  return oracle_neighbours_images(N, S, pos, sptr, cell, pbc, rc, 0, rowptr, recv, send, shift, rvec);
}
int64_t oracle_neighbours_capped(int32_t N, int32_t S, const double* pos, const int32_t* sptr, const double* cell,
                                 const uint8_t* pbc, double rc, int32_t all_images, int32_t max_nb, int32_t* rowptr,
                                 int32_t* recv, int32_t* send, int8_t* shift, double* rvec);
int64_t oracle_neighbours_images(int32_t N, int32_t S, const double* pos, const int32_t* sptr, const double* cell,
                                 const uint8_t* pbc, double rc, int32_t all_images, int32_t* rowptr, int32_t* recv,
                                 int32_t* send, int8_t* shift, double* rvec) {
  return oracle_neighbours_capped(N, S, pos, sptr, cell, pbc, rc, all_images, 0, rowptr, recv, send, shift, rvec);
}
int64_t oracle_neighbours_capped(int32_t N, int32_t S, const double* pos, const int32_t* sptr, const double* cell,
                                 const uint8_t* pbc, double rc, int32_t all_images, int32_t max_nb, int32_t* rowptr,
                                 int32_t* recv, int32_t* send, int8_t* shift, double* rvec) {
  Edges ed;
  neighbours(N, S, pos, sptr, cell, pbc, rc, &ed, all_images, max_nb);
  const int64_t E = (int64_t)ed.recv.size();
  if (rowptr) std::memcpy(rowptr, ed.rowptr.data(), sizeof(int32_t) * (N + 1));
  if (recv) {
    std::memcpy(recv, ed.recv.data(), sizeof(int32_t) * E);
    std::memcpy(send, ed.send.data(), sizeof(int32_t) * E);
    if (shift) std::memcpy(shift, ed.shift.data(), 3 * E);
    if (rvec)
      for (int64_t e = 0; e < E; ++e)
        for (int b = 0; b < 3; ++b)
          rvec[3 * e + b] = pos[3 * ed.send[e] + b] - pos[3 * ed.recv[e] + b] + ed.shift_cart[3 * e + b];
  }
  return E;
}

// Full path.  energy [S]; forces [N][3] or NULL; optional outputs s_out [N][F], v_out [N][3][F],
// eatom [N] (may be NULL).  Returns the number of directed edges.
int64_t oracle_eval_glob(const int32_t* icfg, const double* dcfg, const double* weights, int32_t N, int32_t S,
                         const int32_t* Z, const double* pos, const int32_t* sptr, const double* cell, const uint8_t* pbc,
                         const int32_t* head, const double* glob, double* energy, double* forces, double* s_out,
                         double* v_out, double* eatom);
int64_t oracle_eval(const int32_t* icfg, const double* dcfg /*cutoff, eps*/, const double* weights, int32_t N,
                    int32_t S, const int32_t* Z, const double* pos, const int32_t* sptr, const double* cell,
                    const uint8_t* pbc, const int32_t* head, double* energy, double* forces, double* s_out,
                    double* v_out, double* eatom) {
  return oracle_eval_glob(icfg, dcfg, weights, N, S, Z, pos, sptr, cell, pbc, head, nullptr, energy, forces, s_out, v_out,
                          eatom);
}
// glob [S][n_glob] (host) or NULL: the structures' global attributes (charge, spin)
int64_t oracle_eval_glob(const int32_t* icfg, const double* dcfg, const double* weights, int32_t N, int32_t S,
                         const int32_t* Z, const double* pos, const int32_t* sptr, const double* cell, const uint8_t* pbc,
                         const int32_t* head, const double* glob, double* energy, double* forces, double* s_out,
                         double* v_out, double* eatom) {
  Model m;
  parse_blob(make_cfg(icfg, dcfg), weights, &m);
  Edges ed;
  neighbours(N, S, pos, sptr, cell, pbc, m.c.rc, &ed, m.c.images, m.c.max_nb);
  Tape<double> tp;
  forward<double>(m, N, S, Z, pos, sptr, head, ed, tp, energy, glob);
  if (s_out) std::memcpy(s_out, tp.s_out.data(), sizeof(double) * tp.s_out.size());
  if (v_out) std::memcpy(v_out, tp.v_out.data(), sizeof(double) * tp.v_out.size());
  if (eatom) std::memcpy(eatom, tp.eatom.data(), sizeof(double) * N);
  if (forces) reverse(m, N, S, sptr, head, ed, tp, forces);
  return (int64_t)ed.recv.size();
}

// Forces by forward-mode dual numbers: one forward evaluation per coordinate, seeding
// d x_{i,a} = 1.  Independent of the hand-written reverse sweep.  Small inputs only (3N forwards).
// The edge list is held fixed (built from the values), as it is for the analytic gradient.
void oracle_forces_dual(const int32_t* icfg, const double* dcfg, const double* weights, int32_t N, int32_t S,
                        const int32_t* Z, const double* pos, const int32_t* sptr, const double* cell,
                        const uint8_t* pbc, const int32_t* head, double* forces) {
  Model m;
  parse_blob(make_cfg(icfg, dcfg), weights, &m);
  Edges ed;
  neighbours(N, S, pos, sptr, cell, pbc, m.c.rc, &ed, m.c.images, m.c.max_nb);
  std::vector<int> sof(N);
  for (int g = 0; g < S; ++g) for (int i = sptr[g]; i < sptr[g + 1]; ++i) sof[i] = g;
#pragma omp parallel for schedule(dynamic, 1)
  for (int q = 0; q < 3 * N; ++q) {
    std::vector<Dual> x(3 * (long)N), en(S);
    for (long c = 0; c < 3L * N; ++c) x[c] = Dual(pos[c], c == q ? 1.0 : 0.0);
    Tape<Dual> tp;
    forward<Dual>(m, N, S, Z, x.data(), sptr, head, ed, tp, en.data());
    forces[q] = -en[sof[q / 3]].d;
  }
}

// Radial basis and cutoff envelope alone (for the closed-form pins): g [K], c [1].
void oracle_rbf_cutoff(double d, int32_t K, double rc, double* g, double* c) {
  for (int k = 0; k < K; ++k) g[k] = rbf<double>(d, k, K, rc);
  *c = fcut<double>(d, rc);
}
void oracle_rbf_cutoff_typed(double d, int32_t K, double rc, int32_t type, double* g, double* c) {
  for (int k = 0; k < K; ++k) g[k] = rbf<double>(d, k, K, rc, type);
  *c = fcut<double>(d, rc);
}

}  // extern "C"
