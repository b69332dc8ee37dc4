/* include/pnn.h — C ABI of the B200-native batched PaiNN energy+force library (libpnn.so).
 *
 * The path (the paper names the backbone and the problem only:
 * PAPER.md:147 "PaiNN" [48], PAPER.md:53 forces = energy gradients w.r.t. positions,
 * PAPER.md:126/232 shared trunk + 16 per-dataset heads, PAPER.md:229-231 radial basis / cutoff,
 * PAPER.md:269 periodic boundary conditions, PAPER.md:172 BF16/FP32/FP64):
 *
 *   (Z, positions, optional cell/PBC, per-structure head index, weights, precision)
 *        -> (per-structure energy, per-atom forces = -dE/dx)
 *
 * Conventions
 *   - Every function returns int: 0 = PNN_OK, < 0 = error (pnn_status_string()).  No exceptions, no aborts.
 *   - "DEVICE" pointers are CUDA device pointers owned by the caller (e.g. torch allocations); the library
 *     never frees them and does not use them after the stream work of the call has run.  "HOST" pointers are
 *     ordinary host memory, read or written synchronously inside the call.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls only enqueue work and do
 *     not synchronise unless stated.
 *   - Atoms of a structure are contiguous: struct_ptr[0] = 0, struct_ptr[S] = N.  Units: Angstrom; energies in
 *     the (arbitrary) units of the weights.  Positions are FP64 at the boundary for every model precision so
 *     that the cutoff predicate is evaluated in FP64 (bit-exact edge sets).
 *   - Row-major everywhere.  Weight blob: flat FP64, matrices [out][in], y = W x + b, in the order
 *       emb[Zmax+1][F] (row 0 unused)
 *       per block t: msg_W1[F][F] msg_b1[F] msg_W2[3F][F] msg_b2[3F] flt_W[3F][K] flt_b[3F]
 *                    upd_U[F][F] upd_V[F][F] upd_A1[F][2F] upd_c1[F] upd_A2[3F][F] upd_c2[3F]
 *       per head h:  out_W1[F/2][F] out_b1[F/2] out_w2[F/2] out_b2[1]
 *     3F chunks: rows [0,F) scalar (ss), [F,2F) direction (vs), [2F,3F) vector (vv); upd_A2 rows
 *     [0,F) a_vv, [F,2F) a_sv, [2F,3F) a_ss.
 */
#ifndef PNN_H_
#define PNN_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PNN_OK 0
#define PNN_ERR_INVALID_ARG (-1) /* null pointer, negative size, F not a multiple of 32 or > 256, K > 32 ...  */
#define PNN_ERR_CAPACITY (-2)    /* N / E / S exceed what the workspace was created for                        */
#define PNN_ERR_CUDA (-3)        /* a CUDA runtime call failed; pnn_last_cuda_error() has the text             */
#define PNN_ERR_UNSUPPORTED (-4) /* feature not available in this build / for this precision                   */
#define PNN_ERR_NO_GRAPH (-5)    /* pnn_eval called before pnn_build_graph for these sizes                     */
#define PNN_ERR_BAD_INPUT (-6)   /* device-side check failed: Z outside [1,Zmax] or head outside [0,H)         */

typedef enum { PNN_BF16 = 0, PNN_FP32 = 1, PNN_FP64 = 2 } pnn_precision;

/* F feature width (multiple of 32, 32..256), T interaction blocks, K radial basis functions (<= 32) of type rbf,
 * H heads, Zmax largest atomic number, cutoff r_c [A], norm_eps the epsilon under the sqrt of the update block. */
#define PNN_IMAGES_MINIMUM 0 /* one (nearest) periodic image per ordered pair: exact only for cells >= 2 r_c wide        */
#define PNN_IMAGES_ALL 1     /* every periodic image inside the cutoff, an atom's own images included (narrow cells)     */
#define PNN_RBF_GAUSSIAN 0 /* g_k(d) = exp(-gamma (d - k r_c/(K-1))^2), gamma = (K-1)^2 / (2 r_c^2), k = 0..K-1 (2 <= K) */
#define PNN_RBF_BESSEL 1   /* b_n(d) = sqrt(2/r_c) sin(n pi d / r_c) / d, n = 1..K (the lead model's basis)  */
#define PNN_HEAD_ATOMWISE 0 /* per-atom readout MLP of the structure's head, summed over the atoms      */
#define PNN_BACKBONE_PAINN 0
#define PNN_BACKBONE_SCHNET 1
#define PNN_HEAD_POOLED 1   /* mean pooling, shared layers, per-head branch layers (the paper's graph-level heads)         */
typedef struct {
  int32_t F, T, K, H, Zmax;
  double cutoff;
  double norm_eps;
  int32_t prec; /* pnn_precision */
  int32_t rbf;  /* PNN_RBF_GAUSSIAN or PNN_RBF_BESSEL; both are multiplied by the cosine cutoff */
  int32_t pbc_images; /* PNN_IMAGES_MINIMUM or PNN_IMAGES_ALL (pnn_build_graph) */
  int32_t max_neighbors; /* 0 = every sender inside the cutoff; k > 0 = each receiver keeps its k NEAREST senders (the
                            paper's "Max neighbors": 20 in Table V; 64 with PBC).  Smallest FP64
                            squared distance first, ties by sender index, then lattice shift.  The edge set is then not
                            symmetric: the reverse sweep runs its scatter form (atomic adds; edge_scatter.cu) instead of
                            the gather form, and max_edges still bounds the UNCAPPED edge count of a batch. */
  int32_t n_global; /* global attributes per structure entering the embedding ("global attributes such as charge
                       and spin used as additional input features"; reading Q30): 0 = none; G > 0 appends
                       glob_W[F][G] to the weight blob, s0_i = emb[Z_i] + glob_W . attributes of the atom's structure
                       (pnn_set_globals). */
  int32_t head_type; /* PNN_HEAD_ATOMWISE (0): E_g = sum_i MLP_h(s_i), the blob's heads as listed above.
                        PNN_HEAD_POOLED (1): the paper's graph-level heads ("Output heads 16 (graph-level)",
                        "2 shared layers (dim 50) + 2 branch layers (dim 776)"; reading Q29): x_g = mean_i s_i,
                        y = silu(P2 silu(P1 x_g + p1) + p2), z = silu(B2_h silu(B1_h y + q1_h) + q2_h), E_g = w3_h . z + q3_h.
                        The blob then holds, in place of the atom-wise heads: P1[d1][F] p1[d1] P2[d1][d1] p2[d1], then per
                        head B1[d2][d1] q1[d2] B2[d2][d2] q2[d2] w3[d2] q3[1].  pnn_eval_blended returns PNN_ERR_UNSUPPORTED
                        for such a model. */
  int32_t head_d1;   /* pooled head: width of the two shared layers (paper: 50); ignored for atom-wise heads */
  int32_t head_d2;   /* pooled head: width of the two branch layers (paper: 776) */
  int32_t backbone;  /* PNN_BACKBONE_PAINN (0) or PNN_BACKBONE_SCHNET (1): the second backbone on the same graph (PAPER.md:147,
                        212: SchNet is one of the six backbones of the paper's search; reading Q31).  Per block
                        W_e = (F2 silu(F1 g(d_e) + f1) + f2) c(d_e), m_i = sum_{e=(i<-j)} (A x_j) o W_e,
                        x_i += B2 silu(B1 m_i + b1) + b2; same embedding, radial basis, cutoff and atom-wise heads.  The blob then
                        holds per block flt_W1[F][K] flt_b1[F] flt_W2[F][F] flt_b2[F] in_W[F][F] out_W1[F][F] out_b1[F]
                        out_W2[F][F] out_b2[F] in place of the PaiNN block arrays.  PNN_FP32 / PNN_FP64 only; no neighbour cap,
                        global attributes, pooled heads or blended evaluation (PNN_ERR_UNSUPPORTED / PNN_ERR_INVALID_ARG). */
} pnn_config;

typedef struct pnn_model pnn_model;         /* opaque; owns device copies of the weights in model precision */
typedef struct pnn_workspace pnn_workspace; /* opaque; owns CSR graph, activations and adjoints             */

/* Number of FP64 scalars in the weight blob for this configuration (layout above). */
int pnn_weights_count(const pnn_config* cfg, int64_t* n_scalars);

/* Uploads (and converts / transposes) the weights.  weights_host: HOST, FP64, n_scalars must equal
 * pnn_weights_count().  Synchronous. */
int pnn_model_create(const pnn_config* cfg, const double* weights_host, int64_t n_scalars, pnn_model** out);
void pnn_model_destroy(pnn_model* m);

/* Allocates all device memory needed for batches of up to max_atoms atoms, max_edges directed edges and
 * max_structs structures.  want_forces: 0, or PNN_WS_FORCES (also allocates the per-block tape and the adjoint buffers of
 * the reverse sweep), optionally | PNN_WS_NO_EDGE_TAPE.  A PNN_FP32 model with forces keeps an EDGE
 * TAPE (filter value and its derivative of every edge, feature and block: 24 F T bytes per edge of max_edges) that the
 * reverse edge kernel streams back instead of recomputing the filter; PNN_WS_NO_EDGE_TAPE trades that memory for about 3x
 * slower edge kernels of the reverse sweep.  If the tape (or anything else) cannot be allocated the call fails with
 * PNN_ERR_CUDA: the library never changes kernels silently.  Any other bit in want_forces: PNN_ERR_INVALID_ARG.
 * Synchronous. */
#define PNN_WS_FORCES 1
#define PNN_WS_NO_EDGE_TAPE 2
int pnn_workspace_create(const pnn_model* m, int64_t max_atoms, int64_t max_edges, int64_t max_structs,
                         int want_forces, pnn_workspace** out);
void pnn_workspace_destroy(pnn_workspace* ws);
/* Bytes of device memory the workspace holds (the edge tape included), and the bytes of the edge tape alone (0: none). */
int64_t pnn_workspace_bytes(const pnn_workspace* ws);
int64_t pnn_workspace_edge_tape_bytes(const pnn_workspace* ws);

/* a1 — radius graph (PAPER.md:230 cutoff, PAPER.md:269 PBC).  All ordered pairs (i, j),
 * i != j, in the same structure, with |x_j - x_i + shift.C| < r_c (strict, FP64); under PBC the shift is the
 * per-axis minimum-image rounding of the fractional difference (PNN_IMAGES_MINIMUM), or every shift that satisfies the
 * predicate, pairs i == j with a non-zero shift included (PNN_IMAGES_ALL; several edges per ordered pair then).  Built by a cell list (cells >= r_c wide; a
 * structure narrower than 3 cells along an axis uses one cell on that axis) and emitted as receiver-sorted CSR
 * held inside the workspace, together with the per-edge unit vector and distance in model precision.
 *   pos        DEVICE [N,3] f64        struct_ptr DEVICE [S+1] i32
 *   cell       DEVICE [S,3,3] f64 (rows = lattice vectors) or NULL    pbc DEVICE [S,3] u8 or NULL
 * Edge overflow (E > max_edges) is detected on the device and reported by pnn_check_async_errors /
 * pnn_graph_view / pnn_eval_host (PNN_ERR_CAPACITY); a truncated graph is never evaluated: until the next pnn_build_graph
 * the edge kernels of pnn_eval do nothing, and once the overflow has been reported pnn_eval returns PNN_ERR_NO_GRAPH.
 * Asynchronous. */
int pnn_build_graph(pnn_workspace* ws, int64_t n_atoms, int64_t n_structs, const double* pos,
                    const int32_t* struct_ptr, const double* cell, const uint8_t* pbc, void* cuda_stream);

/* DEVICE views of the last graph: rowptr [N+1] i32 (receiver i owns edges rowptr[i]..rowptr[i+1]), col [E] i32
 * (global sender index), shift [E,3] i8 (integer lattice shift of the sender image).  *n_edges is a host value:
 * this call synchronises the stream of the last pnn_build_graph.  Any out pointer may be NULL. */
int pnn_graph_view(const pnn_workspace* ws, const int32_t** rowptr, const int32_t** col, const int8_t** shift,
                   int64_t* n_edges);

/* Copies the last graph into caller-owned buffers (HOST or DEVICE, sized from pnn_graph_view's n_edges):
 * rowptr [N+1] i32, col [E] i32, shift [E,3] i8.  Any pointer may be NULL.  Synchronous. */
int pnn_graph_copy(const pnn_workspace* ws, int32_t* rowptr, int32_t* col, int8_t* shift);

/* The radius graph WITHOUT any allocation — for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it): no model, no workspace.  Same builder and same result as pnn_build_graph (cell
 * list, strict d < cutoff in FP64, receiver-sorted CSR, bit-identical rowptr / col / shift), but every scratch array of the
 * build (cell lists, scan buffers, per-edge geometry) lives in ONE file-scope static device array of
 * PNN_STATIC_SCRATCH_BYTES inside the library, which every GPU that loads libpnn.so holds until the process exits.  Limits,
 * rejected with PNN_ERR_CAPACITY (pnn_last_cuda_error() then names the argument and the limit): n_atoms <=
 * PNN_STATIC_MAX_ATOMS, n_structs <= PNN_STATIC_MAX_STRUCTS, max_edges <= PNN_STATIC_MAX_EDGES.
 *   pos, struct_ptr, cell, pbc: DEVICE, as pnn_build_graph.  pbc_images: PNN_IMAGES_MINIMUM or PNN_IMAGES_ALL.
 *   rowptr [n_atoms+1] i32, col [max_edges] i32, shift [max_edges,3] i8: DEVICE, caller-owned OUTPUTS; rowptr[n_atoms] is the
 *   number of directed edges.  flags: DEVICE i32 [1] output or NULL: 0, or PNN_STATIC_EDGE_OVERFLOW when the graph has more
 *   than max_edges edges (rowptr is then still complete, col / shift are unspecified).
 * Asynchronous on cuda_stream; calls no cudaMalloc / cudaFree or allocating routine.  The address of the static array is
 * resolved once per device, on the first call made with that device current (make that call outside graph capture).  ALL
 * calls share the array: calls that overlap on the GPU (different streams, or another host thread's call on the same
 * device) race; issue them on one stream or order them with events.  The array keeps the previous call's contents; what
 * must start at zero is cleared on the stream by every call. */
#define PNN_STATIC_MAX_ATOMS 16384
#define PNN_STATIC_MAX_STRUCTS 4096
#define PNN_STATIC_MAX_EDGES 262144
#define PNN_STATIC_SCRATCH_BYTES (6 * 1024 * 1024)
#define PNN_STATIC_EDGE_OVERFLOW 1
int pnn_build_graph_static(int64_t n_atoms, int64_t n_structs, const double* pos, const int32_t* struct_ptr,
                           const double* cell, const uint8_t* pbc, double cutoff, int32_t pbc_images, int64_t max_edges,
                           int32_t* rowptr, int32_t* col, int8_t* shift, int32_t* flags, void* cuda_stream);

#define PNN_ENERGY 1
#define PNN_FORCES 2

/* a2..a7 — embedding, T x (message, update), multi-head readout, and (with PNN_FORCES) the analytic reverse
 * sweep.  Uses the graph last built in the workspace, which must have been built for
 * the same n_atoms and n_structs (PNN_ERR_NO_GRAPH at once otherwise) and the same pos: pos DEVICE [N,3] f64 is
 * checksummed on the device against the positions pnn_build_graph saw, and a mismatch (atoms moved without a rebuild)
 * is reported as PNN_ERR_NO_GRAPH by pnn_check_async_errors; the results of that call are then undefined.
 *   Z DEVICE [N] i32 in [1,Zmax]     head DEVICE [S] i32 in [0,H)
 *   energy DEVICE [S], forces DEVICE [N,3]: f64 for a PNN_FP64 model, f32 for PNN_FP32 and PNN_BF16.
 *   forces may be NULL unless flags has PNN_FORCES (which needs a workspace created with want_forces).
 * Asynchronous. */
int pnn_eval(const pnn_model* m, pnn_workspace* ws, int64_t n_atoms, int64_t n_structs, const int32_t* Z,
             const double* pos, const int32_t* struct_ptr, const int32_t* head, int flags, void* energy,
             void* forces, void* cuda_stream);

/* pnn_build_graph + pnn_eval as ONE replayed CUDA graph, for loops that evaluate the same (n_atoms, n_structs) again and again
 * with positions updated IN PLACE (molecular dynamics, relaxations; small batches are bound by launch overhead: ~60-110
 * launches per evaluation).  Every launch geometry of the path depends on n_atoms / n_structs only (the edge count lives on
 * the device), so the recorded sequence stays valid when the atoms move.  The first call with a new signature — sizes, flags,
 * stream and every pointer argument — and the one after it run the path eagerly (kernel attributes are set then), the third
 * records it into a CUDA graph on an internal stream, and from then on a call is one cudaGraphLaunch on cuda_stream.  Arguments and error behaviour
 * as pnn_build_graph and pnn_eval; the edge-overflow / bad-input / stale-graph flags are still reported by
 * pnn_check_async_errors.  A different signature drops the recorded graph and starts over.  Not available while
 * pnn_profile_enable is on (PNN_ERR_UNSUPPORTED).  Asynchronous. */
int pnn_eval_replay(const pnn_model* m, pnn_workspace* ws, int64_t n_atoms, int64_t n_structs, const int32_t* Z,
                    const double* pos, const int32_t* struct_ptr, const int32_t* head, const double* cell,
                    const uint8_t* pbc, int flags, void* energy, void* forces, void* cuda_stream);

/* Global attributes of the structures of the NEXT evaluations of this workspace (pnn_config.n_global = G > 0): glob DEVICE
 * [n_structs, G] f64 (e.g. total charge, spin multiplicity), read by pnn_eval / pnn_eval_blended when they run — the buffer
 * stays owned by the caller and must stay valid until then; NULL = all attributes zero.  PNN_ERR_INVALID_ARG when the model
 * has n_global = 0 and glob is not NULL.  pnn_eval_host and the streaming driver evaluate with zero attributes. */
int pnn_set_globals(pnn_workspace* ws, int64_t n_structs, const double* glob);

/* Blended multi-head evaluation — the paper's inference pipeline (PAPER.md:166-168 branch weights, :371-373 "encoder
 * reuse", "branch skipping", "fused gradient", Fig. 5 at :420): the shared trunk runs ONCE, every
 * structure g is read out by all heads h with head_weights[g][h] >= skip_below, E_g = sum_h w[g][h] E_g^(h), and ONE
 * reverse sweep gives forces = -dE/dx of that blended energy.  head_weights DEVICE [S,H], f64 for a PNN_FP64 model, f32
 * otherwise (in the paper: a softmax over a composition MLP; here an input).  Other arguments, graph requirement and
 * error behaviour as pnn_eval.  Asynchronous. */
int pnn_eval_blended(const pnn_model* m, pnn_workspace* ws, int64_t n_atoms, int64_t n_structs, const int32_t* Z,
                     const double* pos, const int32_t* struct_ptr, const void* head_weights, double skip_below,
                     int flags, void* energy, void* forces, void* cuda_stream);

/* Composition-conditioned branch weights ("the MLP maps the structure's chemical-composition vector
 * to softmax weights that blend these branch outputs"; "24,500 parameters ... per-element
 * chemical-composition vectors ... softmax-normalized"; reading Q28 for what the paper leaves open):
 *   c_z = (atoms of the structure with atomic number z) / (atoms of the structure), z = 1..widths[0] (c = 0 if empty);
 *   x <- SiLU(W_l x + b_l) for the hidden layers, the last layer linear; w = softmax over the widths[n_layers] heads.
 * pnn_branch_mlp_create: widths HOST [n_layers+1] (1 <= n_layers <= 8, every width in [1,256]); params HOST f64,
 * per layer W [out,in] row-major then b [out], n_params = sum(out*in + out) (PNN_ERR_INVALID_ARG otherwise); copied to
 * the device in FP64 (prec = PNN_FP64) or FP32 (PNN_FP32, PNN_BF16: the router is never evaluated in BF16).  The caller
 * owns *out and frees it with pnn_branch_mlp_destroy. */
typedef struct pnn_branch_mlp pnn_branch_mlp;
int pnn_branch_mlp_create(int32_t n_layers, const int32_t* widths, const double* params, int64_t n_params, int prec,
                          pnn_branch_mlp** out);
void pnn_branch_mlp_destroy(pnn_branch_mlp* b);

/* head_weights[g][h], DEVICE [S, widths[n_layers]] (f64 for a PNN_FP64 router, f32 otherwise) — the array
 * pnn_eval_blended takes.  Z DEVICE [N] i32, struct_ptr DEVICE [S+1] i32.  An atomic number outside [1, widths[0]] is
 * left out of the counts and sets the workspace's bad-input flag (pnn_check_async_errors -> PNN_ERR_BAD_INPUT).  The
 * workspace is used for that flag and the launch count only; no graph is needed.  Asynchronous. */
int pnn_branch_weights(const pnn_branch_mlp* b, pnn_workspace* ws, int64_t n_atoms, int64_t n_structs,
                       const int32_t* Z, const int32_t* struct_ptr, void* head_weights, void* cuda_stream);

/* Convenience for callers with HOST buffers (bench.py's e2e leg): copies Z, pos, struct_ptr, head (and cell /
 * pbc when not NULL) to the device, runs pnn_build_graph + pnn_eval and copies energy [S] / forces [N,3] back.
 * energy_host / forces_host have the dtype pnn_eval documents.  Device-side errors of the call (edge overflow, bad Z /
 * head) are returned by the call itself.  When consecutive calls on a workspace have the same n_atoms and n_structs the
 * device part is replayed as one CUDA graph (pnn_eval_replay on the workspace's staging buffers; not while profiling is
 * on); the streaming driver inherits this for batches of a fixed shape.  Synchronous. */
int pnn_eval_host(const pnn_model* m, pnn_workspace* ws, int64_t n_atoms, int64_t n_structs, const int32_t* Z,
                  const double* pos, const int32_t* struct_ptr, const int32_t* head, const double* cell,
                  const uint8_t* pbc, int flags, void* energy_host, void* forces_host, void* cuda_stream);

/* Streaming driver for screening runs ("1.1 billion atomistic structures in 50 seconds", the per-GPU
 * throughput of PAPER.md:422-426; BASELINE.json configs[3]: 1,048,576 structures "streamed in batches of 16,384";
 * SURVEY.md §7 step 8): `depth` pipeline slots, each with its own workspace, staging buffers and CUDA stream, so that the
 * host-to-device copies of batch k+1 and the device-to-host copies of batch k-1 overlap the kernels of batch k.
 *   pnn_stream_create  flags = PNN_ENERGY [| PNN_FORCES] for every batch; sizes are per batch; 1 <= depth <= 8
 *                      (2 = double buffering).  Device memory: depth workspaces (pnn_stream_bytes).
 *   pnn_stream_submit  enqueues one batch (arguments as pnn_eval_host, all HOST pointers; pinned memory is needed for the
 *                      copies to overlap) into slot (number of batches submitted so far) mod depth and returns without
 *                      waiting for it; the input and output buffers must stay valid and untouched until the batch has been
 *                      waited for.  If that slot still holds an unfinished batch the call first waits for it, and a device
 *                      error of THAT batch is what it returns.
 *   pnn_stream_wait    blocks until the oldest batch not yet waited for is complete (its energy_host / forces_host are
 *                      then valid) and returns its device-side status (PNN_ERR_CAPACITY, PNN_ERR_BAD_INPUT); PNN_OK when
 *                      nothing is in flight.
 *   pnn_stream_drain   waits for everything in flight; returns the first error.
 * Results are bit-identical to pnn_eval_host on the same batch (same kernels, same launch configuration). */
typedef struct pnn_stream pnn_stream;
int pnn_stream_create(const pnn_model* m, int64_t max_atoms, int64_t max_edges, int64_t max_structs, int flags,
                      int depth, pnn_stream** out);
void pnn_stream_destroy(pnn_stream* s);
int pnn_stream_submit(pnn_stream* s, int64_t n_atoms, int64_t n_structs, const int32_t* Z, const double* pos,
                      const int32_t* struct_ptr, const int32_t* head, const double* cell, const uint8_t* pbc,
                      void* energy_host, void* forces_host);
int pnn_stream_wait(pnn_stream* s);
int pnn_stream_drain(pnn_stream* s);
int64_t pnn_stream_launch_count(const pnn_stream* s); /* kernels launched on behalf of the stream so far */
int64_t pnn_stream_bytes(const pnn_stream* s);        /* device memory held by its workspaces          */

/* Reads the device error flags (edge overflow -> PNN_ERR_CAPACITY, positions changed since pnn_build_graph ->
 * PNN_ERR_NO_GRAPH, bad Z / head -> PNN_ERR_BAD_INPUT) and clears them.  Synchronises the device. */
int pnn_check_async_errors(pnn_workspace* ws);

/* Optional per-kernel-family timing: when enabled, pnn_build_graph / pnn_eval bracket each kernel family with CUDA
 * events on the launch stream.  pnn_profile_read synchronises the device, aggregates the records since the last
 * read by family name (names: max_entries x 32 bytes, NUL-padded; total_ms; launches) and clears them. */
int pnn_profile_enable(pnn_workspace* ws, int on);
int pnn_profile_read(pnn_workspace* ws, int max_entries, char* names, double* total_ms, int64_t* launches,
                     int* n_entries);

/* The BF16 node contraction on its own (a3 / a5 building block; also used by the tests and bench.py to measure the
 * tensor pipe): C[M,N] = act( A[M,K] . Wt[N,K]^T + bias ), A / Wt DEVICE BF16 row-major with row strides lda / ldw
 * (elements), FP32 accumulation on tcgen05 tensor cores.  bias DEVICE f32 [N] or NULL; act 0 = none, 1 = SiLU.
 * C DEVICE f32 (row stride ldc) and / or Cb DEVICE bf16 (row stride ldcb); either may be NULL.  N and K multiples of
 * 32, lda / ldw / ldcb multiples of 8, ldc a multiple of 4, all base pointers 16-byte aligned (PNN_ERR_INVALID_ARG
 * otherwise).  Asynchronous. */
int pnn_gemm_bf16(int64_t M, int32_t N, int32_t K, const void* A, int64_t lda, const void* Wt, int64_t ldw,
                  const float* bias, int32_t act, float* C, int64_t ldc, void* Cb, int64_t ldcb, void* cuda_stream);

/* Measured peak of the plain FMA pipe in TFLOP/s (the ALU roofs of the FP32 / FP64 edge kernels and
 * GEMMs "must be measured on the box by a small FMA micro-benchmark"): independent register FMA chains, packed
 * fma.rn.f32x2 for PNN_FP32 and DFMA for PNN_FP64, best of five launches timed with CUDA events.  *tflops is a host
 * value.  PNN_BF16 -> PNN_ERR_INVALID_ARG (its roofs are HBM and the tensor pipe).  Synchronous. */
int pnn_measure_alu_peak(int prec, double* tflops, void* cuda_stream);

/* Measured bandwidth of L2-resident reads in GB/s: a 32 MB buffer (a quarter of the L2, far larger than L1) streamed by
 * every CTA in 512-byte rows per warp, the access shape of the edge kernels' sender-row gathers; best of five launches
 * timed with CUDA events.  Context for the gather-bound edge kernels (cfg3: 61 neighbours per atom, the sender rows live
 * in L2, and SURVEY.md 8(d)'s HBM roof says little about them).  *gbs is a host value.  Synchronous; allocates and frees
 * its buffer. */
int pnn_measure_l2_peak(double* gbs, void* cuda_stream);

/* Number of kernels the library has launched on behalf of this workspace since it was created. */
int64_t pnn_launch_count(const pnn_workspace* ws);

const char* pnn_status_string(int status);
const char* pnn_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PNN_H_ */
