/*
 * wl_refine.h — C ABI of the B200-native randomized 1-WL colour refinement library.
 *
 * Implements, with hand-written sm_100a CUDA kernels, the data-parallel hot path of
 * arxiv/paper_2607_02603 ("Scaling Weisfeiler-Leman Expressiveness Analysis to Massive Graphs with GPUs"):
 *   Algorithm 1, RSC: random weight per colour, z = A w over Z/2^64, relabel (colour, z)
 *   Algorithm 2, RBSC: edge batches, inner nodes (Def. 5), local RSC, merge (Eq. 4), quotient (Def. 4)
 * Citations "L<n>" are line numbers of PAPER.md; "Q<n>" are the readings listed in DESIGN.md.
 *
 * General conventions
 *   - Graph = CSR whose ROWS ARE SOURCES: a_ij = (weighted) number of edges i -> j, sums run over row i (L43, L49, Q8).
 *     row_ptr int64[n+1] (row_ptr[0] = 0, non-decreasing, row_ptr[n] = m), col_idx int32[m] in [0, n),
 *     weights uint32[m] (>= 0) or NULL meaning all ones.  Duplicate (i, j) entries add (a_ij in N_0, L43, Q10).
 *   - Preconditions of Theorem 1 (L129): n <= 2^31 - 2 here (int32 ids; the paper allows 2^32) and every row sum <= 2^32.
 *   - Arithmetic is the ring Z/2^64 (unsigned 64-bit wrap-around, L100, Q3).  No floating point on the path.
 *   - Colours returned to the caller are CANONICAL: ids 0..k-1 in order of first occurrence, so equal partitions give
 *     equal arrays (Q7, Q21).
 *   - "device" pointers are CUDA device memory of the current device, "host" pointers are host memory (pinned
 *     recommended for the *_host / batched entry points).  All buffers are owned by the caller; the library never
 *     frees caller memory.  Entry points taking a workspace allocate nothing on the device.
 *   - cuda_stream is a cudaStream_t cast to void* (NULL = default stream).  Calls return after the result is
 *     complete on that stream (they synchronise the stream to read the convergence state).
 *   - Return value: WL_OK (0) or a negative wl_status.  Functions never throw and never call exit().
 *   - There is NO CPU fallback: without a CUDA device every compute entry point returns WL_ECUDA.
 */
#ifndef WL_REFINE_H_
#define WL_REFINE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum wl_status {
  WL_OK = 0,
  WL_EINVAL = -1,     /* null pointer, negative size, malformed CSR (bad offsets, column out of range)            */
  WL_ERANGE = -2,     /* n too large for int32 ids, or a row sum above 2^32 (Theorem 1 precondition, L129)        */
  WL_ENOMEM = -3,     /* workspace / device cap too small, or a device allocation failed                           */
  WL_ECUDA = -4,      /* a CUDA call failed (wl_last_cuda_error() gives the cudaError_t)                           */
  WL_EMAXROUNDS = -5  /* max_rounds / max_outer_iters reached before the fixed point                               */
} wl_status;

/* Adjacency in CSR form; all three arrays live where the entry point says (device or host). */
typedef struct wl_csr {
  int64_t n;               /* nodes                                            */
  int64_t m;               /* stored entries                                   */
  const int64_t* row_ptr;  /* n + 1 offsets                                    */
  const int32_t* col_idx;  /* m targets                                        */
  const uint32_t* weights; /* m edge weights, or NULL = unweighted (all ones)  */
} wl_csr;

/* flags for wl_options.flags */
#define WL_FLAG_NO_VALIDATE 1u   /* skip the CSR validation pass (one extra read of col_idx)                          */
#define WL_FLAG_NO_PRUNE 2u      /* keep every row in every round (no active-set pruning); results are identical      */
#define WL_FLAG_MERGE_KERNEL 4u  /* use the merge-path (edge-balanced, shared-memory staged) SpMV instead of the default
                                    warp-per-row + hub-chunk kernels; implies no pruning                               */
#define WL_FLAG_AGGRESSIVE_STOP 8u /* batched: stop when the next iteration's N_b would not decrease (L328)            */
#define WL_FLAG_NARROW_COLORS 32u /* wl_spmv_round only: all colour ids are < 65536, gather them as 16-bit (wl_refine
                                    switches by itself while k <= 65536)                                              */
#define WL_FLAG_SYNC_EVERY_ROUND 64u /* never queue several rounds without a host synchronisation (default: after round 6
                                       the device keeps the colour count and the host looks once per window, S5)       */
#define WL_FLAG_EDGE_BALANCED 128u /* use the edge-balanced SpMV kernel (one warp per 2048 consecutive entries, all rows) in
                                      every round instead of the row kernels; results are identical (measured slower on the
                                      headline graph, kept for extreme degree skew)                          */
#define WL_FLAG_NO_DEEP 256u     /* never switch to the worklist regime (below): every round recomputes every active row */
#define WL_FLAG_DEEP_EARLY 512u  /* switch to the worklist regime at round 2 instead of round 7 (testing)                 */
#define WL_FLAG_DEEP_CLUSTER 32768u /* worklist regime: every window of queued rounds as ONE launch by one thread-block cluster
                                       (cluster barriers between the phases instead of kernel boundaries).  Same results; measured
                                       slower than the default two kernels per round on B200, kept for testing                */
#define WL_FLAG_NO_FUSED_RECUT 2048u /* batched, default (re-cut) mode: always upload every batch again for its local refinement
                                        (default: the quotient pass refines the next iteration's greedy batches on the rows it
                                        has just emitted, whenever every row fits a batch).  Same results                       */
#define WL_FLAG_NO_FINAL 1024u   /* do not drop blocks whose whole neighbourhood is final from the active set (R5)        */
#define WL_FLAG_INHERIT_BATCHES 4096u /* batched: from the second outer iteration on, a quotient keeps the batches of its
                                        graph (the rows emitted together) instead of being re-cut by M_b, and its local
                                        refinement runs while those rows are still on the device: one upload pass per
                                        iteration instead of two (reading Q14b)                               */
#define WL_FLAG_CONSUME_INPUT 8192u /* batched, whole-CSR form only: the caller's col_idx (and weights) array is OVERWRITTEN: the
                                      quotient of the first outer iteration is written over the rows it was made from (its rows
                                      come out in row order and never hold more entries, Def. 4), as every later quotient
                                      overwrites its predecessor.  The host scratch then holds no column array
                                      (wl_refine_batched_host_bytes_consume): a graph of 77 GB needs 86 GB of scratch instead of
                                      154 GB.  The arrays must be writable; their contents are undefined afterwards           */
#define WL_FLAG_TAG_TABLE 16384u /* wl_refine from a uniform start: serve the gathers of the highest-degree nodes from a
                                   direct-mapped {tag, colour} table in shared memory during the 16-bit rounds (one persistent
                                   CTA per SM).  Results are identical.  OFF by default: measured slower than the plain row
                                   kernel on the headline graph (19.6 ms against 16.5 ms, profiles/r2_spmv_levers.md)        */
#define WL_FLAG_TEST_SMALL_OVERFLOW 536870912u /* testing: the device-side overflow list of the compressed quotient weights holds 2
                                                  entries, so that the fallback to plain uint32 weights is exercised            */
#define WL_FLAG_NO_CANONICAL 16u /* leave internal dense ids in out_colors (skips S6)                                  */

typedef struct wl_options {
  uint32_t flags;           /* WL_FLAG_*                                                                             */
  int32_t max_rounds;       /* <= 0: n + 1 (Alg. 1 needs at most n refinement steps, L416)                           */
  uint64_t stream_id;       /* second input of the round key (outer iteration / batch id); 0 for plain RSC           */
  int64_t* round_colors;    /* host, optional: number of colours after every round (the trajectory the oracle prints) */
  int32_t round_colors_cap; /* capacity of round_colors                                                              */
  int32_t max_outer_iters;  /* batched only; <= 0: unlimited                                                          */
  void* host_workspace;     /* batched only, optional: PINNED HOST scratch for the quotient graphs of Alg. 2 line 13 (they
                               exceed device memory by assumption, L135).  NULL: the library pins its own (first touch of
                               host pages costs far more than the transfers; callers that refine repeatedly should pass
                               one).  Caller-owned, contents undefined before and after.                               */
  size_t host_workspace_bytes; /* wl_refine_batched_host_bytes(n, m) always suffices; a smaller one is ignored          */
  int32_t ring_bits;        /* Algorithm 1's precision parameter q (L109-L110): the ring is Z/2^q.  0 or >= 64: q = 64, the
                               only setting Theorem 1's 1e-9 guarantee covers (L129).  1..63: every z is reduced mod 2^q where
                               it is compared; used to COUNT collisions (Lemma 1), never for production results          */
  int32_t host_pieces;      /* wl_refine_host only: number of pieces (whole rows each) the column upload is cut into so that the
                               first pass over the columns runs behind the link; <= 0: about 256 MB per piece, at most 32     */
  void* device_workspace;   /* wl_refine_host, optional: DEVICE scratch (256-byte aligned) that holds the uploaded graph and
                               the refinement workspace; NULL: the library allocates its own inside the call and frees it before
                               returning (cudaFree of the 28.6 GB a scale-27 call needs costs 9-17 ms: callers that refine
                               repeatedly pass one).  Caller-owned, contents undefined before and after.                       */
  size_t device_workspace_bytes; /* >= wl_refine_host_device_bytes(n, m, weighted, with_init); a smaller one is WL_ENOMEM.
                               wl_refine_batched, optional: a DEVICE arena all device buffers of the call are cut from (give it
                               device_cap_bytes, or what the graph needs when there is no cap): the call then makes no cudaMalloc /
                               cudaFree (they cost 18 ms per outer iteration and now and then 0.4 s).  A buffer that finds no free
                               block in it is allocated with cudaMalloc as without an arena; the cap is checked as always.       */
  const int32_t* batched_init_colors; /* wl_refine_batched only, optional: HOST int32[n], arbitrary non-negative labels (equal label
                               = same class), the initial partition L94 gives Algorithm 1, carried into Algorithm 2 (L171 has none;
                               reading Q18): the local start of every batch (Eq. 3) is intersected with the classes, a block of
                               a quotient carries the class of its nodes.  The result is a stable colouring that refines the classes,
                               the coarsest such one whenever the loop ends with N_b = 1.  NULL: one class.  8 more bytes per node on
                               the device.  A negative label is WL_EINVAL.                                                       */
} wl_options;

typedef struct wl_stats {
  int32_t rounds;            /* refinement rounds executed (the last one only confirms, Q1/Q2)                        */
  int32_t outer_iters;       /* batched: outer iterations of Alg. 2; 0 for wl_refine                                  */
  int64_t num_colors;        /* |H| of the result                                                                     */
  int64_t last_num_batches;  /* batched: N_b of the last outer iteration                                              */
  int64_t boundary_nodes;    /* batched: boundary nodes (Def. 5) in the first outer iteration                         */
  int64_t edges_streamed;    /* column indices actually consumed by SpMV kernels over all rounds                      */
  int64_t bytes_h2d;         /* host -> device bytes moved by the call                                                */
  int64_t bytes_d2h;         /* device -> host bytes moved by the call                                                */
  double ms_total;           /* device time of the whole call (CUDA events on cuda_stream)                            */
  double ms_spmv;            /* sum over rounds of the S1+S2 kernels                                                  */
  double ms_relabel;         /* sum over rounds of the S3+S4 kernels                                                  */
  int32_t spmv_launches;     /* rounds whose S1+S2 kernels streamed column indices (all rows or an active row list)   */
  int32_t kernel_launches;   /* kernels launched by the call                                                          */
  double ms_spmv_kernel;     /* device time of those S1+S2 kernels alone (CUDA events on cuda_stream)                 */
  int64_t spmv_alg_bytes;    /* algorithmic bytes of those launches: (4+G) per streamed entry (G = 2 or 4 bytes of
                                gathered colour id) + 16 per processed row (offsets + y)        */
  double ms_spmv_top;        /* the longest single S1+S2 launch of the call (row kernel + hub kernel of one round) ...  */
  int64_t spmv_top_alg_bytes;/* ... its algorithmic bytes ...                                                          */
  int64_t spmv_top_edges;    /* ... and the column indices it consumed (bench.py's roofline object)                     */
  double ms_rest_top;        /* S3+S4 (+ compaction) of that same round                                                */
  int64_t rows_top;          /* rows that round processed                                                              */
} wl_stats;

/* ------------------------------------------------------------------------------------------------------------------
 * Single batch: Algorithm 1 (RSC), L106-L127, from an arbitrary initial partition (L94).
 * ---------------------------------------------------------------------------------------------------------------- */

/* Bytes of device workspace wl_refine needs for a graph with n nodes and m entries (0 on invalid sizes). */
size_t wl_refine_workspace_bytes(int64_t n, int64_t m);

/* Bytes of device workspace that also hold the in-neighbour lists and work lists of the deep-round (worklist) regime:
 * from round 7 on only the rows with a changed out-neighbour are recomputed, under one fixed weight key (same partitions
 * per round, same fixed point; S5).  wl_refine uses that regime when the workspace it is given is at least this large. */
size_t wl_refine_deep_workspace_bytes(int64_t n, int64_t m);
/* device bytes one wl_refine_host call needs (CSR + optional weights / initial partition + colours + wl_refine_workspace_bytes) */
size_t wl_refine_host_device_bytes(int64_t n, int64_t m, int weighted, int with_init);

/* Coarsest stable colouring refining init_colors, with error probability <= 1e-9 (Theorem 1).
 *   g            CSR, all arrays DEVICE.
 *   init_colors  DEVICE int32[n], arbitrary non-negative labels (equal label = same block), or NULL = one block.
 *   seed         seeds the per-round weights  w(c) = P_key(c), key = f(seed, opt->stream_id, round)  (Q4, Q5).
 *   out_colors   DEVICE int32[n]; canonical ids on return (may alias init_colors).
 *   stats        HOST, may be NULL.      opt  HOST, may be NULL (defaults).
 *   workspace    DEVICE, >= wl_refine_workspace_bytes(n, m), 256-byte aligned; contents undefined before and after.
 * Errors: WL_EINVAL, WL_ERANGE, WL_ENOMEM (workspace too small), WL_ECUDA, WL_EMAXROUNDS. */
int wl_refine(const wl_csr* g, const int32_t* init_colors, uint64_t seed, int32_t* out_colors, wl_stats* stats,
              const wl_options* opt, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Same computation from HOST buffers (the end-to-end call): allocates its own device memory, copies the CSR and
 * init_colors host -> device, runs wl_refine, copies the colours device -> host.  g arrays, init_colors, out_colors: HOST
 * (pinned memory if the copies are to overlap the rounds).  The uploads run on a stream of the library's own in the order
 * the rounds need them (row offsets, then the columns in opt->host_pieces pieces of whole rows); S0, round 1 and the first
 * pass over the columns (S1+S2 piece by piece) run behind the link.  Same results as wl_refine. */
int wl_refine_host(const wl_csr* g, const int32_t* init_colors, uint64_t seed, int32_t* out_colors, wl_stats* stats,
                   const wl_options* opt, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------------------------
 * Step-level entry points, used by the parity tests and the benchmark.
 * ---------------------------------------------------------------------------------------------------------------- */

/* key(seed, stream_id, round) of the weight bijection (HOST computation, pure). Round numbers start at 1. */
uint64_t wl_round_key(uint64_t seed, uint64_t stream_id, uint64_t round);
/* w(c) = P_key(c) (HOST computation, pure): the weight Algorithm 1 line 3 assigns to colour c (L115-L118). */
uint64_t wl_weight(uint64_t key, uint64_t color);

/* S1+S2: y_i = sum_j a_ij * w(colors[j]) mod 2^64 (Alg. 1 line 5, L120).  colors: DEVICE int32[n] (any non-negative
 * ids); y: DEVICE uint64[n]; workspace as for wl_refine.  flags: WL_FLAG_MERGE_KERNEL selects the merge-path kernel. */
int wl_spmv_round(const wl_csr* g, const int32_t* colors, uint64_t key, uint64_t* y, uint32_t flags, void* workspace,
                  size_t workspace_bytes, void* cuda_stream);

/* S1+S2 restricted to an active row list (the pruned rounds, SURVEY.md §8(d) option 6): y[rows[t]] for t < num_rows as in
 * wl_spmv_round; every other entry of y is left untouched.  rows: DEVICE int32[num_rows], distinct node ids.
 * flags: WL_FLAG_NARROW_COLORS. */
int wl_spmv_rows(const wl_csr* g, const int32_t* colors, uint64_t key, const int32_t* rows, int64_t num_rows, uint64_t* y,
                 uint32_t flags, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* S3+S4: new_colors = dense ids (0..k'-1, unspecified order) of the exact pairs (colors[i], y[i]) (Alg. 1 line 6,
 * L122; Q6).  colors must be dense ids 0..k-1 (k given).  num_colors: HOST, receives k'.  new_colors may alias colors.
 * Blocks that do not split keep their id. */
int wl_relabel(int64_t n, const int32_t* colors, int64_t k, const uint64_t* y, int32_t* new_colors, int64_t* num_colors,
               void* workspace, size_t workspace_bytes, void* cuda_stream);

/* S6: canonical first-occurrence renumbering.  colors: DEVICE int32[n] with ids in [0, n); out may alias colors;
 * num_colors HOST (may be NULL). */
int wl_canonicalize(int64_t n, const int32_t* colors, int32_t* out, int64_t* num_colors, void* workspace,
                    size_t workspace_bytes, void* cuda_stream);

/* S6 for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc):
 * the same renumbering as wl_canonicalize, by the same kernels, with their scratch in a fixed file-scope device array of the
 * library instead of a caller workspace.  The call allocates nothing (no cudaMalloc / cudaFree / cudaHostAlloc, no allocating
 * library routine), copies nothing to the host and never synchronises: it only enqueues its kernels on cuda_stream and returns.
 *   n          at most WL_STATIC_MAX_NODES; a larger n returns WL_ERANGE with nothing enqueued (use wl_canonicalize).
 *   colors     DEVICE int32[n], ids in [0, n); out: DEVICE int32[n], may alias colors.
 *   num_colors DEVICE int64* (8-byte aligned; NOT host memory, unlike wl_canonicalize's) receiving the number of distinct
 *              colours when the stream reaches the end of the call, or NULL.  n == 0 writes nothing.
 * The array (about 8.2 MiB: two int32 per node of the maximum, plus the scan words) is held by every GPU that loads the library
 * until the process exits.  EVERY call on a device shares it and it keeps the last call's contents; each call rewrites all it
 * reads, so calls one after another (same stream, or ordered by events) are independent, but two calls that OVERLAP on one
 * GPU (different streams, or different host threads on unordered streams) race on it and both results are undefined.  The
 * device of cuda_stream must be the current device: the array's address is looked up for the current device on the first call
 * there (cudaGetSymbolAddress; make that first call outside any stream capture).
 * Returns WL_OK once everything is enqueued; WL_EINVAL (negative n, null colors / out), WL_ERANGE (n above the maximum),
 * WL_ECUDA (symbol lookup or launch failure, see wl_last_cuda_error).  Errors of the kernels themselves surface at the caller's
 * next synchronisation of the stream. */
#define WL_STATIC_MAX_NODES 1048576
int wl_canonicalize_static(int64_t n, const int32_t* colors, int32_t* out, int64_t* num_colors, void* cuda_stream);
int64_t wl_canonicalize_static_max_nodes(void); /* = WL_STATIC_MAX_NODES of the library that is loaded */

/* ------------------------------------------------------------------------------------------------------------------
 * Batched: Algorithm 2 (RBSC), L169-L202, over HOST-resident edge batches.
 * ---------------------------------------------------------------------------------------------------------------- */

/* One batch E_k of the edge partition (L137, L180).  Either
 *   CSR-slice form (src == NULL): the batch owns the consecutive CSR edge positions [edge_begin, edge_begin + num_edges) of a
 *     global CSR whose row_ptr (HOST, n + 1 offsets, shared by all batches) is given in every batch; col_idx / weights point at
 *     THIS batch's first entry; or
 *   COO form (src != NULL): arbitrary edges (src[e], col_idx[e]) with optional weights, num_edges of them, any order;
 *     row_ptr and edge_begin are ignored.  All batches of a call have the same form.  The first outer iteration then runs
 *     three streaming passes (inner mask of Def. 5 by the method of L463; local refinement of the gathered rows of V_k;
 *     quotient by block ranges); later iterations run on the library's own quotient CSR.  Nodes without out-edges are inner
 *     to batch 0 (Q9).  WL_FLAG_INHERIT_BATCHES is not defined for this form (WL_EINVAL). */
typedef struct wl_edge_batch {
  int64_t edge_begin;
  int64_t num_edges;
  const int64_t* row_ptr;
  const int32_t* col_idx;
  const uint32_t* weights;
  const int32_t* src;
} wl_edge_batch;

/* Stable colouring of (V, A) by Algorithm 2; equals the coarsest one whenever the loop ends with N_b = 1 (L208).
 *   batches          HOST array of num_batches descriptors = the edge partition of outer iteration 1 (Alg. 2 line 5).
 *                    num_batches == 0: `whole` must be given and the library cuts it itself (Q13).
 *   whole            HOST CSR of the full graph (num_batches == 0), else NULL.
 *   max_batch_edges  M_b (L171): cap on edges per batch for the library's own partitions (later outer iterations, Q14).
 *                    <= 0 (with `whole` and a device cap): the library derives the largest M_b that fits the cap.
 *   device_cap_bytes upper bound on device memory the call may allocate (0 = no cap); WL_ENOMEM if it cannot be met.
 *   out_colors       HOST int32[n], canonical ids on the ORIGINAL nodes (Q16). */
int wl_refine_batched(int64_t n, int32_t num_batches, const wl_edge_batch* batches, const wl_csr* whole, uint64_t seed,
                      size_t device_cap_bytes, int64_t max_batch_edges, int32_t* out_colors, wl_stats* stats,
                      const wl_options* opt, void* cuda_stream);

/* Quotient weights of an UNWEIGHTED input are stored and moved as one byte each plus per-emission overflow lists for the weights
 * >= 255 (at most m / 255 of them: a quotient row sums to the out-degree of its representative, L447); a batch with more heavy
 * weights than the device-side list takes makes the call start over with uint32 weights (with WL_FLAG_CONSUME_INPUT: WL_ENOMEM).
 * Bytes of pinned host scratch that always suffice for wl_options.host_workspace: two offset arrays of n + 1 entries and
 * one weighted entry array of m entries (a quotient never has more nodes or entries than its graph, Def. 4; later
 * quotients overwrite the first one in place). */
size_t wl_refine_batched_host_bytes(int64_t n, int64_t m);
/* the same under WL_FLAG_CONSUME_INPUT: two offset arrays, plus one weight array of m entries unless the input is weighted */
size_t wl_refine_batched_host_bytes_consume(int64_t n, int64_t m, int weighted);
/* optional extra: a host workspace with this many bytes MORE than the size above also holds the overflow lists of the one-byte
 * weights (unweighted inputs); otherwise the library pins them itself in every call (cudaHostAlloc / cudaFreeHost of some tens of
 * megabytes: 50-800 ms per call, measured at scale 26).  wl_refine_batched_host_bytes has that room already (it counts four bytes
 * per weight); add it to wl_refine_batched_host_bytes_consume. */
size_t wl_refine_batched_host_overflow_bytes(int64_t m);

/* B2: inner-node labels of Def. 5 (L139-L145) by the method of L463.  edge_batch: DEVICE int32[m] batch id of every CSR edge
 * slot; sink_batch: DEVICE int32[n] label given to nodes without out-edges (Q9); label: DEVICE int32[n], -1 = boundary. */
int wl_inner_labels(int64_t n, const int64_t* row_ptr, const int32_t* edge_batch, const int32_t* sink_batch, int32_t* label,
                    void* cuda_stream);

/* B6: quotient graph of Def. 4 / Eq. 1 (L59-L65) for canonical colours (representative = first node of a block, Q17).
 * All arrays DEVICE.  q_row_ptr int64[k+1]; q_col / q_weights capacity q_cap entries; *q_m (HOST) receives the entry count.
 * Columns of a row come out sorted with equal targets merged.  WL_ENOMEM if q_cap is too small (q_m is still set). */
int wl_quotient(const wl_csr* g, const int32_t* colors, int64_t k, int64_t* q_row_ptr, int32_t* q_col, uint32_t* q_weights,
                int64_t q_cap, int64_t* q_m, void* workspace, size_t workspace_bytes, void* cuda_stream);
size_t wl_quotient_workspace_bytes(int64_t n, int64_t m);

/* ------------------------------------------------------------------------------------------------------------------
 * One batch at a time on DEVICE buffers: the per-batch work of an outer iteration of Algorithm 2, for callers that spread the
 * batches over several GPUs (L213 "embarrassingly parallel ... scheduled concurrently across GPUs", L239) and exchange the
 * block maps themselves (paper_2607_02603_b200/sharded.py does, over torch.distributed).
 * ---------------------------------------------------------------------------------------------------------------- */

/* B3 + B4 for the inner nodes V_k = [lo, lo + rows->n) of a batch (Eq. 3; Alg. 2 line 9): `rows` holds exactly their rows
 * (DEVICE; row_ptr[0] = 0, row_ptr[0..n] index col_idx / weights, targets are global node ids < n_targets); every target outside V_k is
 * an implicit singleton.  local_colors (DEVICE int32[n]): dense ids in first-occurrence order inside the batch; is_first
 * (DEVICE uint8[n]): 1 for the first node of every block; *num_colors (HOST): their number.  opt: flags, ring_bits, max_rounds,
 * stream_id are honoured.  workspace >= wl_refine_inner_workspace_bytes(n, m), 256-byte aligned. */
size_t wl_refine_inner_workspace_bytes(int64_t n_rows, int64_t m);
int wl_refine_inner(const wl_csr* rows, int64_t lo, int64_t n_targets, uint64_t seed, int32_t* local_colors, uint8_t* is_first,
                    int64_t* num_colors, const wl_options* opt, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* B6 for the whole rows of the nodes [lo, lo + rows->n): the quotient rows (Def. 4) of the blocks whose representative (first node,
 * is_first[i - lo] == 1) lies among them, i.e. the blocks first_block .. first_block + num_blocks - 1 of the canonical block map
 * block_of (DEVICE int32 over ALL nodes).  q_row_ptr: DEVICE int64[num_blocks + 1] starting at 0; columns of a row come out in
 * any order with equal targets merged.  WL_ENOMEM if q_cap is too small (*q_m is still set). */
size_t wl_quotient_rows_workspace_bytes(int64_t n_rows, int64_t m, int64_t num_blocks);
int wl_quotient_rows(const wl_csr* rows, int64_t lo, const int32_t* block_of, const uint8_t* is_first, int64_t first_block,
                     int64_t num_blocks, int64_t* q_row_ptr, int32_t* q_col, uint32_t* q_weights, int64_t q_cap, int64_t* q_m,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------------------------ */
const char* wl_strerror(int code);
int wl_last_cuda_error(void);      /* cudaError_t of the last WL_ECUDA on this thread */
const char* wl_version(void);
int64_t wl_kernel_launches(void);  /* kernels launched by this library on the calling thread since it was loaded */

#ifdef __cplusplus
}
#endif
#endif /* WL_REFINE_H_ */
