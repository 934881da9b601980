/* etx.h — C ABI of libetx: the hits -> edge-scores hot path of the ETX4VELO GNN tracking pipeline
 * (F. Giasemis, arXiv 2508.07423; "P:n" = line n of PAPER.md), written for one NVIDIA B200 (sm_100a).
 *
 * The path (thesis §8.3; GPU pipeline steps P:2585-2593):
 *   a0 features   recentre + rescale hit coordinates
 *   a1 embed      embedding MLP, ReLU hidden layers, linear output (Eqs. 4.24-4.27)
 *   a2 graph      hit i on plane p -> hits j of the same event on planes p+1..p+G with
 *                 d^2(i,j) = |emb_i - emb_j|^2 < r2_max (Eq. 8.1)
 *   a3 encoders   h0 = MLP_n(x,y,z) ; e0_ij = MLP_e([h0_i, h0_j])
 *   a4-a6         n_iter x { m_l = [sum_{l->j} e_lj, sum_{i->l} e_il] (Eq. 8.5);
 *                            h_l += phi_k([h_l, m_l]) ; e_ij += psi_k([h_i, h_j, e_ij]) }
 *   a7 scores     s_ij = sigmoid(MLP_c(e_ij))
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers owned by the caller (e.g. torch tensors); h_* are HOST
 *     pointers.  The library never frees or reallocates caller memory.  `stream` is a cudaStream_t
 *     passed as void* (NULL = default stream).  All work is enqueued on that stream.
 *   - Every call returns an etx_status; no exceptions or aborts cross the ABI.  After a failure
 *     etx_last_error(ctx) holds a message.  There is NO CPU fallback: without a CUDA device every
 *     compute call returns ETX_ERR_CUDA.
 *   - Events are independent; a batch is a CSR list of events: SoA fp32 hit arrays (P:2620,
 *     P:2630) plus prefix-sum offsets.  Hits of an event must be sorted by plane.
 *   - Weights: one flat fp32 host blob, MLPs in the order  embedding, node encoder, edge encoder,
 *     (node network k, edge network k) for k = 0..n_iter-1, classifier; inside an MLP the layers are
 *     consecutive, each W[out][in] row-major followed by b[out].  GNN MLPs have gnn_n_layers
 *     matrices: in -> H -> ... -> H -> out with in = 3 (node enc), 2H (edge enc, [h_src, h_dst]),
 *     3H (node net, [h, m_out, m_in]), 3H (edge net, [h_src, h_dst, e]), H (classifier, out = 1).
 */
#ifndef ETX_H_
#define ETX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ETX_MAX_MLP_LAYERS 8

typedef enum {
  ETX_OK = 0,
  ETX_ERR_INVALID = -1,   /* bad argument, unsupported shape, malformed batch                     */
  ETX_ERR_CAPACITY = -2,  /* graph has more edges than edge_capacity (n_edges holds the need)     */
  ETX_ERR_CUDA = -3,      /* CUDA runtime error or no device                                      */
  ETX_ERR_UNSORTED = -4,  /* hits of an event are not sorted by plane                             */
  ETX_ERR_NOMEM = -5      /* workspace missing or too small                                       */
} etx_status;

typedef enum {
  ETX_PREC_FP32 = 0,    /* fp32 operands, FFMA on the CUDA cores, fp32 accumulate                 */
  ETX_PREC_TF32X3 = 1,  /* tcgen05 tensor cores, error-compensated 3xTF32 split (fp32-equivalent) */
  ETX_PREC_BF16 = 2,    /* tcgen05 tensor cores, bf16 operands, fp32 accumulate, fp32 state: the per-EDGE MLP chains
                           (edge encoder, edge networks) run one kind::f16 MMA pass on bf16-rounded operands; the
                           per-HIT MLPs (node encoder, node networks, per-hit projections of the edge MLPs' first
                           layers) and the classifier run the BF16X3 split below -- they cost N rows instead of E (the
                           classifier: one launch) and keep every edge of config c3 inside its 2e-2 gate             */
  ETX_PREC_BF16X3 = 3,  /* tcgen05, operands split x = hi + lo into two bf16 (16 significand bits),
                           three kind::f16 MMAs (lo.hi + hi.lo + hi.hi), fp32 accumulate and state:
                           meets the fp32 tolerance at half the tensor-core work of 3xTF32          */
  ETX_PREC_INT8 = 4,    /* next row (NEXT-3, GNN part): tcgen05 kind::i8 -- INT8 codes for every GNN MLP layer
                           input and weight (static ranges: etx_set_int8_ranges), exact int32 sums, fp32
                           de-quantisation, biases, state and scatter-sum; the embedding stays 3xTF32      */
  ETX_PREC_FP8 = 5      /* next row (NEXT-3, GNN part): tcgen05 kind::f8f6f4 -- e4m3 values for every GNN MLP layer
                           input and weight (the same static ranges, S = alpha / 448), fp32 accumulation,
                           de-quantisation, biases, state and scatter-sum; the embedding stays 3xTF32      */
} etx_precision;

typedef struct {
  int32_t emb_n_layers;                       /* weight matrices in the embedding MLP             */
  int32_t emb_dims[ETX_MAX_MLP_LAYERS + 1];   /* e.g. {3,128,128,128,4}                           */
  int32_t gnn_hidden;                         /* H = n_h = n_e; 64 or 128                */
  int32_t gnn_n_layers;                       /* weight matrices per GNN MLP (hidden layers + 1)  */
  int32_t n_iter;                             /* message-passing steps, distinct weights */
  int32_t precision;                          /* etx_precision of the GNN / embedding MLPs        */
  int32_t n_planes;                           /* 26                                      */
  float norm_center[5];                       /* r, phi, z, x, y : f = (v - center) / scale       */
  float norm_scale[5];
} etx_model_desc;

typedef struct {                /* CSR batch of events, device resident                           */
  int32_t n_events, n_hits;
  const int32_t* d_event_ptr;   /* [n_events+1] hit offsets, d_event_ptr[0] = 0                   */
  const uint8_t* d_plane;       /* [n_hits] plane id < n_planes, ascending inside an event        */
  const float *d_r, *d_phi, *d_z, *d_x, *d_y; /* [n_hits] raw mm / rad                            */
} etx_batch;

typedef struct {                /* same batch in HOST memory (for etx_infer_host)                 */
  int32_t n_events, n_hits;
  const int32_t* h_event_ptr;
  const uint8_t* h_plane;
  const float *h_r, *h_phi, *h_z, *h_x, *h_y;
} etx_batch_host;

typedef struct {                /* rough hit graph, arrays caller-allocated with capacity         */
  int64_t edge_capacity;        /* in: entries available in d_src, d_dst, d_in_perm               */
  int64_t n_edges;              /* out of etx_build_graph: E (also on ETX_ERR_CAPACITY)           */
  int32_t* d_row_ptr;           /* [n_hits+1] CSR by source: edges of hit i are row_ptr[i]..      */
  int32_t* d_src;               /* [cap] source hit of edge e; edges ordered (src asc, dst asc)   */
  int32_t* d_dst;               /* [cap] destination hit of edge e                                */
  int32_t* d_in_ptr;            /* [n_hits+1] CSR by destination                                  */
  int32_t* d_in_perm;           /* [cap] edge ids entering hit j, in_ptr[j].., ascending edge id  */
} etx_graph;

typedef struct etx_ctx etx_ctx;

/* Number of floats the weight blob must hold for `desc` (layout above); 0 if desc is invalid.     */
size_t etx_weight_count(const etx_model_desc* desc);

/* Create a context on CUDA device `device`: validates desc, copies the weights to the device and
 * pre-arranges them for the kernels.  h_weights: host fp32 blob of n_weights floats.              */
etx_status etx_create(etx_ctx** ctx, const etx_model_desc* desc, const float* h_weights,
                      size_t n_weights, int device);
etx_status etx_destroy(etx_ctx* ctx);
const char* etx_last_error(const etx_ctx* ctx);   /* ctx may be NULL: last create error            */

/* Device scratch the calls need for batches up to these sizes.  with_host_path adds the staging
 * buffers etx_infer_host carves (device copies of the batch, embeddings, graph, encodings).       */
size_t etx_workspace_bytes(const etx_ctx* ctx, int32_t n_events, int32_t n_hits,
                           int64_t edge_capacity, int with_host_path);
/* Hand the context a caller-owned device buffer (256-byte aligned); it stays caller-owned.        */
etx_status etx_set_workspace(etx_ctx* ctx, void* d_workspace, size_t bytes);

/* a0+a1: d_emb[n_hits, emb_dim] fp32 row-major = embedding MLP of ((r,phi,z) - center) / scale.   */
etx_status etx_embed(etx_ctx* ctx, const etx_batch* batch, float* d_emb, void* stream);

/* Report-only variant of etx_embed (reading Q16; BASELINE.json's config 3 says "embedding ... in bf16"): the
 * embedding MLP with its hidden layers' operands rounded to bf16 (round to nearest even), one tcgen05.mma.kind::f16 per
 * K-step, fp32 accumulation; the 3-input first layer and the narrow output layer stay fp32 FMA chains as in etx_embed.
 * The path itself always embeds in 3xTF32 because the embedding decides graph edges; this call exists so that bench.py
 * can report what a bf16 embedding does to the edge set (thesis analogue: +5-10 % edges after INT8 calibration).
 * Needs 128-wide hidden layers (ETX_ERR_INVALID otherwise).                                                           */
etx_status etx_embed_bf16(etx_ctx* ctx, const etx_batch* batch, float* d_emb, void* stream);

/* Next row (embedding part): the embedding MLP of etx_embed with INT8 weights and
 * activations, static post-training quantisation with the symmetric scheme of Eqs. 4.31-4.33:
 * S = alpha / 127, x_q = clip(round(x / S), -127, 127) (round half to even, fp32 division).  Per layer the input
 * is quantised with S_a = h_act_alpha[l] / 127 (HOST array of emb_n_layers calibrated ranges, > 0), the weight
 * with S_w = max|W_l| / 127 (done once at etx_create); y = float(int32 sum) * (S_a * S_w) + b, ReLU on hidden
 * layers, every float step one rounded fp32 operation.  d_emb[n_hits, emb_dim] fp32 as etx_embed.               */
etx_status etx_embed_int8(etx_ctx* ctx, const etx_batch* batch, const float* h_act_alpha, int32_t n_alpha,
                          float* d_emb, void* stream);

/* Next row (NEXT-3, GNN part; "the quantization of the GNN holds the most potential"): a context created with
 * ETX_PREC_INT8 runs every GNN MLP (encoders, node / edge networks, classifier) as an INT8 chain on the tensor cores
 * (tcgen05.mma.kind::i8): static post-training quantisation with the symmetric per-tensor scheme of Eqs. 4.31-4.33
 * exactly as etx_embed_int8 -- layer input codes with S_a = alpha / 127 (calibrated ranges, below), weight
 * codes with S_w = max|W_l| / 127, exact int32 sums, y = float(sum) * (S_a S_w) + b in single rounded fp32 steps.  The
 * state h, e, the aggregate m (sequential fp32 sums in ascending edge id) and the residual adds stay fp32.  Exception: the
 * node encoder's first layer (3 geometry features in) stays fp32 with double accumulation; its ReLU output is the first
 * quantised tensor.  The first layer of the edge MLPs is factorised as in the other tensor-core modes, in exact integer
 * arithmetic (int32 per-hit projections).  etx_set_int8_ranges hands over the ranges: HOST array of (3 + 2 n_iter) x
 * gnn_n_layers positive floats, MLPs in the order node encoder, edge encoder, (node network k, edge network k) for
 * k = 0..n_iter-1, classifier; entry l of an MLP = range of layer l's input (entry 0 of the node encoder is unused).
 * Without it etx_gnn_forward / etx_edge_scores return ETX_ERR_INVALID in this precision.  Needs gnn_hidden = 128.
 * ETX_PREC_FP8 is the same scheme on the e4m3 grid (reading Q26): S = alpha / 448, value = e4m3(clip(x * fl(1 / S),
 * -448, 448)) rounded to nearest even (cvt.rn.satfinite.e4m3x2.f32), weights likewise with S_w = max|W_l| / 448, products
 * accumulated in fp32 by the tensor cores (tcgen05.mma.kind::f8f6f4), y = acc * (S_a S_w) + b; the first-layer projections of
 * the edge MLPs are fp32 sums.  It takes the same ranges through etx_set_int8_ranges.  Results agree with the quantised oracle
 * within a tolerance, not bit for bit: the oracle's sums are exact, the tensor cores' are fp32.                        */
etx_status etx_set_int8_ranges(etx_ctx* ctx, const float* h_alpha, size_t n);

/* a2: fixed-radius search in embedding space.  Edge (i -> j) iff same event,
 * 1 <= plane(j) - plane(i) <= max_plane_gap, and d^2 < r2_max with d^2 evaluated in fp32 as
 * ((e0-f0)^2 + (e1-f1)^2) + ... left to right, each operation rounded (no FMA).  Output is the
 * unique ordered CSR (src asc, dst asc) plus the by-destination lists.  k_max = 0: pure fixed
 * radius (the hot path).  k_max > 0 (next row; Algorithm 1): at most k_max
 * out-edges per hit, the k_max nearest by (d^2 as above, then hit index), still in ascending dst
 * order; k_max < 0 is ETX_ERR_INVALID.  Validates the batch (ETX_ERR_INVALID / ETX_ERR_UNSORTED).
 * Synchronises the stream once to return g->n_edges; if E > edge_capacity returns ETX_ERR_CAPACITY
 * with n_edges = E and d_src/d_dst/d_in_perm untouched.                                           */
etx_status etx_build_graph(etx_ctx* ctx, const etx_batch* batch, const float* d_emb, float r2_max,
                           int32_t max_plane_gap, int32_t k_max, etx_graph* g, void* stream);

/* a3-a6: encoders + n_iter message-passing steps.  d_edge_enc [n_edges, H] fp32 receives e^n;
 * d_hit_enc [n_hits, H] fp32 receives h^n if not NULL.  Both must be 16-byte aligned (ETX_ERR_INVALID).                                            */
etx_status etx_gnn_forward(etx_ctx* ctx, const etx_batch* batch, const etx_graph* g,
                           float* d_edge_enc, float* d_hit_enc, void* stream);

/* a7: d_scores[n_edges] fp32 = sigmoid(classifier(e)).                                            */
etx_status etx_edge_scores(etx_ctx* ctx, const etx_graph* g, const float* d_edge_enc,
                           float* d_scores, void* stream);

/* Next row beyond the hits -> edge-scores path: score cut + track building.  The purified hit graph keeps
 * the edges with score >= score_min; tracks are its weakly connected components
 * (plane-sweep minimum-label propagation repeated until stable, so the result is the exact
 * WCC).  d_labels[n_hits] receives for every hit the smallest hit index of its component (a hit without
 * kept edges gets its own index).  Deterministic.                                                    */
etx_status etx_build_tracks(etx_ctx* ctx, const etx_batch* batch, const etx_graph* g, const float* d_scores,
                            float score_min, int32_t* d_labels, void* stream);

/* Next row: triplet building (Fig. 8.13).  Two edges of the purified hit graph (score >= score_min,
 * the cut of etx_build_tracks) that share a hit C form an articulation (A -> C, C -> B), a left elbow (C -> A,
 * C -> B) or a right elbow (A -> C, B -> C).  Rows are pairs of EDGE IDS (d_first[i], d_second[i]) in three
 * consecutive sections -- n[0] articulations (first = the incoming edge A -> C, second = the outgoing edge
 * C -> B), then n[1] left elbows, then n[2] right elbows (first < second) -- each section ordered by (shared hit,
 * first, second).  d_ptr [3][n_hits + 1] receives, per kind, the offset of every shared hit's rows inside its
 * section (CSR by shared hit; d_ptr[k][n_hits] = n[k]).  All buffers are caller-owned DEVICE memory.
 * Synchronises the stream to return the counts.  n[0] + n[1] + n[2] > capacity: ETX_ERR_CAPACITY with n filled
 * and d_first / d_second untouched.  A kind with more than 2^31 - 1 rows is ETX_ERR_CAPACITY as well.
 * Needs the workspace of etx_build_graph.  Deterministic (integer work, one fixed order).                     */
typedef struct {
  int64_t capacity;           /* in: rows available in d_first / d_second                                   */
  int64_t n[3];               /* out: articulations, left elbows, right elbows                              */
  int32_t* d_ptr;             /* [3][n_hits + 1]                                                            */
  int32_t* d_first;           /* [capacity]                                                                 */
  int32_t* d_second;          /* [capacity]                                                                 */
} etx_triplets;
etx_status etx_build_triplets(etx_ctx* ctx, const etx_batch* batch, const etx_graph* g, const float* d_scores,
                              float score_min, etx_triplets* t, void* stream);

/* etx_build_triplets for callers that cannot allocate device memory and have registered no workspace (code under CUDA
 * graph capture set-up, tight serving loops, harnesses that forbid cudaMalloc).  Same arguments, same rows, same d_ptr
 * and counts as etx_build_triplets, bit for bit.  Its only scratch -- the block sums of the three device-wide scans -- is
 * a fixed file-scope device array inside the library (9 KB, held by every GPU that loads libetx.so until the process
 * exits) instead of the workspace of etx_set_workspace: the call allocates nothing (no cudaMalloc / cudaFree, no
 * allocating library routine) and works on a context without a workspace.
 * Limit: batch->n_hits <= ETX_STATIC_TRIPLET_MAX_HITS, else ETX_ERR_CAPACITY (nothing is launched).
 * The array is shared by EVERY call on a device, whatever the context or stream, and keeps the last call's contents;
 * the part a call uses is cleared on its stream first.  Two calls that overlap on the GPU (different streams, or
 * different host threads) race on it and give undefined counts: serialise them.  Not recorded by etx_profile_read.
 * Other statuses as etx_build_triplets.                                                                          */
#define ETX_STATIC_TRIPLET_MAX_HITS 4194304   /* 2^22: four of the thesis' 2^20-hit GNN batches; config c4 has 3.5 M */
etx_status etx_build_triplets_static(etx_ctx* ctx, const etx_batch* batch, const etx_graph* g, const float* d_scores,
                                     float score_min, etx_triplets* t, void* stream);

/* Next row: triplet classifiers ("edge encodings are sufficient for both the edge classifier and triplet
 * classifier"; Fig. 8.12 caption P:2330, [.,.] = concatenation; "separate triplet classifiers for articulations
 * and elbows", each "an MLP ending with a layer with 1 unit, and a sigmoid").  Reading: s = sigmoid(MLP_k([e_first,
 * e_second])) on the rows of etx_build_triplets; MLP_art scores the articulations, MLP_elb both elbow kinds; each is
 * 2H -> H .. H -> 1 with gnn_n_layers matrices.  The two MLPs come in their own host blob (articulation classifier,
 * then elbow classifier; layer layout as the main blob) of etx_triplet_weight_count(desc) floats, and run in the
 * context's precision.  d_trip_scores [n[0] + n[1] + n[2]] fp32, row for row with d_first / d_second.            */
size_t etx_triplet_weight_count(const etx_model_desc* desc);
etx_status etx_set_triplet_classifiers(etx_ctx* ctx, const float* h_weights, size_t n_weights);
etx_status etx_triplet_scores(etx_ctx* ctx, const etx_graph* g, const float* d_edge_enc, const etx_triplets* t,
                              float* d_trip_scores, void* stream);

/* Next row: track building from triplets, the four steps of P:2363 (section 8.3.5).  The EDGE graph has the kept
 * edges (score >= score_min) as nodes and the kept triplets (triplet score >= trip_min) as connections.
 *   1. the two edges of every kept elbow are merged into one super-edge; a kept articulation (a, b) becomes the pair
 *      (S(a), S(b)); pairs inside one super-edge vanish and equal pairs count once ("duplicate edges ... are removed");
 *   2. a pair (u, v) is SHARED iff u has two or more distinct successors or v two or more distinct predecessors
 *      ("two articulations sharing an edge"); connected sets = components under the elbows and the UNSHARED pairs;
 *   3. every distinct (set of u, set of v) of a shared articulation is a track: the union of the two sets (the shared
 *      set is duplicated into each of its tracks); a set touched by no shared articulation is a track by itself;
 *   4. a track is the ascending list of the hits of its edges.
 * Outputs (caller-owned DEVICE memory): d_edge_set[n_edges] = the set of every edge, named by its smallest edge id
 * (-1 for a cut edge); d_joins [n_joins][2] = the distinct (set of u, set of v) pairs, ascending; tracks in CSR form,
 * d_track_ptr [n_tracks + 1] / d_track_hits: first the n_plain untouched sets by ascending name, then the joins in
 * order.  Everything is one fixed array (integer work).  Synchronises the stream twice to learn the counts; if a
 * capacity is short returns ETX_ERR_CAPACITY with the four counts filled and only d_edge_set written.  Needs a
 * workspace of etx_triplet_tracks_workspace_bytes (the same etx_set_workspace buffer; contents are clobbered).    */
typedef struct {
  int64_t join_capacity, track_capacity, hit_capacity;   /* in: rows of d_joins, tracks (d_track_ptr has +1), hit entries */
  int64_t n_joins, n_plain, n_tracks, n_track_hits;      /* out */
  int32_t* d_edge_set;                                   /* [n_edges]            */
  int32_t* d_joins;                                      /* [join_capacity][2]   */
  int32_t* d_track_ptr;                                  /* [track_capacity + 1] */
  int32_t* d_track_hits;                                 /* [hit_capacity]       */
} etx_tracks;
size_t etx_triplet_tracks_workspace_bytes(const etx_ctx* ctx, int32_t n_hits, int64_t n_edges, int64_t n_articulations);
etx_status etx_build_tracks_from_triplets(etx_ctx* ctx, const etx_batch* batch, const etx_graph* g, const float* d_scores,
                                          float score_min, const etx_triplets* t, const float* d_trip_scores,
                                          float trip_min, etx_tracks* tracks, void* stream);

/* Whole path with HOST buffers: copies the batch host->device, runs a0..a7, copies src/dst/scores
 * back (h_src, h_dst may be NULL; each needs edge_capacity entries).  Host buffers should be pinned for
 * the copies to be asynchronous.  Synchronises the stream before returning.
 * Workspace: one sized with etx_workspace_bytes(..., with_host_path = 1) for the whole batch runs it in one
 * pass.  A SMALLER workspace is not an error: the batch is then split into consecutive event ranges that fit
 * (the thesis bounds its GNN batches the same way: <= 2^20 hits, <= 2^22 edges), run one after the
 * other; events are independent and edges are ordered by source, so the outputs are identical to the
 * single-pass ones, element for element.  ETX_ERR_NOMEM only if a single event does not fit.
 * *n_edges receives E; on ETX_ERR_CAPACITY the edges found so far plus the range that overflowed.       */
etx_status etx_infer_host(etx_ctx* ctx, const etx_batch_host* batch, float r2_max,
                          int32_t max_plane_gap, int64_t edge_capacity, int64_t* n_edges,
                          int32_t* h_src, int32_t* h_dst, float* h_scores, void* stream);

/* Number of kernels the library has launched on this context since creation (for accounting).     */
int64_t etx_launch_count(const etx_ctx* ctx);

/* Measurement utility (not a step of the path): the rate, in arithmetic operations per second, at which `device`
 * retires the instruction mix of two of the library's ALU-bound kernels, measured with a register-resident
 * microbenchmark (8 independent chains per thread, 8 CTAs of 256 threads per SM, best of 4 timed launches):
 *   kind 0  unfused fp32 add + multiply as scalar instructions   -- the distance test of Eq. 8.1 for d != 4
 *   kind 1  the same as packed pairs (add.rn.f32x2 / mul.rn.f32x2) -- the d = 4 distance test (graph.cu)
 *   kind 2  fused multiply-add, 2 flop each                       -- the exact-fp32 MLP kernel (ETX_PREC_FP32)
 * bench.py divides by these instead of a figure derived from unit counts and clocks.  Needs no context; returns
 * ETX_ERR_CUDA without a device, ETX_ERR_INVALID for a bad kind or a NULL result pointer. */
etx_status etx_measure_alu_peak(int32_t device, int32_t kind, double* ops_per_s);

/* Per-stage device timing.  While enabled, every group of launches of one class is bracketed by CUDA
 * events on the call's stream.  etx_profile_read synchronises those events, returns the accumulated
 * milliseconds and launch counts per class since the last read (arrays of ETX_K_COUNT), and resets.  */
typedef enum {
  ETX_K_EMBED = 0,      /* a0+a1 embedding MLP                                */
  ETX_K_GRAPH = 1,      /* a2 plane index, search count/fill, scans           */
  ETX_K_NODE_ENC = 2,   /* a3 node encoder                                    */
  ETX_K_EDGE_ENC = 3,   /* a3 edge encoder                                    */
  ETX_K_SCATTER = 4,    /* a4 message aggregation                             */
  ETX_K_NODE_NET = 5,   /* a5 node network                                    */
  ETX_K_EDGE_NET = 6,   /* a6 edge network (the dominant kernel)              */
  ETX_K_CLS = 7,        /* a7 classifier + sigmoid                            */
  ETX_K_TRACKS = 8,     /* next row: score cut + WCC track building             */
  ETX_K_EDGE_PROJ = 9,  /* a3/a6 per-hit first-layer projections [A h | B h] of the edge MLPs (tensor-core modes) */
  ETX_K_COUNT = 10
} etx_kernel_class;
etx_status etx_profile_enable(etx_ctx* ctx, int on);
etx_status etx_profile_read(etx_ctx* ctx, double* ms /*[ETX_K_COUNT]*/, int64_t* launches /*[ETX_K_COUNT]*/);

#ifdef __cplusplus
}
#endif
#endif /* ETX_H_ */
