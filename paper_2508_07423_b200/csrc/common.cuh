// Internal declarations shared by the translation units of libetx (sm_100a).  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "../../include/etx.h"

namespace etx {

constexpr int kMaxLayers = ETX_MAX_MLP_LAYERS;
constexpr int kMaxDevices = 64;      // per-device launch configuration tables (cudaFuncSetAttribute is per device)

// One MLP on the device.  Wt[l] is the layer's weight TRANSPOSED to [in][out] row-major (k-major, so
// a K-chunk of it is a contiguous slab), b[l] its bias, both fp32.
struct DevMlp {
  int n_layers = 0;
  int dims[kMaxLayers + 1] = {0};
  const float* Wt[kMaxLayers] = {nullptr};
  const float* b[kMaxLayers] = {nullptr};
  const unsigned char* wimg = nullptr;   // tensor-core weight image (mlp_tc.cu), or null
  // First-layer factorisation (edge encoder / edge networks in tensor-core modes): the first layer's
  // weight W1 = [A | B | C] over the inputs [h_src | h_dst | e] is split; wimg_a / wimg_b are the
  // one-layer images of A and B (applied once per HIT), wimg then holds C (if any) and the other layers.
  const unsigned char* wimg_a = nullptr;
  const unsigned char* wimg_b = nullptr;
  // ETX_PREC_INT8 (next row): per-layer weight scales S_w = max|W_l| / 127, and the integer codes of a 1-unit last
  // layer held as floats (the classifier's output unit is evaluated in the epilogue registers)
  float sw[kMaxLayers] = {0};
  const float* wq_last = nullptr;
};

struct Workspace {            // carved from the caller's buffer by carve_workspace()
  int32_t* plane_ptr = nullptr;   // [n_events * (n_planes+1)]
  int32_t* hit_event = nullptr;   // [n_hits]
  int32_t* cursor = nullptr;      // [n_hits] per-destination fill cursors of the graph build
  int32_t* scan_tmp = nullptr;    // block sums for the device scan
  int32_t* flags = nullptr;       // [8] validation flags / counters
  int32_t* sched = nullptr;       // [8] work counters of the dynamically scheduled kernels (scatter)
  uint32_t* ballots = nullptr;    // [n_hits][kBallotWords] vote words of the search's count pass (4-d embeddings)
  uint16_t* prefix16 = nullptr;   // [n_hits][kBallotWords] votes of the source in the words before each word
  int32_t* in_ptr3 = nullptr;     // [3 n_hits + 1] in-degree per (hit, plane gap 3/2/1), scanned into sub-list offsets
  float* h = nullptr;             // [n_hits, H]
  float* m = nullptr;             // [n_hits, 2H]
  float* p = nullptr;             // [n_hits, 2H] per-hit first-layer projections [A h | B h] (tensor-core modes)
  // host-path staging
  int32_t* s_event_ptr = nullptr; uint8_t* s_plane = nullptr;
  float *s_r = nullptr, *s_phi = nullptr, *s_z = nullptr, *s_x = nullptr, *s_y = nullptr;
  float* s_emb = nullptr;
  int32_t *s_row_ptr = nullptr, *s_src = nullptr, *s_dst = nullptr, *s_in_ptr = nullptr, *s_in_perm = nullptr;
  float* s_edge_enc = nullptr; float* s_scores = nullptr;
  size_t total = 0;
};

// ---- triplets.cu (next row: triplet building)
int launch_triplet_count(int n_hits, const int32_t* row_ptr, const int32_t* in_ptr, const int32_t* in_perm,
                         const float* scores, float score_min, int32_t* ptr /*[3][n_hits+1]*/, cudaStream_t s);
int launch_triplet_fill(int n_hits, const int32_t* row_ptr, const int32_t* in_ptr, const int32_t* in_perm,
                        const float* scores, float score_min, const int32_t* ptr, int32_t* first, int32_t* second,
                        cudaStream_t s);

}  // namespace etx

struct etx_ctx {
  etx_model_desc desc;
  int device = 0;
  int sm_count = 148;
  int hit_mode = -1;          // tensor-core mode of the per-hit MLPs (node encoder, node networks, projections) if not the context's
  float* d_weights = nullptr;      // transposed weights + biases, one allocation
  size_t d_weights_floats = 0;
  const float* d_zero_bias = nullptr;  // 128 zeros inside d_weights
  unsigned char* d_wimg = nullptr; // tensor-core weight images, one allocation
  etx::DevMlp emb, node_enc, edge_enc, cls;
  std::vector<etx::DevMlp> node_net, edge_net;
  void* ws = nullptr;
  size_t ws_bytes = 0;
  int64_t launches = 0;
  bool launch_refused = false;          // a launcher returned < 0 during the current API call (see check_cuda)
  std::string err;
  int* d_emb_wq = nullptr;              // INT8 codes of the embedding MLP's weights (next row), packed 4 per word
  int emb_wq_off[etx::kMaxLayers] = {0};
  float emb_sw[etx::kMaxLayers] = {0};  // their per-layer scales max|W| / 127
  // the same embedding for the tensor-core INT8 kernel (128-wide hidden layers): kind::i8 image of the hidden layers,
  // and the 3-input first layer / the narrow last layer as integer codes held in floats (k-major)
  unsigned char* d_emb_bf16_img = nullptr;  // single-pass bf16 image of the embedding's hidden layers (etx_embed_bf16)
  unsigned char* d_embq_img = nullptr;
  float* d_embq_f = nullptr;            // [3][128] first-layer codes, then [128][n_out] last-layer codes
  // next row: the two triplet classifiers (articulations, elbows), set by etx_set_triplet_classifiers
  float* d_trip_weights = nullptr;
  unsigned char* d_trip_wimg = nullptr;
  etx::DevMlp trip_art, trip_elb;
  bool have_trip = false;
  // next row: calibrated activation ranges of ETX_PREC_INT8, [n_mlps][gnn_n_layers] in the order node encoder, edge
  // encoder, (node network k, edge network k)..., classifier (etx_set_int8_ranges)
  std::vector<float> q_alpha;
  cudaStream_t copy_stream = nullptr;   // etx_infer_host: edge-list copy-out underneath the message passing
  cudaEvent_t copy_event = nullptr;
  // per-stage profiling (etx_profile_enable / etx_profile_read)
  bool prof_on = false;
  struct ProfRec { int cls; int n; cudaEvent_t a, b; };
  std::vector<ProfRec> prof_pending;
  std::vector<cudaEvent_t> prof_pool;
  double prof_ms[ETX_K_COUNT] = {0};
  int64_t prof_n[ETX_K_COUNT] = {0};
};

namespace etx {

// ---- graph.cu
struct GraphArgs {
  int n_events, n_hits, n_planes, d, gap;
  float r2_max;
  const int32_t* event_ptr; const uint8_t* plane; const float* emb;
};
// each returns the number of kernels launched; errors are reported through cudaGetLastError
int launch_plane_index(const GraphArgs& a, int32_t* plane_ptr, int32_t* hit_event, int32_t* flags, cudaStream_t s);
constexpr int kBallotWords = 32;   // vote words (32 candidates each) the count pass keeps per source for the fill pass
int launch_search_count(const GraphArgs& a, const int32_t* plane_ptr, const int32_t* hit_event,
                        int32_t* flags, int32_t* out_deg, int32_t* in_deg3, uint32_t* ballots /*[n_hits][kBallotWords] or null*/,
                        uint16_t* prefix16, cudaStream_t s);
int launch_search_kmax_cap(const GraphArgs& a, int k_max, const int32_t* plane_ptr, const int32_t* hit_event, int32_t* flags,
                           int32_t* out_deg, int32_t* in_deg3, uint32_t* ballots, uint16_t* prefix16, cudaStream_t s);
int launch_in_ptr_from3(int n_hits, const int32_t* in_ptr3, int32_t* in_ptr, cudaStream_t s);
int launch_exclusive_scan(int32_t* data /*[n+1], in place, data[n] = total*/, int n, int32_t* tmp, cudaStream_t s);
int launch_search_fill(const GraphArgs& a, const int32_t* plane_ptr, const int32_t* hit_event,
                       const int32_t* flags, const int32_t* row_ptr, int32_t* src, int32_t* dst,
                       const int32_t* in_ptr, int32_t* in_perm, int32_t* cursor /*[n_hits] scratch*/,
                       const uint32_t* ballots, const uint16_t* prefix16, const int32_t* in_ptr3, cudaStream_t s);
size_t scan_tmp_ints(int n);
int launch_add_offset(const int32_t* in, int32_t* out, int64_t n, int32_t offset, cudaStream_t s);
int launch_sort_in_lists(int n_hits, const int32_t* flags, const int32_t* in_ptr, int32_t* in_perm, cudaStream_t s);
// ---- graph_kmax.cu (next row: k_max-capped search)
int launch_kmax_count(const GraphArgs& a, int k_max, const int32_t* plane_ptr, const int32_t* hit_event,
                      const int32_t* flags, int32_t* out_deg, cudaStream_t s);
int launch_kmax_fill(const GraphArgs& a, int k_max, const int32_t* plane_ptr, const int32_t* hit_event,
                     const int32_t* flags, const int32_t* row_ptr, int32_t* src, int32_t* dst, cudaStream_t s);
int launch_kmax_in_count(const GraphArgs& a, int64_t n_edges, const int32_t* dst, int32_t* in_deg, cudaStream_t s);
int launch_kmax_in_fill(const GraphArgs& a, int64_t n_edges, const int32_t* flags, const int32_t* dst, const int32_t* in_ptr,
                        int32_t* in_perm, int32_t* cursor /*[n_hits] scratch*/, cudaStream_t s);

// ---- mlp_simt.cu
struct Segment {              // input row r, column k (k < width): base[(idx ? idx[r] : r) * ld + k]
  const float* base = nullptr; const int32_t* idx = nullptr; int width = 0; int ld = 0;
};
struct MlpArgs {
  int n_rows = 0;
  // first-layer input: either up to 3 gathered segments, or 3 features computed from SoA arrays
  int n_seg = 0; Segment seg[3];
  const float* feat[3] = {nullptr, nullptr, nullptr}; float fc[3] = {0, 0, 0}; float fs[3] = {1, 1, 1};
  // addend: the first layer's pre-activation starts from add[0][idx0[row]] + add[1][idx1[row]]
  // (128 columns each) instead of zero (tensor-core path only; n_add is 0 or 2)
  int n_add = 0; Segment add[2];
  int wide = 0;               // tensor-core path: one layer with 256 outputs (weight image = two 128-output images back to back)
  DevMlp mlp;
  // output: mode 0 store, 1 residual add (out = res + y; res may alias out), 2 small-N linear,
  // 3 small-N sigmoid
  int out_mode = 0; float* out = nullptr; const float* res = nullptr; int out_ld = 0;
  int emb_mode = -1;          // out_mode 2 (embedding): tensor-core mode to run instead of the default 3xTF32 (etx_embed_bf16)
  int tc_mode = -1;           // tensor-core mode of THIS launch if it differs from the context's (per-hit MLPs of ETX_PREC_BF16 run the split mode)
  float q_sa0 = 1.f; float q_sc[kMaxLayers] = {0}; float q_sn[kMaxLayers] = {0};   // ETX_PREC_INT8 scales (see TcArgs)
};
int launch_mlp_simt(const MlpArgs& a, cudaStream_t s);

// ---- mlp_tc.cu (tcgen05 tensor-core path)
struct TcArgs {
  int n_rows = 0;
  int n_seg = 0; Segment seg[3]; int K0 = 0;      // first-layer input: gathered segments, K0 = sum of widths (may be 0 with an addend)
  int n_add = 0; Segment add[2];                  // 0 or 2 addend sources: layer-1 accumulator starts from their sum
  // feature mode (w1 != null): operand of the first tensor-core layer = ReLU(w1^T f + b1), f = (feat - fc) / fs
  const float* feat[3] = {nullptr, nullptr, nullptr}; float fc[3] = {0, 0, 0}; float fs[3] = {1, 1, 1};
  const float* w1 = nullptr;                      // [3][128] fp32 (k-major), the MLP's own first layer
  const float* b1 = nullptr;                      // [128]
  int n_layers = 0;
  int wide = 0;                                   // one layer, two 128-column output halves per row tile (bf16 modes)
  const unsigned char* wimg = nullptr;            // weight image: swizzled 16 KB tiles in consumption order
  const float* bias[kMaxLayers] = {nullptr};
  const float* w_last = nullptr;                  // classifier: fp32 weights of the 1-unit output layer; narrow output: [128][n_out]
  int n_out = 1;                                  // units of a narrow output layer (out_mode 2)
  int out_mode = 0; float* out = nullptr; const float* res = nullptr; int out_ld = 0;
  // ETX_PREC_INT8 (next row): q_sa0 = scale of the first layer's input (the gather warps quantise with it); per GEMM
  // layer l: q_sc[l] = S_a S_w (de-quantisation), q_sn[l] = the NEXT layer's input scale (re-quantisation)
  float q_sa0 = 1.f; float q_sc[kMaxLayers] = {0}; float q_sn[kMaxLayers] = {0};
  float q_sf = 1.f, q_sc0 = 1.f;                  // feature mode (INT8 embedding): scale of the 3 features, S_a S_w of the MLP's own first layer
  float q_rsa0 = 1.f, q_rsn[kMaxLayers] = {0}, q_rsf = 1.f;   // fl(1 / scale) of q_sa0, q_sn[], q_sf (filled by launch_mlp_tc)
  unsigned long long* dbg = nullptr;              // optional [grid][16] cycle counters (ETX_TC_DEBUG)
  int exp_flags = 0;                              // developer builds only (-DETX_DEV_SWITCHES): timing experiments, wrong results
};
int launch_mlp_tc(const TcArgs& a, int mode, int sm_count, cudaStream_t s);
int tc_chunk_k(int mode);

// ---- tracks.cu (next row: score cut + weakly connected components)
int launch_wcc(int n_events, const int32_t* event_ptr, const int32_t* row_ptr, const int32_t* src,
               const int32_t* dst, const float* scores, float score_min, int32_t* labels, cudaStream_t s);

// ---- triplet_tracks.cu (next row: track building from triplets)
size_t triplet_tracks_ws_bytes(int n_hits, long long n_edges, long long n_art);
int run_triplet_tracks(int n_events, int n_hits, long long n_edges, const int32_t* event_ptr, const int32_t* row_ptr,
                       const int32_t* in_ptr, const int32_t* in_perm, const float* scores, float score_min,
                       const int32_t* tptr, const long long n_trip[3], const int32_t* first, const int32_t* second,
                       const float* tscores, float trip_min, char* ws, int32_t* d_edge_set, long long join_capacity,
                       int32_t* d_joins, long long track_capacity, int32_t* d_track_ptr, long long hit_capacity,
                       int32_t* d_track_hits, long long counts[4], bool* capacity_ok, cudaStream_t s);

// ---- q8_aux.cu (next row: ETX_PREC_INT8)
int launch_node_l1(int n_rows, int H, const float* const feat[3], const float fc[3], const float fs[3], const float* Wt,
                   const float* b, float* out, cudaStream_t s);

// ---- embed_int8.cu (next row: INT8 embedding MLP)
struct Int8Args {
  int n_rows = 0, n_layers = 0, n_out = 0;
  const float* feat[3] = {nullptr, nullptr, nullptr}; float fc[3] = {0, 0, 0}; float fs[3] = {1, 1, 1};
  const int* wq = nullptr;                 // packed int8 weight codes, per layer [out][ceil(in/4)] words
  int w_off[kMaxLayers] = {0};             // word offset of every layer inside wq
  const float* bias[kMaxLayers] = {nullptr};
  float sa[kMaxLayers] = {0};              // activation scale of every layer's input (alpha / 127)
  float sc[kMaxLayers] = {0};              // sa * weight scale
  float* out = nullptr;                    // [n_rows, n_out] fp32
};
int launch_embed_int8(const Int8Args& a, int H, cudaStream_t s);

// ---- scatter.cu
int launch_scatter(int n_nodes, int H, const int32_t* row_ptr, const int32_t* in_ptr,
                   const int32_t* in_perm, const float* e, float* m, int32_t* counter /*device, 1 int*/, cudaStream_t s);

#ifdef ETX_DEV_SWITCHES
int launch_scatter_atomic(int n_nodes, long long n_edges, int H, const int32_t* src, const int32_t* dst,
                          const float* e, float* m, cudaStream_t s);   // developer builds: the measured all-atomics alternative
#endif

}  // namespace etx
