// C ABI of libetx (include/etx.h): context, weight staging, workspace carving, and the launch
// sequences of the four path calls.  No arithmetic of the method happens on the host.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>

#include "common.cuh"

namespace etx {
namespace {

std::string g_create_error;

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

bool valid_width(int h) { return h == 64 || h == 128; }

const char* check_desc(const etx_model_desc* d) {
  if (!d) return "desc is NULL";
  if (d->emb_n_layers < 2 || d->emb_n_layers > kMaxLayers) return "emb_n_layers must be 2..8";
  if (d->emb_dims[0] != 3) return "embedding input must be the 3 features (r, phi, z)";
  for (int l = 1; l < d->emb_n_layers; ++l)
    if (!valid_width(d->emb_dims[l]) || d->emb_dims[l] != d->emb_dims[1])
      return "embedding hidden widths must all be 64 or all be 128";
  if (d->emb_dims[d->emb_n_layers] < 1 || d->emb_dims[d->emb_n_layers] > 8) return "embedding dim must be 1..8";
  if (!valid_width(d->gnn_hidden)) return "gnn_hidden must be 64 or 128";
  if (d->gnn_n_layers < 2 || d->gnn_n_layers > kMaxLayers) return "gnn_n_layers must be 2..8";
  if (d->n_iter < 0 || d->n_iter > 64) return "n_iter must be 0..64";
  if (d->n_planes < 2 || d->n_planes > 255) return "n_planes must be 2..255";
  if (d->precision < ETX_PREC_FP32 || d->precision > ETX_PREC_FP8) return "unknown precision";
  for (int i = 0; i < 5; ++i)
    if (!(d->norm_scale[i] != 0.0f)) return "norm_scale entries must be non-zero";
  return nullptr;
}

struct HostMlp { int n_layers; int dims[kMaxLayers + 1]; };

std::vector<HostMlp> mlp_list(const etx_model_desc& d) {
  std::vector<HostMlp> v;
  auto gnn = [&](int in, int out) {
    HostMlp m; m.n_layers = d.gnn_n_layers; m.dims[0] = in;
    for (int l = 1; l < d.gnn_n_layers; ++l) m.dims[l] = d.gnn_hidden;
    m.dims[d.gnn_n_layers] = out;
    return m;
  };
  HostMlp e; e.n_layers = d.emb_n_layers;
  for (int l = 0; l <= d.emb_n_layers; ++l) e.dims[l] = d.emb_dims[l];
  v.push_back(e);
  const int H = d.gnn_hidden;
  v.push_back(gnn(3, H));
  v.push_back(gnn(2 * H, H));
  for (int k = 0; k < d.n_iter; ++k) { v.push_back(gnn(3 * H, H)); v.push_back(gnn(3 * H, H)); }
  v.push_back(gnn(H, 1));
  return v;
}

size_t mlp_floats(const HostMlp& m) {
  size_t n = 0;
  for (int l = 0; l < m.n_layers; ++l) n += (size_t)m.dims[l] * m.dims[l + 1] + m.dims[l + 1];
  return n;
}

// Tensor-core weight image of the first n_gemm layers of an MLP (mlp_tc.cu): for every layer, for every
// K-chunk of one 128-byte swizzle atom (32 tf32 / 64 bf16 values), one 16 KB tile per piece laid out
// exactly as the canonical K-major SWIZZLE_128B shared-memory operand: row n (output neuron) at
// n*128 bytes, its 16-byte groups XOR-ed with (n & 7).  TF32X3 / BF16X3 store two pieces (hi, lo) per chunk.
uint16_t bf16_rne(float f) {
  uint32_t u; std::memcpy(&u, &f, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

float layer_weight_scale(const float* W, int fi, int fo, float qmax = 127.0f) {
  float mx = 0.0f;
  for (size_t i = 0; i < (size_t)fi * fo; ++i) mx = std::max(mx, std::fabs(W[i]));
  return mx / qmax;
}
// e4m3 (1-4-3, bias 7, no infinities, max 448): nearest value of a finite t, ties to even, saturating; and its byte code
float e4m3_round_host(float t) {
  const float a = std::fabs(t);
  if (!(a < 448.0f)) return t < 0.0f ? -448.0f : 448.0f;
  int e;
  std::frexp(a, &e);
  int le = (a == 0.0f) ? -6 : e - 1;
  if (le < -6) le = -6;
  const float ulp = std::ldexp(1.0f, le - 3);
  const float r = std::nearbyintf(a / ulp) * ulp;
  return t < 0.0f ? -r : r;
}
unsigned char e4m3_code_host(float t) {
  const float v = e4m3_round_host(t);
  const float a = std::fabs(v);
  unsigned char code;
  if (a == 0.0f) code = 0;
  else if (a < 0.015625f) code = (unsigned char)std::lround(a * 512.0f);               // subnormal: mantissa = a / 2^-9
  else {
    int e;
    const float m = std::frexp(a, &e);                                                // a = m 2^e, m in [0.5, 1)
    code = (unsigned char)(((e - 1 + 7) << 3) | (int)std::lround((m * 2.0f - 1.0f) * 8.0f));
  }
  return (unsigned char)(code | ((std::signbit(v) && a != 0.0f) ? 0x80 : 0));
}
int quant_code_host(float x, float S) {              // Eq. 4.33 with x / S evaluated as x * fl(1 / S) (DESIGN reading Q21)
  const float r = 1.0f / S;
  float q = std::nearbyintf(x * r);
  q = std::min(std::max(q, -127.0f), 127.0f);
  return (int)q;
}

// Appends the image of input columns [k_begin, k_end) of one layer W [fo = 128][fi] (row-major, fp32).
void append_wimg_slab(std::vector<unsigned char>& img, const float* W, int fi, int fo, int k_begin, int k_end, int mode) {
  const int KA = tc_chunk_k(mode);
  const int pieces = (mode == ETX_PREC_BF16 || mode == ETX_PREC_INT8 || mode == ETX_PREC_FP8) ? 1 : 2;
  if (mode == ETX_PREC_FP8) {
    // e4m3 codes: S_w = max|W| / 448 over the whole layer, code = e4m3(w * fl(1 / S_w)); layout as the INT8 image
    const float rs = 1.0f / layer_weight_scale(W, fi, fo, 448.0f);
    for (int k0 = k_begin; k0 < k_end; k0 += KA) {
      const size_t base = img.size();
      img.resize(base + 128 * 128, 0);
      for (int n = 0; n < fo; ++n)
        for (int kk = 0; kk < KA; ++kk)
          img[base + (size_t)n * 128 + (size_t)(((kk / 16) ^ (n & 7)) * 16) + (kk % 16)] = e4m3_code_host(W[(size_t)n * fi + k0 + kk] * rs);
    }
    return;
  }
  if (mode == ETX_PREC_INT8) {
    // INT8 codes (Eqs. 4.31-4.33): S_w = max|W| / 127 over the WHOLE layer (per-tensor scale), code =
    // clip(round(w / S_w)); one byte per weight, 128 codes per 128-byte row of the swizzled tile
    const float sw = layer_weight_scale(W, fi, fo);
    for (int k0 = k_begin; k0 < k_end; k0 += KA) {
      const size_t base = img.size();
      img.resize(base + 128 * 128, 0);
      for (int n = 0; n < fo; ++n)
        for (int kk = 0; kk < KA; ++kk) {
          const signed char q = (signed char)quant_code_host(W[(size_t)n * fi + k0 + kk], sw);
          img[base + (size_t)n * 128 + (size_t)(((kk / 16) ^ (n & 7)) * 16) + (kk % 16)] = (unsigned char)q;
        }
    }
    return;
  }
  for (int k0 = k_begin; k0 < k_end; k0 += KA) {
    const size_t base = img.size();
    img.resize(base + (size_t)pieces * 128 * 128, 0);
    for (int n = 0; n < fo; ++n)
      for (int kk = 0; kk < KA; ++kk) {
        const float v = W[(size_t)n * fi + k0 + kk];
        if (mode == ETX_PREC_TF32X3) {
          uint32_t u; std::memcpy(&u, &v, 4);
          const uint32_t hi_u = u & 0xffffe000u;
          float hi; std::memcpy(&hi, &hi_u, 4);
          const float lo = v - hi;
          const size_t off = (size_t)n * 128 + (size_t)(((kk / 4) ^ (n & 7)) * 16) + (kk % 4) * 4;
          std::memcpy(&img[base + off], &hi, 4);
          std::memcpy(&img[base + 128 * 128 + off], &lo, 4);
        } else {
          const uint16_t b = bf16_rne(v);
          const size_t off = (size_t)n * 128 + (size_t)(((kk / 8) ^ (n & 7)) * 16) + (kk % 8) * 2;
          std::memcpy(&img[base + off], &b, 2);
          if (pieces == 2) {                          // BF16X3: lo = bf16(w - hi)
            const uint32_t hu = (uint32_t)b << 16;
            float hf; std::memcpy(&hf, &hu, 4);
            const uint16_t lo = bf16_rne(v - hf);
            std::memcpy(&img[base + 128 * 128 + off], &lo, 2);
          }
        }
      }
  }
}

// Image of layers [l_begin, n_gemm) of an MLP; the first of them restricted to input columns >= k_first.
void append_wimg(std::vector<unsigned char>& img, const HostMlp& m, const float* w, int l_begin, int k_first,
                 int n_gemm, int mode) {
  const float* W = w;
  for (int l = 0; l < n_gemm; ++l) {
    const int fi = m.dims[l], fo = m.dims[l + 1];           // fo == 128
    if (l >= l_begin) append_wimg_slab(img, W, fi, fo, l == l_begin ? k_first : 0, fi, mode);
    W += (size_t)fi * fo + fo;
  }
}

Workspace carve(const etx_ctx* c, int32_t n_events, int32_t n_hits, int64_t cap, bool host_path, char* base) {
  Workspace w;
  size_t off = 0;
  auto take = [&](size_t bytes) { char* p = base ? base + off : nullptr; off += align_up(bytes ? bytes : 1, 256); return p; };
  const int L = c->desc.n_planes, H = c->desc.gnn_hidden, d = c->desc.emb_dims[c->desc.emb_n_layers];
  w.plane_ptr = (int32_t*)take(sizeof(int32_t) * (size_t)n_events * (L + 1));
  w.hit_event = (int32_t*)take(sizeof(int32_t) * (size_t)n_hits);
  w.cursor = (int32_t*)take(sizeof(int32_t) * (size_t)n_hits);
  w.scan_tmp = (int32_t*)take(sizeof(int32_t) * scan_tmp_ints(3 * n_hits + 1));
  w.flags = (int32_t*)take(sizeof(int32_t) * 8);
  w.sched = (int32_t*)take(sizeof(int32_t) * 8);
  if (d == 4) {
    w.ballots = (uint32_t*)take(sizeof(uint32_t) * (size_t)n_hits * kBallotWords);
    w.prefix16 = (uint16_t*)take(sizeof(uint16_t) * (size_t)n_hits * kBallotWords);
    w.in_ptr3 = (int32_t*)take(sizeof(int32_t) * ((size_t)3 * n_hits + 1));
  }
  w.h = (float*)take(sizeof(float) * (size_t)n_hits * H);
  w.m = (float*)take(sizeof(float) * (size_t)n_hits * 2 * H);
  if (c->desc.precision != ETX_PREC_FP32) w.p = (float*)take(sizeof(float) * (size_t)n_hits * 2 * H);
  if (host_path) {
    w.s_event_ptr = (int32_t*)take(sizeof(int32_t) * ((size_t)n_events + 1));
    w.s_plane = (uint8_t*)take((size_t)n_hits);
    w.s_r = (float*)take(sizeof(float) * (size_t)n_hits);
    w.s_phi = (float*)take(sizeof(float) * (size_t)n_hits);
    w.s_z = (float*)take(sizeof(float) * (size_t)n_hits);
    w.s_x = (float*)take(sizeof(float) * (size_t)n_hits);
    w.s_y = (float*)take(sizeof(float) * (size_t)n_hits);
    w.s_emb = (float*)take(sizeof(float) * (size_t)n_hits * d);
    w.s_row_ptr = (int32_t*)take(sizeof(int32_t) * ((size_t)n_hits + 1));
    w.s_in_ptr = (int32_t*)take(sizeof(int32_t) * ((size_t)n_hits + 1));
    w.s_src = (int32_t*)take(sizeof(int32_t) * (size_t)cap);
    w.s_dst = (int32_t*)take(sizeof(int32_t) * (size_t)cap);
    w.s_in_perm = (int32_t*)take(sizeof(int32_t) * (size_t)cap);
    w.s_edge_enc = (float*)take(sizeof(float) * (size_t)cap * H);
    w.s_scores = (float*)take(sizeof(float) * (size_t)cap);
  }
  w.total = off;
  return w;
}

etx_status fail(etx_ctx* c, etx_status st, const std::string& msg) {
  if (c) c->err = msg; else g_create_error = msg;
  return st;
}

etx_status check_cuda(etx_ctx* c, const char* where) {
  if (c && c->launch_refused) {
    c->launch_refused = false;
    return fail(c, ETX_ERR_INVALID, std::string(where) + ": a kernel launcher refused its arguments (unsupported layer "
                                    "shape, or an output buffer that is not 16-byte aligned)");
  }
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(c, ETX_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
  return ETX_OK;
}

etx_status need_ws(etx_ctx* c, const Workspace& probe) {
  if (!c->ws) return fail(c, ETX_ERR_NOMEM, "no workspace set (etx_set_workspace)");
  if (probe.total > c->ws_bytes)
    return fail(c, ETX_ERR_NOMEM, "workspace too small: need " + std::to_string(probe.total) + " bytes, have " +
                                      std::to_string(c->ws_bytes));
  return ETX_OK;
}

etx_status check_batch(etx_ctx* c, const etx_batch* b) {
  if (!b) return fail(c, ETX_ERR_INVALID, "batch is NULL");
  if (b->n_events < 0 || b->n_hits < 0) return fail(c, ETX_ERR_INVALID, "negative batch sizes");
  if (!b->d_event_ptr) return fail(c, ETX_ERR_INVALID, "d_event_ptr is NULL");
  if (b->n_hits > 0 && (!b->d_plane || !b->d_r || !b->d_phi || !b->d_z || !b->d_x || !b->d_y))
    return fail(c, ETX_ERR_INVALID, "batch array is NULL");
  return ETX_OK;
}

// Brackets a group of launches of one class with CUDA events when profiling is on.
struct ProfScope {
  etx_ctx* c; int cls; cudaStream_t s; int64_t l0; cudaEvent_t a = nullptr, b = nullptr;
  ProfScope(etx_ctx* c_, int cls_, cudaStream_t s_) : c(c_), cls(cls_), s(s_), l0(c_->launches) {
    if (!c->prof_on) return;
    a = take(); b = take();
    cudaEventRecord(a, s);
  }
  cudaEvent_t take() {
    if (!c->prof_pool.empty()) { cudaEvent_t e = c->prof_pool.back(); c->prof_pool.pop_back(); return e; }
    cudaEvent_t e; cudaEventCreate(&e); return e;
  }
  ~ProfScope() {
    if (!a) return;
    cudaEventRecord(b, s);
    c->prof_pending.push_back(etx_ctx::ProfRec{cls, (int)(c->launches - l0), a, b});
  }
};

// Precision dispatch.  MLPs with a tensor-core weight image run on tcgen05 (mlp_tc.cu).  In the tensor-core modes
// the embedding MLP runs the 3xTF32 chain whatever the GNN's mode (its result decides graph edges); like the node
// encoder, also fed by 3 raw features, it runs its first layer in the gather warps of the tensor-core kernel.
// ETX_PREC_FP32 runs every MLP in the exact fp32 FFMA kernel (mlp_simt.cu).
int run_mlp_raw(etx_ctx* c, const MlpArgs& a, cudaStream_t s);
// A launcher that refuses its arguments (unsupported shape, output not 16-byte aligned for the tensor map)
// must not pass silently: the refusal is recorded and the API call that asked for it returns ETX_ERR_INVALID.
int run_mlp(etx_ctx* c, const MlpArgs& a, cudaStream_t s) {
  const int n = run_mlp_raw(c, a, s);
  if (n < 0) { c->launch_refused = true; return 0; }
  return n;
}
int run_mlp_raw(etx_ctx* c, const MlpArgs& a, cudaStream_t s) {
  if ((c->desc.precision == ETX_PREC_FP32 && a.emb_mode < 0) || !a.mlp.wimg) return launch_mlp_simt(a, s);
  TcArgs t;
  t.n_rows = a.n_rows; t.n_seg = a.n_seg; t.K0 = a.mlp.dims[0];
  for (int i = 0; i < 3; ++i) t.seg[i] = a.seg[i];
  t.n_add = a.n_add; t.add[0] = a.add[0]; t.add[1] = a.add[1];
  t.n_layers = a.mlp.n_layers;
  t.wide = a.wide;
  t.wimg = a.mlp.wimg;
  for (int l = 0; l < a.mlp.n_layers; ++l) t.bias[l] = a.mlp.b[l];
  if (a.n_seg == 0 && a.n_add == 0) {
    // 3 raw features in (node encoder): the MLP's first layer runs in the gather warps, the tensor-core
    // chain is layers 2.. (the weight image starts at layer 2)
    for (int i = 0; i < 3; ++i) { t.feat[i] = a.feat[i]; t.fc[i] = a.fc[i]; t.fs[i] = a.fs[i]; }
    t.w1 = a.mlp.Wt[0]; t.b1 = a.mlp.b[0];
    t.K0 = a.mlp.dims[1];
    t.n_layers = a.mlp.n_layers - 1;
    for (int l = 0; l + 1 < a.mlp.n_layers; ++l) t.bias[l] = a.mlp.b[l + 1];
    t.n_out = a.mlp.dims[a.mlp.n_layers];
  }
  // the embedding (narrow linear output, out_mode 2) always runs the 3xTF32 kernel, whatever the GNN's mode:
  // its result decides graph edges (DESIGN.md section 5 "Embedding on the tensor cores")
  const int mode = (a.out_mode == 2) ? (a.emb_mode >= 0 ? a.emb_mode : (int)ETX_PREC_TF32X3)
                                     : (a.tc_mode >= 0 ? a.tc_mode : (int)c->desc.precision);
  t.w_last = a.mlp.Wt[a.mlp.n_layers - 1];         // [H][1] == [H]
  if (mode == ETX_PREC_INT8 || mode == ETX_PREC_FP8) {
    if (a.out_mode == 3) { if (!a.mlp.wq_last) return -1; t.w_last = a.mlp.wq_last; }
    t.q_sa0 = a.q_sa0;
    for (int l = 0; l < kMaxLayers; ++l) { t.q_sc[l] = a.q_sc[l]; t.q_sn[l] = a.q_sn[l]; }
  }
  t.out_mode = a.out_mode; t.out = a.out; t.res = a.res; t.out_ld = a.out_ld;
#ifdef ETX_DEV_SWITCHES
  static const char* expv = getenv("ETX_TC_EXP");                  // developer build: timing experiments (wrong results)
  t.exp_flags = (expv && a.out_mode != 2) ? atoi(expv) : 0;      // not the embedding: the graph must stay the real one
#endif
#ifdef ETX_DEV_SWITCHES
  if (getenv("ETX_TC_SYNC")) {                                     // developer build: localise a faulting launch
    const int n = launch_mlp_tc(t, mode, c->sm_count, s);
    const cudaError_t e = cudaStreamSynchronize(s);
    fprintf(stderr, "[tc sync] mode=%d rows=%d K0=%d n_add=%d wide=%d layers=%d out_mode=%d -> %d, %s\n", mode, t.n_rows, t.K0, t.n_add,
            t.wide, t.n_layers, t.out_mode, n, cudaGetErrorString(e));
    return n;
  }
#endif
#ifndef ETX_TC_COUNTERS
  return launch_mlp_tc(t, mode, c->sm_count, s);
#else
  static const bool debug = getenv("ETX_TC_DEBUG") != nullptr;     // developer build: per-role cycle counters
  if (!debug) return launch_mlp_tc(t, mode, c->sm_count, s);
  static unsigned long long* d_dbg = nullptr;
  if (!d_dbg) cudaMalloc(&d_dbg, sizeof(unsigned long long) * 32 * 256);
  cudaMemsetAsync(d_dbg, 0, sizeof(unsigned long long) * 32 * 256, s);
  t.dbg = d_dbg;
  const int n = launch_mlp_tc(t, mode, c->sm_count, s);
  std::vector<unsigned long long> h(32 * 256);
  cudaStreamSynchronize(s);
  cudaMemcpy(h.data(), d_dbg, h.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
  const int grid = std::min((a.n_rows + 127) / 128, c->sm_count);
  double avg[32] = {0};
  for (int b = 0; b < grid; ++b) for (int i = 0; i < 32; ++i) avg[i] += (double)h[b * 32 + i] / grid;
  const double tiles = (double)((a.n_rows + 127) / 128) / grid;
  fprintf(stderr, "[tc dbg] rows=%d K0=%d tiles/cta=%.1f | per tile cycles: mma total %.0f = wait acc_free %.0f + a_full %.0f + "
          "hid_ready %.0f + w_full %.0f + issue %.0f | epi: wait acc_full %.0f of %.0f [hid ld %.0f math %.0f st+arrive %.0f | fin ld %.0f fence %.0f io %.0f rdwait %.0f sts %.0f] | gather: wait a_empty %.0f of %.0f [data wait %.0f cvt+sts %.0f fence+arrive %.0f issue loads %.0f]\n",
          a.n_rows, a.mlp.dims[0], tiles, avg[5] / tiles, avg[0] / tiles, avg[1] / tiles, avg[2] / tiles, avg[3] / tiles, avg[4] / tiles,
          avg[6] / tiles, avg[7] / tiles, avg[10] / tiles, avg[11] / tiles, avg[12] / tiles, avg[13] / tiles, avg[14] / tiles, avg[15] / tiles, avg[20] / tiles, avg[21] / tiles, avg[8] / tiles, avg[9] / tiles, avg[16] / tiles, avg[17] / tiles, avg[18] / tiles, avg[19] / tiles);
  return n;
#endif
}

}  // namespace
}  // namespace etx

using namespace etx;

extern "C" {

size_t etx_weight_count(const etx_model_desc* desc) {
  if (check_desc(desc)) return 0;
  size_t n = 0;
  for (const HostMlp& m : mlp_list(*desc)) n += mlp_floats(m);
  return n;
}

etx_status etx_create(etx_ctx** out, const etx_model_desc* desc, const float* h_weights,
                      size_t n_weights, int device) {
  if (!out) return fail(nullptr, ETX_ERR_INVALID, "ctx out pointer is NULL");
  *out = nullptr;
  if (const char* why = check_desc(desc)) return fail(nullptr, ETX_ERR_INVALID, why);
  if (desc->precision != ETX_PREC_FP32 && desc->gnn_hidden != 128)
    return fail(nullptr, ETX_ERR_INVALID, "tensor-core precisions need gnn_hidden == 128");
  if (!h_weights || n_weights != etx_weight_count(desc))
    return fail(nullptr, ETX_ERR_INVALID, "weight blob size does not match desc (see etx_weight_count)");
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) {
    cudaGetLastError();
    return fail(nullptr, ETX_ERR_CUDA, "no such CUDA device (libetx has no CPU fallback)");
  }
  if (cudaSetDevice(device) != cudaSuccess) return fail(nullptr, ETX_ERR_CUDA, "cudaSetDevice failed");
  etx_ctx* c = new etx_ctx();
  c->desc = *desc;
  c->device = device;
  cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);

  // stage weights: per layer W^T [in][out] (k-major) then b, every array 256-byte aligned
  const std::vector<HostMlp> mlps = mlp_list(*desc);
  std::vector<float> staged;
  std::vector<DevMlp> dev(mlps.size());
  std::vector<std::vector<size_t>> offW(mlps.size()), offB(mlps.size());
  size_t src = 0;
  for (size_t i = 0; i < mlps.size(); ++i) {
    const HostMlp& m = mlps[i];
    dev[i].n_layers = m.n_layers;
    for (int l = 0; l <= m.n_layers; ++l) dev[i].dims[l] = m.dims[l];
    for (int l = 0; l < m.n_layers; ++l) {
      const int fi = m.dims[l], fo = m.dims[l + 1];
      staged.resize(align_up(staged.size(), 64));
      offW[i].push_back(staged.size());
      staged.resize(staged.size() + (size_t)fi * fo);
      float* Wt = staged.data() + offW[i].back();
      const float* W = h_weights + src;                  // [out][in]
      for (int o = 0; o < fo; ++o)
        for (int k = 0; k < fi; ++k) Wt[(size_t)k * fo + o] = W[(size_t)o * fi + k];
      src += (size_t)fi * fo;
      staged.resize(align_up(staged.size(), 64));
      offB[i].push_back(staged.size());
      staged.insert(staged.end(), h_weights + src, h_weights + src + fo);
      src += fo;
    }
  }
  staged.resize(align_up(staged.size(), 64));
  const size_t off_zero = staged.size();               // 128 zeros: bias of the per-hit projection launches
  staged.resize(staged.size() + 128, 0.0f);
  // ETX_PREC_INT8: per-layer weight scales of every GNN MLP, and the classifier's 1-unit output layer as integer codes
  // held in floats (evaluated in the epilogue registers: 128 products of codes sum exactly in fp32)
  const size_t off_clsq = staged.size();
  {
    size_t wsrc = 0;
    for (size_t i = 0; i < mlps.size(); ++i) {
      const float* W = h_weights + wsrc;
      for (int l = 0; l < mlps[i].n_layers; ++l) {
        const int fi = mlps[i].dims[l], fo = mlps[i].dims[l + 1];
        const bool fp8 = desc->precision == ETX_PREC_FP8;
        dev[i].sw[l] = layer_weight_scale(W, fi, fo, fp8 ? 448.0f : 127.0f);
        if (i + 1 == mlps.size() && l == mlps[i].n_layers - 1)
          for (int k = 0; k < fi; ++k)
            staged.push_back(fp8 ? e4m3_round_host(W[k] * (1.0f / dev[i].sw[l])) : (float)quant_code_host(W[k], dev[i].sw[l]));
        W += (size_t)fi * fo + fo;
      }
      wsrc += mlp_floats(mlps[i]);
    }
  }
  c->d_weights_floats = staged.size();
  if (cudaMalloc(&c->d_weights, staged.size() * sizeof(float)) != cudaSuccess ||
      cudaMemcpy(c->d_weights, staged.data(), staged.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess) {
    const std::string msg = std::string("weight upload failed: ") + cudaGetErrorString(cudaGetLastError());
    if (c->d_weights) cudaFree(c->d_weights);
    delete c;
    return fail(nullptr, ETX_ERR_CUDA, msg);
  }
  for (size_t i = 0; i < mlps.size(); ++i)
    for (int l = 0; l < mlps[i].n_layers; ++l) {
      dev[i].Wt[l] = c->d_weights + offW[i][l];
      dev[i].b[l] = c->d_weights + offB[i][l];
    }
  c->d_zero_bias = c->d_weights + off_zero;
  c->emb = dev[0];
  c->node_enc = dev[1];
  c->edge_enc = dev[2];
  for (int k = 0; k < desc->n_iter; ++k) { c->node_net.push_back(dev[3 + 2 * k]); c->edge_net.push_back(dev[4 + 2 * k]); }
  c->cls = dev.back();
  c->cls.wq_last = c->d_weights + off_clsq;
  {
    // next row: INT8 codes of the embedding MLP's weights (Eqs. 4.31-4.33): S_w = max|W| / 127,
    // w_q = clip(round(W / S_w), -127, 127), packed 4 consecutive inputs per word, rows padded with zeros
    const HostMlp& m = mlps[0];
    std::vector<int> codes;
    const float* W = h_weights;
    for (int l = 0; l < m.n_layers; ++l) {
      const int fi = m.dims[l], fo = m.dims[l + 1], kw = (fi + 3) / 4;
      float mx = 0.0f;
      for (size_t i = 0; i < (size_t)fi * fo; ++i) mx = std::max(mx, std::fabs(W[i]));
      const float sw = mx / 127.0f;
      c->emb_sw[l] = sw;
      c->emb_wq_off[l] = (int)codes.size();
      codes.resize(codes.size() + (size_t)fo * kw, 0);
      for (int o = 0; o < fo; ++o)
        for (int k = 0; k < fi; ++k) {
          float q = std::nearbyintf(W[(size_t)o * fi + k] * (1.0f / sw));
          q = std::min(std::max(q, -127.0f), 127.0f);
          codes[c->emb_wq_off[l] + (size_t)o * kw + k / 4] |= (int)(((unsigned)(int)q & 0xffu) << (8 * (k % 4)));
        }
      W += (size_t)fi * fo + fo;
    }
    if (cudaMalloc(&c->d_emb_wq, codes.size() * sizeof(int)) != cudaSuccess ||
        cudaMemcpy(c->d_emb_wq, codes.data(), codes.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
      const std::string msg = std::string("int8 weight upload failed: ") + cudaGetErrorString(cudaGetLastError());
      etx_destroy(c);
      return fail(nullptr, ETX_ERR_CUDA, msg);
    }
  }
  if (mlps[0].n_layers >= 3 && mlps[0].dims[1] == 128) {
    // INT8 embedding on the tensor cores (etx_embed_int8): kind::i8 image of layers 2..L-1, float-held codes of the
    // 3-input first layer [k][128] and of the narrow last layer [k][n_out]
    const HostMlp& m = mlps[0];
    std::vector<unsigned char> qimg;
    append_wimg(qimg, m, h_weights, 1, 0, m.n_layers - 1, ETX_PREC_INT8);
    const int n_out = m.dims[m.n_layers];
    std::vector<float> qf((size_t)3 * 128 + (size_t)128 * n_out);
    const float* W = h_weights;
    for (int o = 0; o < 128; ++o)
      for (int k = 0; k < 3; ++k) qf[(size_t)k * 128 + o] = (float)quant_code_host(W[(size_t)o * 3 + k], c->emb_sw[0]);
    for (int l = 0; l + 1 < m.n_layers; ++l) W += (size_t)m.dims[l] * m.dims[l + 1] + m.dims[l + 1];
    for (int o = 0; o < n_out; ++o)
      for (int k = 0; k < 128; ++k) qf[(size_t)3 * 128 + (size_t)k * n_out + o] = (float)quant_code_host(W[(size_t)o * 128 + k], c->emb_sw[m.n_layers - 1]);
    if (cudaMalloc(&c->d_embq_img, qimg.size()) != cudaSuccess ||
        cudaMemcpy(c->d_embq_img, qimg.data(), qimg.size(), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMalloc(&c->d_embq_f, qf.size() * sizeof(float)) != cudaSuccess ||
        cudaMemcpy(c->d_embq_f, qf.data(), qf.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess) {
      const std::string msg = std::string("int8 embedding image upload failed: ") + cudaGetErrorString(cudaGetLastError());
      etx_destroy(c);
      return fail(nullptr, ETX_ERR_CUDA, msg);
    }
  }
  if (mlps[0].n_layers >= 3 && mlps[0].dims[1] == 128) {
    // report-only bf16 embedding (etx_embed_bf16, reading Q16): single-pass bf16 image of layers 2..L-1
    std::vector<unsigned char> bimg;
    append_wimg(bimg, mlps[0], h_weights, 1, 0, mlps[0].n_layers - 1, ETX_PREC_BF16);
    if (cudaMalloc(&c->d_emb_bf16_img, bimg.size()) != cudaSuccess ||
        cudaMemcpy(c->d_emb_bf16_img, bimg.data(), bimg.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
      const std::string msg = std::string("bf16 embedding image upload failed: ") + cudaGetErrorString(cudaGetLastError());
      etx_destroy(c);
      return fail(nullptr, ETX_ERR_CUDA, msg);
    }
  }
  if (desc->precision != ETX_PREC_FP32) {
    // tensor-core weight images: edge encoder, node/edge networks, classifier (first-layer input a multiple of
    // the chunk); node encoder and a 128-wide embedding with >= 2 hidden layers from their second layer on (their
    // 3-feature first layer is computed in the gather warps).  Other embeddings keep the FFMA kernel.
    std::vector<unsigned char> img;
    std::vector<size_t> img_off(mlps.size(), (size_t)-1), img_a(mlps.size(), (size_t)-1), img_b(mlps.size(), (size_t)-1);
    const int H = desc->gnn_hidden, mode = desc->precision;
    // ETX_PREC_BF16: the per-HIT MLPs (node encoder, node networks, the per-hit projections of the edge MLPs' first layers)
    // run the fp32-equivalent split mode -- they cost N rows, not E, and h carries the largest values of the network --
    // the per-EDGE chains stay single-pass bf16
    const int hit_mode = (mode == ETX_PREC_BF16) ? (int)ETX_PREC_BF16X3 : mode;
    c->hit_mode = (hit_mode != mode) ? hit_mode : -1;
    size_t wsrc = 0;
    for (size_t i = 0; i < mlps.size(); ++i) {
      const float* w = h_weights + wsrc;
#ifdef ETX_DEV_SWITCHES
      const bool emb_ffma = getenv("ETX_EMBED_FFMA") != nullptr;   // developer build: keep the exact FFMA embedding
#else
      const bool emb_ffma = false;
#endif
      if (i == 0 && mlps[i].n_layers >= 3 && mlps[i].dims[1] == 128 && !emb_ffma) {
        // embedding: layers 2..L-1 as 3xTF32 MMA chain (layer 1 in the gather warps, the narrow last layer in the epilogue)
        img_off[i] = img.size();
        append_wimg(img, mlps[i], w, 1, 0, mlps[i].n_layers - 1, ETX_PREC_TF32X3);
      }
      if (i == 1 && mlps[i].n_layers >= 2) {             // node encoder: layers 2.. (layer 1 runs in the gather warps)
        img_off[i] = img.size();
        append_wimg(img, mlps[i], w, 1, 0, mlps[i].n_layers, hit_mode);
      }
      if (i >= 2) {
        const bool is_cls = (i + 1 == mlps.size());
        const bool is_node = !is_cls && i >= 3 && ((i - 3) % 2 == 0);
        if (is_cls || is_node) {
          img_off[i] = img.size();
          append_wimg(img, mlps[i], w, 0, 0, is_cls ? mlps[i].n_layers - 1 : mlps[i].n_layers, hit_mode);
        } else {
          // edge encoder ([h_src | h_dst]) and edge networks ([h_src | h_dst | e]): first layer factorised
          // into the per-hit parts A (columns [0,H)), B ([H,2H)) and the per-edge part C ([2H,3H), networks only)
          const int fi = mlps[i].dims[0];
          img_a[i] = img.size(); append_wimg_slab(img, w, fi, H, 0, H, hit_mode);
          img_b[i] = img.size(); append_wimg_slab(img, w, fi, H, H, 2 * H, hit_mode);
          img_off[i] = img.size();
          if (fi > 2 * H) append_wimg(img, mlps[i], w, 0, 2 * H, mlps[i].n_layers, mode);
          else append_wimg(img, mlps[i], w, 1, 0, mlps[i].n_layers, mode);
        }
      }
      wsrc += mlp_floats(mlps[i]);
    }
    if (cudaMalloc(&c->d_wimg, img.size()) != cudaSuccess ||
        cudaMemcpy(c->d_wimg, img.data(), img.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
      const std::string msg = std::string("weight image upload failed: ") + cudaGetErrorString(cudaGetLastError());
      etx_destroy(c);
      return fail(nullptr, ETX_ERR_CUDA, msg);
    }
    auto place = [&](DevMlp& m, size_t i) {
      m.wimg = c->d_wimg + img_off[i];
      if (img_a[i] != (size_t)-1) { m.wimg_a = c->d_wimg + img_a[i]; m.wimg_b = c->d_wimg + img_b[i]; }
    };
    if (img_off[0] != (size_t)-1) place(c->emb, 0);
    place(c->node_enc, 1);
    place(c->edge_enc, 2);
    for (int k = 0; k < desc->n_iter; ++k) { place(c->node_net[k], 3 + 2 * k); place(c->edge_net[k], 4 + 2 * k); }
    place(c->cls, mlps.size() - 1);
  }
  *out = c;
  return ETX_OK;
}

etx_status etx_destroy(etx_ctx* c) {
  if (!c) return ETX_OK;
  cudaSetDevice(c->device);
  if (c->d_weights) cudaFree(c->d_weights);
  if (c->d_wimg) cudaFree(c->d_wimg);
  if (c->d_emb_wq) cudaFree(c->d_emb_wq);
  if (c->d_embq_img) cudaFree(c->d_embq_img);
  if (c->d_emb_bf16_img) cudaFree(c->d_emb_bf16_img);
  if (c->d_embq_f) cudaFree(c->d_embq_f);
  if (c->d_trip_weights) cudaFree(c->d_trip_weights);
  if (c->d_trip_wimg) cudaFree(c->d_trip_wimg);
  for (const etx_ctx::ProfRec& r : c->prof_pending) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  for (cudaEvent_t e : c->prof_pool) cudaEventDestroy(e);
  if (c->copy_stream) { cudaStreamDestroy(c->copy_stream); cudaEventDestroy(c->copy_event); }
  delete c;
  return ETX_OK;
}

const char* etx_last_error(const etx_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

size_t etx_workspace_bytes(const etx_ctx* c, int32_t n_events, int32_t n_hits, int64_t edge_capacity,
                           int with_host_path) {
  if (!c || n_events < 0 || n_hits < 0 || edge_capacity < 0) return 0;
  return carve(c, n_events, n_hits, edge_capacity, with_host_path != 0, nullptr).total;
}

etx_status etx_set_workspace(etx_ctx* c, void* d_workspace, size_t bytes) {
  if (!c) return ETX_ERR_INVALID;
  if (((uintptr_t)d_workspace & 255) != 0) return fail(c, ETX_ERR_INVALID, "workspace must be 256-byte aligned");
  c->ws = d_workspace;
  c->ws_bytes = d_workspace ? bytes : 0;
  return ETX_OK;
}

int64_t etx_launch_count(const etx_ctx* c) { return c ? c->launches : 0; }

etx_status etx_profile_enable(etx_ctx* c, int on) {
  if (!c) return ETX_ERR_INVALID;
  c->prof_on = on != 0;
  return ETX_OK;
}

etx_status etx_profile_read(etx_ctx* c, double* ms, int64_t* launches) {
  if (!c) return ETX_ERR_INVALID;
  cudaSetDevice(c->device);
  for (const etx_ctx::ProfRec& r : c->prof_pending) {
    float t = 0.f;
    if (cudaEventSynchronize(r.b) != cudaSuccess || cudaEventElapsedTime(&t, r.a, r.b) != cudaSuccess)
      return check_cuda(c, "etx_profile_read");
    c->prof_ms[r.cls] += t;
    c->prof_n[r.cls] += r.n;
    c->prof_pool.push_back(r.a);
    c->prof_pool.push_back(r.b);
  }
  c->prof_pending.clear();
  for (int i = 0; i < ETX_K_COUNT; ++i) {
    if (ms) ms[i] = c->prof_ms[i];
    if (launches) launches[i] = c->prof_n[i];
    c->prof_ms[i] = 0; c->prof_n[i] = 0;
  }
  return ETX_OK;
}

etx_status etx_set_int8_ranges(etx_ctx* c, const float* h_alpha, size_t n) {
  if (!c) return ETX_ERR_INVALID;
  const size_t need = (size_t)(3 + 2 * c->desc.n_iter) * c->desc.gnn_n_layers;
  if (!h_alpha || n != need) return fail(c, ETX_ERR_INVALID, "etx_set_int8_ranges needs (3 + 2 n_iter) x gnn_n_layers ranges");
  for (size_t i = 0; i < n; ++i)
    if (!(h_alpha[i] > 0.0f)) return fail(c, ETX_ERR_INVALID, "activation ranges must be positive");
  c->q_alpha.assign(h_alpha, h_alpha + n);
  return ETX_OK;
}

// ETX_PREC_INT8: scales of one launch covering layers [shift, shift + n_l) of GNN MLP number mi (order of etx_set_int8_ranges)
static void fill_q(const etx_ctx* c, MlpArgs& a, int mi, const DevMlp& full, int shift, int n_l) {
  const int L = c->desc.gnn_n_layers;
  const float* al = c->q_alpha.data() + (size_t)mi * L;
  const float qmax = c->desc.precision == ETX_PREC_FP8 ? 448.0f : 127.0f;     // the range maps to the grid's largest value
  a.q_sa0 = al[shift] / qmax;
  for (int l = 0; l < n_l; ++l) {
    const float sa = al[shift + l] / qmax;
    a.q_sc[l] = sa * full.sw[shift + l];
    a.q_sn[l] = (shift + l + 1 < L) ? al[shift + l + 1] / qmax : 1.0f;
  }
}

etx_status etx_embed(etx_ctx* c, const etx_batch* b, float* d_emb, void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (etx_status st = check_batch(c, b)) return st;
  if (b->n_hits > 0 && !d_emb) return fail(c, ETX_ERR_INVALID, "d_emb is NULL");
  cudaSetDevice(c->device);
  MlpArgs a;
  a.n_rows = b->n_hits;
  a.n_seg = 0;
  a.feat[0] = b->d_r; a.feat[1] = b->d_phi; a.feat[2] = b->d_z;
  for (int i = 0; i < 3; ++i) { a.fc[i] = c->desc.norm_center[i]; a.fs[i] = c->desc.norm_scale[i]; }
  a.mlp = c->emb;
  a.out_mode = 2;
  a.out = d_emb;
  a.out_ld = c->emb.dims[c->emb.n_layers];
  {
    ProfScope ps(c, ETX_K_EMBED, (cudaStream_t)stream);
    c->launches += run_mlp(c, a, (cudaStream_t)stream);
  }
  return check_cuda(c, "etx_embed");
}

etx_status etx_embed_bf16(etx_ctx* c, const etx_batch* b, float* d_emb, void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (etx_status st = check_batch(c, b)) return st;
  if (b->n_hits > 0 && !d_emb) return fail(c, ETX_ERR_INVALID, "d_emb is NULL");
  if (!c->d_emb_bf16_img) return fail(c, ETX_ERR_INVALID, "the bf16 embedding needs 128-wide hidden layers (two or more)");
  cudaSetDevice(c->device);
  MlpArgs a;
  a.n_rows = b->n_hits;
  a.n_seg = 0;
  a.feat[0] = b->d_r; a.feat[1] = b->d_phi; a.feat[2] = b->d_z;
  for (int i = 0; i < 3; ++i) { a.fc[i] = c->desc.norm_center[i]; a.fs[i] = c->desc.norm_scale[i]; }
  a.mlp = c->emb;
  a.mlp.wimg = c->d_emb_bf16_img;
  a.emb_mode = ETX_PREC_BF16;
  a.out_mode = 2;
  a.out = d_emb;
  a.out_ld = c->emb.dims[c->emb.n_layers];
  {
    ProfScope ps(c, ETX_K_EMBED, (cudaStream_t)stream);
    c->launches += run_mlp(c, a, (cudaStream_t)stream);
  }
  return check_cuda(c, "etx_embed_bf16");
}

etx_status etx_embed_int8(etx_ctx* c, const etx_batch* b, const float* h_act_alpha, int32_t n_alpha, float* d_emb,
                          void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (etx_status st = check_batch(c, b)) return st;
  if (b->n_hits > 0 && !d_emb) return fail(c, ETX_ERR_INVALID, "d_emb is NULL");
  const int L = c->emb.n_layers;
  if (!h_act_alpha || n_alpha != L) return fail(c, ETX_ERR_INVALID, "act_alpha needs one calibrated range per embedding layer");
  for (int l = 0; l < L; ++l)
    if (!(h_act_alpha[l] > 0.0f)) return fail(c, ETX_ERR_INVALID, "activation ranges must be positive");
  cudaSetDevice(c->device);
  Int8Args a;
  a.n_rows = b->n_hits; a.n_layers = L; a.n_out = c->emb.dims[L];
  a.feat[0] = b->d_r; a.feat[1] = b->d_phi; a.feat[2] = b->d_z;
  for (int i = 0; i < 3; ++i) { a.fc[i] = c->desc.norm_center[i]; a.fs[i] = c->desc.norm_scale[i]; }
  a.wq = c->d_emb_wq;
  for (int l = 0; l < L; ++l) {
    a.w_off[l] = c->emb_wq_off[l];
    a.bias[l] = c->emb.b[l];
    a.sa[l] = h_act_alpha[l] / 127.0f;
    a.sc[l] = a.sa[l] * c->emb_sw[l];
  }
  a.out = d_emb;
  if (c->d_embq_img) {
    // 128-wide hidden layers: the tcgen05 kernel -- first layer in exact integer arithmetic in the gather warps, hidden
    // layers as kind::i8 MMAs, the narrow last layer in the epilogue registers (mlp_tc.cu); same codes, same result
    TcArgs t;
    t.n_rows = b->n_hits; t.K0 = 128;
    for (int i = 0; i < 3; ++i) { t.feat[i] = a.feat[i]; t.fc[i] = a.fc[i]; t.fs[i] = a.fs[i]; }
    t.w1 = c->d_embq_f; t.b1 = c->emb.b[0];
    t.n_layers = L - 1;
    for (int l = 0; l + 1 < L; ++l) t.bias[l] = c->emb.b[l + 1];
    t.n_out = c->emb.dims[L];
    t.wimg = c->d_embq_img;
    t.w_last = c->d_embq_f + 3 * 128;
    t.out_mode = 2; t.out = d_emb; t.out_ld = c->emb.dims[L];
    t.q_sf = a.sa[0]; t.q_sc0 = a.sc[0]; t.q_sa0 = a.sa[1];
    for (int l = 0; l + 1 < L; ++l) { t.q_sc[l] = a.sc[l + 1]; t.q_sn[l] = (l + 2 < L) ? a.sa[l + 2] : 1.0f; }
    ProfScope ps(c, ETX_K_EMBED, (cudaStream_t)stream);
    const int n = launch_mlp_tc(t, ETX_PREC_INT8, c->sm_count, (cudaStream_t)stream);
    if (n < 0) return fail(c, ETX_ERR_INVALID, "the INT8 tensor-core embedding refused its arguments");
    c->launches += n;
    return check_cuda(c, "etx_embed_int8");
  }
  {
    ProfScope ps(c, ETX_K_EMBED, (cudaStream_t)stream);
    const int n = launch_embed_int8(a, c->emb.dims[1], (cudaStream_t)stream);
    if (n < 0) return fail(c, ETX_ERR_INVALID, "unsupported embedding width for the INT8 path");
    c->launches += n;
  }
  return check_cuda(c, "etx_embed_int8");
}

etx_status etx_build_graph(etx_ctx* c, const etx_batch* b, const float* d_emb, float r2_max,
                           int32_t max_plane_gap, int32_t k_max, etx_graph* g, void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (etx_status st = check_batch(c, b)) return st;
  if (!g || !g->d_row_ptr || !g->d_in_ptr) return fail(c, ETX_ERR_INVALID, "graph or its offset arrays are NULL");
  if (k_max < 0) return fail(c, ETX_ERR_INVALID, "k_max must be >= 0 (0 = no cap)");
  if (max_plane_gap < 1) return fail(c, ETX_ERR_INVALID, "max_plane_gap must be >= 1");
  if (b->n_hits > 0 && !d_emb) return fail(c, ETX_ERR_INVALID, "d_emb is NULL");
  if (c->emb.dims[c->emb.n_layers] == 4 && ((uintptr_t)d_emb & 15))
    return fail(c, ETX_ERR_INVALID, "d_emb must be 16-byte aligned for a 4-dimensional embedding (vector loads)");
  if (max_plane_gap > c->desc.n_planes - 1) max_plane_gap = c->desc.n_planes - 1;   // larger gaps reach no plane; keeps p + gap in range
  if (g->edge_capacity < 0 || (g->edge_capacity > 0 && (!g->d_src || !g->d_dst || !g->d_in_perm)))
    return fail(c, ETX_ERR_INVALID, "edge arrays are NULL");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  if (etx_status st = need_ws(c, carve(c, b->n_events, b->n_hits, 0, false, nullptr))) return st;
  const Workspace w = carve(c, b->n_events, b->n_hits, 0, false, (char*)c->ws);
  GraphArgs a;
  a.n_events = b->n_events; a.n_hits = b->n_hits; a.n_planes = c->desc.n_planes;
  a.d = c->emb.dims[c->emb.n_layers]; a.gap = max_plane_gap; a.r2_max = r2_max;
  a.event_ptr = b->d_event_ptr; a.plane = b->d_plane; a.emb = d_emb;

  // A 4-d embedding runs the tiled search (graph.cu): count pass with kept vote words and per-(hit, plane gap) in-degrees,
  // for k_max > 0 a cap kernel that clears the votes beyond the k_max nearest, scans, and one fill pass that writes src, dst
  // and the by-destination lists at their final positions.  Other dimensions, or a window with more candidates than vote
  // words are kept (flags[1]), use the one-warp-per-source kernels (graph.cu / graph_kmax.cu: cursor atomics + in-list sort).
  bool tiled = a.d == 4 && w.ballots;
  int32_t host[3] = {0, 0, 0};
  for (int attempt = 0; attempt < 2; ++attempt) {
    {
      ProfScope ps(c, ETX_K_GRAPH, s);
      c->launches += launch_plane_index(a, w.plane_ptr, w.hit_event, w.flags, s);
      if (tiled) {
        c->launches += launch_search_count(a, w.plane_ptr, w.hit_event, w.flags, g->d_row_ptr, w.in_ptr3, w.ballots, w.prefix16, s);
        if (k_max > 0)
          c->launches += launch_search_kmax_cap(a, k_max, w.plane_ptr, w.hit_event, w.flags, g->d_row_ptr, w.in_ptr3, w.ballots, w.prefix16, s);
        c->launches += launch_exclusive_scan(g->d_row_ptr, b->n_hits + 1, w.scan_tmp, s);
        c->launches += launch_exclusive_scan(w.in_ptr3, 3 * b->n_hits + 1, w.scan_tmp, s);
        c->launches += launch_in_ptr_from3(b->n_hits, w.in_ptr3, g->d_in_ptr, s);
      } else if (k_max == 0) {
        c->launches += launch_search_count(a, w.plane_ptr, w.hit_event, w.flags, g->d_row_ptr, g->d_in_ptr, nullptr, nullptr, s);
        c->launches += launch_exclusive_scan(g->d_row_ptr, b->n_hits + 1, w.scan_tmp, s);
        c->launches += launch_exclusive_scan(g->d_in_ptr, b->n_hits + 1, w.scan_tmp, s);
      } else {                                       // next row: capped search (graph_kmax.cu)
        c->launches += launch_kmax_count(a, k_max, w.plane_ptr, w.hit_event, w.flags, g->d_row_ptr, s);
        c->launches += launch_exclusive_scan(g->d_row_ptr, b->n_hits + 1, w.scan_tmp, s);
      }
    }
    cudaMemcpyAsync(&host[0], w.flags, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, s);
    cudaMemcpyAsync(&host[2], g->d_row_ptr + b->n_hits, sizeof(int32_t), cudaMemcpyDeviceToHost, s);
    if (cudaStreamSynchronize(s) != cudaSuccess) return check_cuda(c, "etx_build_graph (count)");
    if (etx_status st = check_cuda(c, "etx_build_graph (count)")) return st;
    if (tiled && host[1] != 0 && !(host[0] & 3)) { tiled = false; continue; }   // a window longer than the kept vote words: redo
    break;
  }
  if (host[0] & 1) return fail(c, ETX_ERR_INVALID, "malformed batch: event_ptr not monotone / plane id >= n_planes");
  if (host[0] & 2) return fail(c, ETX_ERR_UNSORTED, "hits of an event are not sorted by plane");
  g->n_edges = host[2];
  if (g->n_edges > g->edge_capacity)
    return fail(c, ETX_ERR_CAPACITY, "graph needs " + std::to_string(g->n_edges) + " edges, capacity " +
                                         std::to_string(g->edge_capacity));
  if (k_max > 0 && !tiled) {
    // the by-destination lists depend on which edges survived the cap: forward fill first, then in-degrees,
    // scan, and the incoming side from the capped edge list
    ProfScope ps(c, ETX_K_GRAPH, s);
    if (g->n_edges > 0)
      c->launches += launch_kmax_fill(a, k_max, w.plane_ptr, w.hit_event, w.flags, g->d_row_ptr, g->d_src, g->d_dst, s);
    c->launches += launch_kmax_in_count(a, g->n_edges, g->d_dst, g->d_in_ptr, s);
    c->launches += launch_exclusive_scan(g->d_in_ptr, b->n_hits + 1, w.scan_tmp, s);
    c->launches += launch_kmax_in_fill(a, g->n_edges, w.flags, g->d_dst, g->d_in_ptr, g->d_in_perm, w.cursor, s);
  } else if (g->n_edges > 0) {
    ProfScope ps(c, ETX_K_GRAPH, s);
    c->launches += launch_search_fill(a, w.plane_ptr, w.hit_event, w.flags, g->d_row_ptr, g->d_src, g->d_dst,
                                      g->d_in_ptr, g->d_in_perm, w.cursor, tiled ? w.ballots : nullptr, w.prefix16, w.in_ptr3, s);
  }
  return check_cuda(c, "etx_build_graph (fill)");
}

etx_status etx_gnn_forward(etx_ctx* c, const etx_batch* b, const etx_graph* g, float* d_edge_enc,
                           float* d_hit_enc, void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (etx_status st = check_batch(c, b)) return st;
  if (!g || g->n_edges < 0 || g->n_edges > g->edge_capacity) return fail(c, ETX_ERR_INVALID, "graph is NULL or not built");
  if (g->n_edges > 0 && !d_edge_enc) return fail(c, ETX_ERR_INVALID, "d_edge_enc is NULL");
  if (((uintptr_t)d_edge_enc & 15) || ((uintptr_t)d_hit_enc & 15))
    return fail(c, ETX_ERR_INVALID, "d_edge_enc / d_hit_enc must be 16-byte aligned (vector and TMA accesses)");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  if (etx_status st = need_ws(c, carve(c, b->n_events, b->n_hits, 0, false, nullptr))) return st;
  const Workspace w = carve(c, b->n_events, b->n_hits, 0, false, (char*)c->ws);
  const int H = c->desc.gnn_hidden, N = b->n_hits;
  const int E = (int)g->n_edges;

  const bool q8 = c->desc.precision == ETX_PREC_INT8 || c->desc.precision == ETX_PREC_FP8;   // 8-bit operands, static ranges
  if (q8 && c->q_alpha.empty()) return fail(c, ETX_ERR_INVALID, "ETX_PREC_INT8 / ETX_PREC_FP8 need calibrated ranges (etx_set_int8_ranges)");
  {  // a3: h0 = MLP_n((x,y,z) normalised)
    MlpArgs a;
    a.n_rows = N; a.n_seg = 0;
    a.feat[0] = b->d_x; a.feat[1] = b->d_y; a.feat[2] = b->d_z;
    const int id[3] = {3, 4, 2};
    for (int i = 0; i < 3; ++i) { a.fc[i] = c->desc.norm_center[id[i]]; a.fs[i] = c->desc.norm_scale[id[i]]; }
    a.mlp = c->node_enc; a.out_mode = 0; a.out = w.h; a.out_ld = H;
    a.tc_mode = c->hit_mode;
    ProfScope ps(c, ETX_K_NODE_ENC, s);
    if (q8) {
      // the 3-feature first layer stays fp32 (double accumulation: q8_aux.cu); its ReLU output, parked in m, is the
      // first quantised tensor; layers 2.. run as an INT8 chain
      c->launches += launch_node_l1(N, H, a.feat, a.fc, a.fs, c->node_enc.Wt[0], c->node_enc.b[0], w.m, s);
      const DevMlp& f = c->node_enc;
      a.n_seg = 1; a.seg[0] = Segment{w.m, nullptr, H, H};
      a.mlp.n_layers = f.n_layers - 1;
      for (int l = 0; l < f.n_layers; ++l) { a.mlp.dims[l] = f.dims[l + 1]; }
      for (int l = 0; l + 1 < f.n_layers; ++l) { a.mlp.Wt[l] = f.Wt[l + 1]; a.mlp.b[l] = f.b[l + 1]; }
      fill_q(c, a, 0, f, 1, f.n_layers - 1);
    }
    c->launches += run_mlp(c, a, s);
  }
  // Tensor-core modes factorise the first layer of the edge MLPs: with W1 = [A | B | C]
  // over [h_src | h_dst | e],  W1 [h_i, h_j, e] = (A h_i) + (B h_j) + C e.  The per-hit projections
  // p_l = [A h_l | B h_l] cost 4 H^2 flop per HIT instead of per EDGE; the edge kernel gathers the two
  // 128-wide rows, adds them and starts its layer-1 accumulator from the sum.
  const bool fact = c->desc.precision != ETX_PREC_FP32;
  auto project = [&](const DevMlp& mlp, int mi) {      // p = [A h | B h] over the hits (mi: the MLP's number, for its INT8 ranges)
    ProfScope ps(c, ETX_K_EDGE_PROJ, s);
    // bf16 modes: ONE launch, h read once, both 128-column halves (the images of A and B are adjacent);
    // TF32X3 (one tile in flight, no second accumulator slot): one launch per half
    const bool wide = c->desc.precision != ETX_PREC_TF32X3;
    for (int part = 0; part < (wide ? 1 : 2); ++part) {
      MlpArgs a;
      a.n_rows = N; a.n_seg = 1;
      a.seg[0] = Segment{w.h, nullptr, H, H};
      a.mlp.n_layers = 1; a.mlp.dims[0] = H; a.mlp.dims[1] = H;
      a.mlp.wimg = part == 0 ? mlp.wimg_a : mlp.wimg_b;
      a.mlp.b[0] = c->d_zero_bias; a.mlp.Wt[0] = c->d_zero_bias;
      a.wide = wide ? 1 : 0;
      a.tc_mode = c->hit_mode;
      if (q8) a.q_sa0 = c->q_alpha[(size_t)mi * c->desc.gnn_n_layers] / (c->desc.precision == ETX_PREC_FP8 ? 448.0f : 127.0f);   // the edge MLP's layer-1 input scale; raw sums out
      a.out_mode = 0; a.out = w.p + part * H; a.out_ld = 2 * H;
      c->launches += run_mlp(c, a, s);
    }
  };
  {  // a3: e0 = MLP_e([h0_src, h0_dst])
    MlpArgs a;
    a.n_rows = E;
    a.mlp = c->edge_enc; a.out_mode = 0; a.out = d_edge_enc; a.out_ld = H;
    if (fact) {
      if (E > 0) project(c->edge_enc, 1);
      if (q8) fill_q(c, a, 1, c->edge_enc, 0, c->edge_enc.n_layers);
      a.n_seg = 0; a.n_add = 2;
      a.add[0] = Segment{w.p, g->d_src, H, 2 * H};
      a.add[1] = Segment{w.p + H, g->d_dst, H, 2 * H};
      a.mlp.dims[0] = 0;                               // no per-edge operand in layer 1
    } else {
      a.n_seg = 2;
      a.seg[0] = Segment{w.h, g->d_src, H, H};
      a.seg[1] = Segment{w.h, g->d_dst, H, H};
    }
    ProfScope ps(c, ETX_K_EDGE_ENC, s);
    c->launches += run_mlp(c, a, s);
  }
  for (int k = 0; k < c->desc.n_iter; ++k) {
    // a4: m = [sum out, sum in] of e^k
    {
      ProfScope ps(c, ETX_K_SCATTER, s);
#ifdef ETX_DEV_SWITCHES
      static const bool atomic = getenv("ETX_SCATTER_ATOMIC") != nullptr;   // developer build: the measured alternative
      if (atomic && H == 128) c->launches += launch_scatter_atomic(N, E, H, g->d_src, g->d_dst, (const float*)d_edge_enc, w.m, s);
      else
#endif
      c->launches += launch_scatter(N, H, g->d_row_ptr, g->d_in_ptr, g->d_in_perm, d_edge_enc, w.m, w.sched, s);
    }
    {  // a5: h += phi_k([h, m])
      MlpArgs a;
      a.n_rows = N; a.n_seg = 2;
      a.seg[0] = Segment{w.h, nullptr, H, H};
      a.seg[1] = Segment{w.m, nullptr, 2 * H, 2 * H};
      a.mlp = c->node_net[k]; a.out_mode = 1; a.out = w.h; a.res = w.h; a.out_ld = H;
      a.tc_mode = c->hit_mode;
      if (q8) fill_q(c, a, 2 + 2 * k, c->node_net[k], 0, c->node_net[k].n_layers);
      ProfScope ps(c, ETX_K_NODE_NET, s);
      c->launches += run_mlp(c, a, s);
    }
    {  // a6: e += psi_k([h_src, h_dst, e]) with the UPDATED h
      MlpArgs a;
      a.n_rows = E;
      a.mlp = c->edge_net[k]; a.out_mode = 1; a.out = d_edge_enc; a.res = d_edge_enc; a.out_ld = H;
      if (fact) {
        if (E > 0) project(c->edge_net[k], 3 + 2 * k);
        if (q8) fill_q(c, a, 3 + 2 * k, c->edge_net[k], 0, c->edge_net[k].n_layers);
        a.n_seg = 1; a.n_add = 2;
        a.seg[0] = Segment{d_edge_enc, nullptr, H, H};
        a.add[0] = Segment{w.p, g->d_src, H, 2 * H};
        a.add[1] = Segment{w.p + H, g->d_dst, H, 2 * H};
        a.mlp.dims[0] = H;                             // per-edge operand of layer 1: e only
      } else {
        a.n_seg = 3;
        a.seg[0] = Segment{w.h, g->d_src, H, H};
        a.seg[1] = Segment{w.h, g->d_dst, H, H};
        a.seg[2] = Segment{d_edge_enc, nullptr, H, H};
      }
      ProfScope ps(c, ETX_K_EDGE_NET, s);
      c->launches += run_mlp(c, a, s);
    }
  }
  if (d_hit_enc && N > 0)
    cudaMemcpyAsync(d_hit_enc, w.h, sizeof(float) * (size_t)N * H, cudaMemcpyDeviceToDevice, s);
  return check_cuda(c, "etx_gnn_forward");
}

etx_status etx_edge_scores(etx_ctx* c, const etx_graph* g, const float* d_edge_enc, float* d_scores,
                           void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (!g || g->n_edges < 0) return fail(c, ETX_ERR_INVALID, "graph is NULL or not built");
  if (g->n_edges > 0 && (!d_edge_enc || !d_scores)) return fail(c, ETX_ERR_INVALID, "d_edge_enc / d_scores is NULL");
  if ((uintptr_t)d_edge_enc & 15) return fail(c, ETX_ERR_INVALID, "d_edge_enc must be 16-byte aligned");
  cudaSetDevice(c->device);
  const int H = c->desc.gnn_hidden;
  MlpArgs a;
  a.n_rows = (int)g->n_edges; a.n_seg = 1;
  a.seg[0] = Segment{d_edge_enc, nullptr, H, H};
  a.mlp = c->cls; a.out_mode = 3; a.out = d_scores; a.out_ld = 1;
  a.tc_mode = c->hit_mode;
  if (c->desc.precision == ETX_PREC_INT8 || c->desc.precision == ETX_PREC_FP8) {
    if (c->q_alpha.empty()) return fail(c, ETX_ERR_INVALID, "ETX_PREC_INT8 / ETX_PREC_FP8 need calibrated ranges (etx_set_int8_ranges)");
    fill_q(c, a, 2 + 2 * c->desc.n_iter, c->cls, 0, c->cls.n_layers);
  }
  {
    ProfScope ps(c, ETX_K_CLS, (cudaStream_t)stream);
    c->launches += run_mlp(c, a, (cudaStream_t)stream);
  }
  return check_cuda(c, "etx_edge_scores");
}

etx_status etx_build_tracks(etx_ctx* c, const etx_batch* b, const etx_graph* g, const float* d_scores,
                            float score_min, int32_t* d_labels, void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (etx_status st = check_batch(c, b)) return st;
  if (!g || g->n_edges < 0 || !g->d_row_ptr) return fail(c, ETX_ERR_INVALID, "graph is NULL or not built");
  if (b->n_hits > 0 && !d_labels) return fail(c, ETX_ERR_INVALID, "d_labels is NULL");
  if (g->n_edges > 0 && (!d_scores || !g->d_src || !g->d_dst)) return fail(c, ETX_ERR_INVALID, "scores / edge arrays are NULL");
  cudaSetDevice(c->device);
  {
    ProfScope ps(c, ETX_K_TRACKS, (cudaStream_t)stream);
    c->launches += launch_wcc(b->n_events, b->d_event_ptr, g->d_row_ptr, g->d_src, g->d_dst, d_scores, score_min,
                              d_labels, (cudaStream_t)stream);
  }
  return check_cuda(c, "etx_build_tracks");
}

etx_status etx_build_triplets(etx_ctx* c, const etx_batch* b, const etx_graph* g, const float* d_scores,
                              float score_min, etx_triplets* t, void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (etx_status st = check_batch(c, b)) return st;
  if (!g || g->n_edges < 0 || !g->d_row_ptr || !g->d_in_ptr) return fail(c, ETX_ERR_INVALID, "graph is NULL or not built");
  if (!t || !t->d_ptr || t->capacity < 0) return fail(c, ETX_ERR_INVALID, "triplet buffers are NULL");
  if (t->capacity > 0 && (!t->d_first || !t->d_second)) return fail(c, ETX_ERR_INVALID, "triplet row arrays are NULL");
  if (g->n_edges > 0 && (!d_scores || !g->d_in_perm)) return fail(c, ETX_ERR_INVALID, "scores / in_perm are NULL");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  if (etx_status st = need_ws(c, carve(c, b->n_events, b->n_hits, 0, false, nullptr))) return st;
  const Workspace w = carve(c, b->n_events, b->n_hits, 0, false, (char*)c->ws);
  const int N = b->n_hits;
  const size_t ld = (size_t)N + 1;
  {
    ProfScope ps(c, ETX_K_TRACKS, s);
    c->launches += launch_triplet_count(N, g->d_row_ptr, g->d_in_ptr, g->d_in_perm, d_scores, score_min, t->d_ptr, s);
    for (int k = 0; k < 3; ++k) c->launches += launch_exclusive_scan(t->d_ptr + k * ld, N + 1, w.scan_tmp, s);
  }
  int32_t host[3] = {0, 0, 0};
  for (int k = 0; k < 3; ++k)
    cudaMemcpyAsync(&host[k], t->d_ptr + k * ld + N, sizeof(int32_t), cudaMemcpyDeviceToHost, s);
  if (cudaStreamSynchronize(s) != cudaSuccess) return check_cuda(c, "etx_build_triplets (count)");
  if (etx_status st = check_cuda(c, "etx_build_triplets (count)")) return st;
  bool overflow = false;
  for (int k = 0; k < 3; ++k) { t->n[k] = host[k]; overflow |= host[k] < 0; }
  if (overflow) return fail(c, ETX_ERR_CAPACITY, "more than 2^31 - 1 triplets of one kind");
  const int64_t total = t->n[0] + t->n[1] + t->n[2];
  if (total > t->capacity)
    return fail(c, ETX_ERR_CAPACITY, "triplets need " + std::to_string(total) + " rows, capacity " + std::to_string(t->capacity));
  if (total > 0) {
    ProfScope ps(c, ETX_K_TRACKS, s);
    c->launches += launch_triplet_fill(N, g->d_row_ptr, g->d_in_ptr, g->d_in_perm, d_scores, score_min, t->d_ptr,
                                       t->d_first, t->d_second, s);
  }
  return check_cuda(c, "etx_build_triplets (fill)");
}

// ---------------------------------------------------------------------------------------------------------------------
// etx_build_triplets_static: etx_build_triplets for callers that may not allocate (include/etx.h).  The only scratch the
// triplet build needs is the block sums of its three device-wide scans; here they live in a file-scope device array of
// fixed size instead of the registered workspace, so the call works on a context that has no workspace at all.
constexpr int kStaticTripletMaxHits = ETX_STATIC_TRIPLET_MAX_HITS;
constexpr int kStaticScanInts = 2304;                // >= scan_tmp_ints(kStaticTripletMaxHits + 1) = 2050 (checked at run time), 9 KB
static __device__ __align__(256) int32_t g_static_scan_scratch[kStaticScanInts];

namespace {
// Device address of the array above on the context's device (which the caller has made current).  In host code the symbol
// is only a stand-in for the array: its device address is asked for once per device and kept.
etx_status static_scan_scratch(etx_ctx* c, int32_t** out) {
  static std::mutex mu;
  static int32_t* addr[kMaxDevices] = {nullptr};
  if (c->device < 0 || c->device >= kMaxDevices) return fail(c, ETX_ERR_INVALID, "device index beyond the per-device tables");
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[c->device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scan_scratch);
    if (e != cudaSuccess || !p)
      return fail(c, ETX_ERR_CUDA, std::string("cudaGetSymbolAddress(static scan scratch): ") + cudaGetErrorString(e));
    addr[c->device] = static_cast<int32_t*>(p);
  }
  *out = addr[c->device];
  return ETX_OK;
}
}  // namespace

etx_status etx_build_triplets_static(etx_ctx* c, const etx_batch* b, const etx_graph* g, const float* d_scores,
                                     float score_min, etx_triplets* t, void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (etx_status st = check_batch(c, b)) return st;
  if (!g || g->n_edges < 0 || !g->d_row_ptr || !g->d_in_ptr) return fail(c, ETX_ERR_INVALID, "graph is NULL or not built");
  if (!t || !t->d_ptr || t->capacity < 0) return fail(c, ETX_ERR_INVALID, "triplet buffers are NULL");
  if (t->capacity > 0 && (!t->d_first || !t->d_second)) return fail(c, ETX_ERR_INVALID, "triplet row arrays are NULL");
  if (g->n_edges > 0 && (!d_scores || !g->d_in_perm)) return fail(c, ETX_ERR_INVALID, "scores / in_perm are NULL");
  const int N = b->n_hits;
  if (N > kStaticTripletMaxHits || scan_tmp_ints(N + 1) > (size_t)kStaticScanInts)
    return fail(c, ETX_ERR_CAPACITY, "etx_build_triplets_static handles at most " + std::to_string(kStaticTripletMaxHits) +
                                         " hits per call (its scratch is a fixed device array); got " + std::to_string(N));
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  int32_t* scan_tmp = nullptr;
  if (etx_status st = static_scan_scratch(c, &scan_tmp)) return st;
  const size_t ld = (size_t)N + 1;
  // The array keeps the previous call's block sums.  The scans write every entry they read, so nothing HAS to start at
  // zero; the part this call uses is cleared anyway so that a result can never depend on an earlier call.
  cudaMemsetAsync(scan_tmp, 0, scan_tmp_ints(N + 1) * sizeof(int32_t), s);
  c->launches += launch_triplet_count(N, g->d_row_ptr, g->d_in_ptr, g->d_in_perm, d_scores, score_min, t->d_ptr, s);
  for (int k = 0; k < 3; ++k) c->launches += launch_exclusive_scan(t->d_ptr + k * ld, N + 1, scan_tmp, s);
  int32_t host[3] = {0, 0, 0};
  for (int k = 0; k < 3; ++k)
    cudaMemcpyAsync(&host[k], t->d_ptr + k * ld + N, sizeof(int32_t), cudaMemcpyDeviceToHost, s);
  if (cudaStreamSynchronize(s) != cudaSuccess) return check_cuda(c, "etx_build_triplets_static (count)");
  if (etx_status st = check_cuda(c, "etx_build_triplets_static (count)")) return st;
  bool overflow = false;
  for (int k = 0; k < 3; ++k) { t->n[k] = host[k]; overflow |= host[k] < 0; }
  if (overflow) return fail(c, ETX_ERR_CAPACITY, "more than 2^31 - 1 triplets of one kind");
  const int64_t total = t->n[0] + t->n[1] + t->n[2];
  if (total > t->capacity)
    return fail(c, ETX_ERR_CAPACITY, "triplets need " + std::to_string(total) + " rows, capacity " + std::to_string(t->capacity));
  if (total > 0)
    c->launches += launch_triplet_fill(N, g->d_row_ptr, g->d_in_ptr, g->d_in_perm, d_scores, score_min, t->d_ptr,
                                       t->d_first, t->d_second, s);
  return check_cuda(c, "etx_build_triplets_static (fill)");
}

size_t etx_triplet_weight_count(const etx_model_desc* desc) {
  if (check_desc(desc)) return 0;
  const int H = desc->gnn_hidden, L = desc->gnn_n_layers;
  size_t one = (size_t)2 * H * H + H;
  for (int l = 1; l < L - 1; ++l) one += (size_t)H * H + H;
  one += (size_t)H + 1;
  return 2 * one;
}

etx_status etx_set_triplet_classifiers(etx_ctx* c, const float* h_weights, size_t n_weights) {
  if (!c) return ETX_ERR_INVALID;
  if (!h_weights || n_weights != etx_triplet_weight_count(&c->desc))
    return fail(c, ETX_ERR_INVALID, "triplet classifier blob size does not match (see etx_triplet_weight_count)");
  cudaSetDevice(c->device);
  const int H = c->desc.gnn_hidden, L = c->desc.gnn_n_layers;
  HostMlp m; m.n_layers = L; m.dims[0] = 2 * H;
  for (int l = 1; l < L; ++l) m.dims[l] = H;
  m.dims[L] = 1;
  std::vector<float> staged;
  std::vector<unsigned char> img;
  size_t offW[2][kMaxLayers], offB[2][kMaxLayers], img_off[2] = {0, 0};
  size_t src = 0;
  for (int i = 0; i < 2; ++i) {
    if (c->desc.precision != ETX_PREC_FP32) { img_off[i] = img.size(); append_wimg(img, m, h_weights + src, 0, 0, L - 1, c->desc.precision); }
    for (int l = 0; l < L; ++l) {
      const int fi = m.dims[l], fo = m.dims[l + 1];
      staged.resize(align_up(staged.size(), 64));
      offW[i][l] = staged.size();
      staged.resize(staged.size() + (size_t)fi * fo);
      float* Wt = staged.data() + offW[i][l];
      const float* W = h_weights + src;
      for (int o = 0; o < fo; ++o)
        for (int k = 0; k < fi; ++k) Wt[(size_t)k * fo + o] = W[(size_t)o * fi + k];
      src += (size_t)fi * fo;
      staged.resize(align_up(staged.size(), 64));
      offB[i][l] = staged.size();
      staged.insert(staged.end(), h_weights + src, h_weights + src + fo);
      src += fo;
    }
  }
  if (c->d_trip_weights) { cudaFree(c->d_trip_weights); c->d_trip_weights = nullptr; }
  if (c->d_trip_wimg) { cudaFree(c->d_trip_wimg); c->d_trip_wimg = nullptr; }
  c->have_trip = false;
  if (cudaMalloc(&c->d_trip_weights, staged.size() * sizeof(float)) != cudaSuccess ||
      cudaMemcpy(c->d_trip_weights, staged.data(), staged.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess)
    return check_cuda(c, "etx_set_triplet_classifiers");
  if (!img.empty() && (cudaMalloc(&c->d_trip_wimg, img.size()) != cudaSuccess ||
                       cudaMemcpy(c->d_trip_wimg, img.data(), img.size(), cudaMemcpyHostToDevice) != cudaSuccess))
    return check_cuda(c, "etx_set_triplet_classifiers");
  DevMlp* dm[2] = {&c->trip_art, &c->trip_elb};
  for (int i = 0; i < 2; ++i) {
    *dm[i] = DevMlp();
    dm[i]->n_layers = L;
    for (int l = 0; l <= L; ++l) dm[i]->dims[l] = m.dims[l];
    for (int l = 0; l < L; ++l) { dm[i]->Wt[l] = c->d_trip_weights + offW[i][l]; dm[i]->b[l] = c->d_trip_weights + offB[i][l]; }
    if (c->d_trip_wimg) dm[i]->wimg = c->d_trip_wimg + img_off[i];
  }
  c->have_trip = true;
  return ETX_OK;
}

etx_status etx_triplet_scores(etx_ctx* c, const etx_graph* g, const float* d_edge_enc, const etx_triplets* t,
                              float* d_trip_scores, void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (!c->have_trip) return fail(c, ETX_ERR_INVALID, "no triplet classifiers set (etx_set_triplet_classifiers)");
  if (c->desc.precision == ETX_PREC_INT8 || c->desc.precision == ETX_PREC_FP8)
    return fail(c, ETX_ERR_INVALID, "the triplet classifiers have no ETX_PREC_INT8 / ETX_PREC_FP8 path");
  if (!g || g->n_edges < 0 || !t) return fail(c, ETX_ERR_INVALID, "graph / triplets are NULL");
  const int64_t total = t->n[0] + t->n[1] + t->n[2];
  if (t->n[0] < 0 || t->n[1] < 0 || t->n[2] < 0 || total > t->capacity) return fail(c, ETX_ERR_INVALID, "triplets not built");
  if (total > 0 && (!d_edge_enc || !d_trip_scores || !t->d_first || !t->d_second)) return fail(c, ETX_ERR_INVALID, "triplet buffers are NULL");
  if ((uintptr_t)d_edge_enc & 15) return fail(c, ETX_ERR_INVALID, "d_edge_enc must be 16-byte aligned");
  cudaSetDevice(c->device);
  const int H = c->desc.gnn_hidden;
  for (int part = 0; part < 2; ++part) {                 // articulations, then both elbow kinds (adjacent sections)
    const int64_t r0 = part == 0 ? 0 : t->n[0], nr = part == 0 ? t->n[0] : t->n[1] + t->n[2];
    if (nr <= 0) continue;
    MlpArgs a;
    a.n_rows = (int)nr; a.n_seg = 2;
    a.seg[0] = Segment{d_edge_enc, t->d_first + r0, H, H};
    a.seg[1] = Segment{d_edge_enc, t->d_second + r0, H, H};
    a.mlp = part == 0 ? c->trip_art : c->trip_elb;
    a.out_mode = 3; a.out = d_trip_scores + r0; a.out_ld = 1;
    ProfScope ps(c, ETX_K_TRACKS, (cudaStream_t)stream);
    c->launches += run_mlp(c, a, (cudaStream_t)stream);
  }
  return check_cuda(c, "etx_triplet_scores");
}

size_t etx_triplet_tracks_workspace_bytes(const etx_ctx* c, int32_t n_hits, int64_t n_edges, int64_t n_articulations) {
  if (!c || n_hits < 0 || n_edges < 0 || n_articulations < 0) return 0;
  return triplet_tracks_ws_bytes(n_hits, n_edges, n_articulations);
}

etx_status etx_build_tracks_from_triplets(etx_ctx* c, const etx_batch* b, const etx_graph* g, const float* d_scores,
                                          float score_min, const etx_triplets* t, const float* d_trip_scores,
                                          float trip_min, etx_tracks* out, void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (etx_status st = check_batch(c, b)) return st;
  if (!g || g->n_edges < 0 || !g->d_row_ptr || !g->d_in_ptr) return fail(c, ETX_ERR_INVALID, "graph is NULL or not built");
  if (!t || !t->d_ptr || !out) return fail(c, ETX_ERR_INVALID, "triplets / tracks are NULL");
  const int64_t total = t->n[0] + t->n[1] + t->n[2];
  if (t->n[0] < 0 || t->n[1] < 0 || t->n[2] < 0 || total > t->capacity) return fail(c, ETX_ERR_INVALID, "triplets not built");
  if (total > 0 && (!t->d_first || !t->d_second || !d_trip_scores)) return fail(c, ETX_ERR_INVALID, "triplet rows / scores are NULL");
  if (g->n_edges > 0 && (!d_scores || !g->d_in_perm || !out->d_edge_set)) return fail(c, ETX_ERR_INVALID, "scores / in_perm / d_edge_set are NULL");
  if (out->join_capacity < 0 || out->track_capacity < 0 || out->hit_capacity < 0) return fail(c, ETX_ERR_INVALID, "negative capacity");
  if (!out->d_track_ptr || (out->join_capacity > 0 && !out->d_joins) || (out->hit_capacity > 0 && !out->d_track_hits))
    return fail(c, ETX_ERR_INVALID, "track buffers are NULL");
  cudaSetDevice(c->device);
  if (!c->ws) return fail(c, ETX_ERR_NOMEM, "no workspace set (etx_set_workspace)");
  const size_t need = triplet_tracks_ws_bytes(b->n_hits, g->n_edges, t->n[0]);
  if (need > c->ws_bytes)
    return fail(c, ETX_ERR_NOMEM, "workspace too small: need " + std::to_string(need) + " bytes (etx_triplet_tracks_workspace_bytes), have " +
                                      std::to_string(c->ws_bytes));
  long long counts[4] = {0, 0, 0, 0};
  const long long ntr[3] = {t->n[0], t->n[1], t->n[2]};
  bool ok = true;
  int n;
  {
    ProfScope ps(c, ETX_K_TRACKS, (cudaStream_t)stream);
    n = run_triplet_tracks(b->n_events, b->n_hits, g->n_edges, b->d_event_ptr, g->d_row_ptr, g->d_in_ptr, g->d_in_perm,
                           d_scores, score_min, t->d_ptr, ntr, t->d_first, t->d_second, d_trip_scores, trip_min,
                           (char*)c->ws, out->d_edge_set, out->join_capacity, out->d_joins, out->track_capacity,
                           out->d_track_ptr, out->hit_capacity, out->d_track_hits, counts, &ok, (cudaStream_t)stream);
    if (n > 0) c->launches += n;
  }
  out->n_joins = counts[0]; out->n_plain = counts[1]; out->n_tracks = counts[2]; out->n_track_hits = counts[3];
  if (n < 0) return check_cuda(c, "etx_build_tracks_from_triplets");
  if (etx_status st = check_cuda(c, "etx_build_tracks_from_triplets")) return st;
  if (!ok)
    return fail(c, ETX_ERR_CAPACITY, "tracks need " + std::to_string(counts[0]) + " joins, " + std::to_string(counts[2]) +
                                         " tracks, " + std::to_string(counts[3]) + " hit entries");
  return ETX_OK;
}

// One pass of the whole path over events [e0, e1) of a HOST batch (hits [h0, h1)), results appended at edge
// offset `edge_off` of the host outputs with hit indices made global again.  The workspace must hold the pass.
static etx_status infer_host_pass(etx_ctx* c, const etx_batch_host* hb, int32_t e0, int32_t e1, float r2_max,
                                  int32_t max_plane_gap, int64_t cap, int64_t edge_off, int64_t* n_edges,
                                  int32_t* h_src, int32_t* h_dst, float* h_scores, cudaStream_t s) {
  const int32_t n_ev = e1 - e0, h0 = hb->h_event_ptr[e0], h1 = hb->h_event_ptr[e1];
  const Workspace w = carve(c, n_ev, h1 - h0, cap, true, (char*)c->ws);
  const size_t nh = (size_t)(h1 - h0);
  std::vector<int32_t> local_ptr;
  const int32_t* ep = hb->h_event_ptr + e0;
  if (h0 != 0) {                                       // a chunk's offsets restart at 0
    local_ptr.resize((size_t)n_ev + 1);
    for (int32_t i = 0; i <= n_ev; ++i) local_ptr[i] = ep[i] - h0;
    ep = local_ptr.data();
  }
  cudaMemcpyAsync(w.s_event_ptr, ep, sizeof(int32_t) * ((size_t)n_ev + 1), cudaMemcpyHostToDevice, s);
  if (!local_ptr.empty()) cudaStreamSynchronize(s);    // the pageable temporary must outlive its copy
  if (nh) {
    cudaMemcpyAsync(w.s_plane, hb->h_plane + h0, nh, cudaMemcpyHostToDevice, s);
    cudaMemcpyAsync(w.s_r, hb->h_r + h0, nh * 4, cudaMemcpyHostToDevice, s);
    cudaMemcpyAsync(w.s_phi, hb->h_phi + h0, nh * 4, cudaMemcpyHostToDevice, s);
    cudaMemcpyAsync(w.s_z, hb->h_z + h0, nh * 4, cudaMemcpyHostToDevice, s);
    cudaMemcpyAsync(w.s_x, hb->h_x + h0, nh * 4, cudaMemcpyHostToDevice, s);
    cudaMemcpyAsync(w.s_y, hb->h_y + h0, nh * 4, cudaMemcpyHostToDevice, s);
  }
  etx_batch b;
  b.n_events = n_ev; b.n_hits = h1 - h0;
  b.d_event_ptr = w.s_event_ptr; b.d_plane = w.s_plane;
  b.d_r = w.s_r; b.d_phi = w.s_phi; b.d_z = w.s_z; b.d_x = w.s_x; b.d_y = w.s_y;
  etx_graph g;
  g.edge_capacity = cap; g.n_edges = 0;
  g.d_row_ptr = w.s_row_ptr; g.d_src = w.s_src; g.d_dst = w.s_dst; g.d_in_ptr = w.s_in_ptr; g.d_in_perm = w.s_in_perm;
  if (etx_status st = etx_embed(c, &b, w.s_emb, s)) return st;
  etx_status st = etx_build_graph(c, &b, w.s_emb, r2_max, max_plane_gap, 0, &g, s);
  *n_edges = g.n_edges;
  if (st) return st;
  // the edge list is final once the graph is built: its device-to-host copy runs on the context's copy stream
  // underneath the message passing; only the scores are copied after the last kernel
  const size_t ne = (size_t)g.n_edges;
  if (!c->copy_stream) {
    cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
    cudaEventCreateWithFlags(&c->copy_event, cudaEventDisableTiming);
  }
  if (ne && (h_src || h_dst)) {
    int32_t *o_src = w.s_src, *o_dst = w.s_dst;
    if (h0 != 0) {                                     // global hit indices: shifted copies in the (still unused) score / encoding buffers
      o_src = reinterpret_cast<int32_t*>(w.s_scores);
      o_dst = reinterpret_cast<int32_t*>(w.s_edge_enc);
      c->launches += launch_add_offset(w.s_src, o_src, (int64_t)ne, h0, s);
      c->launches += launch_add_offset(w.s_dst, o_dst, (int64_t)ne, h0, s);
    }
    cudaEventRecord(c->copy_event, s);
    cudaStreamWaitEvent(c->copy_stream, c->copy_event, 0);
    if (h_src) cudaMemcpyAsync(h_src + edge_off, o_src, ne * 4, cudaMemcpyDeviceToHost, c->copy_stream);
    if (h_dst) cudaMemcpyAsync(h_dst + edge_off, o_dst, ne * 4, cudaMemcpyDeviceToHost, c->copy_stream);
    if (h0 != 0) {                                     // the shifted copies live where the GNN writes next
      cudaEventRecord(c->copy_event, c->copy_stream);
      cudaStreamWaitEvent(s, c->copy_event, 0);
    }
  }
  if (!(st = etx_gnn_forward(c, &b, &g, w.s_edge_enc, nullptr, s)))
    st = etx_edge_scores(c, &g, w.s_edge_enc, w.s_scores, s);
  if (!st && ne && h_scores) cudaMemcpyAsync(h_scores + edge_off, w.s_scores, ne * 4, cudaMemcpyDeviceToHost, s);
  const cudaError_t e1c = cudaStreamSynchronize(c->copy_stream), e2c = cudaStreamSynchronize(s);
  if (st) return st;
  (void)e1c; (void)e2c;
  return check_cuda(c, "etx_infer_host");
}

etx_status etx_infer_host(etx_ctx* c, const etx_batch_host* hb, float r2_max, int32_t max_plane_gap,
                          int64_t edge_capacity, int64_t* n_edges, int32_t* h_src, int32_t* h_dst,
                          float* h_scores, void* stream) {
  if (!c) return ETX_ERR_INVALID;
  if (!hb || hb->n_events < 0 || hb->n_hits < 0 || !hb->h_event_ptr || edge_capacity < 0)
    return fail(c, ETX_ERR_INVALID, "host batch is NULL or malformed");
  if (hb->n_hits > 0 && (!hb->h_plane || !hb->h_r || !hb->h_phi || !hb->h_z || !hb->h_x || !hb->h_y))
    return fail(c, ETX_ERR_INVALID, "host batch array is NULL");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  if (!c->ws) return fail(c, ETX_ERR_NOMEM, "no workspace set (etx_set_workspace)");
  int64_t total = 0;
  if (carve(c, hb->n_events, hb->n_hits, edge_capacity, true, nullptr).total <= c->ws_bytes) {
    const etx_status st = infer_host_pass(c, hb, 0, hb->n_events, r2_max, max_plane_gap, edge_capacity, 0, &total,
                                          h_src, h_dst, h_scores, s);
    if (n_edges) *n_edges = total;
    return st;
  }
  // The batch does not fit the workspace: split it into consecutive event ranges that do (the thesis bounds its
  // GNN batches the same way, <= 2^20 hits / 2^22 edges).  Events are independent and edges are
  // ordered by source, so the passes' outputs concatenate into exactly the single-pass result.  A range gets the
  // edge capacity the workspace has room for (at most what is left of the caller's), sized from the caller's own
  // edges-per-hit ratio; a range whose graph still overflows its share is halved and retried.
  const int32_t* ep = hb->h_event_ptr;
  for (int32_t i = 0; i < hb->n_events; ++i)
    if (ep[i + 1] < ep[i]) return fail(c, ETX_ERR_INVALID, "malformed batch: event_ptr not monotone");
  if (hb->n_events > 0 && (ep[0] != 0 || ep[hb->n_events] != hb->n_hits))
    return fail(c, ETX_ERR_INVALID, "malformed batch: event_ptr does not span the hits");
  const double per_hit = hb->n_hits > 0 ? (double)edge_capacity / hb->n_hits : 0.0;
  auto cap_of = [&](int32_t a, int32_t b2) {
    const int64_t want = (int64_t)std::ceil(per_hit * (ep[b2] - ep[a])) + 1024;
    return std::min<int64_t>(want, edge_capacity - total);
  };
  auto fits = [&](int32_t a, int32_t b2) {
    return carve(c, b2 - a, ep[b2] - ep[a], cap_of(a, b2), true, nullptr).total <= c->ws_bytes;
  };
  int32_t e0 = 0, limit = hb->n_events;
  while (e0 < hb->n_events) {
    if (!fits(e0, e0 + 1))
      return fail(c, ETX_ERR_NOMEM, "workspace too small for event " + std::to_string(e0) + " alone (" +
                                        std::to_string(ep[e0 + 1] - ep[e0]) + " hits)");
    int32_t lo = e0 + 1, hi = std::min(limit, hb->n_events);     // largest range [e0, e1) that fits, by bisection
    while (lo < hi) { const int32_t mid = lo + (hi - lo + 1) / 2; if (fits(e0, mid)) lo = mid; else hi = mid - 1; }
    const int32_t e1 = lo;
    // give the range all the edge room the workspace still has
    int64_t cap = cap_of(e0, e1);
    {
      const size_t base0 = carve(c, e1 - e0, ep[e1] - ep[e0], 0, true, nullptr).total;
      const size_t base1 = carve(c, e1 - e0, ep[e1] - ep[e0], 4096, true, nullptr).total;
      const double per_edge = (double)(base1 - base0) / 4096.0;
      const int64_t room = (int64_t)((double)(c->ws_bytes - base0) / per_edge) - 4096;
      cap = std::max(cap, std::min<int64_t>(room, edge_capacity - total));
      while (cap > 0 && carve(c, e1 - e0, ep[e1] - ep[e0], cap, true, nullptr).total > c->ws_bytes) cap -= 1024;
      if (cap < 0) cap = 0;
    }
    int64_t got = 0;
    const etx_status st = infer_host_pass(c, hb, e0, e1, r2_max, max_plane_gap, cap, total, &got, h_src, h_dst, h_scores, s);
    if (st == ETX_ERR_CAPACITY && e1 - e0 > 1 && total + got <= edge_capacity) { limit = e0 + (e1 - e0) / 2; continue; }
    if (st) { if (n_edges) *n_edges = total + got; return st; }
    total += got;
    e0 = e1; limit = hb->n_events;
  }
  if (n_edges) *n_edges = total;
  return ETX_OK;
}

}  // extern "C"
