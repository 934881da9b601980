// TEST INFRASTRUCTURE — CPU oracle for the hits -> edge-scores path of ETX4VELO (arXiv 2508.07423).
//
// Plain, slow, obviously-correct C++17 written from the thesis' definitions (P:n = PAPER.md line n).
// It shares no code with the CUDA path (paper_2508_07423_b200/csrc) and neither includes the other.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
//
// Arithmetic convention: parameters and stored activations are
// fp32; every dot product and every scatter sum accumulates in double and is rounded to fp32 once;
// the radius predicate is evaluated in fp32, left to right, every operation individually rounded
// (compile with -ffp-contract=off); the sigmoid is evaluated in double and stored as fp32.
// OpenMP is used only over independent rows (hits / edges / events): no sum is ever reordered.
//
// Pins (tests/test_oracle_*.py): brute-force N^2 search, dense incidence-matrix scatter, torch float64
// linear layers, closed forms (r -> inf edge counts, zero/constant networks), invariants.
// Track building (orc_wcc): scipy connected_components, hand-built graphs, partition invariants.
// Whole path vs the thesis' TRAINED network: parity unpinned (no weights, data or printed outputs exist).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <utility>
#include <vector>

extern "C" {

// ---- a0 features: "normalized cylindrical (r, phi, z)" P:2285, "normalized Cartesian" P:2316,
//      "recentering and rescaling" P:2585.  f = (v - center) / scale, feature order r,phi,z,x,y.
void orc_features(int64_t n, const float* r, const float* phi, const float* z, const float* x,
                  const float* y, const float* center, const float* scale,
                  float* f_emb /*[n,3] r,phi,z*/, float* f_node /*[n,3] x,y,z*/) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    const float fr = (r[i] - center[0]) / scale[0];
    const float fp = (phi[i] - center[1]) / scale[1];
    const float fz = (z[i] - center[2]) / scale[2];
    const float fx = (x[i] - center[3]) / scale[3];
    const float fy = (y[i] - center[4]) / scale[4];
    f_emb[3 * i + 0] = fr; f_emb[3 * i + 1] = fp; f_emb[3 * i + 2] = fz;
    f_node[3 * i + 0] = fx; f_node[3 * i + 1] = fy; f_node[3 * i + 2] = fz;
  }
}

// ---- MLP: f_l(z) = g_l(W_l z + b_l), Eq. 4.27; chain Eq. 4.26; g = ReLU on hidden layers
//      (P:1305), identity on the last layer.  W_l stored [out][in] row-major, then b_l [out].
//      `w` points at the first layer's W; layers are consecutive.  in [n, dims[0]] -> out [n, dims[L]].
void orc_mlp(int64_t n, int32_t n_layers, const int32_t* dims, const float* w, const float* in,
             float* out) {
  int32_t maxw = 0;
  for (int l = 0; l <= n_layers; ++l) maxw = dims[l] > maxw ? dims[l] : maxw;
#pragma omp parallel
  {
    std::vector<float> a(maxw), b(maxw);
#pragma omp for schedule(static)
    for (int64_t row = 0; row < n; ++row) {
      for (int i = 0; i < dims[0]; ++i) a[i] = in[row * dims[0] + i];
      const float* p = w;
      for (int l = 0; l < n_layers; ++l) {
        const int fi = dims[l], fo = dims[l + 1];
        const float* W = p;
        const float* bias = p + (int64_t)fi * fo;
        for (int o = 0; o < fo; ++o) {          // per-neuron loop
          double acc = 0.0;
          for (int i = 0; i < fi; ++i) acc += (double)W[(int64_t)o * fi + i] * (double)a[i];
          acc += (double)bias[o];
          float v = (float)acc;
          if (l < n_layers - 1 && !(v > 0.0f)) v = 0.0f;   // ReLU(x) = max(0, x)
          b[o] = v;
        }
        a.swap(b);
        p = bias + fo;
      }
      for (int o = 0; o < dims[n_layers]; ++o) out[row * dims[n_layers] + o] = a[o];
    }
  }
}

// ---- next row (embedding part): the embedding MLP in INT8 by static post-training
//      quantisation, symmetric scheme of Eqs. 4.31-4.33:
//        S = alpha / 127 (alpha mapped to the highest INT8 value),  x_q = clip(round(x / S), -127, 127).
//      Per layer l (the Q -> quantised node -> DQ chain of P:2725): the layer's input is quantised with the
//      per-tensor scale S_a[l] = alpha_a[l] / 127 (alpha_a = calibrated range of that activation, an INPUT of
//      this function), its weight with S_w[l] = max|W_l| / 127 (the weight range is known), the
//      products are summed exactly in integers and de-quantised:
//        y_o = float(sum_k x_q[k] w_q[o][k]) * (S_a S_w) + b_o ;  ReLU on hidden layers (biases stay fp32).
//      Every float step is a single fp32 operation (1 / S, x * that, rint = round-half-even, S_a * S_w, * , +; compile
//      with -ffp-contract=off), so the integer codes -- and with them the outputs -- are reproducible bit
//      for bit (reading Q21).
//      Round 2 (reading Q21, revised): the quotient x / S of Eq. 4.31 is evaluated as x * fl(1 / S) -- one
//      rounded fp32 multiplication by the rounded reciprocal of the scale, the arithmetic of INT8 inference pipelines and
//      of the FP8 row below.  It is the same real number; in fp32 it differs from the divided form on ~6e-5 of the values
//      (those within 3e-5 of a tie), by one code.
static inline int32_t quant_code(float x, float S) {
  const float r = 1.0f / S;
  float q = std::nearbyintf(x * r);                 // default rounding mode: to nearest, ties to even
  if (q > 127.0f) q = 127.0f;
  if (q < -127.0f) q = -127.0f;
  return (int32_t)q;
}

void orc_quantize(int64_t n, const float* x, float alpha, int8_t* codes, float* scale_out) {
  const float S = alpha / 127.0f;
  if (scale_out) *scale_out = S;
  for (int64_t i = 0; i < n; ++i) codes[i] = (int8_t)quant_code(x[i], S);
}

void orc_mlp_int8(int64_t n, int32_t n_layers, const int32_t* dims, const float* w, const float* in,
                  const float* act_alpha /*[n_layers]*/, float* out) {
  int32_t maxw = 0;
  for (int l = 0; l <= n_layers; ++l) maxw = dims[l] > maxw ? dims[l] : maxw;
  // weight codes and scales, once
  std::vector<std::vector<int32_t>> wq(n_layers);
  std::vector<float> sw(n_layers);
  {
    const float* p = w;
    for (int l = 0; l < n_layers; ++l) {
      const int64_t cnt = (int64_t)dims[l] * dims[l + 1];
      float m = 0.0f;
      for (int64_t i = 0; i < cnt; ++i) m = std::fabs(p[i]) > m ? std::fabs(p[i]) : m;
      sw[l] = m / 127.0f;
      wq[l].resize(cnt);
      for (int64_t i = 0; i < cnt; ++i) wq[l][i] = quant_code(p[i], sw[l]);
      p += cnt + dims[l + 1];
    }
  }
#pragma omp parallel
  {
    std::vector<float> a(maxw), b(maxw);
    std::vector<int32_t> aq(maxw);
#pragma omp for schedule(static)
    for (int64_t row = 0; row < n; ++row) {
      for (int i = 0; i < dims[0]; ++i) a[i] = in[row * dims[0] + i];
      const float* p = w;
      for (int l = 0; l < n_layers; ++l) {
        const int fi = dims[l], fo = dims[l + 1];
        const float* bias = p + (int64_t)fi * fo;
        const float sa = act_alpha[l] / 127.0f;
        const float sc = sa * sw[l];
        for (int i = 0; i < fi; ++i) aq[i] = quant_code(a[i], sa);
        for (int o = 0; o < fo; ++o) {
          int64_t acc = 0;
          for (int i = 0; i < fi; ++i) acc += (int64_t)aq[i] * wq[l][(int64_t)o * fi + i];
          const float prod = (float)acc * sc;
          float v = prod + bias[o];
          if (l < n_layers - 1 && !(v > 0.0f)) v = 0.0f;
          b[o] = v;
        }
        a.swap(b);
        p = bias + fo;
      }
      for (int o = 0; o < dims[n_layers]; ++o) out[row * dims[n_layers] + o] = a[o];
    }
  }
}

// ---- next row (GNN part): the message aggregation of Eq. 8.5 in PLAIN fp32 -- every sum
//      starts from 0 and adds its edges' encodings one by one in ascending edge id, each add a single rounded fp32
//      operation ("fp32 scatter").  The hot path's oracle (orc_scatter) accumulates in double; the
//      quantised path needs the aggregate itself reproducible bit for bit, because it feeds a quantiser (a last-bit
//      difference in m can move an INT8 code).  m [n_nodes, 2H] = [outgoing sum, incoming sum].
void orc_scatter_f32(int64_t n_nodes, int64_t n_edges, const int32_t* src, const int32_t* dst, const float* e, int32_t H,
                     float* m) {
  for (int64_t i = 0; i < n_nodes * 2 * H; ++i) m[i] = 0.0f;
  for (int64_t k = 0; k < n_edges; ++k) {               // ascending edge id
    float* mo = m + (int64_t)src[k] * 2 * H;
    float* mi = m + (int64_t)dst[k] * 2 * H + H;
    for (int c = 0; c < H; ++c) { mo[c] = mo[c] + e[k * H + c]; mi[c] = mi[c] + e[k * H + c]; }
  }
}

// ---- a2 rough graph: hit i on plane p connects to hits j of the same event on planes
//      p+1 .. min(p+G, L-1) iff d^2(i,j) < r2_max (Eq. 8.1; strict "<": P:2674).
//      Sequential loop over candidates in ascending index, as P:2674 describes, so edges come out in
//      (src asc, dst asc) order.  Hits of an event must be sorted by plane.
//      d^2 in fp32: ((a0-b0)^2 + (a1-b1)^2) + ... left to right, no FMA.
//      Returns E; writes at most `capacity` edges.  borderline (may be null): per emitted-or-not pair
//      inside |sqrt(d2_double) - sqrt(r2)| <= band, appended as (i, j) up to border_cap pairs.
static inline float d2_fp32(const float* a, const float* b, int d) {
  float s = 0.0f;
  for (int c = 0; c < d; ++c) {
    const float diff = a[c] - b[c];
    const float sq = diff * diff;
    s = (c == 0) ? sq : s + sq;
  }
  return s;
}

int64_t orc_build_graph(int32_t n_events, const int32_t* event_ptr, const uint8_t* plane,
                        int32_t n_planes, const float* emb, int32_t d, float r2_max, int32_t gap,
                        int32_t* src, int32_t* dst, int64_t capacity, double band,
                        int32_t* border_pairs, int64_t border_cap, int64_t* n_border) {
  int64_t E = 0, nb = 0;
  const double rr = std::sqrt((double)r2_max);
  for (int32_t ev = 0; ev < n_events; ++ev) {
    const int32_t lo = event_ptr[ev], hi = event_ptr[ev + 1];
    for (int32_t i = lo; i < hi; ++i) {
      const int pi = plane[i];
      if (pi > n_planes - 2) continue;
      for (int32_t j = i + 1; j < hi; ++j) {            // plane-sorted: candidates lie after i
        const int dp = (int)plane[j] - pi;
        if (dp < 1) continue;
        if (dp > gap) break;
        const float d2 = d2_fp32(emb + (int64_t)i * d, emb + (int64_t)j * d, d);
        if (d2 < r2_max) {
          if (E < capacity) { src[E] = i; dst[E] = j; }
          ++E;
        }
        if (border_pairs) {
          double dd = 0.0;
          for (int c = 0; c < d; ++c) {
            const double df = (double)emb[(int64_t)i * d + c] - (double)emb[(int64_t)j * d + c];
            dd += df * df;
          }
          if (std::fabs(std::sqrt(dd) - rr) <= band) {
            if (nb < border_cap) { border_pairs[2 * nb] = i; border_pairs[2 * nb + 1] = j; }
            ++nb;
          }
        }
      }
    }
  }
  if (n_border) *n_border = nb;
  return E;
}

// ---- next row: k_max-capped rough graph, P:2290 ("a maximum of k_max edges per
//      node is imposed ... a k_max-NN algorithm ... under a maximum squared distance") and Algorithm 1
//      (P:2664-2672): list L of (j, d_j) over the candidates of source i, sort by d ascending, take the
//      first k.  Candidates are the hits of planes p+1..p+G of the same event inside the radius
//      (d^2 < r2_max, same fp32 predicate as orc_build_graph); the sort is STABLE on the fp32 d^2, so
//      equal distances keep ascending j (reading Q2: order (d^2, then j)) -- this is also what
//      the thesis' streaming "replace the farthest if the new hit is closer" loop retains.
//      The kept neighbours are emitted in ascending j (edge order convention Q13).  k_max <= 0: no cap.
int64_t orc_build_graph_kmax(int32_t n_events, const int32_t* event_ptr, const uint8_t* plane,
                             int32_t n_planes, const float* emb, int32_t d, float r2_max, int32_t gap,
                             int32_t k_max, int32_t* src, int32_t* dst, int64_t capacity) {
  int64_t E = 0;
  std::vector<std::pair<float, int32_t>> L;
  std::vector<int32_t> keep;
  for (int32_t ev = 0; ev < n_events; ++ev) {
    const int32_t lo = event_ptr[ev], hi = event_ptr[ev + 1];
    for (int32_t i = lo; i < hi; ++i) {
      const int pi = plane[i];
      if (pi > n_planes - 2) continue;
      L.clear();
      for (int32_t j = i + 1; j < hi; ++j) {
        const int dp = (int)plane[j] - pi;
        if (dp < 1) continue;
        if (dp > gap) break;
        const float d2 = d2_fp32(emb + (int64_t)i * d, emb + (int64_t)j * d, d);
        if (d2 < r2_max) L.emplace_back(d2, j);
      }
      if (k_max > 0 && (int64_t)L.size() > k_max) {
        std::stable_sort(L.begin(), L.end(),
                         [](const std::pair<float, int32_t>& a, const std::pair<float, int32_t>& b) { return a.first < b.first; });
        L.resize(k_max);
      }
      keep.clear();
      for (const auto& q : L) keep.push_back(q.second);
      std::sort(keep.begin(), keep.end());
      for (int32_t j : keep) {
        if (E < capacity) { src[E] = i; dst[E] = j; }
        ++E;
      }
    }
  }
  return E;
}

// all candidate squared distances in double (for the radius calibration)
int64_t orc_candidate_d2(int32_t n_events, const int32_t* event_ptr, const uint8_t* plane,
                         int32_t n_planes, const float* emb, int32_t d, int32_t gap, double* out,
                         int64_t capacity) {
  int64_t n = 0;
  for (int32_t ev = 0; ev < n_events; ++ev) {
    const int32_t lo = event_ptr[ev], hi = event_ptr[ev + 1];
    for (int32_t i = lo; i < hi; ++i) {
      const int pi = plane[i];
      if (pi > n_planes - 2) continue;
      for (int32_t j = i + 1; j < hi; ++j) {
        const int dp = (int)plane[j] - pi;
        if (dp < 1) continue;
        if (dp > gap) break;
        double dd = 0.0;
        for (int c = 0; c < d; ++c) {
          const double df = (double)emb[(int64_t)i * d + c] - (double)emb[(int64_t)j * d + c];
          dd += df * df;
        }
        if (n < capacity) out[n] = dd;
        ++n;
      }
    }
  }
  return n;
}

// ---- a4 message, Eq. 8.5: m_l = [ sum_{l->j} e_lj , sum_{i->l} e_il ]; outgoing first.
//      Edge-order loop with double accumulators, rounded to fp32 once.  m is [n_nodes, 2H].
void orc_scatter(int64_t n_nodes, int64_t n_edges, const int32_t* src, const int32_t* dst,
                 const float* e, int32_t H, float* m) {
  std::vector<double> acc((size_t)n_nodes * 2 * H, 0.0);
  for (int64_t k = 0; k < n_edges; ++k) {
    double* mo = acc.data() + (int64_t)src[k] * 2 * H;        // outgoing sum of the source
    double* mi = acc.data() + (int64_t)dst[k] * 2 * H + H;    // incoming sum of the destination
    for (int c = 0; c < H; ++c) {
      mo[c] += (double)e[k * H + c];
      mi[c] += (double)e[k * H + c];
    }
  }
  for (int64_t i = 0; i < n_nodes * 2 * H; ++i) m[i] = (float)acc[i];
}

// ---- a3 encoders + a4-a6 message passing.
//      h0 = MLP_n(f_node); e0_ij = MLP_e([h0_i, h0_j]) (source first);
//      for k < n_iter: m = scatter(e^k); h^{k+1} = h^k + phi_k([h^k, m]);
//                      e^{k+1} = e^k + psi_k([h_i^{k+1}, h_j^{k+1}, e^k])   (distinct weights per k).
//      All GNN MLPs: n_layers matrices; hidden width H.  Weight pointers are given per MLP.
void orc_gnn_forward(int64_t n_nodes, int64_t n_edges, const int32_t* src, const int32_t* dst,
                     const float* f_node, int32_t H, int32_t n_layers, int32_t n_iter,
                     const float* w_node_enc, const float* w_edge_enc,
                     const float* const* w_node_net, const float* const* w_edge_net,
                     float* h /*[n_nodes,H] out*/, float* e /*[n_edges,H] out*/) {
  std::vector<int32_t> dn(n_layers + 1, H), de(n_layers + 1, H), d3(n_layers + 1, H);
  dn[0] = 3; de[0] = 2 * H; d3[0] = 3 * H;
  orc_mlp(n_nodes, n_layers, dn.data(), w_node_enc, f_node, h);
  std::vector<float> cat((size_t)(n_edges > n_nodes ? n_edges : n_nodes) * 3 * H);
  std::vector<float> upd((size_t)(n_edges > n_nodes ? n_edges : n_nodes) * H);
  std::vector<float> m((size_t)n_nodes * 2 * H);
  for (int64_t k = 0; k < n_edges; ++k) {
    std::memcpy(&cat[k * 2 * H], h + (int64_t)src[k] * H, sizeof(float) * H);
    std::memcpy(&cat[k * 2 * H + H], h + (int64_t)dst[k] * H, sizeof(float) * H);
  }
  orc_mlp(n_edges, n_layers, de.data(), w_edge_enc, cat.data(), e);
  for (int it = 0; it < n_iter; ++it) {
    orc_scatter(n_nodes, n_edges, src, dst, e, H, m.data());
    for (int64_t l = 0; l < n_nodes; ++l) {
      std::memcpy(&cat[l * 3 * H], h + l * H, sizeof(float) * H);
      std::memcpy(&cat[l * 3 * H + H], &m[l * 2 * H], sizeof(float) * 2 * H);
    }
    orc_mlp(n_nodes, n_layers, d3.data(), w_node_net[it], cat.data(), upd.data());
    for (int64_t i = 0; i < n_nodes * H; ++i) h[i] = h[i] + upd[i];          // residual
    for (int64_t k = 0; k < n_edges; ++k) {
      std::memcpy(&cat[k * 3 * H], h + (int64_t)src[k] * H, sizeof(float) * H);
      std::memcpy(&cat[k * 3 * H + H], h + (int64_t)dst[k] * H, sizeof(float) * H);
      std::memcpy(&cat[k * 3 * H + 2 * H], e + k * H, sizeof(float) * H);
    }
    orc_mlp(n_edges, n_layers, d3.data(), w_edge_net[it], cat.data(), upd.data());
    for (int64_t i = 0; i < n_edges * H; ++i) e[i] = e[i] + upd[i];          // residual
  }
}

// ---- a7 edge classifier: MLP ending in 1 unit + sigmoid; sigma(x) = 1/(1+e^-x)
void orc_edge_scores(int64_t n_edges, const float* e, int32_t H, int32_t n_layers, const float* w_cls,
                     float* scores, float* logits /*may be null*/) {
  std::vector<int32_t> dc(n_layers + 1, H);
  dc[n_layers] = 1;
  std::vector<float> lg((size_t)n_edges);
  orc_mlp(n_edges, n_layers, dc.data(), w_cls, e, lg.data());
  for (int64_t k = 0; k < n_edges; ++k) {
    scores[k] = (float)(1.0 / (1.0 + std::exp(-(double)lg[k])));
    if (logits) logits[k] = lg[k];
  }
}

// ---- NEXT-1: score cut + track building.  Purified hit graph = edges with
//      score >= score_min; tracks = its weakly connected components.  Plain union-find over the kept
//      edges (the textbook alternative to the DFS of Algs. 2-3, same result); the label of a hit is the
//      smallest hit index of its component (a hit without kept edges keeps its own index).
static int32_t uf_find(std::vector<int32_t>& parent, int32_t x) {
  while (parent[x] != x) { parent[x] = parent[parent[x]]; x = parent[x]; }
  return x;
}

void orc_wcc(int64_t n_hits, int64_t n_edges, const int32_t* src, const int32_t* dst, const float* scores,
             float score_min, int32_t* labels) {
  std::vector<int32_t> parent((size_t)n_hits);
  for (int64_t i = 0; i < n_hits; ++i) parent[i] = (int32_t)i;
  for (int64_t k = 0; k < n_edges; ++k) {
    if (!(scores[k] >= score_min)) continue;              // edges below the minimum score are removed
    const int32_t a = uf_find(parent, src[k]), b = uf_find(parent, dst[k]);
    if (a != b) { if (a < b) parent[b] = a; else parent[a] = b; }   // root = smallest index of the set
  }
  for (int64_t i = 0; i < n_hits; ++i) labels[i] = uf_find(parent, (int32_t)i);
}

// ---- next row: the GNN's MLPs in FP8 (e4m3: 1 sign, 4 exponent, 3 mantissa bits, bias 7, no
//      infinities, largest finite value 448, subnormals down to 2^-9) with static per-tensor scales.  The thesis treats INT8
//      only (Eqs. 4.31-4.33; "the quantization of the GNN holds the most potential"); this is the same
//      symmetric per-tensor scheme with the integer grid replaced by the e4m3 grid (reading Q26):
//        S = alpha / 448 (alpha mapped to the largest e4m3 value, as P:1487 maps it to 127),
//        x_q = e4m3( clip( x * fl(1 / S), -448, 448 ) ), round to nearest, ties to even (the scaling is ONE rounded fp32
//        multiplication by the rounded reciprocal, the arithmetic of hardware FP8 pipelines; every x_q is decided in that
//        precision on both sides),
//        y_o = float(sum_k x_q[k] w_q[o][k]) * (S_a S_w) + b_o ;  ReLU on hidden layers, biases fp32.
//      The products of two e4m3 values and their sum over <= 512 terms are exact in double, so the oracle's sum is the
//      exact one, rounded to fp32 once; the tensor core accumulates in fp32, so the GPU is compared within a tolerance.
static inline float e4m3_round(float t) {                // nearest e4m3 value of a finite t, ties to even, saturating
  const float a = std::fabs(t);
  if (!(a < 448.0f)) return t < 0.0f ? -448.0f : 448.0f;
  int e;
  std::frexp(a, &e);                                     // a = m 2^e, m in [0.5, 1)  ->  floor(log2 a) = e - 1
  int le = (a == 0.0f) ? -6 : e - 1;
  if (le < -6) le = -6;                                  // subnormal range: spacing 2^-9
  const float ulp = std::ldexp(1.0f, le - 3);            // 3 mantissa bits
  const float r = std::nearbyintf(a / ulp) * ulp;        // power-of-two scaling is exact; nearbyint rounds half to even
  return t < 0.0f ? -r : r;
}

void orc_quantize_fp8(int64_t n, const float* x, float alpha, float* values, float* scale_out) {
  const float S = alpha / 448.0f;
  const float rS = 1.0f / S;
  if (scale_out) *scale_out = S;
  for (int64_t i = 0; i < n; ++i) values[i] = e4m3_round(x[i] * rS);
}

void orc_mlp_fp8(int64_t n, int32_t n_layers, const int32_t* dims, const float* w, const float* in,
                 const float* act_alpha /*[n_layers]*/, float* out) {
  int32_t maxw = 0;
  for (int l = 0; l <= n_layers; ++l) maxw = dims[l] > maxw ? dims[l] : maxw;
  std::vector<std::vector<float>> wq(n_layers);          // e4m3 VALUES of the scaled weights
  std::vector<float> sw(n_layers);
  {
    const float* p = w;
    for (int l = 0; l < n_layers; ++l) {
      const int64_t cnt = (int64_t)dims[l] * dims[l + 1];
      float m = 0.0f;
      for (int64_t i = 0; i < cnt; ++i) m = std::fabs(p[i]) > m ? std::fabs(p[i]) : m;
      sw[l] = m / 448.0f;
      const float rs = 1.0f / sw[l];
      wq[l].resize(cnt);
      for (int64_t i = 0; i < cnt; ++i) wq[l][i] = e4m3_round(p[i] * rs);
      p += cnt + dims[l + 1];
    }
  }
#pragma omp parallel
  {
    std::vector<float> a(maxw), b(maxw), aq(maxw);
#pragma omp for schedule(static)
    for (int64_t row = 0; row < n; ++row) {
      for (int i = 0; i < dims[0]; ++i) a[i] = in[row * dims[0] + i];
      const float* p = w;
      for (int l = 0; l < n_layers; ++l) {
        const int fi = dims[l], fo = dims[l + 1];
        const float* bias = p + (int64_t)fi * fo;
        const float sa = act_alpha[l] / 448.0f;
        const float rsa = 1.0f / sa;
        const float sc = sa * sw[l];
        for (int i = 0; i < fi; ++i) aq[i] = e4m3_round(a[i] * rsa);
        for (int o = 0; o < fo; ++o) {
          double acc = 0.0;                              // exact: products have <= 8 significant bits, <= 512 terms
          for (int i = 0; i < fi; ++i) acc += (double)aq[i] * (double)wq[l][(int64_t)o * fi + i];
          const float prod = (float)acc * sc;
          float v = prod + bias[o];
          if (l < n_layers - 1 && !(v > 0.0f)) v = 0.0f;
          b[o] = v;
        }
        a.swap(b);
        p = bias + fo;
      }
      for (int o = 0; o < dims[n_layers]; ++o) out[row * dims[n_layers] + o] = a[o];
    }
  }
}

}  // extern "C"
