// Next row: the thesis' own rough-graph definition — the fixed-radius graph with at
// most k_max out-edges per hit, the k_max nearest candidates ("a maximum of k_max edges per node is
// imposed", Algorithm 1; k_max = 50, d2_max = 0.9 in the thesis).  Order of candidates:
// (d^2 in fp32, then hit index), so equal distances keep the lower index — what the thesis' streaming
// "replace the farthest if the new hit is closer" loop retains (reading Q2).
//
// The thesis kept a k_max-slot list per thread and replaced its farthest entry.  Here one warp owns a source
// hit, as in graph.cu: a count pass (degree = min(in-radius candidates, k_max)), a scan, and a fill pass.
// A source over the cap (the thesis: < 0.1 % of hits) with at most 128 candidates inside the radius compacts
// their keys (d^2 bits : index) into a per-warp shared-memory list and every lane ranks its own keys against
// the list (rank < k_max = kept); a longer list finds the k_max-th smallest key by a bitwise bisection (64
// warp-wide counting sweeps over the candidate window, no list, no sort).  Either way the kept candidates
// are emitted in ascending index through the same ballot / popc compaction, so the CSR is again the unique
// ordered array.  The by-destination lists are built from the
// capped edge list with integer counters, a cursor and graph.cu's per-segment sort (no second search).
//
// Since round 2 a 4-dimensional embedding takes the tiled search of graph.cu with a vote-clearing cap kernel
// (search_kmax_cap_kernel); these kernels serve the other dimensions and windows longer than the kept vote words.
#include "common.cuh"

namespace etx {
namespace {

constexpr int kWarpsPerBlock = 8;
constexpr unsigned kFull = 0xffffffffu;
constexpr int kListMax = 128;                   // in-radius candidates ranked in shared memory (4 per lane)

__device__ __forceinline__ float dist2(const float* __restrict__ emb, int i, int j, int d) {
  float s = 0.0f;
  for (int c = 0; c < d; ++c) {                    // fp32, left to right, no FMA contraction (as graph.cu)
    const float diff = __fsub_rn(__ldg(emb + (size_t)i * d + c), __ldg(emb + (size_t)j * d + c));
    const float sq = __fmul_rn(diff, diff);
    s = (c == 0) ? sq : __fadd_rn(s, sq);
  }
  return s;
}

__device__ __forceinline__ unsigned long long key_of(float d2, int j) {
  return ((unsigned long long)__float_as_uint(d2) << 32) | (unsigned)j;   // d2 >= 0: bit pattern is monotone
}

// FILL = false: out_deg[i] = min(#candidates inside the radius, k_max).   FILL = true: write src / dst.
template <bool FILL>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
kmax_forward_kernel(GraphArgs a, int k_max, const int32_t* __restrict__ plane_ptr,
                    const int32_t* __restrict__ hit_event, const int32_t* __restrict__ flags,
                    int32_t* __restrict__ out_deg, const int32_t* __restrict__ row_ptr,
                    int32_t* __restrict__ src, int32_t* __restrict__ dst) {
  if (flags[0] != 0) return;
  __shared__ unsigned long long s_keys[FILL ? kWarpsPerBlock : 1][FILL ? kListMax : 1];
  const int lane = threadIdx.x & 31;
  const int warp = blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  const int n_warps = gridDim.x * kWarpsPerBlock;
  const unsigned lt = (1u << lane) - 1u;
  const int L = a.n_planes;
  for (int i = warp; i < a.n_hits; i += n_warps) {
    const int p = a.plane[i];
    int j0 = 0, j1 = 0;
    if (p <= L - 2) {
      const int32_t* pp = plane_ptr + (size_t)hit_event[i] * (L + 1);
      const int top = (p + a.gap < L - 1) ? p + a.gap : L - 1;
      j0 = pp[p + 1];
      j1 = pp[top + 1];
    }
    if (!FILL) {
      int cnt = 0;
      for (int base = j0; base < j1; base += 32) {
        const int j = base + lane;
        const bool ok = j < j1 && dist2(a.emb, i, j, a.d) < a.r2_max;
        cnt += __popc(__ballot_sync(kFull, ok));
      }
      if (lane == 0) out_deg[i] = cnt < k_max ? cnt : k_max;
      continue;
    }
    const int begin = row_ptr[i], deg = row_ptr[i + 1] - begin;
    if (deg == 0) continue;
    unsigned long long thr = ~0ull;                // keep every candidate inside the radius ...
    if (deg == k_max) {                            // ... unless the cap may bind: threshold = k_max-th smallest key
      int total = 0;
      for (int base = j0; base < j1; base += 32) {
        const int j = base + lane;
        const bool ok = j < j1 && dist2(a.emb, i, j, a.d) < a.r2_max;
        total += __popc(__ballot_sync(kFull, ok));
      }
      if (total > k_max && total <= kListMax) {
        // short list: compact the keys (ascending index = ascending slot), rank, emit
        unsigned long long* keys = s_keys[FILL ? (threadIdx.x >> 5) : 0];
        int n = 0;
        for (int base = j0; base < j1; base += 32) {
          const int j = base + lane;
          bool ok = false;
          float d2 = 0.f;
          if (j < j1) { d2 = dist2(a.emb, i, j, a.d); ok = d2 < a.r2_max; }
          const unsigned b = __ballot_sync(kFull, ok);
          if (ok) keys[n + __popc(b & lt)] = key_of(d2, j);
          n += __popc(b);
        }
        __syncwarp();
        int cnt = 0;
        for (int t0 = 0; t0 < total; t0 += 32) {
          const int slot = t0 + lane;
          bool keep = false;
          unsigned long long mine = 0ull;
          if (slot < total) {
            mine = keys[slot];
            int rank = 0;
            for (int m = 0; m < total; ++m) rank += keys[m] < mine;
            keep = rank < k_max;
          }
          const unsigned b = __ballot_sync(kFull, keep);
          if (keep) {
            const int pos = begin + cnt + __popc(b & lt);
            src[pos] = i;
            dst[pos] = (int)(unsigned)(mine & 0xffffffffull);
          }
          cnt += __popc(b);
        }
        __syncwarp();
        continue;
      }
      if (total > k_max) {
        thr = 0ull;                                // invariant: thr <= k-th smallest key
        for (int bit = 63; bit >= 0; --bit) {
          const unsigned long long cand = thr | (1ull << bit);
          int below = 0;
          for (int base = j0; base < j1; base += 32) {
            const int j = base + lane;
            bool ok = false;
            if (j < j1) {
              const float d2 = dist2(a.emb, i, j, a.d);
              ok = d2 < a.r2_max && key_of(d2, j) < cand;
            }
            below += __popc(__ballot_sync(kFull, ok));
          }
          if (below < k_max) thr = cand;           // fewer than k keys below cand: the k-th one is >= cand
        }
      }
    }
    int cnt = 0;
    for (int base = j0; base < j1; base += 32) {
      const int j = base + lane;
      bool ok = false;
      if (j < j1) {
        const float d2 = dist2(a.emb, i, j, a.d);
        ok = d2 < a.r2_max && key_of(d2, j) <= thr;
      }
      const unsigned b = __ballot_sync(kFull, ok);
      if (ok) {
        const int pos = begin + cnt + __popc(b & lt);
        src[pos] = i;
        dst[pos] = j;
      }
      cnt += __popc(b);
    }
  }
}

// Destination side, after the capped forward lists exist: in-degrees by integer atomics over the edge list,
// scan, every edge id dropped into its destination's segment through an integer cursor; graph.cu's segment
// sort then orders each list ascending.
__global__ void __launch_bounds__(256) kmax_in_degree_kernel(int64_t n_edges, const int32_t* __restrict__ dst,
                                                             int32_t* __restrict__ in_deg) {
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n_edges; e += (int64_t)gridDim.x * blockDim.x)
    atomicAdd(&in_deg[dst[e]], 1);
}
__global__ void __launch_bounds__(256) kmax_in_scatter_kernel(int64_t n_edges, const int32_t* __restrict__ dst,
                                                              const int32_t* __restrict__ in_ptr, int32_t* __restrict__ cursor,
                                                              int32_t* __restrict__ in_perm) {
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n_edges; e += (int64_t)gridDim.x * blockDim.x) {
    const int j = dst[e];
    in_perm[in_ptr[j] + atomicAdd(&cursor[j], 1)] = (int32_t)e;
  }
}

inline int search_grid(int n_hits) {
  const int need = (n_hits + kWarpsPerBlock - 1) / kWarpsPerBlock;
  const int cap = 148 * 8;
  return need < 1 ? 1 : (need < cap ? need : cap);
}

}  // namespace

int launch_kmax_count(const GraphArgs& a, int k_max, const int32_t* plane_ptr, const int32_t* hit_event,
                      const int32_t* flags, int32_t* out_deg, cudaStream_t s) {
  kmax_forward_kernel<false><<<search_grid(a.n_hits), kWarpsPerBlock * 32, 0, s>>>(a, k_max, plane_ptr, hit_event, flags,
                                                                                   out_deg, nullptr, nullptr, nullptr);
  cudaMemsetAsync(out_deg + a.n_hits, 0, sizeof(int32_t), s);
  return 1;
}

int launch_kmax_fill(const GraphArgs& a, int k_max, const int32_t* plane_ptr, const int32_t* hit_event,
                     const int32_t* flags, const int32_t* row_ptr, int32_t* src, int32_t* dst, cudaStream_t s) {
  kmax_forward_kernel<true><<<search_grid(a.n_hits), kWarpsPerBlock * 32, 0, s>>>(a, k_max, plane_ptr, hit_event, flags,
                                                                                  nullptr, row_ptr, src, dst);
  return 1;
}

int launch_kmax_in_count(const GraphArgs& a, int64_t n_edges, const int32_t* dst, int32_t* in_deg, cudaStream_t s) {
  cudaMemsetAsync(in_deg, 0, sizeof(int32_t) * ((size_t)a.n_hits + 1), s);
  if (n_edges <= 0) return 0;
  const int64_t need = (n_edges + 255) / 256;
  kmax_in_degree_kernel<<<(int)(need < 148 * 16 ? need : 148 * 16), 256, 0, s>>>(n_edges, dst, in_deg);
  return 1;
}

int launch_kmax_in_fill(const GraphArgs& a, int64_t n_edges, const int32_t* flags, const int32_t* dst, const int32_t* in_ptr,
                        int32_t* in_perm, int32_t* cursor, cudaStream_t s) {
  if (n_edges <= 0) return 0;
  cudaMemsetAsync(cursor, 0, sizeof(int32_t) * (size_t)a.n_hits, s);
  const int64_t need = (n_edges + 255) / 256;
  kmax_in_scatter_kernel<<<(int)(need < 148 * 16 ? need : 148 * 16), 256, 0, s>>>(n_edges, dst, in_ptr, cursor, in_perm);
  return 1 + launch_sort_in_lists(a.n_hits, flags, in_ptr, in_perm, s);
}

}  // namespace etx
