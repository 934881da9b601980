// Next row: the thesis' own rough-graph definition — the fixed-radius graph with at
// most k_max out-edges per hit, the k_max nearest candidates ("a maximum of k_max edges per node is
// imposed", Algorithm 1; k_max = 50, d2_max = 0.9 in the thesis).  Order of candidates:
// (d^2 in fp32, then hit index), so equal distances keep the lower index — what the thesis' streaming
// "replace the farthest if the new hit is closer" loop retains (reading Q2).
//
// The thesis kept a k_max-slot list per thread and replaced its farthest entry.  Here one warp owns a source
// hit, as in graph.cu: a count pass (degree = min(in-radius candidates, k_max)), a scan, and a fill pass.
// A source over the cap (the thesis: < 0.1 % of hits) finds the k_max-th smallest key (d^2 bits : index) by
// a bitwise bisection — 64 warp-wide counting sweeps over its candidate window, no list, no sort, no
// shared memory — and then emits the candidates with key <= threshold in ascending index through the same
// ballot / popc compaction, so the CSR is again the unique ordered array.  The by-destination lists need
// the capped forward lists: a hit counts (and then locates, by binary search) itself in the neighbour
// lists of its in-radius source candidates, sources ascending = edge ids ascending.
#include "common.cuh"

namespace etx {
namespace {

constexpr int kWarpsPerBlock = 8;
constexpr unsigned kFull = 0xffffffffu;

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

// Destination side, after the forward lists exist.  FILL = false: in_deg[i]; FILL = true: in_perm.
template <bool FILL>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
kmax_backward_kernel(GraphArgs a, const int32_t* __restrict__ plane_ptr, const int32_t* __restrict__ hit_event,
                     const int32_t* __restrict__ flags, const int32_t* __restrict__ row_ptr,
                     const int32_t* __restrict__ dst, int32_t* __restrict__ in_deg,
                     const int32_t* __restrict__ in_ptr, int32_t* __restrict__ in_perm) {
  if (flags[0] != 0) return;
  const int lane = threadIdx.x & 31;
  const int warp = blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  const int n_warps = gridDim.x * kWarpsPerBlock;
  const unsigned lt = (1u << lane) - 1u;
  const int L = a.n_planes;
  for (int i = warp; i < a.n_hits; i += n_warps) {
    const int p = a.plane[i];
    int cnt = 0;
    if (p >= 1) {
      const int32_t* pp = plane_ptr + (size_t)hit_event[i] * (L + 1);
      const int bot = (p - a.gap > 0) ? p - a.gap : 0;
      const int s0 = pp[bot], s1 = pp[p];
      const int base_in = FILL ? in_ptr[i] : 0;
      for (int base = s0; base < s1; base += 32) {
        const int sidx = base + lane;
        bool ok = false;
        int lo = 0;
        if (sidx < s1 && dist2(a.emb, sidx, i, a.d) < a.r2_max) {       // source first, as in the forward pass
          int hi = row_ptr[sidx + 1];
          lo = row_ptr[sidx];
          const int end = hi;
          while (lo < hi) {                                              // is i in the source's (capped) list?
            const int mid = (lo + hi) >> 1;
            if (dst[mid] < i) lo = mid + 1; else hi = mid;
          }
          ok = lo < end && dst[lo] == i;
        }
        const unsigned b = __ballot_sync(kFull, ok);
        if (FILL && ok) in_perm[base_in + cnt + __popc(b & lt)] = lo;
        cnt += __popc(b);
      }
    }
    if (!FILL && lane == 0) in_deg[i] = cnt;
  }
  if (!FILL && blockIdx.x == 0 && threadIdx.x == 0) in_deg[a.n_hits] = 0;
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

int launch_kmax_in_count(const GraphArgs& a, const int32_t* plane_ptr, const int32_t* hit_event, const int32_t* flags,
                         const int32_t* row_ptr, const int32_t* dst, int32_t* in_deg, cudaStream_t s) {
  kmax_backward_kernel<false><<<search_grid(a.n_hits), kWarpsPerBlock * 32, 0, s>>>(a, plane_ptr, hit_event, flags, row_ptr,
                                                                                    dst, in_deg, nullptr, nullptr);
  return 1;
}

int launch_kmax_in_fill(const GraphArgs& a, const int32_t* plane_ptr, const int32_t* hit_event, const int32_t* flags,
                        const int32_t* row_ptr, const int32_t* dst, const int32_t* in_ptr, int32_t* in_perm,
                        cudaStream_t s) {
  kmax_backward_kernel<true><<<search_grid(a.n_hits), kWarpsPerBlock * 32, 0, s>>>(a, plane_ptr, hit_event, flags, row_ptr,
                                                                                   dst, nullptr, in_ptr, in_perm);
  return 1;
}

}  // namespace etx
