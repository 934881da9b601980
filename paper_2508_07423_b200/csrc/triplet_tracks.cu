// NEXT-4 (rest) — track building from triplets, the four steps of P:2363 (section 8.3.5), on the GPU.
// The thesis ran this step in Python only.  Reading of the four steps: DESIGN.md Q23 and include/etx.h.
// Integer work throughout: every output is one fixed array (the tests compare them bit for bit with a CPU reference).
//
// Nodes of the EDGE graph = kept edges (score >= score_min); connections = kept triplets (triplet score >= trip_min).
//   1. elbows connect: min-label propagation over the kept elbow rows -> super-edges (label = smallest edge id);
//      a kept articulation row (a, b) becomes the pair (S(a), S(b)); pairs inside one super-edge vanish; duplicates
//      need no removal here because "shared" is decided by min != max over the partners:
//   2. (u, v) is SHARED iff u has two distinct successors (min successor != max successor) or v two distinct
//      predecessors.  A second propagation over elbows + unshared articulations gives the connected sets.
//   3. every distinct (set(u), set(v)) of a shared articulation is a joined track; an untouched set is a track.
//   4. edges -> hits: (set, hit) memberships are sorted per event, so every set's hits come out ascending.
// One CTA owns an event in the iterative kernels (an event's edge ids, triplet rows and hits are contiguous ranges,
// so CTAs never touch each other's entries of the batch-wide scratch arrays).
#include <algorithm>
#include <climits>

#include "common.cuh"

namespace etx {
namespace {

constexpr int kThreads = 256;
constexpr unsigned long long kInfKey = ~0ull;

struct TtArgs {
  int n_events, n_hits;
  long long n_edges, n_art, n_left, n_right;
  const int32_t* event_ptr; const int32_t* row_ptr; const int32_t* in_ptr; const int32_t* in_perm;
  const float* scores; float score_min;
  const int32_t* tptr;                 // [3][n_hits + 1] CSR of the triplet rows by shared hit
  const int32_t* first; const int32_t* second; const float* tscores; float trip_min;
  int32_t* label;                      // [E] out: connected set of every edge (-1 = cut)
  int32_t *mn_out, *mx_out, *mn_in, *mx_in;   // [E + 1] scratch (later: set_start, set_end, touched, plain flags / scan)
  unsigned char* art_flag;             // [n_art] 0 = dropped / vanished, 1 = unshared, 2 = shared
  unsigned long long* jkey;            // [n_art] (set(a) << 32 | set(b)) of a shared row, else kInfKey
};

// ---- steps 1-3 on one event per CTA
__global__ void __launch_bounds__(kThreads) tt_sets_kernel(TtArgs a) {
  __shared__ int changed;
  const size_t ld = (size_t)a.n_hits + 1;
  for (int ev = blockIdx.x; ev < a.n_events; ev += gridDim.x) {
    const int h0 = a.event_ptr[ev], h1 = a.event_ptr[ev + 1];
    const int e0 = a.row_ptr[h0], e1 = a.row_ptr[h1];
    const long long a0 = a.tptr[h0], a1 = a.tptr[h1];                                   // articulation rows
    const long long l0 = a.n_art + a.tptr[ld + h0], l1 = a.n_art + a.tptr[ld + h1];       // left elbows
    const long long r0 = a.n_art + a.n_left + a.tptr[2 * ld + h0], r1 = a.n_art + a.n_left + a.tptr[2 * ld + h1];
    for (int e = e0 + threadIdx.x; e < e1; e += kThreads) {
      a.label[e] = a.scores[e] >= a.score_min ? e : -1;
      a.mn_out[e] = INT_MAX; a.mx_out[e] = -1; a.mn_in[e] = INT_MAX; a.mx_in[e] = -1;
    }
    __syncthreads();
    // min-label propagation over connection rows until nothing changes; `with_art`: also the unshared articulations
    auto propagate = [&](bool with_art) {
      for (;;) {
        if (threadIdx.x == 0) changed = 0;
        __syncthreads();
        int local = 0;
        auto relax = [&](long long row) {
          const int x = a.first[row], y = a.second[row];
          const int lx = ((volatile int32_t*)a.label)[x], ly = ((volatile int32_t*)a.label)[y];
          if (lx < 0 || ly < 0) return;                   // a row over a cut edge (triplets built with another cut): no connection
          if (lx < ly) { if (atomicMin(&a.label[y], lx) > lx) local = 1; }
          else if (ly < lx) { if (atomicMin(&a.label[x], ly) > ly) local = 1; }
        };
        for (long long r = l0 + threadIdx.x; r < l1; r += kThreads) if (a.tscores[r] >= a.trip_min) relax(r);
        for (long long r = r0 + threadIdx.x; r < r1; r += kThreads) if (a.tscores[r] >= a.trip_min) relax(r);
        if (with_art)
          for (long long r = a0 + threadIdx.x; r < a1; r += kThreads) if (a.art_flag[r] == 1) relax(r);
        if (local) changed = 1;
        __syncthreads();
        const int again = changed;
        __syncthreads();
        if (!again) break;
      }
    };
    propagate(false);                                     // step 1: super-edges
    for (long long r = a0 + threadIdx.x; r < a1; r += kThreads) {
      if (!(a.tscores[r] >= a.trip_min)) continue;
      const int u = a.label[a.first[r]], v = a.label[a.second[r]];
      if (u == v || u < 0 || v < 0) continue;
      atomicMin(&a.mn_out[u], v); atomicMax(&a.mx_out[u], v);
      atomicMin(&a.mn_in[v], u); atomicMax(&a.mx_in[v], u);
    }
    __syncthreads();
    for (long long r = a0 + threadIdx.x; r < a1; r += kThreads) {
      unsigned char f = 0;
      if (a.tscores[r] >= a.trip_min) {
        const int u = a.label[a.first[r]], v = a.label[a.second[r]];
        if (u != v && u >= 0 && v >= 0) f = (a.mn_out[u] != a.mx_out[u] || a.mn_in[v] != a.mx_in[v]) ? 2 : 1;
      }
      a.art_flag[r] = f;
    }
    __syncthreads();
    propagate(true);                                      // step 2: connected sets without the shared articulations
    for (int e = e0 + threadIdx.x; e < e1; e += kThreads) a.mn_in[e] = 0;        // mn_in becomes `touched`
    __syncthreads();
    for (long long r = a0 + threadIdx.x; r < a1; r += kThreads) {                // step 3: the joins
      unsigned long long key = kInfKey;
      if (a.art_flag[r] == 2) {
        const int sa = a.label[a.first[r]], sb = a.label[a.second[r]];
        key = ((unsigned long long)(unsigned)sa << 32) | (unsigned)sb;
        a.mn_in[sa] = 1; a.mn_in[sb] = 1;
      }
      a.jkey[r] = key;
    }
    __syncthreads();
  }
}

// ---- ascending sort of every event's segment [off[h0], off[h1]) of 64-bit keys (bitonic network in its all-ascending
// "flip" form, so the virtual +inf padding up to a power of two never moves and is simply skipped)
__global__ void __launch_bounds__(kThreads) seg_sort_kernel(int n_events, const int32_t* __restrict__ event_ptr,
                                                            const int32_t* __restrict__ off, unsigned long long* keys) {
  for (int ev = blockIdx.x; ev < n_events; ev += gridDim.x) {
    const long long b = off[event_ptr[ev]];
    const int n = (int)(off[event_ptr[ev + 1]] - b);
    if (n > 1) {
      unsigned long long* k = keys + b;
      int p = 1;
      while (p < n) p <<= 1;
      for (int size = 2; size <= p; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
          for (int t = threadIdx.x; t < (p >> 1); t += kThreads) {
            int lo, hi;
            if (stride == (size >> 1)) {                  // first step of a merge: mirror pairs inside the block
              const int blk = t / stride, j = t % stride;
              lo = blk * size + j; hi = blk * size + size - 1 - j;
            } else {
              lo = (t / stride) * 2 * stride + (t % stride); hi = lo + stride;
            }
            if (hi < n) {
              const unsigned long long x = k[lo], y = k[hi];
              if (x > y) { k[lo] = y; k[hi] = x; }
            }
          }
          __syncthreads();
        }
      }
    }
    __syncthreads();
  }
}

__global__ void __launch_bounds__(kThreads) tt_join_heads_kernel(long long n, const unsigned long long* __restrict__ jkey,
                                                                 int32_t* __restrict__ head /*[n+1]*/) {
  const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (i == 0) head[n] = 0;
  if (i >= n) return;
  const unsigned long long k = jkey[i];
  head[i] = (k != kInfKey && (i == 0 || jkey[i - 1] != k)) ? 1 : 0;
}

__global__ void __launch_bounds__(kThreads) tt_join_compact_kernel(long long n, const unsigned long long* __restrict__ jkey,
                                                                   const int32_t* __restrict__ pos,
                                                                   unsigned long long* __restrict__ out) {
  const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (i >= n) return;
  if (pos[i + 1] != pos[i]) out[pos[i]] = jkey[i];
}

__global__ void __launch_bounds__(kThreads) tt_plain_flags_kernel(long long n, const int32_t* __restrict__ label,
                                                                  const int32_t* __restrict__ touched, int32_t* __restrict__ flag) {
  const long long e = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (e == 0) flag[n] = 0;
  if (e >= n) return;
  flag[e] = (label[e] == (int)e && !touched[e]) ? 1 : 0;
}

__global__ void __launch_bounds__(kThreads) tt_plain_scatter_kernel(long long n, const int32_t* __restrict__ pos,
                                                                    int32_t* __restrict__ plain_label) {
  const long long e = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (e >= n) return;
  if (pos[e + 1] != pos[e]) plain_label[pos[e]] = (int)e;
}

// ---- step 4: (set, hit) memberships.  A hit belongs to the sets of its kept incident edges (each set once).
template <bool FILL>
__global__ void __launch_bounds__(kThreads) tt_member_kernel(int n_hits, const int32_t* __restrict__ row_ptr,
                                                             const int32_t* __restrict__ in_ptr,
                                                             const int32_t* __restrict__ in_perm,
                                                             const int32_t* __restrict__ label, int32_t* __restrict__ mptr,
                                                             unsigned long long* __restrict__ mkey) {
  const int h = blockIdx.x * kThreads + threadIdx.x;
  if (!FILL && h == 0) mptr[n_hits] = 0;
  if (h >= n_hits) return;
  const int o0 = row_ptr[h], no = row_ptr[h + 1] - o0, i0 = in_ptr[h], ni = in_ptr[h + 1] - i0;
  auto lab_at = [&](int q) { return label[q < no ? o0 + q : in_perm[i0 + q - no]]; };
  int cnt = 0;
  long long w = FILL ? mptr[h] : 0;
  for (int q = 0; q < no + ni; ++q) {
    const int L = lab_at(q);
    if (L < 0) continue;
    bool seen = false;
    for (int p = 0; p < q && !seen; ++p) seen = lab_at(p) == L;
    if (seen) continue;
    if (FILL) mkey[w + cnt] = ((unsigned long long)(unsigned)L << 32) | (unsigned)h;
    ++cnt;
  }
  if (!FILL) mptr[h] = cnt;
}

__global__ void __launch_bounds__(kThreads) tt_set_ranges_kernel(long long m, const unsigned long long* __restrict__ mkey,
                                                                 int32_t* __restrict__ set_start, int32_t* __restrict__ set_end) {
  const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (i >= m) return;
  const int L = (int)(mkey[i] >> 32);
  if (i == 0 || (int)(mkey[i - 1] >> 32) != L) set_start[L] = (int)i;
  if (i == m - 1 || (int)(mkey[i + 1] >> 32) != L) set_end[L] = (int)(i + 1);
}

// track t < n_plain: the untouched set plain_label[t]; else the join (a, b): ascending duplicate-free merge of two sets
template <bool FILL>
__global__ void __launch_bounds__(kThreads) tt_tracks_kernel(long long n_plain, long long n_joins,
                                                             const int32_t* __restrict__ plain_label,
                                                             const unsigned long long* __restrict__ joins,
                                                             const unsigned long long* __restrict__ mkey,
                                                             const int32_t* __restrict__ set_start,
                                                             const int32_t* __restrict__ set_end, int32_t* __restrict__ track_ptr,
                                                             int32_t* __restrict__ track_hits) {
  const long long t = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (!FILL && t == 0) track_ptr[n_plain + n_joins] = 0;
  if (t >= n_plain + n_joins) return;
  int sa, sb = -1;
  if (t < n_plain) sa = plain_label[t];
  else { const unsigned long long k = joins[t - n_plain]; sa = (int)(k >> 32); sb = (int)(k & 0xffffffffu); }
  int i = set_start[sa];
  const int ie = set_end[sa];
  int j = (sb >= 0 && sb != sa) ? set_start[sb] : 0;
  const int je = (sb >= 0 && sb != sa) ? set_end[sb] : 0;
  long long w = FILL ? track_ptr[t] : 0;
  int cnt = 0;
  while (i < ie || j < je) {
    const unsigned hi = i < ie ? (unsigned)(mkey[i] & 0xffffffffu) : 0xffffffffu;
    const unsigned hj = j < je ? (unsigned)(mkey[j] & 0xffffffffu) : 0xffffffffu;
    const unsigned hmin = hi < hj ? hi : hj;
    if (FILL) track_hits[w + cnt] = (int)hmin;
    ++cnt;
    if (hi == hmin) ++i;
    if (hj == hmin) ++j;
  }
  if (!FILL) track_ptr[t] = cnt;
}

__global__ void __launch_bounds__(kThreads) tt_unpack_joins_kernel(long long n, const unsigned long long* __restrict__ joins,
                                                                   int32_t* __restrict__ out /*[n][2]*/) {
  const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
  if (i >= n) return;
  out[2 * i] = (int)(joins[i] >> 32);
  out[2 * i + 1] = (int)(joins[i] & 0xffffffffu);
}

inline int grid_for(long long n) { return (int)((n + kThreads - 1) / kThreads > 0 ? (n + kThreads - 1) / kThreads : 1); }
inline size_t up256(size_t x) { return (x + 255) / 256 * 256; }

}  // namespace

size_t triplet_tracks_ws_bytes(int n_hits, long long n_edges, long long n_art) {
  const size_t E1 = (size_t)n_edges + 1, A1 = (size_t)n_art + 1;
  size_t b = 0;
  b += 4 * up256(4 * E1);                      // mn_out, mx_out, mn_in, mx_in
  b += up256(4 * E1);                          // plain_label
  b += up256(A1) + 2 * up256(8 * A1) + up256(4 * A1);   // art_flag, jkey, joins (compacted), join heads / positions
  b += up256(4 * ((size_t)n_hits + 1));        // mptr
  b += up256(8 * (2 * (size_t)n_edges + 1));   // mkey (a hit is in at most one set per incident edge)
  b += up256(4 * (E1 + A1));                   // track sizes / offsets until the capacities are known
  b += up256(4 * scan_tmp_ints((int)(n_edges + n_art + n_hits) + 2));
  b += 256;
  return b;
}

// Runs the whole procedure.  counts[4] = {n_joins, n_plain, n_tracks, n_track_hits}.  Returns the number of launches,
// or -1 after a CUDA error on the synchronisations; outputs are written only if every capacity suffices
// (*capacity_ok says so).
int run_triplet_tracks(int n_events, int n_hits, long long n_edges, const int32_t* event_ptr, const int32_t* row_ptr,
                       const int32_t* in_ptr, const int32_t* in_perm, const float* scores, float score_min,
                       const int32_t* tptr, const long long n_trip[3], const int32_t* first, const int32_t* second,
                       const float* tscores, float trip_min, char* ws, int32_t* d_edge_set, long long join_capacity,
                       int32_t* d_joins, long long track_capacity, int32_t* d_track_ptr, long long hit_capacity,
                       int32_t* d_track_hits, long long counts[4], bool* capacity_ok, cudaStream_t s) {
  const size_t E1 = (size_t)n_edges + 1, A1 = (size_t)n_trip[0] + 1;
  size_t off = 0;
  auto take = [&](size_t bytes) { char* p = ws + off; off += up256(bytes); return p; };
  TtArgs a;
  a.n_events = n_events; a.n_hits = n_hits; a.n_edges = n_edges;
  a.n_art = n_trip[0]; a.n_left = n_trip[1]; a.n_right = n_trip[2];
  a.event_ptr = event_ptr; a.row_ptr = row_ptr; a.in_ptr = in_ptr; a.in_perm = in_perm;
  a.scores = scores; a.score_min = score_min; a.tptr = tptr; a.first = first; a.second = second;
  a.tscores = tscores; a.trip_min = trip_min; a.label = d_edge_set;
  a.mn_out = (int32_t*)take(4 * E1); a.mx_out = (int32_t*)take(4 * E1);
  a.mn_in = (int32_t*)take(4 * E1); a.mx_in = (int32_t*)take(4 * E1);
  int32_t* plain_label = (int32_t*)take(4 * E1);
  a.art_flag = (unsigned char*)take(A1);
  a.jkey = (unsigned long long*)take(8 * A1);
  unsigned long long* joins = (unsigned long long*)take(8 * A1);
  int32_t* jpos = (int32_t*)take(4 * A1);
  int32_t* mptr = (int32_t*)take(4 * ((size_t)n_hits + 1));
  unsigned long long* mkey = (unsigned long long*)take(8 * (2 * (size_t)n_edges + 1));
  int32_t* tptr_tmp = (int32_t*)take(4 * (E1 + A1));      // T + 1 <= (kept sets) + (articulation rows) + 1 entries
  int32_t* scan_tmp = (int32_t*)take(4 * scan_tmp_ints((int)(n_edges + n_trip[0] + n_hits) + 2));
  int launches = 0;
  const int ev_grid = n_events < 148 * 8 ? (n_events < 1 ? 1 : n_events) : 148 * 8;
  counts[0] = counts[1] = counts[2] = counts[3] = 0;
  *capacity_ok = true;
  if (n_events <= 0 || n_hits <= 0) return 0;

  tt_sets_kernel<<<ev_grid, kThreads, 0, s>>>(a); ++launches;
  // joins: per-event sort of the shared rows' keys, then the distinct ones in order
  seg_sort_kernel<<<ev_grid, kThreads, 0, s>>>(n_events, event_ptr, tptr, a.jkey); ++launches;
  tt_join_heads_kernel<<<grid_for(a.n_art + 1), kThreads, 0, s>>>(a.n_art, a.jkey, jpos); ++launches;
  launches += launch_exclusive_scan(jpos, (int)a.n_art + 1, scan_tmp, s);
  if (a.n_art > 0) { tt_join_compact_kernel<<<grid_for(a.n_art), kThreads, 0, s>>>(a.n_art, a.jkey, jpos, joins); ++launches; }
  // untouched sets, ascending label  (mx_in: flags then positions; mn_in holds `touched`)
  tt_plain_flags_kernel<<<grid_for(n_edges + 1), kThreads, 0, s>>>(n_edges, a.label, a.mn_in, a.mx_in); ++launches;
  launches += launch_exclusive_scan(a.mx_in, (int)n_edges + 1, scan_tmp, s);
  if (n_edges > 0) { tt_plain_scatter_kernel<<<grid_for(n_edges), kThreads, 0, s>>>(n_edges, a.mx_in, plain_label); ++launches; }
  // memberships (set, hit), sorted per event: every set's hits ascending, sets ascending
  tt_member_kernel<false><<<grid_for(n_hits), kThreads, 0, s>>>(n_hits, row_ptr, in_ptr, in_perm, a.label, mptr, mkey); ++launches;
  launches += launch_exclusive_scan(mptr, n_hits + 1, scan_tmp, s);
  tt_member_kernel<true><<<grid_for(n_hits), kThreads, 0, s>>>(n_hits, row_ptr, in_ptr, in_perm, a.label, mptr, mkey); ++launches;
  seg_sort_kernel<<<ev_grid, kThreads, 0, s>>>(n_events, event_ptr, mptr, mkey); ++launches;
  int32_t h3[3] = {0, 0, 0};
  cudaMemcpyAsync(&h3[0], jpos + a.n_art, 4, cudaMemcpyDeviceToHost, s);
  cudaMemcpyAsync(&h3[1], a.mx_in + n_edges, 4, cudaMemcpyDeviceToHost, s);
  cudaMemcpyAsync(&h3[2], mptr + n_hits, 4, cudaMemcpyDeviceToHost, s);
  if (cudaStreamSynchronize(s) != cudaSuccess) return -1;
  const long long n_joins = h3[0], n_plain = h3[1], n_member = h3[2], T = n_joins + n_plain;
  counts[0] = n_joins; counts[1] = n_plain; counts[2] = T;
  if (n_member > 0) { tt_set_ranges_kernel<<<grid_for(n_member), kThreads, 0, s>>>(n_member, mkey, a.mn_out, a.mx_out); ++launches; }
  // track sizes -> offsets; they stay in scratch until the capacities are known
  tt_tracks_kernel<false><<<grid_for(T + 1), kThreads, 0, s>>>(n_plain, n_joins, plain_label, joins, mkey, a.mn_out, a.mx_out, tptr_tmp, nullptr); ++launches;
  launches += launch_exclusive_scan(tptr_tmp, (int)T + 1, scan_tmp, s);
  int32_t total = 0;
  cudaMemcpyAsync(&total, tptr_tmp + T, 4, cudaMemcpyDeviceToHost, s);
  if (cudaStreamSynchronize(s) != cudaSuccess) return -1;
  counts[3] = total;
  if (n_joins > join_capacity || T > track_capacity || total > hit_capacity) { *capacity_ok = false; return launches; }
  cudaMemcpyAsync(d_track_ptr, tptr_tmp, 4 * ((size_t)T + 1), cudaMemcpyDeviceToDevice, s);
  if (T > 0) { tt_tracks_kernel<true><<<grid_for(T), kThreads, 0, s>>>(n_plain, n_joins, plain_label, joins, mkey, a.mn_out, a.mx_out, d_track_ptr, d_track_hits); ++launches; }
  if (n_joins > 0) { tt_unpack_joins_kernel<<<grid_for(n_joins), kThreads, 0, s>>>(n_joins, joins, d_joins); ++launches; }
  return launches;
}

}  // namespace etx
