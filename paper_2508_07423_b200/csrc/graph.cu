// a2 — rough graph construction by fixed-radius search in embedding space (Eq. 8.1; P:2290;
// sequential reference loop P:2674).  The thesis' kernel ran one thread per source hit looping over
// the candidates ("lacks parallelization over neighbors").  Here one WARP owns a hit and its
// 32 lanes test 32 candidates at a time; the candidates of a hit on plane p are the contiguous index
// range of planes p+1..p+G of the same event (hits are plane-sorted, per-(event, plane) offsets are
// the buckets), so loads are coalesced float4 reads that stay in L1/L2 (an event's embeddings are
// ~25 KB).  A count pass, a device scan and a fill pass with ballot / popc compaction give the unique
// ordered CSR (src asc, dst asc).  The by-destination lists need no second search: the count pass bumps
// an integer in-degree counter per found edge, the fill pass drops each edge id into its destination's
// segment through an integer cursor, and a last pass sorts every (short) segment ascending -- integer
// atomics only, so the result is still one unique array.
//
// d^2 is evaluated exactly as the ABI states: fp32, left to right, __fsub_rn/__fmul_rn/__fadd_rn so
// that ptxas cannot contract to FMA — graph edges must match the oracle bit for bit.
#include "common.cuh"

namespace etx {
namespace {

constexpr int kWarpsPerBlock = 8;
constexpr unsigned kFull = 0xffffffffu;

__global__ void plane_index_kernel(GraphArgs a, int32_t* __restrict__ plane_ptr,
                                   int32_t* __restrict__ hit_event, int32_t* __restrict__ flags) {
  const int L = a.n_planes;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    if (a.event_ptr[0] != 0 || a.event_ptr[a.n_events] != a.n_hits) atomicOr(&flags[0], 1);
  }
  for (int ev = blockIdx.x; ev < a.n_events; ev += gridDim.x) {
    const int lo = a.event_ptr[ev], hi = a.event_ptr[ev + 1];
    if (lo < 0 || hi < lo || hi > a.n_hits) {
      if (threadIdx.x == 0) atomicOr(&flags[0], 1);
      continue;
    }
    int32_t* pp = plane_ptr + (size_t)ev * (L + 1);
    for (int i = lo + threadIdx.x; i < hi; i += blockDim.x) {
      const int cur = a.plane[i];
      const int prev = (i == lo) ? -1 : (int)a.plane[i - 1];
      hit_event[i] = ev;
      if (cur >= L) { atomicOr(&flags[0], 1); continue; }
      if (cur < prev) { atomicOr(&flags[0], 2); continue; }
      for (int p = prev + 1; p <= cur; ++p) pp[p] = i;     // first hit of planes prev+1..cur
    }
    if (threadIdx.x == 0) {
      const int last = (hi > lo) ? (int)a.plane[hi - 1] : -1;
      for (int p = last + 1; p <= L; ++p) pp[p] = hi;
    }
  }
}

template <int D>
__device__ __forceinline__ void load_emb(const float* __restrict__ emb, int i, int d, float (&v)[8]) {
  if (D == 4) {
    const float4 t = __ldg(reinterpret_cast<const float4*>(emb) + i);
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  } else {
#pragma unroll
    for (int c = 0; c < 8; ++c) v[c] = (c < d) ? __ldg(emb + (size_t)i * d + c) : 0.0f;
  }
}

// Packed fp32 pairs (sm_100 add/mul.rn.f32x2): two IEEE round-to-nearest operations per instruction, each lane
// rounded on its own, never contracted -- the same values as the scalar __fsub_rn / __fmul_rn, half the issue slots.
__device__ __forceinline__ unsigned long long pack2(float x, float y) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
  return r;
}
__device__ __forceinline__ unsigned long long add2_rn(unsigned long long a, unsigned long long b) {
  unsigned long long r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ unsigned long long mul2_rn(unsigned long long a, unsigned long long b) {
  unsigned long long r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
// d = 4: d^2 = ((q0 + q1) + q2) + q3 with q_c = (b_c - a_c)^2 = (a_c - b_c)^2 exactly (negation is exact), the
// differences and squares as packed pairs, the sum left to right as Eq. 8.1's oracle evaluates it.
// na01 / na23 hold the NEGATED coordinates of the source hit.
__device__ __forceinline__ float dist2_d4(unsigned long long na01, unsigned long long na23, const float4& b) {
  const unsigned long long t01 = add2_rn(pack2(b.x, b.y), na01), t23 = add2_rn(pack2(b.z, b.w), na23);
  const unsigned long long q01 = mul2_rn(t01, t01), q23 = mul2_rn(t23, t23);
  float q0, q1, q2, q3;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(q0), "=f"(q1) : "l"(q01));
  asm("mov.b64 {%0, %1}, %2;" : "=f"(q2), "=f"(q3) : "l"(q23));
  return __fadd_rn(__fadd_rn(__fadd_rn(q0, q1), q2), q3);
}

template <int D>
__device__ __forceinline__ float dist2(const float (&a)[8], const float (&b)[8], int d) {
  float s = 0.0f;
  const int n = (D == 4) ? 4 : d;
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    if (c < n) {
      const float diff = __fsub_rn(a[c], b[c]);
      const float sq = __fmul_rn(diff, diff);
      s = (c == 0) ? sq : __fadd_rn(s, sq);
    }
  }
  return s;
}

// MODE 0: count out-degree (and in-degree, by integer atomics).  MODE 1: fill the edges and drop every edge
// id into its destination's segment of in_perm (unordered; sort_in_lists_kernel orders it).
template <int D, int MODE>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
search_kernel(GraphArgs a, const int32_t* __restrict__ plane_ptr, const int32_t* __restrict__ hit_event,
              const int32_t* __restrict__ flags, int32_t* __restrict__ out_deg,
              int32_t* __restrict__ in_deg, const int32_t* __restrict__ row_ptr,
              int32_t* __restrict__ src, int32_t* __restrict__ dst,
              const int32_t* __restrict__ in_ptr, int32_t* __restrict__ in_perm, int32_t* __restrict__ cursor) {
  if (flags[0] != 0) return;                       // malformed batch: plane_ptr is not trustworthy
  const int lane = threadIdx.x & 31;
  const int warp = blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  const int n_warps = gridDim.x * kWarpsPerBlock;
  const unsigned lt = (1u << lane) - 1u;
  const int L = a.n_planes;
  for (int i = warp; i < a.n_hits; i += n_warps) {
    const int ev = hit_event[i];
    const int p = a.plane[i];
    const int32_t* pp = plane_ptr + (size_t)ev * (L + 1);
    float me[8], other[8];
    load_emb<D>(a.emb, i, a.d, me);
    int cnt = 0;
    if (p <= L - 2) {
      const int j0 = pp[p + 1];
      const int top = (p + a.gap < L - 1) ? p + a.gap : L - 1;
      const int j1 = pp[top + 1];
      const int base_out = (MODE == 1) ? row_ptr[i] : 0;
      // fill pass: the count pass already fixed this hit's out-degree -- stop as soon as all its edges are written
      // (a hit without neighbours tests nothing, the others skip the candidates behind their last neighbour)
      const int deg = (MODE == 1) ? row_ptr[i + 1] - base_out : 0x7fffffff;
      const float r2 = a.r2_max;
      const unsigned long long nme01 = pack2(-me[0], -me[1]), nme23 = pack2(-me[2], -me[3]);
      for (int base = j0; base < j1 && cnt < deg; base += 32) {
        const int j = base + lane;
        // branch-free body: lanes past the end test the last candidate again and are masked out of the vote
        const int jc = j < j1 ? j : j1 - 1;
        bool ok;
        if constexpr (D == 4) {
          ok = (dist2_d4(nme01, nme23, __ldg(reinterpret_cast<const float4*>(a.emb) + jc)) < r2) & (j < j1);
        } else {
          load_emb<D>(a.emb, jc, a.d, other);
          ok = (dist2<D>(me, other, a.d) < r2) & (j < j1);
        }
        const unsigned b = __ballot_sync(kFull, ok);
        if (ok) {
          if (MODE == 0) {
            atomicAdd(&in_deg[j], 1);
          } else {
            const int pos = base_out + cnt + __popc(b & lt);
            src[pos] = i;
            dst[pos] = j;
            in_perm[in_ptr[j] + atomicAdd(&cursor[j], 1)] = pos;
          }
        }
        cnt += __popc(b);
      }
    }
    if (MODE == 0 && lane == 0) out_deg[i] = cnt;
  }
  if (MODE == 0 && blockIdx.x == 0 && threadIdx.x == 0) out_deg[a.n_hits] = 0;
}

// ------------------------------------------------------------------ d = 4: tiled count pass + candidate-major pair fill pass
// One CTA owns an (event, source plane) window: the candidates -- the hits of planes p+1..p+G of the event, a
// contiguous index range -- are staged ONCE in shared memory as float4 and every warp tests them against FOUR source
// hits at a time (register-blocked: one shared-memory load per candidate and four distance tests), instead of one warp
// per source re-reading its ~190-candidate window from L1/L2.  The count pass also KEEPS its vote words (kBallotWords
// 32-candidate words per source), so the fill pass expands bits into edges and computes no distance at all; a window
// longer than kBallotWords x 32 candidates re-tests only the words that did not fit.
constexpr int kTileCand = 1024;                    // candidates staged per chunk (16 KB)

// b[k & 3] as three selects (a chain of comparisons became a jump table in the inner loop)
__device__ __forceinline__ unsigned sel4(unsigned b0, unsigned b1, unsigned b2, unsigned b3, int k) {
  const unsigned lo = (k & 1) ? b1 : b0, hi = (k & 1) ? b3 : b2;
  return (k & 2) ? hi : lo;
}
// shared-memory counter update on a 32-bit shared address (atomicAdd on the generic pointer re-derived the window base from
// the CTA id in every iteration)
__device__ __forceinline__ void red_shared_add(uint32_t addr, int v) {
  asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

__global__ void __launch_bounds__(kWarpsPerBlock * 32)
search_tile_count_kernel(GraphArgs a, const int32_t* __restrict__ plane_ptr, int32_t* __restrict__ flags,
                         int32_t* __restrict__ out_deg /*zeroed*/, int32_t* __restrict__ in_deg3 /*[n_hits][3], zeroed*/,
                         uint32_t* __restrict__ ballots /*[n_hits][kBallotWords]*/,
                         uint16_t* __restrict__ prefix16 /*[n_hits][kBallotWords]*/) {
  if (flags[0] != 0) return;
  __shared__ float4 cand[kTileCand];
  __shared__ int s_in[kTileCand];                  // edges of THIS plane's sources into every candidate of the window
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int L = a.n_planes;
  const long long n_work = (long long)a.n_events * (L - 1);
  const float4* __restrict__ emb4 = reinterpret_cast<const float4*>(a.emb);
  const float r2 = a.r2_max;
  for (long long work = blockIdx.x; work < n_work; work += gridDim.x) {
    const int ev = (int)(work / (L - 1)), p = (int)(work % (L - 1));
    const int32_t* pp = plane_ptr + (size_t)ev * (L + 1);
    const int s0 = pp[p], s1 = pp[p + 1];
    const int top = (p + a.gap < L - 1) ? p + a.gap : L - 1;
    const int j0 = s1, j1 = pp[top + 1];
    if (s1 <= s0 || j1 <= j0) continue;            // uniform over the CTA
    const int ncc = j1 - j0;
    if (ncc > kTileCand) {                         // more candidates than vote words are kept: the caller redoes the build
      if (threadIdx.x == 0) atomicOr(&flags[1], 1);  // with the one-warp-per-source kernels
      continue;
    }
    __syncthreads();                               // the previous window is no longer read
    for (int t = threadIdx.x; t < ncc; t += blockDim.x) { cand[t] = __ldg(emb4 + j0 + t); s_in[t] = 0; }
    __syncthreads();
    const int nw = (ncc + 31) >> 5;
    const uint32_t s_in_lane = (uint32_t)__cvta_generic_to_shared(s_in + lane);
    for (int i0 = s0 + 4 * warp; i0 < s1; i0 += 4 * kWarpsPerBlock) {
      unsigned long long n01[4], n23[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        // a source slot past the plane's last hit sits infinitely far away: its d^2 overflows to +inf and it never votes
        const float4 m = (i0 + k < s1) ? __ldg(emb4 + i0 + k) : make_float4(1e30f, 1e30f, 1e30f, 1e30f);
        n01[k] = pack2(-m.x, -m.y); n23[k] = pack2(-m.z, -m.w);
      }
      const bool owner = lane < 4 && i0 + lane < s1;               // lane k < 4 keeps source i0 + k's words and count
      uint32_t* const my_words = ballots + (size_t)(i0 + (lane & 3)) * kBallotWords;
      uint16_t* const my_prefix = prefix16 + (size_t)(i0 + (lane & 3)) * kBallotWords;
      int cnt = 0;
      for (int t = 0; t < nw; ++t) {
        const int idx = t * 32 + lane;
        const bool vld = idx < ncc;
        const float4 cq = cand[vld ? idx : ncc - 1];
        const bool ok0 = (dist2_d4(n01[0], n23[0], cq) < r2) & vld, ok1 = (dist2_d4(n01[1], n23[1], cq) < r2) & vld;
        const bool ok2 = (dist2_d4(n01[2], n23[2], cq) < r2) & vld, ok3 = (dist2_d4(n01[3], n23[3], cq) < r2) & vld;
        const unsigned b0 = __ballot_sync(kFull, ok0), b1 = __ballot_sync(kFull, ok1);
        const unsigned b2 = __ballot_sync(kFull, ok2), b3 = __ballot_sync(kFull, ok3);
        if (owner) {
          const unsigned mine = sel4(b0, b1, b2, b3, lane);
          my_words[t] = mine;
          my_prefix[t] = (uint16_t)cnt;            // votes of this source in the words before this one (<= 1024)
          cnt += __popc(mine);
        }
        const int n_in = (int)ok0 + (int)ok1 + (int)ok2 + (int)ok3;
        if (n_in) red_shared_add(s_in_lane + (uint32_t)t * 128u, n_in);  // this CTA is the only writer of (candidate, plane gap)
      }
      if (owner) out_deg[i0 + lane] = cnt;
    }
    __syncthreads();
    // The in-list of a hit is ordered by source index = by source plane first: three sub-lists (gap 3, 2, 1), each counted
    // by exactly one CTA -- no global atomics, and the fill pass can place every edge id at its final position.
    const int q2 = pp[(p + 2 < L) ? p + 2 : L], q3 = pp[(p + 3 < L) ? p + 3 : L];
    for (int t = threadIdx.x; t < ncc; t += blockDim.x) {
      const int j = j0 + t;
      const int g = 1 + (int)(j >= q2) + (int)(j >= q3);
      in_deg3[(size_t)3 * j + (3 - g)] = s_in[t];
    }
  }
}

// Next row NEXT-2 on the tiled search (k_max > 0, d = 4; Algorithm 1): after the count pass a source
// with more than k_max votes keeps its k_max nearest candidates by (d^2 in fp32, then hit index) -- the order of
// graph_kmax.cu and of the oracle -- by CLEARING the other votes: the vote words then describe the capped graph, and the scans and
// the pair fill pass run unchanged.  One warp per hit, almost all of which leave at once (the thesis:
// < 0.1 % of hits exceed k_max = 50); lane t owns vote word t (a window has at most kBallotWords = 32 words, else the
// caller falls back to graph_kmax.cu: flags[1]).  <= 128 votes: their keys (d^2 bits : index) are compacted into a
// per-warp shared-memory list and every lane ranks its keys against the list; more: the k_max-th smallest key by bitwise
// bisection (64 counting sweeps over the lane's own word).  Dropped votes give their in-degree count back.
constexpr int kCapListMax = 128;
static_assert(kBallotWords <= 32, "one vote word per lane");

__device__ __forceinline__ unsigned long long cap_key(float d2, int j) {
  return ((unsigned long long)__float_as_uint(d2) << 32) | (unsigned)j;   // d2 >= 0: the bit pattern is monotone
}

__global__ void __launch_bounds__(kWarpsPerBlock * 32)
search_kmax_cap_kernel(GraphArgs a, int k_max, const int32_t* __restrict__ plane_ptr, const int32_t* __restrict__ hit_event,
                       int32_t* __restrict__ flags, int32_t* __restrict__ out_deg, int32_t* __restrict__ in_deg3,
                       uint32_t* __restrict__ ballots, uint16_t* __restrict__ prefix16) {
  if (flags[0] != 0) return;
  __shared__ unsigned long long s_keys[kWarpsPerBlock][kCapListMax];
  const int lane = threadIdx.x & 31;
  const int n_warps = gridDim.x * kWarpsPerBlock;
  const int L = a.n_planes;
  const float4* __restrict__ emb4 = reinterpret_cast<const float4*>(a.emb);
  unsigned long long* keys = s_keys[threadIdx.x >> 5];
  for (int i = blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5); i < a.n_hits; i += n_warps) {
    const int total = out_deg[i];
    if (total <= k_max) continue;
    const int p = a.plane[i];                      // total > 0 implies p <= L - 2
    const int32_t* pp = plane_ptr + (size_t)hit_event[i] * (L + 1);
    const int j0 = pp[p + 1];
    const int top = (p + a.gap < L - 1) ? p + a.gap : L - 1;
    const int j1 = pp[top + 1];
    const int nw = (j1 - j0 + 31) >> 5;
    if (nw > kBallotWords) continue;               // flagged by the count pass: the caller redoes the build with graph_kmax.cu
    const float4 m = __ldg(emb4 + i);
    const unsigned long long n01 = pack2(-m.x, -m.y), n23 = pack2(-m.z, -m.w);
    const unsigned word = lane < nw ? ballots[(size_t)i * kBallotWords + lane] : 0u;
    const int jw = j0 + lane * 32;                 // first candidate of this lane's word
    unsigned keep = word;                          // votes that survive the cap
    if (total <= kCapListMax) {
      // short list: every lane writes its votes' keys behind the votes of the lanes before it (ascending index = ascending slot)
      int off = __popc(word);
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(kFull, off, o);
        if (lane >= o) off += t;
      }
      off -= __popc(word);
      for (unsigned w = word; w; w &= w - 1) {
        const int bit = __ffs(w) - 1;
        keys[off++] = cap_key(dist2_d4(n01, n23, __ldg(emb4 + jw + bit)), jw + bit);
      }
      __syncwarp();
      for (unsigned w = word; w; w &= w - 1) {
        const int bit = __ffs(w) - 1;
        const unsigned long long mine = cap_key(dist2_d4(n01, n23, __ldg(emb4 + jw + bit)), jw + bit);
        int rank = 0;
        for (int q = 0; q < total; ++q) rank += keys[q] < mine;
        if (rank >= k_max) keep &= ~(1u << bit);
      }
      __syncwarp();
    } else {
      unsigned long long thr = 0ull;               // invariant: thr <= the k_max-th smallest key
      for (int b = 63; b >= 0; --b) {
        const unsigned long long cand = thr | (1ull << b);
        int below = 0;
        for (unsigned w = word; w; w &= w - 1) {
          const int bit = __ffs(w) - 1;
          below += cap_key(dist2_d4(n01, n23, __ldg(emb4 + jw + bit)), jw + bit) < cand;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) below += __shfl_xor_sync(kFull, below, o);
        if (below < k_max) thr = cand;             // fewer than k_max keys below cand: the k_max-th one is >= cand
      }
      for (unsigned w = word; w; w &= w - 1) {
        const int bit = __ffs(w) - 1;
        if (cap_key(dist2_d4(n01, n23, __ldg(emb4 + jw + bit)), jw + bit) > thr) keep &= ~(1u << bit);
      }
    }
    const int q2 = pp[(p + 2 < L) ? p + 2 : L], q3 = pp[(p + 3 < L) ? p + 3 : L];
    for (unsigned w = word & ~keep; w; w &= w - 1) {
      const int j = jw + __ffs(w) - 1;
      const int g = 1 + (int)(j >= q2) + (int)(j >= q3);
      atomicSub(&in_deg3[(size_t)3 * j + (3 - g)], 1);
    }
    int before = __popc(keep);                     // the surviving votes' prefix counts replace the count pass's
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(kFull, before, o);
      if (lane >= o) before += t;
    }
    before -= __popc(keep);
    if (lane < nw) {
      ballots[(size_t)i * kBallotWords + lane] = keep;
      prefix16[(size_t)i * kBallotWords + lane] = (uint16_t)before;
    }
    if (lane == 0) out_deg[i] = k_max;
  }
}

// Fill pass for d = 4: the same (event, source plane) tiling as the count pass, candidate-major.  A warp takes one vote word of
// the window -- 32 candidates, one per lane -- and walks the plane's sources in ascending order: a set bit is the edge
// (i -> j); its id is row_ptr[i] + (votes of i before this word) + (votes of i below this bit), and because the sources come
// in ascending order the lane's running count is the edge's rank inside the candidate's sub-list of this plane gap.  So src,
// dst AND the by-destination lists are written at their final positions: no cursor atomics, no sort pass.
// Transposes a 32 x 32 bit matrix held one row per lane (bit c of lane l's word = element (l, c)); on return bit l of lane
// c's word = element (l, c).  Five stages; stage j swaps the off-diagonal j x j blocks of every 2j x 2j block.
__device__ __forceinline__ unsigned transpose_bits(unsigned x, int lane) {
  unsigned lo_cols = 0x0000ffffu;                  // columns whose index has bit j clear
#pragma unroll
  for (int j = 16; j >= 1; j >>= 1) {
    const unsigned other = __shfl_xor_sync(kFull, x, j);
    x = (lane & j) ? ((x & ~lo_cols) | ((other >> j) & lo_cols)) : ((x & lo_cols) | ((other << j) & ~lo_cols));
    lo_cols ^= lo_cols << (j >> 1);
  }
  return x;
}

constexpr int kFillSrc = 64;                       // sources whose vote words are staged per step

__global__ void __launch_bounds__(kWarpsPerBlock * 32)
search_pair_fill_kernel(GraphArgs a, const int32_t* __restrict__ plane_ptr, const int32_t* __restrict__ flags,
                        const uint32_t* __restrict__ ballots, const uint16_t* __restrict__ prefix16,
                        const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ in_ptr3,
                        int32_t* __restrict__ src, int32_t* __restrict__ dst, int32_t* __restrict__ in_perm) {
  if (flags[0] != 0) return;
  // the sources' vote words, prefix counts and first edge ids are staged in shared memory by all threads at once (read
  // one by one from global memory in the source loop they cost a DRAM latency each: 0.83 ms instead of 0.2)
  __shared__ uint32_t s_w[kFillSrc * kBallotWords];
  __shared__ uint16_t s_pre[kFillSrc * kBallotWords];
  __shared__ int32_t s_row[kFillSrc];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  const int L = a.n_planes;
  const long long n_work = (long long)a.n_events * (L - 1);
  for (long long work = blockIdx.x; work < n_work; work += gridDim.x) {
    const int ev = (int)(work / (L - 1)), p = (int)(work % (L - 1));
    const int32_t* pp = plane_ptr + (size_t)ev * (L + 1);
    const int s0 = pp[p], s1 = pp[p + 1];
    const int top = (p + a.gap < L - 1) ? p + a.gap : L - 1;
    const int j0 = s1, j1 = pp[top + 1];
    if (s1 <= s0 || j1 <= j0 || j1 - j0 > kTileCand) continue;
    const int q2 = pp[(p + 2 < L) ? p + 2 : L], q3 = pp[(p + 3 < L) ? p + 3 : L];
    const int nw = (j1 - j0 + 31) >> 5;
    int at[(kBallotWords + kWarpsPerBlock - 1) / kWarpsPerBlock];     // next free position of this lane's candidates' sub-lists
#pragma unroll
    for (int r = 0; r < (kBallotWords + kWarpsPerBlock - 1) / kWarpsPerBlock; ++r) {
      const int j = j0 + (warp + r * kWarpsPerBlock) * 32 + lane;
      const int g = 1 + (int)(j >= q2) + (int)(j >= q3);
      at[r] = (warp + r * kWarpsPerBlock < nw && j < j1) ? in_ptr3[(size_t)3 * j + (3 - g)] : 0;
    }
    for (int c0 = s0; c0 < s1; c0 += kFillSrc) {
      const int ns = (s1 - c0) < kFillSrc ? (s1 - c0) : kFillSrc;
      __syncthreads();                             // the previous step's words are no longer read
      // staged word-major, [t][source], so that the 32 sources of a block sit in 32 consecutive banks
      for (int x = threadIdx.x; x < ns * nw; x += blockDim.x) {
        const int ii = x / nw, t = x - ii * nw;
        s_w[t * kFillSrc + ii] = __ldg(ballots + (size_t)(c0 + ii) * kBallotWords + t);
        s_pre[t * kFillSrc + ii] = __ldg(prefix16 + (size_t)(c0 + ii) * kBallotWords + t);
      }
      for (int x = threadIdx.x; x < ns; x += blockDim.x) s_row[x] = row_ptr[c0 + x];
      __syncthreads();
#pragma unroll
      for (int r = 0; r < (kBallotWords + kWarpsPerBlock - 1) / kWarpsPerBlock; ++r) {
        const int t = warp + r * kWarpsPerBlock;
        if (t >= nw) break;                        // uniform over the warp
        const int j = j0 + t * 32 + lane;
        for (int b0 = 0; b0 < ns; b0 += 32) {
          // 32 sources x 32 candidates of votes: lane = source on the way in, lane = candidate after the transposition
          // (five block-swap stages), so that every lane walks only ITS candidate's votes, sources ascending -- the order of
          // the by-destination list -- instead of all lanes stepping through every (source, word) pair for one vote each.
          unsigned v = (b0 + lane < ns) ? s_w[t * kFillSrc + b0 + lane] : 0u;
          if (__ballot_sync(kFull, v != 0u) == 0u) continue;
          v = transpose_bits(v, lane);
          while (v != 0u) {
            const int ii = b0 + __ffs((int)v) - 1;
            v &= v - 1u;
            const int eid = s_row[ii] + (int)s_pre[t * kFillSrc + ii] + __popc(s_w[t * kFillSrc + ii] & lt);
            src[eid] = c0 + ii;
            dst[eid] = j;
            in_perm[at[r]++] = eid;
          }
        }
      }
    }
  }
}

// in_ptr[j] = start of hit j's in-list = start of its first sub-list; in_ptr[n_hits] = E
__global__ void __launch_bounds__(256) in_ptr_from3_kernel(int n_hits, const int32_t* __restrict__ in_ptr3, int32_t* __restrict__ in_ptr) {
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j <= n_hits; j += gridDim.x * blockDim.x) in_ptr[j] = in_ptr3[(size_t)3 * j];
}

// Orders every destination's list of edge ids ascending.  One warp per hit: a list of <= 32 ids (in-degrees are
// ~6-10) sits one id per lane, each lane ranks its id with shuffles and writes it to its place (coalesced both
// ways); up to 128 ids sit four per lane and are ranked the same way (at C4, in-degree ~10 with a tail, the single-lane
// insertion sort these lists used to fall back to made this kernel 4.1 ms of a 8.6 ms graph build); longer lists are
// insertion-sorted by one lane.
__global__ void __launch_bounds__(256) sort_in_lists_kernel(int n_hits, const int32_t* __restrict__ flags,
                                                            const int32_t* __restrict__ in_ptr, int32_t* __restrict__ in_perm) {
  if (flags[0] != 0) return;
  const int lane = threadIdx.x & 31;
  const int n_warps = gridDim.x * (blockDim.x >> 5);
  for (int j = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); j < n_hits; j += n_warps) {
    const int k0 = in_ptr[j], n = in_ptr[j + 1] - k0;
    if (n <= 1) continue;
    if (n <= 32) {
      const int v = lane < n ? in_perm[k0 + lane] : 0x7fffffff;
      int rank = 0;
      for (int m = 0; m < n; ++m) rank += __shfl_sync(kFull, v, m) < v;      // ids are distinct
      __syncwarp();
      if (lane < n) in_perm[k0 + rank] = v;
    } else if (n <= 128) {
      int v[4], rank[4] = {0, 0, 0, 0};
#pragma unroll
      for (int q = 0; q < 4; ++q) v[q] = (lane + 32 * q < n) ? in_perm[k0 + lane + 32 * q] : 0x7fffffff;
#pragma unroll
      for (int q2 = 0; q2 < 4; ++q2) {
        if (32 * q2 >= n) break;                                             // uniform over the warp
        const int cnt = n - 32 * q2 < 32 ? n - 32 * q2 : 32;
        for (int m = 0; m < cnt; ++m) {
          const int o = __shfl_sync(kFull, v[q2], m);
#pragma unroll
          for (int q = 0; q < 4; ++q) rank[q] += o < v[q];
        }
      }
      __syncwarp();
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if (lane + 32 * q < n) in_perm[k0 + rank[q]] = v[q];
    } else if (lane == 0) {
      for (int k = k0 + 1; k < k0 + n; ++k) {
        const int v = in_perm[k];
        int q = k - 1;
        while (q >= k0 && in_perm[q] > v) { in_perm[q + 1] = in_perm[q]; --q; }
        in_perm[q + 1] = v;
      }
    }
  }
}

// ------------------------------------------------------------------ device-wide exclusive scan
constexpr int kScanThreads = 256;
constexpr int kScanPerThread = 8;
constexpr int kScanTile = kScanThreads * kScanPerThread;

__device__ __forceinline__ int block_exclusive_scan(int v, int* total) {
  __shared__ int warp_sums[kScanThreads / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(kFull, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) warp_sums[w] = inc;
  __syncthreads();
  if (w == 0) {
    int s = (lane < kScanThreads / 32) ? warp_sums[lane] : 0;
#pragma unroll
    for (int o = 1; o < kScanThreads / 32; o <<= 1) {
      const int t = __shfl_up_sync(kFull, s, o);
      if (lane >= o) s += t;
    }
    if (lane < kScanThreads / 32) warp_sums[lane] = s;
  }
  __syncthreads();
  const int before = (w == 0) ? 0 : warp_sums[w - 1];
  *total = warp_sums[kScanThreads / 32 - 1];
  __syncthreads();
  return before + inc - v;
}

__global__ void __launch_bounds__(kScanThreads) scan_block_sums(const int32_t* __restrict__ data, int n,
                                                                int32_t* __restrict__ tmp) {
  const int base = blockIdx.x * kScanTile + threadIdx.x * kScanPerThread;
  int s = 0;
#pragma unroll
  for (int k = 0; k < kScanPerThread; ++k) s += (base + k < n) ? data[base + k] : 0;
  int total;
  block_exclusive_scan(s, &total);
  if (threadIdx.x == 0) tmp[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanThreads) scan_tmp_kernel(int32_t* __restrict__ tmp, int nb) {
  int carry = 0;
  for (int base = 0; base < nb; base += kScanThreads) {
    const int i = base + threadIdx.x;
    const int v = (i < nb) ? tmp[i] : 0;
    int total;
    const int ex = block_exclusive_scan(v, &total);
    if (i < nb) tmp[i] = carry + ex;
    carry += total;
  }
}

__global__ void __launch_bounds__(kScanThreads) scan_apply(int32_t* __restrict__ data, int n,
                                                           const int32_t* __restrict__ tmp) {
  const int base = blockIdx.x * kScanTile + threadIdx.x * kScanPerThread;
  int v[kScanPerThread];
  int s = 0;
#pragma unroll
  for (int k = 0; k < kScanPerThread; ++k) { v[k] = (base + k < n) ? data[base + k] : 0; s += v[k]; }
  int total;
  int run = block_exclusive_scan(s, &total) + tmp[blockIdx.x];
#pragma unroll
  for (int k = 0; k < kScanPerThread; ++k) {
    if (base + k < n) data[base + k] = run;
    run += v[k];
  }
}

inline int search_grid(int n_hits) {
  const int need = (n_hits + kWarpsPerBlock - 1) / kWarpsPerBlock;
  const int cap = 148 * 8;                         // 8 resident CTAs of 256 threads per SM
  return need < 1 ? 1 : (need < cap ? need : cap);
}

}  // namespace

size_t scan_tmp_ints(int n) { return (size_t)((n + kScanTile - 1) / kScanTile) + 1; }

int launch_plane_index(const GraphArgs& a, int32_t* plane_ptr, int32_t* hit_event, int32_t* flags,
                       cudaStream_t s) {
  cudaMemsetAsync(flags, 0, 8 * sizeof(int32_t), s);
  const int grid = a.n_events < 1 ? 1 : (a.n_events < 148 * 16 ? a.n_events : 148 * 16);
  plane_index_kernel<<<grid, 128, 0, s>>>(a, plane_ptr, hit_event, flags);
  return 1;
}

template <int MODE>
static void launch_search(const GraphArgs& a, const int32_t* plane_ptr, const int32_t* hit_event,
                          const int32_t* flags, int32_t* out_deg, int32_t* in_deg,
                          const int32_t* row_ptr, int32_t* src, int32_t* dst, const int32_t* in_ptr,
                          int32_t* in_perm, int32_t* cursor, cudaStream_t s) {
  const int grid = search_grid(a.n_hits);
  if (a.d == 4)
    search_kernel<4, MODE><<<grid, kWarpsPerBlock * 32, 0, s>>>(a, plane_ptr, hit_event, flags, out_deg, in_deg,
                                                               row_ptr, src, dst, in_ptr, in_perm, cursor);
  else
    search_kernel<0, MODE><<<grid, kWarpsPerBlock * 32, 0, s>>>(a, plane_ptr, hit_event, flags, out_deg, in_deg,
                                                               row_ptr, src, dst, in_ptr, in_perm, cursor);
}

// d = 4 with the tiled kernels (ballots != null): out_deg and in_deg3 [n_hits][3] (+1) are filled; otherwise the
// one-warp-per-source count pass fills out_deg and in_deg [n_hits] (passed as in_deg3).
int launch_search_count(const GraphArgs& a, const int32_t* plane_ptr, const int32_t* hit_event,
                        int32_t* flags, int32_t* out_deg, int32_t* in_deg3, uint32_t* ballots, uint16_t* prefix16, cudaStream_t s) {
  if (a.d == 4 && ballots) {                       // tiled count pass (shared-memory candidate windows, kept vote words)
    cudaMemsetAsync(in_deg3, 0, sizeof(int32_t) * ((size_t)3 * a.n_hits + 1), s);
    cudaMemsetAsync(out_deg, 0, sizeof(int32_t) * ((size_t)a.n_hits + 1), s);
    const long long n_work = (long long)a.n_events * (a.n_planes - 1);
    const int cap = 148 * 8;
    search_tile_count_kernel<<<(int)(n_work < 1 ? 1 : (n_work < cap ? n_work : cap)), kWarpsPerBlock * 32, 0, s>>>(
        a, plane_ptr, flags, out_deg, in_deg3, ballots, prefix16);
    return 1;
  }
  cudaMemsetAsync(in_deg3, 0, sizeof(int32_t) * ((size_t)a.n_hits + 1), s);
  launch_search<0>(a, plane_ptr, hit_event, flags, out_deg, in_deg3, nullptr, nullptr, nullptr, nullptr,
                   nullptr, nullptr, s);
  return 1;
}

int launch_search_kmax_cap(const GraphArgs& a, int k_max, const int32_t* plane_ptr, const int32_t* hit_event, int32_t* flags,
                           int32_t* out_deg, int32_t* in_deg3, uint32_t* ballots, uint16_t* prefix16, cudaStream_t s) {
  search_kmax_cap_kernel<<<search_grid(a.n_hits), kWarpsPerBlock * 32, 0, s>>>(a, k_max, plane_ptr, hit_event, flags, out_deg,
                                                                               in_deg3, ballots, prefix16);
  return 1;
}

int launch_in_ptr_from3(int n_hits, const int32_t* in_ptr3, int32_t* in_ptr, cudaStream_t s) {
  const int need = (n_hits + 256) / 256;
  in_ptr_from3_kernel<<<need < 148 * 8 ? need : 148 * 8, 256, 0, s>>>(n_hits, in_ptr3, in_ptr);
  return 1;
}

int launch_exclusive_scan(int32_t* data, int n, int32_t* tmp, cudaStream_t s) {
  const int nb = (n + kScanTile - 1) / kScanTile;
  scan_block_sums<<<nb, kScanThreads, 0, s>>>(data, n, tmp);
  scan_tmp_kernel<<<1, kScanThreads, 0, s>>>(tmp, nb);
  scan_apply<<<nb, kScanThreads, 0, s>>>(data, n, tmp);
  return 3;
}

// ballots != null: the tiled pair fill (in_ptr3 = scanned sub-list offsets, no cursor, no sort); else the one-warp-per-source
// fill with cursor atomics and the in-list sort
int launch_search_fill(const GraphArgs& a, const int32_t* plane_ptr, const int32_t* hit_event,
                       const int32_t* flags, const int32_t* row_ptr, int32_t* src, int32_t* dst,
                       const int32_t* in_ptr, int32_t* in_perm, int32_t* cursor /*[n_hits] scratch*/,
                       const uint32_t* ballots, const uint16_t* prefix16, const int32_t* in_ptr3, cudaStream_t s) {
  if (a.d == 4 && ballots) {
    const long long n_work = (long long)a.n_events * (a.n_planes - 1);
    const int cap = 148 * 8;
    search_pair_fill_kernel<<<(int)(n_work < 1 ? 1 : (n_work < cap ? n_work : cap)), kWarpsPerBlock * 32, 0, s>>>(
        a, plane_ptr, flags, ballots, prefix16, row_ptr, in_ptr3, src, dst, in_perm);
    return 1;
  }
  cudaMemsetAsync(cursor, 0, sizeof(int32_t) * (size_t)a.n_hits, s);
  launch_search<1>(a, plane_ptr, hit_event, flags, nullptr, nullptr, row_ptr, src, dst, in_ptr, in_perm, cursor, s);
  return 1 + launch_sort_in_lists(a.n_hits, flags, in_ptr, in_perm, s);
}

int launch_sort_in_lists(int n_hits, const int32_t* flags, const int32_t* in_ptr, int32_t* in_perm, cudaStream_t s) {
  const int need = (n_hits + 7) / 8;
  sort_in_lists_kernel<<<need < 148 * 8 ? (need < 1 ? 1 : need) : 148 * 8, 256, 0, s>>>(n_hits, flags, in_ptr, in_perm);
  return 1;
}

// out[i] = in[i] + offset (etx_infer_host's event-range passes: chunk-local hit indices -> indices of the whole batch)
namespace {
__global__ void add_offset_kernel(const int32_t* __restrict__ in, int32_t* __restrict__ out, int64_t n, int32_t offset) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) out[i] = in[i] + offset;
}
}  // namespace
int launch_add_offset(const int32_t* in, int32_t* out, int64_t n, int32_t offset, cudaStream_t s) {
  if (n <= 0) return 0;
  const int64_t need = (n + 255) / 256;
  add_offset_kernel<<<(int)(need < 148 * 8 ? need : 148 * 8), 256, 0, s>>>(in, out, n, offset);
  return 1;
}

}  // namespace etx
