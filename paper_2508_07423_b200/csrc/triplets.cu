// NEXT-4 (triplet part) — triplet building, Fig. 8.13.
// The edge connections of the purified hit graph (edges with score >= score_min, the cut of tracks.cu): two kept
// edges sharing a hit C form an articulation (A -> C, C -> B), a left elbow (C -> A, C -> B) or a right elbow
// (A -> C, B -> C).  The thesis built them in Python only; here they come straight from the two
// CSR structures etx_build_graph already made: a hit's outgoing edges are the contiguous ids
// row_ptr[C] .. row_ptr[C+1], its incoming edges the ascending ids in_perm[in_ptr[C] ..].
// Count pass (per hit: kept in-degree x kept out-degree, and the two binomials) -> three device scans -> fill pass,
// so every list is written in ONE fixed order (shared hit, first edge id, second edge id): integer work, compared
// bit for bit with the oracle.  One thread per hit: the lists of a hit are a handful of ids.
#include "common.cuh"

namespace etx {
namespace {

constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads) triplet_count_kernel(int n_hits, const int32_t* __restrict__ row_ptr,
                                                                 const int32_t* __restrict__ in_ptr,
                                                                 const int32_t* __restrict__ in_perm,
                                                                 const float* __restrict__ scores, float score_min,
                                                                 int32_t* __restrict__ ptr /*[3][n_hits+1]*/) {
  const int c = blockIdx.x * kThreads + threadIdx.x;
  const size_t ld = (size_t)n_hits + 1;
  if (c == 0) { ptr[n_hits] = 0; ptr[ld + n_hits] = 0; ptr[2 * ld + n_hits] = 0; }
  if (c >= n_hits) return;
  int kout = 0, kin = 0;
  for (int e = row_ptr[c]; e < row_ptr[c + 1]; ++e) kout += scores[e] >= score_min;
  for (int k = in_ptr[c]; k < in_ptr[c + 1]; ++k) kin += scores[in_perm[k]] >= score_min;
  ptr[c] = kin * kout;
  ptr[ld + c] = kout * (kout - 1) / 2;
  ptr[2 * ld + c] = kin * (kin - 1) / 2;
}

__global__ void __launch_bounds__(kThreads) triplet_fill_kernel(int n_hits, const int32_t* __restrict__ row_ptr,
                                                                const int32_t* __restrict__ in_ptr,
                                                                const int32_t* __restrict__ in_perm,
                                                                const float* __restrict__ scores, float score_min,
                                                                const int32_t* __restrict__ ptr,
                                                                int32_t* __restrict__ first, int32_t* __restrict__ second) {
  const int c = blockIdx.x * kThreads + threadIdx.x;
  if (c >= n_hits) return;
  const size_t ld = (size_t)n_hits + 1;
  const long long n_art = ptr[n_hits], n_left = ptr[ld + n_hits];
  const int o0 = row_ptr[c], o1 = row_ptr[c + 1], i0 = in_ptr[c], i1 = in_ptr[c + 1];
  long long w = ptr[c];                                   // articulations: I(C) x O(C), the incoming edge slowest
  for (int k = i0; k < i1; ++k) {
    const int a = in_perm[k];
    if (!(scores[a] >= score_min)) continue;
    for (int b = o0; b < o1; ++b)
      if (scores[b] >= score_min) { first[w] = a; second[w] = b; ++w; }
  }
  w = n_art + ptr[ld + c];                                // left elbows: pairs of O(C)
  for (int a = o0; a < o1; ++a) {
    if (!(scores[a] >= score_min)) continue;
    for (int b = a + 1; b < o1; ++b)
      if (scores[b] >= score_min) { first[w] = a; second[w] = b; ++w; }
  }
  w = n_art + n_left + ptr[2 * ld + c];                   // right elbows: pairs of I(C)
  for (int k = i0; k < i1; ++k) {
    const int a = in_perm[k];
    if (!(scores[a] >= score_min)) continue;
    for (int q = k + 1; q < i1; ++q) {
      const int b = in_perm[q];
      if (scores[b] >= score_min) { first[w] = a; second[w] = b; ++w; }
    }
  }
}

}  // namespace

int launch_triplet_count(int n_hits, const int32_t* row_ptr, const int32_t* in_ptr, const int32_t* in_perm,
                         const float* scores, float score_min, int32_t* ptr, cudaStream_t s) {
  triplet_count_kernel<<<(n_hits + kThreads) / kThreads, kThreads, 0, s>>>(n_hits, row_ptr, in_ptr, in_perm, scores,
                                                                             score_min, ptr);
  return 1;
}

int launch_triplet_fill(int n_hits, const int32_t* row_ptr, const int32_t* in_ptr, const int32_t* in_perm,
                        const float* scores, float score_min, const int32_t* ptr, int32_t* first, int32_t* second,
                        cudaStream_t s) {
  if (n_hits <= 0) return 0;
  triplet_fill_kernel<<<(n_hits + kThreads - 1) / kThreads, kThreads, 0, s>>>(n_hits, row_ptr, in_ptr, in_perm, scores,
                                                                                score_min, ptr, first, second);
  return 1;
}

}  // namespace etx
