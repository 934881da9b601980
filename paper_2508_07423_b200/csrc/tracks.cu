// NEXT-1 — score cut + track building.
// Purified hit graph = edges with score >= score_min; tracks = its weakly connected components; the
// label of a hit is the smallest hit index of its component.
//
// The thesis propagates minimum labels in two plane sweeps (forward over the left neighbours, backward
// over the right ones).  Two sweeps are not always enough (a zig-zag component keeps a wrong
// label), so the sweeps are repeated here until no label changes, which makes the result the exact WCC.
// One CTA owns an event.  Edges are source-sorted and hits plane-sorted, so walking the event's edge
// list in ascending chunks IS a forward plane sweep (labels flow src -> dst through edges handled
// earlier in the same pass) and walking it in descending chunks is the backward sweep; the order needs
// no plane table.  Labels live in global memory (an event's labels are ~6-14 KB: L1/L2 resident);
// min-propagation is order-independent, so atomicMin gives a deterministic result.
#include "common.cuh"

namespace etx {
namespace {

constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads) wcc_kernel(int n_events, const int32_t* __restrict__ event_ptr,
                                                       const int32_t* __restrict__ row_ptr,
                                                       const int32_t* __restrict__ src,
                                                       const int32_t* __restrict__ dst,
                                                       const float* __restrict__ scores, float score_min,
                                                       int32_t* labels) {
  __shared__ int changed;
  for (int ev = blockIdx.x; ev < n_events; ev += gridDim.x) {
    const int h0 = event_ptr[ev], h1 = event_ptr[ev + 1];
    const int e0 = row_ptr[h0], e1 = row_ptr[h1];
    for (int i = h0 + threadIdx.x; i < h1; i += kThreads) labels[i] = i;
    __syncthreads();
    const int n_chunks = (e1 - e0 + kThreads - 1) / kThreads;
    for (;;) {                                           // until stable: labels only decrease, so this terminates (2-3 rounds on tracks)
      if (threadIdx.x == 0) changed = 0;
      __syncthreads();
      int local = 0;
      for (int c = 0; c < n_chunks; ++c) {               // forward sweep: dst takes the min of its left neighbours
        const int k = e0 + c * kThreads + threadIdx.x;
        if (k < e1 && scores[k] >= score_min) {
          const int ls = ((volatile int32_t*)labels)[src[k]];
          if (atomicMin(&labels[dst[k]], ls) > ls) local = 1;
        }
        __syncthreads();
      }
      for (int c = n_chunks - 1; c >= 0; --c) {          // backward sweep: src takes the min of its right neighbours
        const int k = e0 + c * kThreads + threadIdx.x;
        if (k < e1 && scores[k] >= score_min) {
          const int ld = ((volatile int32_t*)labels)[dst[k]];
          if (atomicMin(&labels[src[k]], ld) > ld) local = 1;
        }
        __syncthreads();
      }
      if (local) changed = 1;
      __syncthreads();
      const int again = changed;
      __syncthreads();
      if (!again) break;
    }
  }
}

}  // namespace

int launch_wcc(int n_events, const int32_t* event_ptr, const int32_t* row_ptr, const int32_t* src,
               const int32_t* dst, const float* scores, float score_min, int32_t* labels, cudaStream_t s) {
  if (n_events <= 0) return 0;
  const int cap = 148 * 8;
  wcc_kernel<<<n_events < cap ? n_events : cap, kThreads, 0, s>>>(n_events, event_ptr, row_ptr, src, dst, scores,
                                                                   score_min, labels);
  return 1;
}

}  // namespace etx
