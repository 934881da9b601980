// a4 — message aggregation, Eq. 8.5: m_l = [ sum_{l->j} e_lj , sum_{i->l} e_il ].
// The thesis' pipeline did this with a scatter_add operator / TensorRT plugin, i.e.
// atomics.  Here both halves are SEGMENTED REDUCTIONS with a fixed summation order (deterministic):
// edges are source-sorted, so the outgoing sum of hit l is a contiguous run of rows of e; the incoming
// sum walks the by-destination list in_perm (ascending edge id).  One warp owns a hit; a lane owns
// H/32 consecutive features, so every row read is one fully coalesced 512-byte (H=128) request, and
// four rows are kept in flight per lane.  fp32 accumulation always (BASELINE.json C3).
// Roofline: HBM — e is needed twice (once per half) but, with the in-order work distribution below, the
// second use hits in L2: DRAM traffic ~ E x H x 4 B (+ 4 B per edge of in_perm) read, N x 2H x 4 B written.
#include "common.cuh"

namespace etx {
namespace {

template <int V> struct Vec;
template <> struct Vec<4> { using T = float4; };
template <> struct Vec<2> { using T = float2; };

__device__ __forceinline__ void add(float4& a, const float4& b) { a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w; }
__device__ __forceinline__ void add(float2& a, const float2& b) { a.x += b.x; a.y += b.y; }
__device__ __forceinline__ void zero(float4& a) { a = make_float4(0.f, 0.f, 0.f, 0.f); }
__device__ __forceinline__ void zero(float2& a) { a = make_float2(0.f, 0.f); }

template <int H>
__global__ void __launch_bounds__(256) scatter_kernel(int n_nodes, const int32_t* __restrict__ row_ptr,
                                                      const int32_t* __restrict__ in_ptr,
                                                      const int32_t* __restrict__ in_perm,
                                                      const float* __restrict__ e, float* __restrict__ m,
                                                      int* __restrict__ next_hit) {
  using T = typename Vec<H / 32>::T;
  const int lane = threadIdx.x & 31;
  __shared__ int s_base;
  const T* __restrict__ ev = reinterpret_cast<const T*>(e);
  T* __restrict__ mv = reinterpret_cast<T*>(m);
  constexpr int RV = H / (H / 32);                 // vectors per row of e  (= 32)
  // Hits are handed out IN ORDER, 8 at a time (one per warp), through a global counter: whatever the
  // relative speed of the CTAs, the hits in flight are always the most recent ~9.5k, so a row of e read
  // as an outgoing edge of its source is still in L2 when its destination (<= G planes later in the same
  // event) reads it as an incoming edge.  (A static grid-stride assignment lets CTAs drift apart by more
  // than the L2 holds: measured 9.2 GB of DRAM reads per launch for 4.9 GB of e.)
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) s_base = atomicAdd(next_hit, (int)(blockDim.x >> 5));
    __syncthreads();
    const int base = s_base;
    if (base >= n_nodes) break;
    const int l = base + (int)(threadIdx.x >> 5);
    if (l >= n_nodes) continue;
    T acc_out, acc_in;
    zero(acc_out); zero(acc_in);
    {                                              // outgoing: contiguous rows row_ptr[l] .. row_ptr[l+1]
      const int k0 = __ldg(row_ptr + l), k1 = __ldg(row_ptr + l + 1);
      int k = k0;
      for (; k + 4 <= k1; k += 4) {
        const T a = __ldg(ev + (size_t)(k + 0) * RV + lane), b = __ldg(ev + (size_t)(k + 1) * RV + lane);
        const T c = __ldg(ev + (size_t)(k + 2) * RV + lane), d = __ldg(ev + (size_t)(k + 3) * RV + lane);
        add(acc_out, a); add(acc_out, b); add(acc_out, c); add(acc_out, d);
      }
      for (; k < k1; ++k) add(acc_out, __ldg(ev + (size_t)k * RV + lane));
    }
    {                                              // incoming: gathered rows in_perm[in_ptr[l] ..]
      const int k0 = __ldg(in_ptr + l), k1 = __ldg(in_ptr + l + 1);
      int k = k0;
      for (; k + 4 <= k1; k += 4) {
        const int i0 = __ldg(in_perm + k), i1 = __ldg(in_perm + k + 1);
        const int i2 = __ldg(in_perm + k + 2), i3 = __ldg(in_perm + k + 3);
        const T a = __ldg(ev + (size_t)i0 * RV + lane), b = __ldg(ev + (size_t)i1 * RV + lane);
        const T c = __ldg(ev + (size_t)i2 * RV + lane), d = __ldg(ev + (size_t)i3 * RV + lane);
        add(acc_in, a); add(acc_in, b); add(acc_in, c); add(acc_in, d);
      }
      for (; k < k1; ++k) add(acc_in, __ldg(ev + (size_t)__ldg(in_perm + k) * RV + lane));
    }
    mv[(size_t)l * 2 * RV + lane] = acc_out;       // outgoing first (Eq. 8.5)
    mv[(size_t)l * 2 * RV + RV + lane] = acc_in;
  }
}

#ifdef ETX_DEV_SWITCHES
// The alternative the thesis' pipeline used (scatter_add), kept ONLY as a measured comparison
// (developer builds, -DETX_DEV_SWITCHES, with ETX_SCATTER_ATOMIC=1): one warp per edge row, one vector reduction
// (red.global.add.v4.f32) per lane into m[src] (outgoing half) and m[dst] (incoming half) of a zeroed m.
// Summation order is whatever the L2 serialises: not deterministic, and measured slower.
__global__ void __launch_bounds__(256) scatter_atomic_kernel(long long n_edges, const int32_t* __restrict__ src,
                                                             const int32_t* __restrict__ dst,
                                                             const float* __restrict__ e, float* __restrict__ m) {
  const int lane = threadIdx.x & 31;
  const long long n_warps = (long long)gridDim.x * (blockDim.x >> 5);
  for (long long k = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); k < n_edges; k += n_warps) {
    const float4 v = __ldg(reinterpret_cast<const float4*>(e) + k * 32 + lane);
    float* po = m + (size_t)__ldg(src + k) * 256 + lane * 4;
    float* pi = m + (size_t)__ldg(dst + k) * 256 + 128 + lane * 4;
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(po), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(pi), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
  }
}
#endif

}  // namespace

#ifdef ETX_DEV_SWITCHES
int launch_scatter_atomic(int n_nodes, long long n_edges, int H, const int32_t* src, const int32_t* dst,
                          const float* e, float* m, cudaStream_t s) {
  if (n_nodes <= 0 || H != 128) return n_nodes <= 0 ? 0 : -1;
  cudaMemsetAsync(m, 0, sizeof(float) * (size_t)n_nodes * 2 * H, s);
  if (n_edges <= 0) return 0;
  const long long need = (n_edges + 7) / 8;
  scatter_atomic_kernel<<<(int)(need < 148 * 8 ? need : 148 * 8), 256, 0, s>>>(n_edges, src, dst, e, m);
  return 1;
}
#endif

int launch_scatter(int n_nodes, int H, const int32_t* row_ptr, const int32_t* in_ptr,
                   const int32_t* in_perm, const float* e, float* m, int32_t* counter, cudaStream_t s) {
  if (n_nodes <= 0) return 0;
  cudaMemsetAsync(counter, 0, sizeof(int32_t), s);
  const int need = (n_nodes + 7) / 8;
  const int cap = 148 * 8;                         // 8 resident CTAs of 256 threads per SM
  const int grid = need < cap ? need : cap;
  if (H == 128) scatter_kernel<128><<<grid, 256, 0, s>>>(n_nodes, row_ptr, in_ptr, in_perm, e, m, counter);
  else if (H == 64) scatter_kernel<64><<<grid, 256, 0, s>>>(n_nodes, row_ptr, in_ptr, in_perm, e, m, counter);
  else return -1;
  return 1;
}

}  // namespace etx
