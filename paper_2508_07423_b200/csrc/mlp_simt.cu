// Fused MLP chain on the CUDA cores in exact fp32 (ETX_PREC_FP32): one CTA owns a tile of 128 rows
// (hits or edges), gathers the first layer's input straight from the node / edge arrays (the
// concatenations [h_src, h_dst, e], [h, m] of P:2332-2339 are never materialised), keeps every hidden
// activation in shared memory, and writes only the final result (+ residual, or the sigmoid score).
// Each layer is f_l(z) = g_l(W_l z + b_l), Eq. 4.27, ReLU on hidden layers.
//
// Tiling: 256 threads, each an 8 x (H/16) register tile; activations are kept k-major (Xs[k][row]) so
// the per-k operand fetch is two broadcast LDS.128; weights are pre-transposed to [in][out] on the
// host side so a K-chunk is one contiguous slab streamed by cp.async (they live in L2: ~0.3 MB per
// network, read by every CTA).  Double-buffered K-chunks of 16; 2 CTAs per SM.
//
// This is the exact-fp32 path (FFMA roofline).  The tensor-core paths live in mlp_tc.cu.
#include "common.cuh"

namespace etx {
namespace {

constexpr int TM = 128;        // rows per CTA
constexpr int KC = 16;         // K chunk
constexpr int NT = 256;        // threads per CTA
constexpr int LDA = TM + 4;    // padded leading dimension of k-major tiles (keeps float4 alignment)

template <int H>
struct Smem {
  float Hs[H][LDA];            // hidden activations, Hs[k][row]
  float As[2][KC][LDA];        // first-layer input chunks, As[buf][k][row]
  float Ws[2][KC][H];          // weight chunks, Ws[buf][k][n]
};

__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(src));
}
__device__ __forceinline__ void cp_async4(void* dst, const void* src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(d), "l"(src));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

template <int H>
__global__ void __launch_bounds__(NT, 2) mlp_simt_kernel(const MlpArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem<H>& sm = *reinterpret_cast<Smem<H>*>(smem_raw);
  constexpr int TN = H / 16;               // columns per thread (8 or 4)
  constexpr int NG = TN / 4;               // float4 column groups per thread
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int row0 = blockIdx.x * TM;
  const int lr = tid & (TM - 1);           // the input row this thread gathers
  const int kph = tid >> 7;                // and the parity of the k it copies
  const int grow = (row0 + lr < a.n_rows) ? row0 + lr : a.n_rows - 1;

  const float* segp[3] = {nullptr, nullptr, nullptr};
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    if (s < a.n_seg) {
      const int r = a.seg[s].idx ? __ldg(a.seg[s].idx + grow) : grow;
      segp[s] = a.seg[s].base + (size_t)r * a.seg[s].ld;
    }
  }
  const int L = a.mlp.n_layers;
  const bool small_out = a.out_mode >= 2;
  const int n_gemm = small_out ? L - 1 : L;     // layers run through the tiled GEMM

  for (int l = 0; l < n_gemm; ++l) {
    const int K = a.mlp.dims[l];
    const float* __restrict__ Wt = a.mlp.Wt[l];
    const bool from_input = (l == 0);
    const int n_chunks = (K + KC - 1) / KC;

    auto load_chunk = [&](int c, int buf) {
      const int k0 = c * KC;
      // weights: KC rows of H floats
#pragma unroll
      for (int i = 0; i < (KC * H / 4) / NT; ++i) {
        const int q = tid + i * NT;                // float4 index inside the chunk
        const int kk = q / (H / 4), n4 = q % (H / 4);
        float* dst = &sm.Ws[buf][kk][n4 * 4];
        if (k0 + kk < K) cp_async16(dst, Wt + (size_t)(k0 + kk) * H + n4 * 4);
        else *reinterpret_cast<float4*>(dst) = make_float4(0.f, 0.f, 0.f, 0.f);
      }
      if (!from_input) return;
      if (a.n_seg == 0) {                          // a0: features computed on the fly (one chunk)
        for (int q = tid; q < KC * TM; q += NT) {
          const int kk = q / TM, r = q % TM;
          float v = 0.f;
          if (kk < 3) {
            const int gr = (row0 + r < a.n_rows) ? row0 + r : a.n_rows - 1;
            v = __fdiv_rn(__fsub_rn(__ldg(a.feat[kk] + gr), a.fc[kk]), a.fs[kk]);
          }
          sm.As[buf][kk][r] = v;
        }
      } else {                                     // gathered segments; a chunk lies inside one segment
        int s = 0, start = 0;
        while (s < a.n_seg - 1 && k0 >= start + a.seg[s].width) { start += a.seg[s].width; ++s; }
        const float* src = (s == 0 ? segp[0] : (s == 1 ? segp[1] : segp[2])) + (k0 - start);
#pragma unroll
        for (int i = 0; i < KC / 2; ++i) {
          const int kk = kph + 2 * i;
          cp_async4(&sm.As[buf][kk][lr], src + kk);
        }
      }
    };

    float acc[8][TN];
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int j = 0; j < TN; ++j) acc[r][j] = 0.f;

    load_chunk(0, 0);
    cp_async_commit();
    for (int c = 0; c < n_chunks; ++c) {
      if (c + 1 < n_chunks) {
        load_chunk(c + 1, (c + 1) & 1);
        cp_async_commit();
        cp_async_wait<1>();
      } else {
        cp_async_wait<0>();
      }
      __syncthreads();
      const float(*A)[LDA] = from_input ? sm.As[c & 1] : &sm.Hs[c * KC];
      const float(*W)[H] = sm.Ws[c & 1];
#pragma unroll
      for (int kk = 0; kk < KC; ++kk) {
        const float4 a0 = *reinterpret_cast<const float4*>(&A[kk][ty * 8]);
        const float4 a1 = *reinterpret_cast<const float4*>(&A[kk][ty * 8 + 4]);
        const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
#pragma unroll
        for (int g = 0; g < NG; ++g) {
          const float4 w = *reinterpret_cast<const float4*>(&W[kk][g * 64 + tx * 4]);
          const float wv[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
          for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[r][g * 4 + j] = fmaf(av[r], wv[j], acc[r][g * 4 + j]);
        }
      }
      __syncthreads();
    }

    const float* __restrict__ bias = a.mlp.b[l];
    if (l < L - 1) {                               // hidden layer: bias + ReLU -> Hs (k-major)
#pragma unroll
      for (int g = 0; g < NG; ++g)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int col = g * 64 + tx * 4 + j;
          const float b = __ldg(bias + col);
          float4 v0, v1;
          v0.x = fmaxf(acc[0][g * 4 + j] + b, 0.f); v0.y = fmaxf(acc[1][g * 4 + j] + b, 0.f);
          v0.z = fmaxf(acc[2][g * 4 + j] + b, 0.f); v0.w = fmaxf(acc[3][g * 4 + j] + b, 0.f);
          v1.x = fmaxf(acc[4][g * 4 + j] + b, 0.f); v1.y = fmaxf(acc[5][g * 4 + j] + b, 0.f);
          v1.z = fmaxf(acc[6][g * 4 + j] + b, 0.f); v1.w = fmaxf(acc[7][g * 4 + j] + b, 0.f);
          *reinterpret_cast<float4*>(&sm.Hs[col][ty * 8]) = v0;
          *reinterpret_cast<float4*>(&sm.Hs[col][ty * 8 + 4]) = v1;
        }
      __syncthreads();
    } else {                                       // output layer of width H: linear (+ residual)
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int row = row0 + ty * 8 + r;
        if (row < a.n_rows) {
#pragma unroll
          for (int g = 0; g < NG; ++g) {
            const int col = g * 64 + tx * 4;
            const float4 b = __ldg(reinterpret_cast<const float4*>(bias + col));
            float4 y = make_float4(acc[r][g * 4 + 0] + b.x, acc[r][g * 4 + 1] + b.y,
                                   acc[r][g * 4 + 2] + b.z, acc[r][g * 4 + 3] + b.w);
            if (a.out_mode == 1) {
              const float4 q = *reinterpret_cast<const float4*>(a.res + (size_t)row * a.out_ld + col);
              y.x += q.x; y.y += q.y; y.z += q.z; y.w += q.w;
            }
            *reinterpret_cast<float4*>(a.out + (size_t)row * a.out_ld + col) = y;
          }
        }
      }
    }
  }

  if (small_out) {                                 // narrow output layer (embedding dim, classifier)
    const int K = a.mlp.dims[L - 1], N = a.mlp.dims[L];
    const float* __restrict__ Wt = a.mlp.Wt[L - 1];
    const float* __restrict__ bias = a.mlp.b[L - 1];
    for (int q = tid; q < TM * N; q += NT) {
      const int r = q % TM, n = q / TM;
      float s = 0.f;
      for (int k = 0; k < K; ++k) s = fmaf(sm.Hs[k][r], __ldg(Wt + (size_t)k * N + n), s);
      s += __ldg(bias + n);
      if (a.out_mode == 3) s = 1.0f / (1.0f + expf(-s));     // sigma(x) = 1/(1+e^-x)
      const int row = row0 + r;
      if (row < a.n_rows) a.out[(size_t)row * a.out_ld + n] = s;
    }
  }
}

template <int H>
int launch_h(const MlpArgs& a, cudaStream_t s) {
  static bool configured[kMaxDevices] = {false};    // the shared-memory opt-in is a per-DEVICE attribute of the function
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return -1;
  const size_t smem = sizeof(Smem<H>);
  if (!configured[dev]) {
    if (cudaFuncSetAttribute(mlp_simt_kernel<H>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
    configured[dev] = true;
  }
  const int grid = (a.n_rows + TM - 1) / TM;
  mlp_simt_kernel<H><<<grid, NT, smem, s>>>(a);
  return 1;
}

}  // namespace

// Requirements (checked by the caller, etx_api.cu): hidden widths all equal H in {64,128}; segment
// widths multiples of 16; out_mode < 2 needs dims[L] == H; out_mode >= 2 needs L >= 2, dims[L] <= 8.
int launch_mlp_simt(const MlpArgs& a, cudaStream_t s) {
  if (a.n_rows <= 0) return 0;
  const int H = a.mlp.dims[1];
  if (H == 128) return launch_h<128>(a, s);
  if (H == 64) return launch_h<64>(a, s);
  return -1;
}

}  // namespace etx
