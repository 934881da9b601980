// Measured denominators for the rooflines bench.py reports that MEASURED_PEAKS.json does not hold: the rate at which
// one B200 retires UNFUSED fp32 additions / multiplications -- the operation mix of the radius search's distance test
// (Eq. 8.1: differences, squares and their sum, each individually rounded; graph.cu), as scalar instructions
// (FADD / FMUL) and as the packed pairs the d = 4 path uses (add.rn.f32x2 / mul.rn.f32x2) -- and fused FFMA, the
// exact-fp32 MLP kernel's instruction (mlp_simt.cu).  A measurement utility, not a step of the path.
#include "common.cuh"

namespace etx {
namespace {

constexpr int kChains = 8;          // independent dependency chains per thread (hides the 4-cycle ALU latency)
constexpr int kIters = 4096;

template <int KIND>
__global__ void __launch_bounds__(256) alu_peak_kernel(float* __restrict__ out, float seed) {
  float x[kChains], y[kChains];
#pragma unroll
  for (int c = 0; c < kChains; ++c) { x[c] = seed + (float)(threadIdx.x + c); y[c] = 1.0f + 1e-7f * (float)c; }
  if constexpr (KIND == 0) {         // scalar, unfused: one addition and one multiplication per chain and iteration
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
      for (int c = 0; c < kChains; ++c) x[c] = __fmul_rn(__fadd_rn(x[c], y[c]), y[c]);
    }
  } else if constexpr (KIND == 1) {  // packed pairs: two additions and two multiplications per instruction pair
    unsigned long long p[kChains], q[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) {
      asm("mov.b64 %0, {%1, %2};" : "=l"(p[c]) : "f"(x[c]), "f"(x[c] + 0.5f));
      asm("mov.b64 %0, {%1, %2};" : "=l"(q[c]) : "f"(y[c]), "f"(y[c]));
    }
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
      for (int c = 0; c < kChains; ++c) {
        asm("add.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(q[c]));
        asm("mul.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(q[c]));
      }
    }
#pragma unroll
    for (int c = 0; c < kChains; ++c) {
      float lo, hi;
      asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p[c]));
      x[c] = lo + hi;
    }
  } else {                           // fused multiply-add: 2 flop per instruction
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
      for (int c = 0; c < kChains; ++c) { x[c] = fmaf(x[c], y[c], y[c]); x[c] = fmaf(x[c], y[c], y[c]); }
    }
  }
  float s = 0.0f;
#pragma unroll
  for (int c = 0; c < kChains; ++c) s += x[c];
  if (s == 12345.678f) out[0] = s;   // never true for these inputs: keeps the chains alive without a store per thread
}

}  // namespace
}  // namespace etx

extern "C" etx_status etx_measure_alu_peak(int32_t device, int32_t kind, double* ops_per_s) {
  using namespace etx;
  if (!ops_per_s || kind < 0 || kind > 2) return ETX_ERR_INVALID;
  if (cudaSetDevice(device) != cudaSuccess) return ETX_ERR_CUDA;
  int sms = 0;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return ETX_ERR_CUDA;
  float* d_out = nullptr;
  cudaEvent_t e0, e1;
  if (cudaMalloc(&d_out, sizeof(float)) != cudaSuccess) return ETX_ERR_CUDA;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int grid = sms * 8, threads = 256;
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {              // first repetitions warm up; the best of the rest is the burst peak
    cudaEventRecord(e0, 0);
    if (kind == 0) alu_peak_kernel<0><<<grid, threads>>>(d_out, 1.0f);
    else if (kind == 1) alu_peak_kernel<1><<<grid, threads>>>(d_out, 1.0f);
    else alu_peak_kernel<2><<<grid, threads>>>(d_out, 1.0f);
    cudaEventRecord(e1, 0);
    if (cudaEventSynchronize(e1) != cudaSuccess) break;
    float ms = 0.0f;
    cudaEventElapsedTime(&ms, e0, e1);
    // arithmetic operations retired: scalar 2 per chain step, packed 4, fused 4 (2 FFMA x 2 flop)
    const double per_step = (kind == 0) ? 2.0 : 4.0;
    const double ops = (double)grid * threads * kIters * kChains * per_step;
    if (rep >= 2 && ms > 0.0f) best = best > ops / (ms * 1e-3) ? best : ops / (ms * 1e-3);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(d_out);
  if (cudaGetLastError() != cudaSuccess || best == 0.0) return ETX_ERR_CUDA;
  *ops_per_s = best;
  return ETX_OK;
}
