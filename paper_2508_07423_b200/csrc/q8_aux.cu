// Next row (NEXT-3, GNN part), helper of ETX_PREC_INT8: the node encoder's FIRST layer (3 normalised geometry features
// in) stays an fp32 layer (DESIGN Q24); its ReLU output is the first tensor the INT8 chain quantises, so it must
// be reproducible to the last bit: the 3-term dot product accumulates in double, products exact, adds individually
// rounded (no FMA), then one rounding to fp32 -- the arithmetic convention of the hot path's definition.
#include "common.cuh"

namespace etx {
namespace {

__global__ void __launch_bounds__(256) node_l1_kernel(int n_rows, int H, const float* __restrict__ f0, const float* __restrict__ f1,
                                                      const float* __restrict__ f2, float c0, float c1, float c2, float s0,
                                                      float s1, float s2, const float* __restrict__ Wt /*[3][H]*/,
                                                      const float* __restrict__ b, float* __restrict__ out /*[n_rows][H]*/) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)n_rows * H) return;
  const int row = (int)(i / H), o = (int)(i % H);
  const double x = (double)__fdiv_rn(__fsub_rn(__ldg(f0 + row), c0), s0);
  const double y = (double)__fdiv_rn(__fsub_rn(__ldg(f1 + row), c1), s1);
  const double z = (double)__fdiv_rn(__fsub_rn(__ldg(f2 + row), c2), s2);
  double acc = __dmul_rn((double)__ldg(Wt + o), x);                                  // 0 + w0 x is exact
  acc = __dadd_rn(acc, __dmul_rn((double)__ldg(Wt + H + o), y));
  acc = __dadd_rn(acc, __dmul_rn((double)__ldg(Wt + 2 * H + o), z));
  acc = __dadd_rn(acc, (double)__ldg(b + o));
  const float v = (float)acc;
  out[i] = v > 0.0f ? v : 0.0f;
}

}  // namespace

int launch_node_l1(int n_rows, int H, const float* const feat[3], const float fc[3], const float fs[3], const float* Wt,
                   const float* b, float* out, cudaStream_t s) {
  if (n_rows <= 0) return 0;
  const long long n = (long long)n_rows * H;
  node_l1_kernel<<<(int)((n + 255) / 256), 256, 0, s>>>(n_rows, H, feat[0], feat[1], feat[2], fc[0], fc[1], fc[2], fs[0], fs[1],
                                                         fs[2], Wt, b, out);
  return 1;
}

}  // namespace etx
