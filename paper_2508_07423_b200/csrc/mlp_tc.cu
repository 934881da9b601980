// Fused MLP chain on the 5th-generation tensor cores (tcgen05 + TMEM), sm_100a only.
//
// Computes, for a tile of 128 rows (edges or hits), the whole chain of Eq. 4.27 layers of one
// GNN MLP — edge encoder, node/edge network or classifier — without any
// intermediate leaving the SM:
//
//   * one persistent CTA per SM, six warps:
//       warps 0-3  "row workers": thread r owns tile row r = TMEM lane r.  They gather the first
//                  layer's input rows ([h_src | h_dst | e], [h | m], ...) straight from global memory,
//                  convert them to the MMA operand type and write them into a TMEM operand ring with
//                  tcgen05.st; after each layer they read the accumulator with tcgen05.ld, apply
//                  bias + ReLU and write the next layer's A operand back into TMEM; after the last
//                  layer they add the residual and store (or apply the 1-unit head + sigmoid).
//       warp 4     weight loader: streams pre-swizzled weight tiles (16 KB, canonical K-major
//                  SWIZZLE_128B images prepared once at etx_create) from L2 into a shared-memory ring
//                  with cp.async.bulk (TMA bulk copy) completing on mbarriers.
//       warp 5     MMA issuer: one thread issues tcgen05.mma with A from TMEM and B from shared
//                  memory, accumulating in TMEM; tcgen05.commit releases ring slots and hands the
//                  accumulator to the workers.
//   * hidden activations never touch shared or global memory: accumulator -> registers -> TMEM.
//   * TMEM map (512 columns): [0,128) accumulator | hidden A operand | first-layer A operand ring.
//
// Precision modes:
//   ETX_PREC_TF32X3: x = hi + lo with hi = x & 0xffffe000 (top 11 significand bits), lo = x - hi;
//                    x.w ~ lo.w_hi + hi.w_lo + hi.w_hi as three kind::tf32 MMAs, fp32 accumulate.
//                    The dropped lo.w_lo term is ~2^-22 relative: fp32-equivalent.
//   ETX_PREC_BF16:   operands rounded to bf16 (RNE), one kind::f16 MMA, fp32 accumulate; the state
//                    (h, e, m) and the residual adds stay fp32.
#include "common.cuh"

namespace etx {
namespace {

constexpr int TM = 128;
constexpr int kThreads = 192;
constexpr int HW = 128;                       // hidden width handled by this kernel

template <int MODE> struct Cfg;
template <> struct Cfg<ETX_PREC_TF32X3> {
  static constexpr int KA = 32;               // K elements per 128-byte swizzle atom
  static constexpr int PIECES = 2;            // hi, lo
  static constexpr int NSTAGE = 6;            // weight ring stages
  static constexpr int NSLOT = 2;             // first-layer A operand ring slots (TMEM)
  static constexpr int A_COLS = 32;           // TMEM columns per piece per chunk
  static constexpr uint32_t IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((HW >> 3) << 17) | ((TM >> 4) << 24);
};
template <> struct Cfg<ETX_PREC_BF16> {
  static constexpr int KA = 64;
  static constexpr int PIECES = 1;
  static constexpr int NSTAGE = 8;
  static constexpr int NSLOT = 4;
  static constexpr int A_COLS = 32;           // 64 bf16 = 32 columns
  static constexpr uint32_t IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((HW >> 3) << 17) | ((TM >> 4) << 24);
};
constexpr int kAtomBytes = 128 * 128;         // one weight tile: 128 rows (n) x 128 bytes (k)

// ------------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred P1;\n\t"
      "WAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
      "@P1 bra DONE;\n\t"
      "bra WAIT_LOOP;\n\t"
      "DONE:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]^T     (TS form: A operand in tensor memory)
template <int MODE>
__device__ __forceinline__ void mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t accumulate) {
  if constexpr (MODE == ETX_PREC_TF32X3)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(Cfg<MODE>::IDESC), "r"(accumulate) : "memory");
  else
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(Cfg<MODE>::IDESC), "r"(accumulate) : "memory");
}
// 32 lanes x 32 consecutive columns: thread i of the warp owns lane (base + i)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
        "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
        "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
      "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
      ::"r"(taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
        "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]),
        "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]), "r"(v[20]), "r"(v[21]), "r"(v[22]), "r"(v[23]),
        "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]), "r"(v[31])
      : "memory");
}
// K-major SWIZZLE_128B shared-memory matrix descriptor: 8-row groups 1024 B apart (SBO), version 1
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr) {
  return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) |
         ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {   // lo -> bits [0,16)
  uint32_t d;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}
__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }

// Writes one chunk (KA k-values of this thread's row) of an A operand into TMEM at column `col`.
// TF32X3: hi piece at col, lo piece at col + lo_off.  BF16: packed pairs at col.
template <int MODE>
__device__ __forceinline__ void store_operand_chunk(uint32_t lane_addr, uint32_t col, uint32_t lo_off,
                                                    const float (&x)[Cfg<MODE>::KA]) {
  uint32_t v[32];
  if constexpr (MODE == ETX_PREC_TF32X3) {
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(x[i]) & 0xffffe000u;
    tmem_st32(lane_addr + col, v);
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(x[i] - __uint_as_float(v[i]));
    tmem_st32(lane_addr + col + lo_off, v);
  } else {
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = pack_bf16x2(x[2 * i], x[2 * i + 1]);
    tmem_st32(lane_addr + col, v);
  }
}

struct Bars {                                   // mbarriers (8 bytes each) + TMEM base
  uint64_t w_full[8], w_empty[8], a_full[4], a_empty[4], acc_full, work_done;
  uint32_t tmem_base;
};

template <int MODE>
__global__ void __launch_bounds__(kThreads, 1) mlp_tc_kernel(const TcArgs a) {
  using C = Cfg<MODE>;
  constexpr int KA = C::KA, P = C::PIECES, NSTAGE = C::NSTAGE, NSLOT = C::NSLOT, AC = C::A_COLS;
  constexpr uint32_t kStageBytes = P * kAtomBytes;
  constexpr int HID_COLS = HW * (MODE == ETX_PREC_TF32X3 ? 4 : 2) / 4;   // columns per piece of a hidden operand
  constexpr uint32_t COL_ACC = 0, COL_HID = 128, COL_A = COL_HID + P * HID_COLS;
  constexpr int HCH = HW / KA;                  // chunks per hidden layer

  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t wring = (raw + 1023u) & ~1023u;                         // SWIZZLE_128B needs 1024-byte alignment
  Bars* bars = reinterpret_cast<Bars*>(smem_raw + (wring - raw) + NSTAGE * kStageBytes);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_tiles = (a.n_rows + TM - 1) / TM;
  const int n_gemm = (a.out_mode == 3) ? a.n_layers - 1 : a.n_layers;
  const int nc1 = a.K0 / KA;

  if (threadIdx.x == 0) {
    for (int i = 0; i < NSTAGE; ++i) { mbar_init(smem_u32(&bars->w_full[i]), 1); mbar_init(smem_u32(&bars->w_empty[i]), 1); }
    for (int i = 0; i < NSLOT; ++i) { mbar_init(smem_u32(&bars->a_full[i]), 128); mbar_init(smem_u32(&bars->a_empty[i]), 1); }
    mbar_init(smem_u32(&bars->acc_full), 1);
    mbar_init(smem_u32(&bars->work_done), 128);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 5) {                               // TMEM: all 512 columns of this SM (1 CTA per SM)
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&bars->tmem_base)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;

  if (warp < 4) {
    // =========================== row workers ===========================
    const int r = threadIdx.x;
    const uint32_t lane_addr = tmem + ((uint32_t)(warp * 32) << 16);
    uint32_t a_cnt = 0, layer_cnt = 0;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
      const int row = tile * TM + r;
      const int grow = row < a.n_rows ? row : a.n_rows - 1;
      const float* segp[3];
#pragma unroll
      for (int s = 0; s < 3; ++s) {
        segp[s] = nullptr;
        if (s < a.n_seg) {
          const int idx = a.seg[s].idx ? __ldg(a.seg[s].idx + grow) : grow;
          segp[s] = a.seg[s].base + (size_t)idx * a.seg[s].ld;
        }
      }
      // ---- first layer: gather chunks into the TMEM operand ring
      for (int c = 0; c < nc1; ++c, ++a_cnt) {
        const uint32_t slot = a_cnt % NSLOT, n = a_cnt / NSLOT;
        const int k0 = c * KA;
        int s = 0, start = 0;
        while (s < a.n_seg - 1 && k0 >= start + a.seg[s].width) { start += a.seg[s].width; ++s; }
        const float4* src = reinterpret_cast<const float4*>((s == 0 ? segp[0] : (s == 1 ? segp[1] : segp[2])) + (k0 - start));
        float x[KA];
#pragma unroll
        for (int i = 0; i < KA / 4; ++i) {
          const float4 t = __ldg(src + i);
          x[4 * i] = t.x; x[4 * i + 1] = t.y; x[4 * i + 2] = t.z; x[4 * i + 3] = t.w;
        }
        mbar_wait(smem_u32(&bars->a_empty[slot]), (n & 1) ^ 1);
        tc_fence_after();
        store_operand_chunk<MODE>(lane_addr, COL_A + slot * P * AC, AC, x);
        tc_wait_st();
        tc_fence_before();
        mbar_arrive(smem_u32(&bars->a_full[slot]));
      }
      // ---- epilogues
      for (int l = 0; l < n_gemm; ++l, ++layer_cnt) {
        const float* __restrict__ bias = a.bias[l];
        mbar_wait(smem_u32(&bars->acc_full), layer_cnt & 1);
        tc_fence_after();
        const bool last = (l == n_gemm - 1);
        if (!last) {                             // hidden layer: ReLU(x + b) -> next A operand in TMEM
#pragma unroll 1
          for (int q = 0; q < HW / 32; ++q) {
            uint32_t v[32];
            tmem_ld32(lane_addr + COL_ACC + q * 32, v);
            tc_wait_ld();
            if constexpr (MODE == ETX_PREC_TF32X3) {
              float x[32];
#pragma unroll
              for (int i = 0; i < 32; ++i) x[i] = fmaxf(__uint_as_float(v[i]) + __ldg(bias + q * 32 + i), 0.f);
              store_operand_chunk<MODE>(lane_addr, COL_HID + q * 32, HID_COLS, reinterpret_cast<const float(&)[KA]>(x));
            } else {                             // 32 accumulator columns -> 16 packed bf16 columns
              uint32_t w[16];
#pragma unroll
              for (int i = 0; i < 16; ++i) {
                const float x0 = fmaxf(__uint_as_float(v[2 * i]) + __ldg(bias + q * 32 + 2 * i), 0.f);
                const float x1 = fmaxf(__uint_as_float(v[2 * i + 1]) + __ldg(bias + q * 32 + 2 * i + 1), 0.f);
                w[i] = pack_bf16x2(x0, x1);
              }
              asm volatile(
                  "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
                  "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
                  ::"r"(lane_addr + COL_HID + q * 16),
                    "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]),
                    "r"(w[8]), "r"(w[9]), "r"(w[10]), "r"(w[11]), "r"(w[12]), "r"(w[13]), "r"(w[14]), "r"(w[15])
                  : "memory");
            }
          }
          tc_wait_st();
        } else if (a.out_mode == 3) {            // classifier: last hidden layer, then 1 unit + sigmoid
          float logit = 0.f;
#pragma unroll 1
          for (int q = 0; q < HW / 32; ++q) {
            uint32_t v[32];
            tmem_ld32(lane_addr + COL_ACC + q * 32, v);
            tc_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; ++i) {
              const float x = fmaxf(__uint_as_float(v[i]) + __ldg(bias + q * 32 + i), 0.f);
              logit = fmaf(x, __ldg(a.w_last + q * 32 + i), logit);
            }
          }
          logit += __ldg(a.bias[a.n_layers - 1]);
          if (row < a.n_rows) a.out[row] = 1.0f / (1.0f + expf(-logit));
        } else {                                 // linear output (+ residual) -> global
          float* __restrict__ out = a.out + (size_t)grow * a.out_ld;
          const float* __restrict__ res = a.res ? a.res + (size_t)grow * a.out_ld : nullptr;
#pragma unroll 1
          for (int q = 0; q < HW / 32; ++q) {
            uint32_t v[32];
            tmem_ld32(lane_addr + COL_ACC + q * 32, v);
            tc_wait_ld();
            if (row < a.n_rows) {
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                const float4 b = __ldg(reinterpret_cast<const float4*>(bias + q * 32) + i);
                float4 y = make_float4(__uint_as_float(v[4 * i]) + b.x, __uint_as_float(v[4 * i + 1]) + b.y,
                                       __uint_as_float(v[4 * i + 2]) + b.z, __uint_as_float(v[4 * i + 3]) + b.w);
                if (a.out_mode == 1) {
                  const float4 t = *(reinterpret_cast<const float4*>(res + q * 32) + i);
                  y.x += t.x; y.y += t.y; y.z += t.z; y.w += t.w;
                }
                *(reinterpret_cast<float4*>(out + q * 32) + i) = y;
              }
            }
          }
        }
        tc_fence_before();
        mbar_arrive(smem_u32(&bars->work_done));
      }
    }
  } else if (warp == 4) {
    // =========================== weight loader ===========================
    if (lane == 0) {
      const int chunks_per_tile = nc1 + (n_gemm - 1) * HCH;
      uint32_t w_cnt = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        for (int q = 0; q < chunks_per_tile; ++q, ++w_cnt) {
          const uint32_t ws = w_cnt % NSTAGE, wn = w_cnt / NSTAGE;
          mbar_wait(smem_u32(&bars->w_empty[ws]), (wn & 1) ^ 1);
          mbar_expect_tx(smem_u32(&bars->w_full[ws]), kStageBytes);
          bulk_g2s(wring + ws * kStageBytes, a.wimg + (size_t)q * kStageBytes, kStageBytes, smem_u32(&bars->w_full[ws]));
        }
      }
    }
  } else {
    // =========================== MMA issuer ===========================
    if (lane == 0) {
      uint32_t w_cnt = 0, a_cnt = 0, g = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        for (int l = 0; l < n_gemm; ++l, ++g) {
          if (g > 0) {                           // previous epilogue done: accumulator free, hidden operand written
            mbar_wait(smem_u32(&bars->work_done), (g - 1) & 1);
            tc_fence_after();
          }
          const int nch = (l == 0) ? nc1 : HCH;
          for (int c = 0; c < nch; ++c, ++w_cnt) {
            const uint32_t ws = w_cnt % NSTAGE, wn = w_cnt / NSTAGE;
            uint32_t a_col, lo_off, slot = 0;
            if (l == 0) {
              slot = a_cnt % NSLOT;
              mbar_wait(smem_u32(&bars->a_full[slot]), (a_cnt / NSLOT) & 1);
              a_col = COL_A + slot * P * AC; lo_off = AC;
            } else {
              a_col = COL_HID + c * AC; lo_off = HID_COLS;
            }
            mbar_wait(smem_u32(&bars->w_full[ws]), wn & 1);
            tc_fence_after();
            const uint32_t wb = wring + ws * kStageBytes;
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {       // 4 MMA k-steps of 32 bytes inside the 128-byte atom
              const uint32_t acc = (c > 0 || ks > 0) ? 1u : 0u;
              const uint32_t a_hi = tmem + a_col + ks * 8;
              const uint64_t b_hi = smem_desc(wb + ks * 32);
              if constexpr (MODE == ETX_PREC_TF32X3) {
                const uint32_t a_lo = a_hi + lo_off;
                const uint64_t b_lo = smem_desc(wb + kAtomBytes + ks * 32);
                mma_ts<MODE>(tmem + COL_ACC, a_lo, b_hi, acc);       // small terms first
                mma_ts<MODE>(tmem + COL_ACC, a_hi, b_lo, 1u);
                mma_ts<MODE>(tmem + COL_ACC, a_hi, b_hi, 1u);
              } else {
                mma_ts<MODE>(tmem + COL_ACC, a_hi, b_hi, acc);
              }
            }
            tc_commit(smem_u32(&bars->w_empty[ws]));
            if (l == 0) { tc_commit(smem_u32(&bars->a_empty[slot])); ++a_cnt; }
          }
          tc_commit(smem_u32(&bars->acc_full));
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 5) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
  }
}

template <int MODE>
int launch_mode(const TcArgs& a, int sm_count, cudaStream_t s) {
  using C = Cfg<MODE>;
  static bool configured = false;
  const size_t smem = 1024 + (size_t)C::NSTAGE * C::PIECES * kAtomBytes + sizeof(Bars) + 64;
  if (!configured) {
    cudaFuncSetAttribute(mlp_tc_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    configured = true;
  }
  const int n_tiles = (a.n_rows + TM - 1) / TM;
  const int grid = n_tiles < sm_count ? n_tiles : sm_count;
  mlp_tc_kernel<MODE><<<grid, kThreads, smem, s>>>(a);
  return 1;
}

}  // namespace

int tc_chunk_k(int mode) { return mode == ETX_PREC_TF32X3 ? Cfg<ETX_PREC_TF32X3>::KA : Cfg<ETX_PREC_BF16>::KA; }

// Requirements (checked by the caller): hidden width 128; K0 a multiple of the chunk (32 / 64) and
// segment widths multiples of it; out_mode 0/1 needs dims[L] == 128; out_mode 3 needs dims[L] == 1.
int launch_mlp_tc(const TcArgs& a, int mode, int sm_count, cudaStream_t s) {
  if (a.n_rows <= 0) return 0;
  if (mode == ETX_PREC_TF32X3) return launch_mode<ETX_PREC_TF32X3>(a, sm_count, s);
  if (mode == ETX_PREC_BF16) return launch_mode<ETX_PREC_BF16>(a, sm_count, s);
  return -1;
}

}  // namespace etx
