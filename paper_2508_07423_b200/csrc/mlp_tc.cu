// Fused MLP chain on the 5th-generation tensor cores (tcgen05 + TMEM), sm_100a only.
//
// Computes, for a tile of 128 rows (edges or hits), the whole chain of Eq. 4.27 layers of one
// GNN MLP — edge encoder, node/edge network or classifier — without any
// intermediate leaving the SM.  One persistent CTA per SM, 28 warps in 7 warpgroups (register budgets
// re-partitioned with setmaxnreg: gather 64, epilogue 104, loader/MMA 40):
//
//   warps 0-15 gather:   coalesced 16-byte loads of the first layer's input rows ([h_src | h_dst | e],
//                        [h | m], ...) straight from the node / edge arrays (8 or 16 lanes per row, a
//                        ring of K-chunks prefetched in registers: 64 KB in flight per SM), conversion
//                        to the MMA operand type and st.shared into a ring of canonical K-major
//                        SWIZZLE_128B operand tiles.
//   warps 16-23 epilogue (lane quarter = warp & 3, column half = (warp-16) >> 2): thread r owns tile row r = TMEM lane r.  After a hidden layer: tcgen05.ld the
//                        accumulator 32 columns at a time, bias + ReLU, convert, tcgen05.st the next
//                        layer's A operand back into TMEM and release that K-chunk to the MMA warp at
//                        once, so the next layer's MMAs start while the rest of the epilogue runs.
//                        After the last layer: bias (+ residual) through a swizzled staging tile so
//                        the global read-modify-write is coalesced, or the 1-unit head + sigmoid.
//   warp 24    loader:   streams pre-swizzled weight tiles (prepared once at etx_create) from L2 into a
//                        shared-memory ring with cp.async.bulk (TMA bulk copy) completing on mbarriers.
//   warp 25    MMA:      one thread issues tcgen05.mma — SS form (A, B in shared memory) for the first
//                        layer, TS form (A in TMEM) for the others — into one of two 128-column TMEM
//                        accumulators (ping-pong), and tcgen05.commit-s ring slots / accumulators.
//
// TMEM map (512 columns): acc0 [0,128) | acc1 [128,256) | hidden A operand [256, ...).
// Hidden activations never touch shared or global memory.
//
// Precision modes:
//   ETX_PREC_TF32X3: x = hi + lo with hi = x & 0xffffe000 (top 11 significand bits), lo = x - hi;
//                    x.w ~ lo.w_hi + hi.w_lo + hi.w_hi as three kind::tf32 MMAs, fp32 accumulate.
//                    The dropped lo.w_lo term is ~2^-22 relative: fp32-equivalent.
//   ETX_PREC_BF16:   operands rounded to bf16 (RNE), one kind::f16 MMA, fp32 accumulate; the state
//                    (h, e, m) and the residual adds stay fp32.
//   ETX_PREC_BF16X3: x = hi + lo with hi = bf16(x), lo = bf16(x - hi) (16 significand bits), three
//                    kind::f16 MMAs lo.w_hi + hi.w_lo + hi.w_hi.  Half the MMA steps, shared-memory and
//                    L2 bytes of TF32X3.  Measured score error is the same ~1e-5 as TF32X3, because both
//                    are dominated by the tensor core's truncating fp32 accumulation.
#include <cuda.h>
#include <cuda_fp16.h>
#include <cstring>

#include "common.cuh"
#include "tc_ptx.cuh"

// Per-role cycle counters (developer aid).  Compiled in only with -DETX_TC_COUNTERS (build.py:
// ETX_TC_COUNTERS=1), because their 64-bit registers do not fit the 64-register gather budget.
#ifdef ETX_TC_COUNTERS
#define ETX_DBG(a) ((a).dbg != nullptr)
#else
#define ETX_DBG(a) false
#endif

// Timing experiments that deliberately produce WRONG results (gather every tile from the same rows, skip the weight
// copies) exist only in developer builds (-DETX_DEV_SWITCHES, build.py: ETX_DEV_SWITCHES=1).  The default library
// contains none of them: no environment variable can change what it computes.
#ifdef ETX_DEV_SWITCHES
#define ETX_EXP(a, bit) (((a).exp_flags & (bit)) != 0)
#else
#define ETX_EXP(a, bit) false
#endif

namespace etx {
namespace {

constexpr int TM = 128;
constexpr int kGatherThreads = 512;      // warpgroups 0-3 (warps 0-15)
constexpr int kEpiThreads = 256;         // warpgroups 4-5 (warps 16-23): lane quarter = warp & 3, column half = (warp - 16) >> 2
constexpr int kThreads = kGatherThreads + kEpiThreads + 128;   // + warpgroup 6: loader warp 24, MMA warp 25, two idle warps
constexpr int kWarpEpi0 = kGatherThreads / 32, kWarpLoader = kWarpEpi0 + kEpiThreads / 32, kWarpMma = kWarpLoader + 1, kWarpCommit = kWarpMma + 1;
constexpr uint32_t kBarEntry0 = 2;       // named barriers 2 .. 2 + NSTAGE_A - 1: one per operand-ring entry
// Register re-partitioning (setmaxnreg, per warpgroup): the kernel launches at <= 72 registers per
// thread (896 threads), then the gather warpgroups shrink to 64, loader/MMA to 40, and the epilogue
// warpgroups grow to 104.  More, thinner warps: the SIMT roles are latency-bound, not issue-bound.
constexpr int kRegGather = 64, kRegEpi = 104, kRegCtl = 40;
constexpr int HW = 128;                       // hidden width handled by this kernel
constexpr int kAtomBytes = 128 * 128;         // one operand tile: 128 rows x 128 bytes (one swizzle atom wide)
constexpr int kStageBoxBytes = 8 * 4096;      // output staging: 4 KB boxes [32 rows x 32 fp32 columns], Cfg::STAGE_BOXES per epilogue warp

template <int MODE> struct Cfg;
template <> struct Cfg<ETX_PREC_TF32X3> {
  static constexpr int KA = 32;               // K elements per 128-byte swizzle atom
  static constexpr int KG = 32;               // columns of one gather unit (= KA except for 8-bit operands)
  static constexpr int PIECES = 2;            // hi, lo
  // Ring split (measured, edge network at C2): the operand ring wants depth (a whole tile of entries in
  // flight), the weight ring does not (2 stages = one hidden layer; weights are never late): 4+2 -> 2+4
  // stages gave -5 % (TF32X3), -7 % (BF16X3), -9 % (BF16, 8+4 -> 4+8).
  static constexpr int NSTAGE_W = 2;          // weight ring stages (32 KB each)
  static constexpr int NSTAGE_A = 4;          // first-layer A operand ring stages (32 KB each)
  static constexpr int PREFETCH = 4;          // K-chunks a gather thread keeps in flight in registers
  static constexpr int STAGE_BOXES = 1;
  static constexpr int HID_COLS = 128;        // TMEM columns per piece of a hidden operand
  static constexpr uint32_t IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((HW >> 3) << 17) | ((TM >> 4) << 24);
};
template <> struct Cfg<ETX_PREC_BF16> {
  static constexpr int KA = 64;
  static constexpr int KG = 64;
  static constexpr int PIECES = 1;
  static constexpr int NSTAGE_W = 4;          // 16 KB each
  static constexpr int NSTAGE_A = 8;          // 16 KB each
  static constexpr int PREFETCH = 2;
  static constexpr int STAGE_BOXES = 1;
  static constexpr int HID_COLS = 64;         // 128 bf16 = 64 columns
  static constexpr uint32_t IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((HW >> 3) << 17) | ((TM >> 4) << 24);
};
template <> struct Cfg<ETX_PREC_BF16X3> {
  static constexpr int KA = 64;
  static constexpr int KG = 64;
  static constexpr int PIECES = 2;            // hi, lo (bf16 each)
  static constexpr int NSTAGE_W = 2;          // 32 KB each
  static constexpr int NSTAGE_A = 4;          // 32 KB each
  static constexpr int PREFETCH = 2;
  static constexpr int STAGE_BOXES = 1;
  static constexpr int HID_COLS = 64;
  static constexpr uint32_t IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((HW >> 3) << 17) | ((TM >> 4) << 24);
};

// Next row (NEXT-3, GNN part): INT8 codes for every layer input and weight (Eqs. 4.31-4.33), one
// kind::i8 MMA per K-step (K = 32), int32 accumulators, fp32 de-quantisation / bias / state.  A 128-byte atom holds 128
// codes, so a K-chunk is 128 wide; the fp32 rows are still gathered in 64-column units (two units fill one ring entry),
// which keeps the gather geometry -- and the fp32 / int32 addend path -- of the single-pass bf16 mode.
template <> struct Cfg<ETX_PREC_INT8> {
  static constexpr int KA = 128;
  static constexpr int KG = 64;
  static constexpr int PIECES = 1;
  static constexpr int NSTAGE_W = 4;          // 16 KB each
  static constexpr int NSTAGE_A = 8;          // 16 KB each
  static constexpr int PREFETCH = 2;
  static constexpr int STAGE_BOXES = 1;
  static constexpr int HID_COLS = 32;         // 128 codes = 32 columns
  static constexpr uint32_t IDESC = (2u << 4) | (1u << 7) | (1u << 10) | ((HW >> 3) << 17) | ((TM >> 4) << 24);   // D = s32, A = B = s8
};

// Next row (NEXT-3, GNN part) in FP8: e4m3 values for every layer input and weight (reading Q26), one
// kind::f8f6f4 MMA per K-step (K = 32), fp32 accumulators.  Same 8-bit operand geometry as the INT8 mode.
template <> struct Cfg<ETX_PREC_FP8> {
  static constexpr int KA = 128;
  static constexpr int KG = 64;
  static constexpr int PIECES = 1;
  static constexpr int NSTAGE_W = 4;          // 16 KB each
  static constexpr int NSTAGE_A = 8;          // 16 KB each
  static constexpr int PREFETCH = 2;
  static constexpr int STAGE_BOXES = 1;
  static constexpr int HID_COLS = 32;         // 128 codes = 32 columns
  static constexpr uint32_t IDESC = (1u << 4) | (0u << 7) | (0u << 10) | ((HW >> 3) << 17) | ((TM >> 4) << 24);   // D = f32, A = B = e4m3
};

// Shared-memory split per launch variant.  The wide per-hit projection launches (VAR 1: one layer, 256 output columns,
// output-bound) trade one operand-ring entry for a second staging slice per epilogue warp, so that a warp's two output
// boxes never wait for each other's TMA read (projections 3.79 -> 3.38 ms per step at C2); the multi-layer launches keep
// the deeper ring (edge network +2.5 % with 3 entries: its fp32 addend alone takes two).  Same trade in the single-pass
// bf16 mode (two of its eight 16 KB entries): projections 3.41 -> 3.26 ms at C3; on its multi-layer launches it nets zero
// (edge encoder -0.11 ms, node network -0.06, edge network +0.18).
template <int MODE, int VAR> struct Split {
  static constexpr bool kTwoBoxes = (MODE == ETX_PREC_BF16X3 || MODE == ETX_PREC_BF16) && VAR == 1;
  static constexpr int NSTAGE_A = Cfg<MODE>::NSTAGE_A - (kTwoBoxes ? 2 / Cfg<MODE>::PIECES : 0);   // 32 KB of ring entries
  static constexpr int STAGE_BOXES = kTwoBoxes ? 2 : Cfg<MODE>::STAGE_BOXES;
};

using namespace tcp;

// two floats -> two e4m3 codes (round to nearest even, saturating at +-448); `lo` goes to bits [0,8)
__device__ __forceinline__ uint32_t cvt_e4m3x2(float lo, float hi) {
  uint16_t d;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(d) : "f"(hi), "f"(lo));
  return (uint32_t)d;
}
__device__ __forceinline__ uint32_t pack_e4m3x4(float a, float b, float c, float d) {
  return cvt_e4m3x2(a, b) | (cvt_e4m3x2(c, d) << 16);
}
// the float value of the e4m3 rounding of t (exact: e4m3 is a subset of fp16)
__device__ __forceinline__ float e4m3_value(float t) {
  const uint16_t c = (uint16_t)cvt_e4m3x2(t, 0.0f);
  uint32_t h2;
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"(c));
  return __half2float(__ushort_as_half((unsigned short)(h2 & 0xffffu)));
}

// Eq. 4.33 with alpha_q = 127: clip(round(x / S), -127, 127), round half to even -- the oracle's arithmetic, in which the
// quotient is ONE rounded fp32 multiplication by the rounded reciprocal of the scale (reading Q21, revised in
// round 2).  Round 1's reading divided (x / S in fp32): reproducing IEEE division bit for bit needed a tie test per value and
// a division on the rare ambiguous ones, which made the INT8 instantiation 12k instructions long (instruction-cache misses:
// stall_no_inst 39 % in the epilogue warps) and slower than the fp32-equivalent mode it approximates.
struct QScale { float S, r; };                  // scale and fl(1 / S)
template <int N>
__device__ __forceinline__ void quant_codes(const float (&x)[N], float (&q)[N], QScale s) {
#pragma unroll
  for (int i = 0; i < N; ++i) q[i] = fminf(fmaxf(rintf(__fmul_rn(x[i], s.r)), -127.0f), 127.0f);
}
__device__ __forceinline__ uint32_t pack_codes(float a, float b, float c, float d) {
  return ((uint32_t)(int)a & 0xffu) | (((uint32_t)(int)b & 0xffu) << 8) | (((uint32_t)(int)c & 0xffu) << 16) | (((uint32_t)(int)d & 0xffu) << 24);
}
__device__ __forceinline__ float quant_f(float x, QScale s) {
  float xi[1] = {x}, q[1];
  quant_codes<1>(xi, q, s);
  return q[0];
}
// y = float(sum) * (S_a S_w) + b, each step one rounded fp32 operation
__device__ __forceinline__ float dequant(uint32_t acc_bits, float sc, float b) {
  return __fadd_rn(__fmul_rn(__int2float_rn((int)acc_bits), sc), b);
}

// D[tmem] (+)= A * B^T with B in shared memory; A in shared memory (SS) or tensor memory (TS)
template <int MODE>
__device__ __forceinline__ void mma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t accumulate) {
  if constexpr (MODE == ETX_PREC_TF32X3)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(Cfg<MODE>::IDESC), "r"(accumulate) : "memory");
  else if constexpr (MODE == ETX_PREC_INT8)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(Cfg<MODE>::IDESC), "r"(accumulate) : "memory");
  else if constexpr (MODE == ETX_PREC_FP8)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(Cfg<MODE>::IDESC), "r"(accumulate) : "memory");
  else
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(Cfg<MODE>::IDESC), "r"(accumulate) : "memory");
}
template <int MODE>
__device__ __forceinline__ void mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t accumulate) {
  if constexpr (MODE == ETX_PREC_TF32X3)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(Cfg<MODE>::IDESC), "r"(accumulate) : "memory");
  else if constexpr (MODE == ETX_PREC_INT8)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(Cfg<MODE>::IDESC), "r"(accumulate) : "memory");
  else if constexpr (MODE == ETX_PREC_FP8)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(Cfg<MODE>::IDESC), "r"(accumulate) : "memory");
  else
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(Cfg<MODE>::IDESC), "r"(accumulate) : "memory");
}

constexpr int kTcLayers = 4;                    // layers whose biases fit in shared memory beside the rings and the output staging

struct Unit {                                   // one gather unit: KA columns of one source (16 bytes)
  const char* base;                             // source base + column offset (bytes)
  uint32_t ldb;                                 // row stride in bytes
  int32_t sel;                                  // row index: 0 / 1 = first / second index array, -1 = the tile row itself
};
constexpr int kMaxUnits = 24;

struct Bars {                                   // mbarriers (8 bytes each) + TMEM base + gather unit table
  uint64_t w_full[8], w_empty[8], a_full[8], a_empty[8], acc_full[3], acc_free[3], hid_ready[12];
  uint32_t tmem_base;
  // Progress counters for the two MMA issuer warps (see there): weight stages the loader has started to fill, operand
  // entries the commit warp has published.  An mbarrier parity wait is only meaningful for the barrier's CURRENT phase;
  // an issuer that reaches a stage / entry one ring revolution ahead of its sibling would read the other parity as
  // "complete".  It first waits for the counter to pass its index, which implies the previous phase has completed.
  uint32_t w_issued, a_produced;
  Unit utab[kMaxUnits];
};

// tcgen05.cp: 128 lanes x 256 bits (8 fp32 columns) from a K-major SWIZZLE_128B shared-memory tile into
// tensor memory.  Reads exactly the slab a kind::tf32 MMA k-step reads as its A operand (measured:
// [tmem + 8 ks] <- desc + 2 ks gives lane r, column c = tile element (r, c)); ordered with the
// tcgen05.mma issued after it by the same thread, tracked by tcgen05.commit.
__device__ __forceinline__ void tmem_cp_128x256b(uint32_t taddr, uint64_t desc) {
  asm volatile("tcgen05.cp.cta_group::1.128x256b [%0], %1;" ::"r"(taddr), "l"(desc) : "memory");
}

// VAR: 0 regular, 1 wide (one layer, 256 outputs), 2 feat (first-layer operand computed from 3 raw features),
//      3 feat + narrow linear output layer of <= 8 units computed in the epilogue registers (embedding MLP)
template <int MODE, int VAR>
__global__ void __launch_bounds__(kThreads, 1) mlp_tc_kernel(const TcArgs a, const __grid_constant__ CUtensorMap tmap) {
  using C = Cfg<MODE>;
  constexpr int KA = C::KA, P = C::PIECES, NSW = C::NSTAGE_W, NSA = Split<MODE, VAR>::NSTAGE_A, HID_COLS = C::HID_COLS;
  constexpr uint32_t kStageBytes = P * kAtomBytes;
  static_assert(NSW <= 8 && NSA <= 8, "Bars holds 8 mbarriers per ring");
  constexpr uint32_t COL_ACC = 0;
  // Tiles in flight per CTA.  The bf16 modes keep TWO 128-row tiles in flight (slot s: accumulator s,
  // hidden operand region s): the MMA warp issues layer l of tile A, then of tile B, while the epilogue
  // warps turn A's accumulator into its next operand; both tiles use each weight stage before it is
  // released, so the weight ring moves half the bytes.  TF32X3 needs 256 columns per hidden operand
  // and keeps one tile in flight with ping-pong accumulators.
  // 8-bit operands (INT8 / FP8): a hidden operand is 32 columns, so THREE tiles would fit (3 x (128 + 32) = 480 columns);
  // the slot logic below is written for up to three and that was measured: FP8 edge network -2 %, edge encoder +13 %,
  // INT8 embedding +10 % -- a third tile in flight does not help, because the eight epilogue warps process the tiles'
  // jobs one after the other and are busy whatever the number of tiles waiting for them.  Two it stays.
  constexpr int NSLOT = (MODE == ETX_PREC_TF32X3) ? 1 : 2;
  constexpr uint32_t COL_HID = (NSLOT == 3) ? 384 : 256;   // hidden operand regions behind the accumulators
  // MMA issuer warps.  2 (one per tile in flight, each walking its own tile's chain of waits) is implemented and correct,
  // and measured SLOWER (edge network 23.5 -> 25.4 ms per step, classifier 1.9 -> 2.4): issued concurrently, the two tiles'
  // MMAs interleave in the tensor pipe and both tiles finish their layer late and together, which destroys the stagger
  // (layer l of tile A, then of tile B) that lets the epilogue warps work on one tile while the other one's MMAs run.
  constexpr int NMW = 1;
  constexpr uint32_t HIDW = P * HID_COLS;       // TMEM columns of one hidden operand region (256 / 128 / 64)
  constexpr int HCH = HW / KA;                  // K-chunks per hidden layer (4 / 2; 1 for 8-bit operands)
  constexpr int KG = C::KG;                     // columns of one gather unit
  constexpr int GCH = HW / KG;                  // gather units per 128 columns
  constexpr int UPE = KA / KG;                  // gather units per ring entry (2 for 8-bit operands, else 1)
  constexpr bool q8 = (MODE == ETX_PREC_INT8);
  constexpr bool f8 = (MODE == ETX_PREC_FP8);
  constexpr bool op8 = q8 || f8;                // 8-bit operands: one 128-code K-chunk per 128 inputs
  constexpr int LPR = KG * 4 / 16;              // gather lanes per row: 16-byte pieces of a unit row (8 / 16)
  constexpr int RPP = kGatherThreads / LPR;     // rows covered by one pass of the gather threads (32 / 16)
  constexpr int NPASS = TM / RPP;               // passes per chunk (4 / 8)
  constexpr int D = C::PREFETCH;                // nc1 is a multiple of D for every MLP this kernel serves

  // SWIZZLE_128B tiles need 1024-byte alignment: the dynamic window is declared with that alignment (checked below), so
  // no slack is reserved -- every byte of the 227 KB counts (rings 192 KB + output staging + biases + barriers)
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const uint32_t base = smem_u32(smem_raw);
  const uint32_t wring = base;
  const uint32_t aring = wring + NSW * kStageBytes;
  const uint32_t stage_out = aring + NSA * kStageBytes;                  // 32 KB: one swizzled 4 KB staging box per epilogue warp
  unsigned char* gen = smem_raw;
  float* wlast_s = reinterpret_cast<float*>(gen + (NSW + NSA) * kStageBytes);   // [128] / [128][8]: classifier and narrow-output launches stage no output, so this aliases the staging boxes
  constexpr int kStageOutBytes = Split<MODE, VAR>::STAGE_BOXES * kStageBoxBytes;
  float* bias_s = reinterpret_cast<float*>(gen + (NSW + NSA) * kStageBytes + kStageOutBytes);   // [kTcLayers][128]
  Bars* bars = reinterpret_cast<Bars*>(bias_s + kTcLayers * HW);
  if (base & 1023u) __trap();

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_tiles = (a.n_rows + TM - 1) / TM;
  const int n_gemm = (a.out_mode == 3 || VAR == 3) ? a.n_layers - 1 : a.n_layers;
  const int nc1 = a.K0 / KA;
  const int my_tiles = (n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;   // tiles blockIdx.x + i * gridDim.x
  // Wide mode (one layer, 256 outputs: the per-hit projections [A h | B h] of the factorised edge MLPs):
  // the two slots of a "pair" are the two 128-column output halves of ONE row tile -- the operand entries
  // are gathered once and serve both halves, each half has its own weight chunks and accumulator.
  constexpr bool wide = (VAR == 1);             // (compile-time switches: the regular kernels carry none of it)
  constexpr bool feat = (VAR == 2 || VAR == 3);
  constexpr bool narrow = (VAR == 3);
  static_assert(!wide || NSLOT >= 2, "wide mode needs two accumulator slots");
  const int n_pairs = wide ? my_tiles : (my_tiles + NSLOT - 1) / NSLOT;
  auto slots_of = [&](int pi) { return wide ? 2 : ((my_tiles - pi * NSLOT) < NSLOT ? (my_tiles - pi * NSLOT) : NSLOT); };
  auto tile_of = [&](int pi, int sl) { return (int)blockIdx.x + (wide ? pi : pi * NSLOT + sl) * (int)gridDim.x; };
  const bool share1 = !wide && nc1 <= NSW;      // first-layer weight stages shared by the tiles of a pair
  // Addend (first-layer factorisation): the accumulator of layer 1 starts from
  // add[0][idx0[row]] + add[1][idx1[row]] (128 fp32 columns) instead of zero.
  const int n_addu = a.n_add ? 2 * GCH : 0;     // addend gather units per tile (two sources x 128 / KG column chunks)
  const int n_addg = n_addu / D;                // = 2 groups of 64 columns
  const int n_units = n_addu + a.K0 / KG;
  Unit* utab = bars->utab;
  if ((int)threadIdx.x < n_units) {
    const int u = threadIdx.x;
    Unit un;
    if (u < n_addu) {
      const bool second = (u & 1) != 0;
      const float* b = second ? a.add[1].base : a.add[0].base;
      const int ld = second ? a.add[1].ld : a.add[0].ld;
      const bool has_idx = (second ? a.add[1].idx : a.add[0].idx) != nullptr;
      un.base = reinterpret_cast<const char*>(b + (u >> 1) * KG);
      un.ldb = (uint32_t)ld * 4u;
      un.sel = has_idx ? (u & 1) : -1;
    } else {
      int k = (u - n_addu) * KG, sg = 0;
      if (a.n_seg > 1 && k >= a.seg[0].width) { k -= a.seg[0].width; sg = 1; }
      if (sg == 1 && a.n_seg > 2 && k >= a.seg[1].width) { k -= a.seg[1].width; sg = 2; }
      const float* b = sg == 0 ? a.seg[0].base : (sg == 1 ? a.seg[1].base : a.seg[2].base);
      const int ld = sg == 0 ? a.seg[0].ld : (sg == 1 ? a.seg[1].ld : a.seg[2].ld);
      const bool has_idx = (sg == 0 ? a.seg[0].idx : (sg == 1 ? a.seg[1].idx : nullptr)) != nullptr;
      un.base = reinterpret_cast<const char*>(b + k);
      un.ldb = (uint32_t)ld * 4u;
      un.sel = (has_idx && !a.n_add) ? sg : -1;
    }
    utab[u] = un;
  }

  for (int i = threadIdx.x; i < n_gemm * HW; i += kThreads) bias_s[i] = __ldg(a.bias[i / HW] + i % HW);
  if constexpr (narrow) {                        // last layer's weights [k][n_out] (k-major) padded to 8 units per k
    for (int i = threadIdx.x; i < HW * 8; i += kThreads)
      wlast_s[i] = (i % 8) < a.n_out ? __ldg(a.w_last + (i / 8) * a.n_out + (i % 8)) : 0.f;
  } else if (a.out_mode == 3)
    for (int i = threadIdx.x; i < HW; i += kThreads) wlast_s[i] = __ldg(a.w_last + i);
  if (threadIdx.x == 0) {
    for (int i = 0; i < NSW; ++i) { mbar_init(smem_u32(&bars->w_full[i]), 1); mbar_init(smem_u32(&bars->w_empty[i]), NMW); }
    for (int i = 0; i < NSA; ++i) { mbar_init(smem_u32(&bars->a_full[i]), 1); mbar_init(smem_u32(&bars->a_empty[i]), wide ? 2 : 1); }
    for (int i = 0; i < 3; ++i) { mbar_init(smem_u32(&bars->acc_full[i]), 1); mbar_init(smem_u32(&bars->acc_free[i]), kEpiThreads / 32); }
    for (int i = 0; i < 12; ++i) mbar_init(smem_u32(&bars->hid_ready[i]), op8 ? 8 : 4);   // 8-bit: ONE chunk per layer, written by all 8 warps
    bars->w_issued = 0; bars->a_produced = 0;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == kWarpMma) {                        // TMEM: all 512 columns of this SM (1 CTA per SM)
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&bars->tmem_base)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;

  if (warp < kWarpEpi0) {
    // =========================== gather warps ===========================
    reg_dec<kRegGather>();
    const int t = threadIdx.x;                   // 0..511
    const int jl = t % LPR;                      // 16-byte piece of the chunk row this thread moves
    const int r0 = t / LPR;                      // first of its rows; then r0 + RPP, r0 + 2 RPP, ...
    float4 buf[D][NPASS];
    long long g_wait = 0, gp[4] = {0, 0, 0, 0}, tq = 0;
    const bool gdbg = ETX_DBG(a);
#define GP_T0() if (gdbg) tq = clock64()
#define GP_ACC(i) if (gdbg) { const long long tn = clock64(); gp[i] += tn - tq; tq = tn; }
    const long long g_start = gdbg ? clock64() : 0;

    // Producer cursor (tile, unit).  A unit is KA consecutive columns of one source for the 128 rows of a
    // tile; the per-unit source (base + column offset, row stride, which row-index array) sits in a
    // small shared-memory table built once per launch, so the per-unit path has no segment search, no
    // division and no dynamic indexing of kernel parameters (these warps have almost no ILP: every
    // scalar instruction costs its full latency).  Units of a tile: first the addend units (source 0 /
    // source 1 alternating, column chunk by column chunk), then the K-chunks of the MMA operand.
    const int32_t* sidx0 = a.n_add ? a.add[0].idx : (a.n_seg > 0 ? a.seg[0].idx : nullptr);
    const int32_t* sidx1 = a.n_add ? a.add[1].idx : (a.n_seg > 1 ? a.seg[1].idx : nullptr);
    const int total_groups = my_tiles * (n_units / D);
    int ptile = blockIdx.x, pu = 0;
    int ridx[2][NPASS], rown[NPASS];
    auto load_unit = [&](float4 (&dst)[NPASS]) {
      if constexpr (feat) {
        // Feature mode (node encoder): the operand of the first tensor-core layer is the output of the
        // MLP's own first layer, ReLU(W1 f + b1) with f = the 3 normalised features of the row -- 3 FMAs per
        // value, computed here instead of being loaded.  ridx[0..1] / rown hold the row's 3 features.
        // 8-bit (INT8 embedding): the features become INT8 codes (held as floats), w1 holds weight codes as floats, so
        // the 3-term sums below are exact integers; de-quantisation + bias + ReLU follow the oracle's single steps and
        // the store path re-quantises with the next layer's scale
        auto feat_val = [&](float f) { if constexpr (q8) return quant_f(f, QScale{a.q_sf, a.q_rsf}); else return f; };
        if (pu == 0) {
          // all feature loads first, then the normalisations: the IEEE division has a slow-path branch the loads are
          // not hoisted across, and a load -> divide -> load chain costs one DRAM latency per feature (12 per tile)
          // (measured: node encoder 0.80 -> 0.46 ms at C2; with 2 passes per thread, the 3xTF32 embedding, the
          // in-order form is 6 % faster, so it keeps it)
          float f0[NPASS], f1[NPASS], f2[NPASS];
#pragma unroll
          for (int p = 0; p < NPASS; ++p) {
            int row = ptile * TM + r0 + p * RPP;
            row = row < a.n_rows ? row : a.n_rows - 1;
            f0[p] = __ldg(a.feat[0] + row); f1[p] = __ldg(a.feat[1] + row); f2[p] = __ldg(a.feat[2] + row);
            if constexpr (NPASS <= 2) {
              ridx[0][p] = __float_as_int(feat_val(__fdiv_rn(__fsub_rn(f0[p], a.fc[0]), a.fs[0])));
              ridx[1][p] = __float_as_int(feat_val(__fdiv_rn(__fsub_rn(f1[p], a.fc[1]), a.fs[1])));
              rown[p] = __float_as_int(feat_val(__fdiv_rn(__fsub_rn(f2[p], a.fc[2]), a.fs[2])));
            }
          }
          if constexpr (NPASS > 2) {
#pragma unroll
            for (int p = 0; p < NPASS; ++p) {
              ridx[0][p] = __float_as_int(feat_val(__fdiv_rn(__fsub_rn(f0[p], a.fc[0]), a.fs[0])));
              ridx[1][p] = __float_as_int(feat_val(__fdiv_rn(__fsub_rn(f1[p], a.fc[1]), a.fs[1])));
              rown[p] = __float_as_int(feat_val(__fdiv_rn(__fsub_rn(f2[p], a.fc[2]), a.fs[2])));
            }
          }
        }
        const int c0 = pu * KG + jl * 4;             // this thread's 4 columns of the layer-1 output
        const float4 w0 = __ldg(reinterpret_cast<const float4*>(a.w1 + c0));
        const float4 w1 = __ldg(reinterpret_cast<const float4*>(a.w1 + HW + c0));
        const float4 w2 = __ldg(reinterpret_cast<const float4*>(a.w1 + 2 * HW + c0));
        const float4 bb = __ldg(reinterpret_cast<const float4*>(a.b1 + c0));
#pragma unroll
        for (int p = 0; p < NPASS; ++p) {
          const float fx = __int_as_float(ridx[0][p]), fy = __int_as_float(ridx[1][p]), fz = __int_as_float(rown[p]);
          if constexpr (q8) {
            dst[p].x = fmaxf(__fadd_rn(__fmul_rn(fmaf(w2.x, fz, fmaf(w1.x, fy, w0.x * fx)), a.q_sc0), bb.x), 0.f);
            dst[p].y = fmaxf(__fadd_rn(__fmul_rn(fmaf(w2.y, fz, fmaf(w1.y, fy, w0.y * fx)), a.q_sc0), bb.y), 0.f);
            dst[p].z = fmaxf(__fadd_rn(__fmul_rn(fmaf(w2.z, fz, fmaf(w1.z, fy, w0.z * fx)), a.q_sc0), bb.z), 0.f);
            dst[p].w = fmaxf(__fadd_rn(__fmul_rn(fmaf(w2.w, fz, fmaf(w1.w, fy, w0.w * fx)), a.q_sc0), bb.w), 0.f);
          } else {
          dst[p].x = fmaxf(fmaf(w2.x, fz, fmaf(w1.x, fy, fmaf(w0.x, fx, bb.x))), 0.f);
          dst[p].y = fmaxf(fmaf(w2.y, fz, fmaf(w1.y, fy, fmaf(w0.y, fx, bb.y))), 0.f);
          dst[p].z = fmaxf(fmaf(w2.z, fz, fmaf(w1.z, fy, fmaf(w0.z, fx, bb.z))), 0.f);
          dst[p].w = fmaxf(fmaf(w2.w, fz, fmaf(w1.w, fy, fmaf(w0.w, fx, bb.w))), 0.f);
          }
        }
        if (++pu == n_units) { pu = 0; ptile += gridDim.x; }
        return;
      }
      if (pu == 0) {
#pragma unroll
        for (int p = 0; p < NPASS; ++p) {
          const int row = ptile * TM + r0 + p * RPP;
          rown[p] = row < a.n_rows ? row : a.n_rows - 1;
          if (ETX_EXP(a, 4)) rown[p] = r0 + p * RPP;      // timing experiment: every tile reads the same rows
        }
        if (sidx0) {
#pragma unroll
          for (int p = 0; p < NPASS; ++p) ridx[0][p] = ETX_EXP(a, 4) ? rown[p] : __ldg(sidx0 + rown[p]);
        }
        if (sidx1) {
#pragma unroll
          for (int p = 0; p < NPASS; ++p) ridx[1][p] = ETX_EXP(a, 4) ? rown[p] : __ldg(sidx1 + rown[p]);
        }
      }
      const Unit un = utab[pu];
      const char* base = un.base + jl * 16;
      if (ETX_EXP(a, 32)) {                        // timing experiment (wrong results): no global loads in the gather warps
#pragma unroll
        for (int p = 0; p < NPASS; ++p) dst[p] = make_float4(1.f, 2.f, 3.f, 4.f);
        if (++pu == n_units) { pu = 0; ptile += gridDim.x; }
        return;
      }
#pragma unroll
      for (int p = 0; p < NPASS; ++p) {
        const uint32_t idx = (uint32_t)(un.sel == 0 ? ridx[0][p] : (un.sel == 1 ? ridx[1][p] : rown[p]));
        dst[p] = __ldg(reinterpret_cast<const float4*>(base + (size_t)idx * un.ldb));
      }
      if (++pu == n_units) { pu = 0; ptile += gridDim.x; }
    };
    // store one K-chunk of the MMA operand (converted / split) into ring entry `slot`
    auto store_operand = [&](const float4 (&src)[NPASS], uint32_t slot) {
      const uint32_t tile_hi = aring + slot * kStageBytes;
      if (ETX_EXP(a, 512)) return;                 // timing experiment (wrong results): the gather warps store nothing
#pragma unroll
      for (int p = 0; p < NPASS; ++p) {
        const int r = r0 + p * RPP;
        const float4 v = src[p];
        if constexpr (MODE == ETX_PREC_TF32X3) {
          const uint32_t off = r * 128 + ((jl ^ (r & 7)) << 4);
          const uint32_t hx = __float_as_uint(v.x) & 0xffffe000u, hy = __float_as_uint(v.y) & 0xffffe000u;
          const uint32_t hz = __float_as_uint(v.z) & 0xffffe000u, hw = __float_as_uint(v.w) & 0xffffe000u;
          st_shared_v4(tile_hi + off, hx, hy, hz, hw);
          st_shared_v4(tile_hi + kAtomBytes + off,
                       __float_as_uint(v.x - __uint_as_float(hx)), __float_as_uint(v.y - __uint_as_float(hy)),
                       __float_as_uint(v.z - __uint_as_float(hz)), __float_as_uint(v.w - __uint_as_float(hw)));
        } else {                             // 4 floats -> 4 bf16 = 8 bytes at k-byte offset 8*jl
          const uint32_t off = r * 128 + (((jl >> 1) ^ (r & 7)) << 4) + ((jl & 1) << 3);
          if constexpr (P == 2) {
            uint32_t h0, l0, h1, l1;
            split_bf16x2(v.x, v.y, h0, l0);
            split_bf16x2(v.z, v.w, h1, l1);
            st_shared_v2(tile_hi + off, h0, h1);
            st_shared_v2(tile_hi + kAtomBytes + off, l0, l1);
          } else {
            st_shared_v2(tile_hi + off, pack_bf16x2(v.x, v.y), pack_bf16x2(v.z, v.w));
          }
        }
      }
    };
    auto wait_entry = [&](uint32_t cnt) {
      const long long tg0 = gdbg ? clock64() : 0;
      mbar_wait_warp(smem_u32(&bars->a_empty[cnt % NSA]), ((cnt / NSA) & 1) ^ 1, lane);
      if (gdbg) g_wait += clock64() - tg0;
    };

    if (total_groups > 0) {
#pragma unroll
      for (int d = 0; d < D; ++d) load_unit(buf[d]);
    }
    uint32_t ecnt = 0;                         // ring entries produced so far (the MMA warp counts the same)
    int gi = 0;                                // group of D units inside the tile
    for (int g = 0; g < total_groups; ++g) {
      const bool more = g + 1 < total_groups;
      if (gi < n_addg) {
        // ---- addend group: 64 fp32 columns of add[0][idx0[row]] + add[1][idx1[row]] as two 16 KB tiles in
        // the operand layout (tcgen05.cp moves them into the accumulator, see the MMA warp).  P == 2:
        // both tiles in one ring entry; P == 1 (16 KB entries): two consecutive entries.
        constexpr int ENT = (P == 2) ? 1 : 2;
        wait_entry(ecnt);
        if constexpr (ENT == 2) wait_entry(ecnt + 1);
        GP_T0();
#pragma unroll
        for (int p = 0; p < (ETX_EXP(a, 512) ? 0 : NPASS); ++p) {
          const int r = r0 + p * RPP;
          if constexpr (LPR == 8) {            // unit = 32 columns: (buf0 + buf1) -> tile 0, (buf2 + buf3) -> tile 1
            const uint32_t dst0 = aring + (ecnt % NSA) * kStageBytes + r * 128 + ((jl ^ (r & 7)) << 4);
            const float4 x = buf[0][p], y = buf[1][p], z = buf[D - 2][p], w = buf[D - 1][p];
            st_shared_v4(dst0, __float_as_uint(x.x + y.x), __float_as_uint(x.y + y.y), __float_as_uint(x.z + y.z), __float_as_uint(x.w + y.w));
            st_shared_v4(dst0 + kAtomBytes, __float_as_uint(z.x + w.x), __float_as_uint(z.y + w.y), __float_as_uint(z.z + w.z), __float_as_uint(z.w + w.w));
          } else {                             // unit = 64 columns: lanes 0-7 of a row -> tile 0, lanes 8-15 -> tile 1
            const uint32_t tsel = jl >> 3;
            const uint32_t tbase = (P == 2) ? aring + (ecnt % NSA) * kStageBytes + tsel * kAtomBytes
                                            : aring + ((ecnt + tsel) % NSA) * kStageBytes;
            const float4 x = buf[0][p], y = buf[1][p];
            if constexpr (q8)                  // the projections are exact int32 sums: integer add of the bit patterns
              st_shared_v4(tbase + r * 128 + (((jl & 7) ^ (r & 7)) << 4),
                           (uint32_t)(__float_as_int(x.x) + __float_as_int(y.x)), (uint32_t)(__float_as_int(x.y) + __float_as_int(y.y)),
                           (uint32_t)(__float_as_int(x.z) + __float_as_int(y.z)), (uint32_t)(__float_as_int(x.w) + __float_as_int(y.w)));
            else
            st_shared_v4(tbase + r * 128 + (((jl & 7) ^ (r & 7)) << 4),
                         __float_as_uint(x.x + y.x), __float_as_uint(x.y + y.y), __float_as_uint(x.z + y.z), __float_as_uint(x.w + y.w));
          }
        }
        GP_ACC(1);
        // Hand-off without a release arrive or a proxy fence in THESE warps (either would wait for their
        // in-flight prefetch loads): bar.arrive on the entry's named barrier; the commit warp completes that
        // barrier, fences and arrives on a_full (see below).
        named_bar_arrive(kBarEntry0 + ecnt % NSA, kGatherThreads + 32);
        if constexpr (ENT == 2) named_bar_arrive(kBarEntry0 + (ecnt + 1) % NSA, kGatherThreads + 32);
        ecnt += ENT;
        GP_ACC(2);
        if (more) {
#pragma unroll
          for (int d = 0; d < D; ++d) load_unit(buf[d]);
        }
        GP_ACC(3);
      } else if constexpr (UPE == 2) {
        // 8-bit operands: the D = 2 units of a group are the two 64-column halves of ONE K-chunk (128 codes per row)
        static_assert(UPE == 1 || D == UPE, "a group of gather units fills exactly one ring entry");
        wait_entry(ecnt);
        GP_T0();
        const uint32_t tile_q = aring + (ecnt % NSA) * kStageBytes;
#pragma unroll
        for (int d = 0; d < D; ++d) {
#pragma unroll
          for (int p2 = 0; p2 < NPASS; p2 += 2) {           // 8 values per tie test (these warps have 64 registers)
            float xq[8] = {buf[d][p2].x, buf[d][p2].y, buf[d][p2].z, buf[d][p2].w,
                           buf[d][p2 + 1].x, buf[d][p2 + 1].y, buf[d][p2 + 1].z, buf[d][p2 + 1].w};
            float cq[8];
            if constexpr (f8) {                             // e4m3: scale by fl(1/S), the conversion rounds and saturates
#pragma unroll
              for (int i = 0; i < 8; ++i) cq[i] = __fmul_rn(xq[i], a.q_rsa0);
            } else {
              quant_codes<8>(xq, cq, QScale{a.q_sa0, a.q_rsa0});
            }
#pragma unroll
            for (int h2 = 0; h2 < 2; ++h2) {
              const int r = r0 + (p2 + h2) * RPP;
              const uint32_t byte = d * 64 + jl * 4;        // K position of this thread's 4 codes inside the 128-byte row
              const uint32_t word = f8 ? pack_e4m3x4(cq[4 * h2], cq[4 * h2 + 1], cq[4 * h2 + 2], cq[4 * h2 + 3])
                                       : pack_codes(cq[4 * h2], cq[4 * h2 + 1], cq[4 * h2 + 2], cq[4 * h2 + 3]);
              asm volatile("st.shared.b32 [%0], %1;" ::"r"(tile_q + r * 128 + (((byte >> 4) ^ (r & 7)) << 4) + (byte & 15)),
                           "r"(word) : "memory");
            }
          }
          if (more) load_unit(buf[d]);                       // this buffer's next loads fly while the other half is converted
        }
        GP_ACC(1);
        named_bar_arrive(kBarEntry0 + ecnt % NSA, kGatherThreads + 32);
        ++ecnt;
        GP_ACC(2);
      } else {
#pragma unroll
        for (int d = 0; d < D; ++d) {
          wait_entry(ecnt);
          GP_T0();
          store_operand(buf[d], ecnt % NSA);
          GP_ACC(1);
          named_bar_arrive(kBarEntry0 + ecnt % NSA, kGatherThreads + 32);
          ++ecnt;
          GP_ACC(2);
          if (more) load_unit(buf[d]);
          GP_ACC(3);
        }
      }
      if (++gi == n_units / D) gi = 0;
    }
    if (gdbg && t == 0) {
      a.dbg[(size_t)blockIdx.x * 32 + 8] = (unsigned long long)g_wait;
      a.dbg[(size_t)blockIdx.x * 32 + 9] = (unsigned long long)(clock64() - g_start);
      for (int i = 0; i < 4; ++i) a.dbg[(size_t)blockIdx.x * 32 + 16 + i] = (unsigned long long)gp[i];
    }
  } else if (warp < kWarpLoader) {
    // =========================== epilogue warps ===========================
    reg_inc<kRegEpi>();
    const int ew = warp - kWarpEpi0;             // 0..7
    const int q4 = ew & 3;                       // TMEM lane quarter this warp may access (= warp & 3)
    const int hh = ew >> 2;                      // column half this warp owns
    const int et = q4 * 32 + lane;               // tile row = TMEM lane
    const uint32_t lane_addr = tmem + ((uint32_t)(q4 * 32) << 16);
    uint32_t g = 0;
    long long e_wait = 0, ep[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}, tp = 0;
    const bool edbg = ETX_DBG(a);
#define EP_T0() if (edbg) tp = clock64()
#define EP_ACC(i) if (edbg) { const long long tn = clock64(); ep[i] += tn - tp; tp = tn; }
    const long long e_start = edbg ? clock64() : 0;
    uint32_t uacc[3] = {0, 0, 0};                // jobs seen per accumulator (mbarrier phase)
    for (int pi = 0; pi < n_pairs; ++pi) {
      const int ns = slots_of(pi);
      for (int l = 0; l < n_gemm; ++l)
      for (int sl = 0; sl < ns; ++sl, ++g) {
        const uint32_t b = (NSLOT >= 2) ? (uint32_t)sl : (g & 1);
        const int tile = tile_of(pi, sl);
        const uint32_t hid = lane_addr + COL_HID + (NSLOT >= 2 ? sl * HIDW : 0);
        uint64_t* hid_ready = bars->hid_ready + (NSLOT >= 2 ? sl * 4 : 0);
        long long te0 = edbg ? clock64() : 0;
        mbar_wait_warp(smem_u32(&bars->acc_full[b]), uacc[b] & 1, lane);
        ++uacc[b];
        if (edbg) e_wait += clock64() - te0;
        tc_fence_after();
        const uint32_t acc = lane_addr + COL_ACC + b * 128;
        {
        const int L = l, HH = hh;
        const float* bias = bias_s + L * HW;
        if (L < n_gemm - 1) {
          // ---- hidden layer: ReLU(x + b) -> next A operand in TMEM, released chunk by chunk.
          // This warp's column half holds K-chunks HH*HCH/2 .. of the next layer.
          if constexpr (op8) {
            // 8-bit: de-quantise the int32 (INT8) / fp32 (FP8) sums, bias, ReLU, re-quantise with the NEXT layer's input scale
            // (the Q -> node -> DQ chain of P:2725); this warp's 64 columns become 16 packed columns of the single K-chunk
            EP_T0();
            uint32_t va[32], vb[32], w[16];
            tmem_ld32(acc + HH * 64, va);
            tmem_ld32(acc + HH * 64 + 32, vb);
            tc_wait_ld();
            EP_ACC(0);
            const float sc = a.q_sc[L];
            const QScale sn{a.q_sn[L], a.q_rsn[L]};
            const float* bq = bias + HH * 64;
#pragma unroll
            for (int g4 = 0; g4 < 4; ++g4) {         // 16 values per tie test
              float xv[16], cv[16];
#pragma unroll
              for (int i = 0; i < 16; ++i) {
                const uint32_t acc_bits = g4 < 2 ? va[16 * g4 + i] : vb[16 * (g4 - 2) + i];
                if constexpr (f8) xv[i] = fmaxf(__fadd_rn(__fmul_rn(__uint_as_float(acc_bits), sc), bq[16 * g4 + i]), 0.f);
                else xv[i] = fmaxf(dequant(acc_bits, sc, bq[16 * g4 + i]), 0.f);
              }
              if constexpr (f8) {
#pragma unroll
                for (int i = 0; i < 16; ++i) cv[i] = __fmul_rn(xv[i], sn.r);
#pragma unroll
                for (int i = 0; i < 4; ++i) w[4 * g4 + i] = pack_e4m3x4(cv[4 * i], cv[4 * i + 1], cv[4 * i + 2], cv[4 * i + 3]);
              } else {
              quant_codes<16>(xv, cv, sn);
#pragma unroll
              for (int i = 0; i < 4; ++i) w[4 * g4 + i] = pack_codes(cv[4 * i], cv[4 * i + 1], cv[4 * i + 2], cv[4 * i + 3]);
              }
            }
            asm volatile(
                "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
                "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
                ::"r"(hid + HH * 16), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]),
                  "r"(w[8]), "r"(w[9]), "r"(w[10]), "r"(w[11]), "r"(w[12]), "r"(w[13]), "r"(w[14]), "r"(w[15]) : "memory");
            EP_ACC(1);
            tc_wait_st();
            tc_fence_before();
            mbar_arrive_relaxed_warp(smem_u32(&hid_ready[0]), lane);
            EP_ACC(2);
          }
#pragma unroll
          for (int c = HH * (HCH / 2); c < (HH + 1) * (HCH / 2); ++c) {
            EP_T0();
            if constexpr (MODE == ETX_PREC_TF32X3) {
              uint32_t v[32], w[32];
              tmem_ld32(acc + c * 32, v);
              tc_wait_ld();
              EP_ACC(0);
#pragma unroll
              for (int i = 0; i < 32; ++i) {
                const float x = fmaxf(__uint_as_float(v[i]) + bias[c * 32 + i], 0.f);
                w[i] = __float_as_uint(x) & 0xffffe000u;
                v[i] = __float_as_uint(x - __uint_as_float(w[i]));
              }
              tmem_st32(hid + c * 32, w);
              tmem_st32(hid + HID_COLS + c * 32, v);
            } else if constexpr (P == 2) {       // BF16X3: 64 accumulator columns -> 32 hi + 32 lo packed columns
              uint32_t va[32], vb[32], wh[32], wl[32];     // both loads in flight, one wait (va/vb die pair by pair as wh/wl are born)
              if (ETX_EXP(a, 256)) {               // timing experiment (wrong results): no tensor-memory traffic in the hidden epilogue
                tc_fence_before();
                mbar_arrive_relaxed_warp(smem_u32(&hid_ready[c]), lane);
                continue;
              }
              tmem_ld32(acc + c * 64, va);
              tmem_ld32(acc + c * 64 + 32, vb);
              // the first half's biases are fetched while the tensor-memory loads fly: tcgen05.wait::ld is an asm volatile
              // with a memory clobber, so a load written after it is issued after it (ncu: the short scoreboard of these
              // LDS was the epilogue warps' largest stall)
              float4 bp[8];
#pragma unroll
              for (int i = 0; i < 8; ++i) bp[i] = *reinterpret_cast<const float4*>(bias + c * 64 + 4 * i);
              tc_wait_ld();
              EP_ACC(0);
              if (ETX_EXP(a, 8)) {                 // timing experiment (wrong results): no bias / ReLU / split arithmetic
                tmem_st32(hid + c * 32, va);
                tmem_st32(hid + HID_COLS + c * 32, vb);
              } else {
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                split_bf16x2(fmaxf(__uint_as_float(va[4 * i]) + bp[i].x, 0.f), fmaxf(__uint_as_float(va[4 * i + 1]) + bp[i].y, 0.f), wh[2 * i], wl[2 * i]);
                split_bf16x2(fmaxf(__uint_as_float(va[4 * i + 2]) + bp[i].z, 0.f), fmaxf(__uint_as_float(va[4 * i + 3]) + bp[i].w, 0.f), wh[2 * i + 1], wl[2 * i + 1]);
              }
#pragma unroll
              for (int i = 0; i < 16; ++i)
                split_bf16x2(fmaxf(__uint_as_float(vb[2 * i]) + bias[c * 64 + 32 + 2 * i], 0.f),
                             fmaxf(__uint_as_float(vb[2 * i + 1]) + bias[c * 64 + 32 + 2 * i + 1], 0.f), wh[16 + i], wl[16 + i]);
              tmem_st32(hid + c * 32, wh);
              tmem_st32(hid + HID_COLS + c * 32, wl);
              }
            } else {
              uint32_t va[32], vb[32], w[32];
              tmem_ld32(acc + c * 64, va);
              tmem_ld32(acc + c * 64 + 32, vb);
              tc_wait_ld();
              EP_ACC(0);
#pragma unroll
              for (int i = 0; i < 16; ++i)
                w[i] = pack_bf16x2(fmaxf(__uint_as_float(va[2 * i]) + bias[c * 64 + 2 * i], 0.f),
                                   fmaxf(__uint_as_float(va[2 * i + 1]) + bias[c * 64 + 2 * i + 1], 0.f));
#pragma unroll
              for (int i = 0; i < 16; ++i)
                w[16 + i] = pack_bf16x2(fmaxf(__uint_as_float(vb[2 * i]) + bias[c * 64 + 32 + 2 * i], 0.f),
                                        fmaxf(__uint_as_float(vb[2 * i + 1]) + bias[c * 64 + 32 + 2 * i + 1], 0.f));
              tmem_st32(hid + c * 32, w);
            }
            EP_ACC(1);
            tc_wait_st();
            tc_fence_before();
            mbar_arrive_relaxed_warp(smem_u32(&hid_ready[c]), lane);
            EP_ACC(2);
          }
          tc_fence_before();
          mbar_arrive_relaxed_warp(smem_u32(&bars->acc_free[b]), lane);
        } else if (narrow) {
          // ---- narrow linear output (embedding, Eq. 4.27 with identity output): last hidden layer, then
          // n_out <= 8 units as fp32 FMA chains over the 128 hidden values of the row, in registers
          if (HH == 0) {
            float o8[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll 1
            for (int q = 0; q < HW / 32; ++q) {
              uint32_t v[32];
              tmem_ld32(acc + q * 32, v);
              tc_wait_ld();
#pragma unroll
              for (int i = 0; i < 32; ++i) {
                float hv;
                if constexpr (q8) hv = quant_f(fmaxf(dequant(v[i], a.q_sc[L], bias[q * 32 + i]), 0.f), QScale{a.q_sn[L], a.q_rsn[L]});   // code x weight codes: exact
                else hv = fmaxf(__uint_as_float(v[i]) + bias[q * 32 + i], 0.f);
                const float4 w0 = *reinterpret_cast<const float4*>(wlast_s + (q * 32 + i) * 8);
                const float4 w1 = *reinterpret_cast<const float4*>(wlast_s + (q * 32 + i) * 8 + 4);
                o8[0] = fmaf(hv, w0.x, o8[0]); o8[1] = fmaf(hv, w0.y, o8[1]); o8[2] = fmaf(hv, w0.z, o8[2]); o8[3] = fmaf(hv, w0.w, o8[3]);
                o8[4] = fmaf(hv, w1.x, o8[4]); o8[5] = fmaf(hv, w1.y, o8[5]); o8[6] = fmaf(hv, w1.z, o8[6]); o8[7] = fmaf(hv, w1.w, o8[7]);
              }
            }
            tc_fence_before();
            mbar_arrive_relaxed_warp(smem_u32(&bars->acc_free[b]), lane);
            const int row = tile * TM + et;
            if (row < a.n_rows) {
#pragma unroll
              for (int o = 0; o < 8; ++o)
                if (o < a.n_out) {
                  if constexpr (q8) a.out[(size_t)row * a.out_ld + o] = __fadd_rn(__fmul_rn(o8[o], a.q_sc[a.n_layers - 1]), __ldg(a.bias[a.n_layers - 1] + o));
                  else a.out[(size_t)row * a.out_ld + o] = o8[o] + __ldg(a.bias[a.n_layers - 1] + o);
                }
            }
          } else {
            mbar_arrive_relaxed_warp(smem_u32(&bars->acc_free[b]), lane);
          }
        } else if (a.out_mode == 3) {
          // ---- classifier: last hidden layer, then 1 unit + sigmoid; column half 0
          // warps do all 128 columns of their rows (a cross-warp sum is not worth it for 1 unit).
          if (HH == 0) {
            float logit = 0.f;
#pragma unroll 1
            for (int q = 0; q < HW / 32; ++q) {
              uint32_t v[32];
              tmem_ld32(acc + q * 32, v);
              tc_wait_ld();
              if constexpr (q8) {              // codes of the last hidden activation x integer weight codes (held as floats):
                float xv[32], cv[32];          // exact below 2^24
#pragma unroll
                for (int i = 0; i < 32; ++i) xv[i] = fmaxf(dequant(v[i], a.q_sc[L], bias[q * 32 + i]), 0.f);
                quant_codes<32>(xv, cv, QScale{a.q_sn[L], a.q_rsn[L]});
#pragma unroll
                for (int i = 0; i < 32; ++i) logit = fmaf(cv[i], wlast_s[q * 32 + i], logit);
              } else if constexpr (f8) {       // e4m3 values of the last hidden activation x e4m3 values of the weights, fp32 sum
#pragma unroll
                for (int i = 0; i < 32; ++i) {
                  const float x = fmaxf(__fadd_rn(__fmul_rn(__uint_as_float(v[i]), a.q_sc[L]), bias[q * 32 + i]), 0.f);
                  logit = fmaf(e4m3_value(__fmul_rn(x, a.q_rsn[L])), wlast_s[q * 32 + i], logit);
                }
              } else {
#pragma unroll
              for (int i = 0; i < 32; ++i)
                logit = fmaf(fmaxf(__uint_as_float(v[i]) + bias[q * 32 + i], 0.f), wlast_s[q * 32 + i], logit);
              }
            }
            tc_fence_before();
            mbar_arrive_relaxed_warp(smem_u32(&bars->acc_free[b]), lane);
            if constexpr (op8) logit = __fadd_rn(__fmul_rn(logit, a.q_sc[a.n_layers - 1]), __ldg(a.bias[a.n_layers - 1]));
            else
            logit += __ldg(a.bias[a.n_layers - 1]);
            const int row = tile * TM + et;
            if (row < a.n_rows) a.out[row] = 1.0f / (1.0f + expf(-logit));
          } else {
            mbar_arrive_relaxed_warp(smem_u32(&bars->acc_free[b]), lane);
          }
        } else {
          // ---- linear output (+ residual).  Each warp moves 32 columns of its own 32 rows at a time:
          // thread = row = TMEM lane writes its 128 bytes (+ bias) into the warp's private 4 KB staging box, laid out
          // as the SWIZZLE_128B tensor-map box [32 rows x 32 columns], and one lane hands the box to the TMA
          // unit -- a tensor store, or for the residual e += y a tensor REDUCE-ADD on the in-place
          // state: one IEEE fp32 add per element, performed at L2, no residual load, deterministic (each
          // element is touched exactly once).  No SIMT global traffic, no read-back of the staging tile,
          // rows past n_rows are clipped by the tensor map.
          // The warp's 64 accumulator columns go to registers first and the accumulator is released at once (the MMA
          // warp starts the next tile's first layer while the boxes drain).  Two TMA operations per warp and tile:
          // in-kernel counters put the issue of one operation at ~420 cycles of the issuing warp with all eight
          // epilogue warps at it (16 boxes of 4 KB per tile instead of round 1's 32 of 2 KB).
          constexpr int SB = Split<MODE, VAR>::STAGE_BOXES;
          const uint32_t stg0 = stage_out + ew * (SB * 4096);
          const bool in_place_add = (a.out_mode == 1);
          const int row0 = tile * TM + q4 * 32;
          EP_T0();
          uint32_t va[32], vb[32];
          if (!ETX_EXP(a, 256)) {
          tmem_ld32(acc + HH * 64, va);
          tmem_ld32(acc + HH * 64 + 32, vb);
          }
          tc_wait_ld();
          tc_fence_before();
          mbar_arrive_relaxed_warp(smem_u32(&bars->acc_free[b]), lane);
          EP_ACC(3);
#pragma unroll
          for (int q = 0; q < (ETX_EXP(a, 16) ? 0 : 2); ++q) {       // (timing experiment 16, wrong results: no output at all)
            const int col0 = HH * 64 + q * 32;
            EP_T0();
            const uint32_t stg = stg0 + (SB == 2 ? q * 4096 : 0);
            if (lane == 0) {                       // the TMA unit has read the slice's previous box (with a slice per box that
              if constexpr (SB == 2) bulk_wait_read1(); else bulk_wait_read0();   // is the LAST tile's: one newer group may be pending)
            }
            __syncwarp();
            EP_ACC(6);
            // The box's 32 biases first, all eight 128-bit loads in flight together: st_shared_v4 is an asm volatile
            // with a memory clobber, so a bias load written between two stores is issued only after the store before it
            // and the loop pays one shared-memory latency per store (in-kernel counters: 2.2k cycles per tile for these
            // 16 stores in the edge network, 3.7k for the 32 of the projection launches).
            float4 bq[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) bq[j] = *reinterpret_cast<const float4*>(bias + col0 + 4 * j);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const uint32_t v0 = q == 0 ? va[4 * j] : vb[4 * j], v1 = q == 0 ? va[4 * j + 1] : vb[4 * j + 1];
              const uint32_t v2 = q == 0 ? va[4 * j + 2] : vb[4 * j + 2], v3 = q == 0 ? va[4 * j + 3] : vb[4 * j + 3];
              const uint32_t dst = stg + lane * 128 + ((j ^ (lane & 7)) << 4);
              if constexpr (q8 && wide)        // 8-bit per-hit projections: the raw int32 sums (they are added as integers)
                st_shared_v4(dst, v0, v1, v2, v3);
              else if constexpr (q8) {
                const float sc = a.q_sc[L];
                st_shared_v4(dst, __float_as_uint(dequant(v0, sc, bq[j].x)), __float_as_uint(dequant(v1, sc, bq[j].y)),
                             __float_as_uint(dequant(v2, sc, bq[j].z)), __float_as_uint(dequant(v3, sc, bq[j].w)));
              } else if constexpr (f8 && !wide) {   // fp32 sums of e4m3 products: y = acc * (S_a S_w) + b (the projections stay raw sums)
                const float sc = a.q_sc[L];
                st_shared_v4(dst, __float_as_uint(__fadd_rn(__fmul_rn(__uint_as_float(v0), sc), bq[j].x)),
                             __float_as_uint(__fadd_rn(__fmul_rn(__uint_as_float(v1), sc), bq[j].y)),
                             __float_as_uint(__fadd_rn(__fmul_rn(__uint_as_float(v2), sc), bq[j].z)),
                             __float_as_uint(__fadd_rn(__fmul_rn(__uint_as_float(v3), sc), bq[j].w)));
              } else
              st_shared_v4(dst, __float_as_uint(__uint_as_float(v0) + bq[j].x), __float_as_uint(__uint_as_float(v1) + bq[j].y),
                           __float_as_uint(__uint_as_float(v2) + bq[j].z), __float_as_uint(__uint_as_float(v3) + bq[j].w));
            }
            EP_ACC(7);
            fence_async_smem();                    // generic-proxy writes -> async proxy (TMA)
            __syncwarp();
            EP_ACC(4);
            if (lane == 0) {
              const int cg = (wide ? sl * HW : 0) + col0;
              if (in_place_add) tma_reduce_add_2d(&tmap, stg, cg, row0);
              else tma_store_2d(&tmap, stg, cg, row0);
              bulk_commit();
            }
            EP_ACC(5);
          }
        }
        }
      }
    }
    if (lane == 0) bulk_wait_all();              // every output box has left the SM before the CTA retires
    __syncwarp();
    if (edbg && ew == 0 && lane == 0) {
      a.dbg[(size_t)blockIdx.x * 32 + 6] = (unsigned long long)e_wait;
      a.dbg[(size_t)blockIdx.x * 32 + 7] = (unsigned long long)(clock64() - e_start);
      for (int i = 0; i < 6; ++i) a.dbg[(size_t)blockIdx.x * 32 + 10 + i] = (unsigned long long)ep[i];
      for (int i = 6; i < 9; ++i) a.dbg[(size_t)blockIdx.x * 32 + 14 + i] = (unsigned long long)ep[i];
    }
  } else if (warp == kWarpLoader) {
    // =========================== weight loader ===========================
    reg_dec<kRegCtl>();
    if (lane == 0) {
      const int chunks_per_tile = nc1 + (n_gemm - 1) * HCH;
      uint32_t w_cnt = 0;
      for (int pi = 0; pi < n_pairs; ++pi) {        // per tile pair: a shared stage serves both tiles before its release
        const int ns = slots_of(pi);
        const int rep1 = share1 ? 1 : ns;           // an unshared first layer is streamed once per tile
        for (int qq = 0; qq < chunks_per_tile + (rep1 - 1) * nc1; ++qq, ++w_cnt) {
          const int q = wide ? qq : (qq < rep1 * nc1 ? qq % (nc1 > 0 ? nc1 : 1) : qq - (rep1 - 1) * nc1);
          const uint32_t ws = w_cnt % NSW, wn = w_cnt / NSW;
          mbar_wait(smem_u32(&bars->w_empty[ws]), (wn & 1) ^ 1);
          if (ETX_EXP(a, 2)) { mbar_arrive(smem_u32(&bars->w_full[ws])); if (NMW == 2) st_release_shared(smem_u32(&bars->w_issued), w_cnt + 1); continue; }
          mbar_expect_tx(smem_u32(&bars->w_full[ws]), kStageBytes);
          bulk_g2s(wring + ws * kStageBytes, a.wimg + (size_t)q * kStageBytes, kStageBytes, smem_u32(&bars->w_full[ws]));
          if (NMW == 2) st_release_shared(smem_u32(&bars->w_issued), w_cnt + 1);
        }
      }
    }
  } else if (warp == kWarpCommit) {
    // =========================== operand-ring commit warp ===========================
    // Completes, entry by entry, the named barrier the 16 gather warps bar.arrive on after their
    // st.shared, then makes those generic-proxy writes visible to the tensor core (fence.proxy.async)
    // and arrives on the entry's a_full mbarrier.  This warp has no memory traffic of its own, so the
    // release + fence cost nothing; in the gather warps they cost a global-load latency per entry.
    reg_dec<kRegCtl>();
    const int ent_per_tile = (a.n_add ? ((P == 2) ? 2 : 4) : 0) + nc1;
    const uint32_t total = (uint32_t)my_tiles * (uint32_t)ent_per_tile;
    for (uint32_t cnt = 0; cnt < total; ++cnt) {
      named_bar_sync(kBarEntry0 + cnt % NSA, kGatherThreads + 32);
      fence_async_smem();
      if (lane == 0) {
        mbar_arrive(smem_u32(&bars->a_full[cnt % NSA]));
        if (NMW == 2) st_release_shared(smem_u32(&bars->a_produced), cnt + 1);
      }
      __syncwarp();
    }
  } else if (warp > kWarpMma && NMW == 1) {
    reg_dec<kRegCtl>();                          // idle warp that completes the control warpgroup
  } else {
    // =========================== MMA issuers ===========================
    reg_dec<kRegCtl>();
    // Warp-uniform control flow: every lane waits on the barriers, one elected lane issues.  (Issuing
    // from a divergent `if (lane == 0)` region makes ptxas wrap every UTCHMMA in an election loop,
    // which left the tensor pipe idle half of the time.)
    // NMW == 2 (measured alternative, see NMW): the two tiles in flight have one issuer warp each (warp kWarpMma: slot 0,
    // the control warpgroup's fourth warp: slot 1).  What the tiles share is counted: a weight stage is released by two
    // arrivals (a stage only one tile uses is committed twice), the wide mode's operand entries likewise; the progress
    // counters in Bars keep an issuer from waiting on a parity one ring revolution ahead.  The motivation: with
    // everything else switched off (no MMAs, loads, stores or tensor-memory traffic: developer build, ETX_TC_EXP) the
    // hand-shakes alone cost 4.3k cycles per tile -- one warp walks both tiles' chains of ~17 mbarrier waits (>= 90
    // cycles each even when already complete), fences and commits.
    const int mw = (warp == kWarpMma) ? 0 : 1;
    const int ept = (a.n_add ? ((P == 2) ? 2 : 4) : 0) + nc1;      // operand-ring entries per tile
    uint32_t w_base = 0, a_base = 0, g = 0;
    long long dt[6] = {0, 0, 0, 0, 0, 0};
    const bool dbg = ETX_DBG(a) && mw == 0;
    long long t_start = dbg ? clock64() : 0, t0 = 0;
#define DBG_T0() if (dbg) t0 = clock64()
#define DBG_ACC(i) if (dbg) dt[i] += clock64() - t0
    uint32_t uacc[3] = {0, 0, 0}, uhid[3] = {0, 0, 0};  // jobs issued per accumulator / per hidden region (mbarrier phases)
    for (int pi = 0; pi < n_pairs; ++pi) {
      const int ns = slots_of(pi);
      for (int l = 0; l < n_gemm; ++l) {
       const int nch = (l == 0) ? nc1 : HCH;
       // The tiles of a pair share the weight stages of a layer when the whole layer fits in half the
       // ring (every hidden layer; a first layer of <= NSW/2 chunks); otherwise the loader streams the
       // layer once per tile.
       const bool shared_w = (l > 0) || share1;
       for (int sl = 0; sl < ns; ++sl, ++g) {
        if (NMW == 2 && sl != mw) continue;         // the other issuer's tile
        const uint32_t b = (NSLOT >= 2) ? (uint32_t)sl : (g & 1);
        const uint32_t hs = (NSLOT >= 2) ? (uint32_t)sl : 0u;
        uint32_t w_cnt = shared_w ? w_base : w_base + (uint32_t)(sl * nch);       // first weight stage this tile uses
        uint32_t a_cnt = a_base + (wide ? 0u : (uint32_t)(sl * ept));             // first operand entry of this tile
        // arrivals this issuer owes a weight stage: two complete it (one per issuer; both from the stage's only user)
        const int n_wc = (NMW == 2) ? ((!shared_w || ns == 1) ? 2 : 1) : 1;
        DBG_T0();
        if (uacc[b] >= 1) mbar_wait(smem_u32(&bars->acc_free[b]), (uacc[b] - 1) & 1);   // epilogue done with acc[b]
        DBG_ACC(0);
        const uint32_t d_tmem = tmem + COL_ACC + b * 128;
        if (l == 0 && a.n_add) {
          // addend tiles -> accumulator (tcgen05.cp, ordered before the MMAs issued below)
          constexpr int NENT = (P == 2) ? 2 : 4, TPE = (P == 2) ? 2 : 1;     // ring entries per tile, 16 KB tiles per entry
          for (int en = 0; en < NENT; ++en, ++a_cnt) {
            const uint32_t slot = a_cnt % NSA;
            DBG_T0();
            if (NMW == 2) spin_until_above(smem_u32(&bars->a_produced), a_cnt);
            mbar_wait(smem_u32(&bars->a_full[slot]), (a_cnt / NSA) & 1);
            DBG_ACC(1);
            fence_async_smem();                  // gather warps' st.shared (generic proxy) -> tcgen05.cp (async proxy)
            tc_fence_after();
            if (elect_one()) {
#pragma unroll
              for (int t = 0; t < TPE; ++t) {
                const uint64_t sd = smem_desc(aring + slot * kStageBytes + t * kAtomBytes);
                if (ETX_EXP(a, 128)) continue;     // timing experiment (wrong results): no tcgen05.cp of the addend
#pragma unroll
                for (int ks = 0; ks < 4; ++ks) tmem_cp_128x256b(d_tmem + (en * TPE + t) * 32 + ks * 8, sd + ks * 2);
              }
              tc_commit(smem_u32(&bars->a_empty[slot]));
              if (nch == 0 && en == NENT - 1) tc_commit(smem_u32(&bars->acc_full[b]));
            }
            __syncwarp();
          }
        }
        for (int c = 0; c < nch; ++c, ++w_cnt) {
          const uint32_t ws = w_cnt % NSW, wn = w_cnt / NSW;
          uint32_t slot = 0;
          DBG_T0();
          if (l == 0) {
            slot = a_cnt % NSA;
            if (NMW == 2) spin_until_above(smem_u32(&bars->a_produced), a_cnt);
            mbar_wait(smem_u32(&bars->a_full[slot]), (a_cnt / NSA) & 1);
            // The proxy fence that makes the gather warps' st.shared (generic proxy) visible to the
            // tensor core (async proxy) sits HERE, on the consumer side of the mbarrier: the writes are
            // ordered before it by the barrier's release/acquire, and it precedes the MMAs in program
            // order.  Executed by the writers it would also wait for their in-flight prefetch loads
            // (measured: ~1.2k cycles per K-chunk, the whole global-load latency, on every chunk).
            fence_async_smem();
            DBG_ACC(1);
          } else {
            mbar_wait(smem_u32(&bars->hid_ready[hs * 4 + c]), uhid[hs] & 1);
            DBG_ACC(2);
          }
          DBG_T0();
          if (NMW == 2) spin_until_above(smem_u32(&bars->w_issued), w_cnt);
          if (NMW == 2 || !shared_w || sl == 0) mbar_wait(smem_u32(&bars->w_full[ws]), wn & 1);   // one issuer: the pair's second tile finds a shared stage already there
          DBG_ACC(3);
          tc_fence_after();
          DBG_T0();
          if (elect_one()) {
            const uint64_t wd = smem_desc(wring + ws * kStageBytes);          // weight tile (hi piece)
            const uint32_t accum0 = (c > 0 || (l == 0 && a.n_add)) ? 1u : 0u;
            if (ETX_EXP(a, 64)) {                  // timing experiment (wrong results): no MMAs, only the commits
            } else if (l == 0) {
              const uint64_t ad = smem_desc(aring + slot * kStageBytes);      // gathered operand tile (hi piece)
#pragma unroll
              for (int ks = 0; ks < 4; ++ks) {     // 4 MMA k-steps of 32 bytes inside the 128-byte atom
                const uint32_t accum = ks > 0 ? 1u : accum0;
                if constexpr (P == 2) {
                  mma_ss<MODE>(d_tmem, ad + (kAtomBytes >> 4) + ks * 2, wd + ks * 2, accum);   // lo.hi  (small terms first)
                  mma_ss<MODE>(d_tmem, ad + ks * 2, wd + (kAtomBytes >> 4) + ks * 2, 1u);      // hi.lo
                  mma_ss<MODE>(d_tmem, ad + ks * 2, wd + ks * 2, 1u);                          // hi.hi
                } else {
                  mma_ss<MODE>(d_tmem, ad + ks * 2, wd + ks * 2, accum);
                }
              }
            } else {
              const uint32_t at = tmem + COL_HID + hs * HIDW + c * 32;
#pragma unroll
              for (int ks = 0; ks < 4; ++ks) {
                const uint32_t accum = ks > 0 ? 1u : accum0;
                if constexpr (P == 2) {
                  mma_ts<MODE>(d_tmem, at + HID_COLS + ks * 8, wd + ks * 2, accum);
                  mma_ts<MODE>(d_tmem, at + ks * 8, wd + (kAtomBytes >> 4) + ks * 2, 1u);
                  mma_ts<MODE>(d_tmem, at + ks * 8, wd + ks * 2, 1u);
                } else {
                  mma_ts<MODE>(d_tmem, at + ks * 8, wd + ks * 2, accum);
                }
              }
            }
            if (NMW == 2 || !shared_w || sl == ns - 1) tc_commit(smem_u32(&bars->w_empty[ws]));   // one issuer: a shared stage is released after the pair's last tile
            if (n_wc == 2) tc_commit(smem_u32(&bars->w_empty[ws]));
            if (l == 0) tc_commit(smem_u32(&bars->a_empty[slot]));       // wide: the entry is released by both halves' arrivals
            if (c == nch - 1) tc_commit(smem_u32(&bars->acc_full[b]));
          }
          __syncwarp();
          DBG_ACC(4);
          if (l == 0) ++a_cnt;
        }
        ++uacc[b];
        if (l > 0) ++uhid[hs];
       }
       w_base += shared_w ? (uint32_t)nch : (uint32_t)(ns * nch);
      }
      a_base += wide ? (uint32_t)ept : (uint32_t)(ns * ept);
    }
    if (dbg && lane == 0) {
      unsigned long long* o = a.dbg + (size_t)blockIdx.x * 32;
      for (int i = 0; i < 5; ++i) o[i] = (unsigned long long)dt[i];
      o[5] = (unsigned long long)(clock64() - t_start);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kWarpMma) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
  }
}

// Tensor map of the output [n_rows][n_cols] fp32 (row stride out_ld floats) with the epilogue's box: 32 columns
// (128 bytes, SWIZZLE_128B) x 32 rows.  cuTensorMapEncodeTiled is fetched through the runtime (no link-time
// dependency on libcuda: the library must still load on a machine without a driver).
bool encode_out_map(CUtensorMap* m, float* out, int n_rows, int n_cols, int out_ld) {
  using Fn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                          const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                          CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static Fn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return reinterpret_cast<Fn>(p);
  }();
  if (!fn || (reinterpret_cast<uintptr_t>(out) & 15) || (out_ld & 3)) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)n_cols, (cuuint64_t)n_rows};
  const cuuint64_t strides[1] = {(cuuint64_t)out_ld * sizeof(float)};
  const cuuint32_t box[2] = {32, 32}, estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, out, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int MODE, int VAR>
int launch_mode(const TcArgs& a, int sm_count, cudaStream_t s) {
  using C = Cfg<MODE>;
  static int configured[kMaxDevices] = {0};         // the shared-memory opt-in is a per-DEVICE attribute of the function
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return -1;
  // rings (192 KB) + output staging (32 KB; the classifier's / narrow output's last-layer weights alias it) + biases +
  // barriers: 226.8 of the 227 KB an SM offers
  const size_t smem = (size_t)(C::NSTAGE_W + Split<MODE, VAR>::NSTAGE_A) * C::PIECES * kAtomBytes + Split<MODE, VAR>::STAGE_BOXES * kStageBoxBytes +
                      kTcLayers * HW * sizeof(float) + sizeof(Bars) + 16;
  if (!configured[dev]) {
    if (cudaFuncSetAttribute(mlp_tc_kernel<MODE, VAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
    configured[dev] = 1;
  }
  const int n_gemm = (a.out_mode == 3 || VAR == 3) ? a.n_layers - 1 : a.n_layers;
  if (n_gemm > kTcLayers) return -1;                // the shared-memory bias table holds kTcLayers layers
  const int n_tiles = (a.n_rows + TM - 1) / TM;
  const int grid = n_tiles < sm_count ? n_tiles : sm_count;
  CUtensorMap tmap;
  std::memset(&tmap, 0, sizeof(tmap));
  if (a.out_mode != 3 && VAR != 3 && !encode_out_map(&tmap, a.out, a.n_rows, VAR == 1 ? 2 * HW : HW, a.out_ld)) return -1;
  mlp_tc_kernel<MODE, VAR><<<grid, kThreads, smem, s>>>(a, tmap);
  return 1;
}

}  // namespace

int tc_chunk_k(int mode) {
  return mode == ETX_PREC_TF32X3 ? Cfg<ETX_PREC_TF32X3>::KA
                                 : ((mode == ETX_PREC_INT8 || mode == ETX_PREC_FP8) ? Cfg<ETX_PREC_INT8>::KA : Cfg<ETX_PREC_BF16>::KA);
}

// Requirements (checked by the caller): hidden width 128; K0 a multiple of the chunk (32 / 64) and
// segment widths multiples of it; out_mode 0/1 needs dims[L] == 128; out_mode 3 needs dims[L] == 1.
int launch_mlp_tc(const TcArgs& a_in, int mode, int sm_count, cudaStream_t s) {
  if (a_in.n_rows <= 0) return 0;
  TcArgs a = a_in;
  if (mode == ETX_PREC_INT8 || mode == ETX_PREC_FP8) {
    a.q_rsa0 = 1.0f / a.q_sa0; a.q_rsf = 1.0f / a.q_sf;
    for (int l = 0; l < kMaxLayers; ++l) a.q_rsn[l] = a.q_sn[l] != 0.0f ? 1.0f / a.q_sn[l] : 0.0f;
  }
  if (a.wide) {                                  // one layer, no addend, two output halves; bf16 modes only
    if (a.n_layers != 1 || a.n_add != 0 || a.out_mode != 0) return -1;
    if (mode == ETX_PREC_BF16) return launch_mode<ETX_PREC_BF16, 1>(a, sm_count, s);
    if (mode == ETX_PREC_BF16X3) return launch_mode<ETX_PREC_BF16X3, 1>(a, sm_count, s);
    if (mode == ETX_PREC_INT8) return launch_mode<ETX_PREC_INT8, 1>(a, sm_count, s);
    if (mode == ETX_PREC_FP8) return launch_mode<ETX_PREC_FP8, 1>(a, sm_count, s);
    return -1;
  }
  if (a.w1) {                                    // first-layer operand computed from 3 features (node encoder, embedding)
    if (a.n_add != 0 || a.n_seg != 0 || a.K0 != HW || !a.b1 || !a.feat[0] || !a.feat[1] || !a.feat[2]) return -1;
    if (a.out_mode == 2) {                       // narrow linear output (embedding): 3xTF32, or the INT8 embedding
      if ((mode != ETX_PREC_TF32X3 && mode != ETX_PREC_INT8 && mode != ETX_PREC_BF16) || a.n_out < 1 || a.n_out > 8 || a.n_layers < 2) return -1;
      if (mode == ETX_PREC_INT8) return launch_mode<ETX_PREC_INT8, 3>(a, sm_count, s);
      if (mode == ETX_PREC_BF16) return launch_mode<ETX_PREC_BF16, 3>(a, sm_count, s);     // report-only (etx_embed_bf16)
      return launch_mode<ETX_PREC_TF32X3, 3>(a, sm_count, s);
    }
    if (mode == ETX_PREC_TF32X3) return launch_mode<ETX_PREC_TF32X3, 2>(a, sm_count, s);
    if (mode == ETX_PREC_BF16) return launch_mode<ETX_PREC_BF16, 2>(a, sm_count, s);
    if (mode == ETX_PREC_BF16X3) return launch_mode<ETX_PREC_BF16X3, 2>(a, sm_count, s);
    return -1;
  }
  if (mode == ETX_PREC_TF32X3) return launch_mode<ETX_PREC_TF32X3, 0>(a, sm_count, s);
  if (mode == ETX_PREC_BF16) return launch_mode<ETX_PREC_BF16, 0>(a, sm_count, s);
  if (mode == ETX_PREC_BF16X3) return launch_mode<ETX_PREC_BF16X3, 0>(a, sm_count, s);
  if (mode == ETX_PREC_INT8) return launch_mode<ETX_PREC_INT8, 0>(a, sm_count, s);
  if (mode == ETX_PREC_FP8) return launch_mode<ETX_PREC_FP8, 0>(a, sm_count, s);
  return -1;
}

}  // namespace etx
