// mq_gemm.cu -- the fused base + residual int4 GEMM (ZipperEngine; Eq.4).
//
// Orientation ("swap-AB"): the WEIGHT tile is the MMA's M operand (128 output channels),
// the TOKEN tile is the MMA's N operand (BT = 16..128 tokens), so the same kernel serves
// decode (M = 1..32 tokens) and prefill.  Accumulators live in TMEM as D[n, t]:
// lane = output channel, column = token; acc0 (base, scale s_w) and acc1 (residual, scale
// s_r) are separate column ranges because the scales differ (north_star (iii)).
//
// The weight operand never exists as int8 in shared memory: the unpack warps read the packed
// int4 tile (one thread per output channel), expand it in registers and write it straight
// into TENSOR MEMORY (tcgen05.st), from where tcgen05.mma reads it as its A operand.  Shared
// memory therefore carries 0.5 B (TMA write) + 0.5 B (read) per weight instead of 3 B.
//
// Granularity.  A K-STEP is 128 input channels (one 8 KB packed weight tile).  The single-thread
// roles pay a fixed instruction cost per hand-off, so hand-offs are coarser than a K-step:
//   P stage  = SK consecutive K-steps of one output tile: ONE 1-D bulk copy of SK*8 KB packed
//              weights (the device layout keeps a tile's K-steps contiguous) + SK 2-D tensor
//              copies of the packed token tile, [BT][64 B] per K-step;
//   U stage  = UK K-steps unpacked: 32*UK TMEM columns (weights, MMA A operand) + UK token
//              sub-tiles [BT][128 B] in the K-major SWIZZLE_128B layout (MMA B operand).
// Decode (BT <= 32): SK = UK = 4 (32 KB per hand-off), two unpack groups.  Prefill (BT = 128):
// SK = 2, UK = 1, four unpack groups; its 512 TMEM columns hold two 128-column accumulators (the
// base one single-buffered) and four operand stages of 32 weight + 32 residual-cell columns.
//
// Warp roles (6 + 4G warps, one persistent CTA per SM; G = 2 unpack groups, 4 for BT = 128), control
// flow warp-uniform, single instructions issued by an elected lane:
//   warp 0      producer : TMA.  Also fetches the residual metadata of its K-steps (32 K-steps per
//                          load, two batches ahead), writes the per-K-step metadata words and, for
//                          K-steps that own a residual cell, loads the cell's 2 KB quarters.
//   warps 6..   unpack groups of 4 warps, taking U stages in rotation: int4 -> int8 (value x16:
//                          nibble moved to the high half of a byte, two logic ops per 8
//                          elements; both operands use the same element order inside 32 bytes, so
//                          dot products are unchanged and accumulators are 256 x the true value).
//   warp 1      MMA      : tcgen05.mma kind::i8, A from TMEM: 4 per K-step for the base, 2 per
//                          present k-half of a residual cell re-using the SAME token tile.
//   warps 2-5   epilogue : tcgen05.ld both accumulators, y = s_a * (s_w*acc0 + s_r*acc1) in
//                          fp32, bf16/fp16 store.
//
// Work distribution ("stream-K"): the K-steps of all output tiles form one sequence that is
// cut into gridDim.x equal contiguous ranges, so every SM streams the same number of weight
// bytes whatever N is.  A tile whose K range is shared by S CTAs: each writes its int32 partial
// tile to a private workspace slot (plain coalesced stores, integer adds are exact so the result
// stays bit-identical), waits until all S partials are visible and finishes 1/S of the tile.  The
// wait needs the S contributors co-resident (grid <= SM count, one CTA per SM): an environment that
// exposes fewer SMs than cudaDevAttrMultiProcessorCount (MPS active-thread percentage, green contexts)
// must run this kernel with option split_k = 1 (whole tiles, nothing waits).  Decode shapes (M <= 32) and
// prefill shapes (M >= 64) do not come here by default: mq_decode.cu (row slabs: no CTA ever waits for another)
// and mq_prefill.cu (whole tiles; CTA pairs are co-scheduled by the hardware as clusters) serve them.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <mutex>
#include <cstring>

#include "mq_internal.h"
#include <type_traits>
#include "mq_ptx.cuh"

namespace {

using namespace mq;
using namespace mq::ptx;

constexpr int FIRST_EPI_WARP = 2;
constexpr int FIRST_UNPACK_WARP = 6;
constexpr int A_COLS = BK / 4;               // 32 TMEM columns hold 128 int8 per lane (one K-step)

// per-K-step metadata word handed from the producer to the unpack groups and the MMA warp
constexpr int META_VALID = (int)0x80000000;  // the K-step exists (a P stage may hold fewer than SK)
constexpr int META_FIRST = 1 << 30;          // first K-step of this CTA's segment of a tile
constexpr int META_LAST = 1 << 29;           // last K-step of the segment: accumulators complete
// bits 0-3: residual quarter mask; bits 4-11: sequence number of the residual cell among the cells
// of its unpack group in this CTA (mod 256); bits 12-27: sequence number of the cell's first
// stored quarter among the quarters of its unpack group (mod 65536)

// A8: W4A8 variant (the paper's other precision): per-token int8 activations, 1 byte per element in
// the token area; the unpack groups only re-order them (no expansion), accumulators are 16 x the true value.
#ifndef MQ_BT128_UK2
#define MQ_BT128_UK2 0
#endif
template <int BT, bool FUSED = false, bool A8 = false>
struct Cfg {
  // Unpack groups (4 warps each).  An item costs a group ~1000 cycles of mostly latency (loads,
  // TMEM/shared stores, proxy fences), so prefill runs four groups side by side.
  static constexpr int G = (BT == 128 && !MQ_BT128_UK2) ? 4 : 2;
  static constexpr int NUM_THREADS = 32 * (FIRST_UNPACK_WARP + 4 * G);
  static constexpr int SK = BT <= 32 ? 4 : 2;                    // K-steps per P stage
  static constexpr int UK = BT <= 32 ? 4 : (BT == 64 ? 2 : (MQ_BT128_UK2 ? 2 : 1));   // K-steps per U stage (item)
  static constexpr int IPS = SK / UK;                            // items per P stage
  // PAIR (prefill tile): the two U stages that hold the two K-steps of one P stage share ONE full / empty barrier pair,
  // and the MMA warp issues their 8 base MMAs (+ residual MMAs) as one elected block: the MMA queue is shallow, so every
  // instruction between two K-steps' MMAs is pipe idle time (profiles/r2_probe_int8.md)
  static constexpr bool PAIR = BT == 128 && UK == 1 && SK == 2;
  static constexpr int PSTAGES = A8 ? (BT == 16 ? 4 : (BT == 32 ? 3 : (BT == 64 ? 4 : 3)))
                                    : (BT <= 32 ? 4 : (BT == 64 ? 6 : 4));
  static constexpr int USTAGES = G;                                   // one per unpack group
  // Unpacked residual cells (TMEM): every unpack group owns a private ring of RG stages.  A ring
  // shared between the groups would be unsafe: mbarrier parity waits cannot tell "my turn" from
  // "two phases early", and cells fall on the groups irregularly.
  static constexpr int RG = BT <= 32 ? 2 : 1;
  static constexpr int RSTAGES = G * RG;
  static constexpr int QG = BT == 16 ? 8 : (BT == 128 ? 2 : 4);       // packed residual quarter slots (2 KB) per group,
  static constexpr int NQ = G * QG;                   // private for the same reason
  // BT = 128: two 128-column accumulators + four operand stages fill the 512 TMEM columns, so the
  // base accumulator is single-buffered there (the epilogue of a tile is not overlapped).
  static constexpr int ACC0_STAGES = BT == 128 ? 1 : 2;
  static constexpr int ACC1_STAGES = BT <= 64 ? 2 : 1;
  static constexpr int P_W = SK * TILE_BYTES;
  // token area of a P stage: packed int4 tokens [SK][BT][64 B], or (FUSED) raw 16-bit activations
  // [SK][8 rows][256 B] fetched by a tensor map over A itself
  static constexpr int TOK_KSTEP = FUSED ? 8 * BK * 2 : (A8 ? BT * BK : BT * (BK / 2));
  static constexpr float ACC_INV = A8 ? 0.0625f : 0.00390625f;   // accumulators are x16 (A8) or x256
  static constexpr int ACC_SHIFT = A8 ? 4 : 8;
  static_assert(!(FUSED && A8), "the fused quantizer is 4-bit only");
  static constexpr int P_TOK = SK * TOK_KSTEP;
  static constexpr int P_STAGE = P_W + P_TOK;
  static constexpr int U_SUB = BT * BK;                          // one int8 token sub-tile
  static constexpr int U_STAGE = UK * U_SUB;
  // tensor memory columns
  static constexpr int ACC1_COL0 = ACC0_STAGES * BT;
  static constexpr int A_COL0 = ACC1_COL0 + ACC1_STAGES * BT;
  static constexpr int R_COL0 = A_COL0 + USTAGES * UK * A_COLS;
  static constexpr int TMEM_NEED = R_COL0 + RSTAGES * A_COLS;
  static constexpr int TMEM_COLS = TMEM_NEED <= 32 ? 32 : (TMEM_NEED <= 64 ? 64 : (TMEM_NEED <= 128 ? 128 : (TMEM_NEED <= 256 ? 256 : 512)));
  static_assert(TMEM_NEED <= 512, "tensor memory budget");
  static_assert((G & (G - 1)) == 0 && USTAGES >= G, "ring safety: groups <= stages");
  // shared memory map (offsets from a 1024-aligned base)
  static constexpr int OFF_U = 0;
  static constexpr int OFF_P = OFF_U + USTAGES * U_STAGE;
  static constexpr int OFF_RP = OFF_P + PSTAGES * P_STAGE;
  static constexpr int OFF_BAR = OFF_RP + NQ * QUARTER_BYTES;
  static constexpr int NUM_BARS = 2 * PSTAGES + 2 * USTAGES + 2 * NQ + 2 * RSTAGES + 2 + ACC0_STAGES + ACC1_STAGES + 1;
  static constexpr int OFF_META = OFF_BAR + NUM_BARS * 8;
  static constexpr int SA_TILE = BT >= 64 ? 2 * BT + 4 : 0;   // token scales of the tile being drained (two tiles deep)
  static constexpr int META_WORDS = PSTAGES * SK + USTAGES * UK + 12 + 16 + SA_TILE;   // + token scales (FUSED)
  static constexpr int OFF_END = OFF_META + META_WORDS * 4;
  static constexpr int SMEM_BYTES = OFF_END + 1024;  // slack for the 1024-byte alignment
  static_assert(SMEM_BYTES <= 232448, "shared memory budget");
  static_assert(P_STAGE % 1024 == 0 && U_SUB % 1024 == 0, "swizzle atoms need 1024-byte alignment");
};

// Exact division of n < 2^31 by a run-time constant d: q = umulhi(n, mul) >> shr with
// l = ceil(log2 d), mul = floor(2^(31+l) / d) + 1, shr = l - 1 (d = 1: mul = 0 marks the identity).
// A hardware 32-bit division costs a single-warp role ~100 cycles, this costs ~10.
struct FastDiv {
  uint32_t mul, shr, d;
};
__device__ __forceinline__ uint32_t fdiv(uint32_t n, const FastDiv& f) {
  return f.mul ? (__umulhi(n, f.mul) >> f.shr) : n;
}

struct GemmParams {
  const uint8_t* base;
  const float* sw;
  const float* sr;
  const uint8_t* res;
  const int2* unit_meta;  // [NT*KS] {quarter mask, first quarter index}; mask 0 = no residual cell
  const float* sa;
  void* Y;
  int32_t* dbg0;
  int32_t* dbg1;
  int32_t* ws_cnt;    // [tiles] partials published (zero between calls)
  int32_t* ws_done;   // [tiles] contributors finished (zero between calls)
  int32_t* ws_flag;   // [grid][2] did this partial receive residual MMAs?
  int32_t* ws_part;   // [grid][2 slots][2 accs][BT][128] int32 partial tiles
  int64_t ldy;
  uint32_t units;     // NT*TT*KS (< 2^31, checked by the host)
  uint32_t gran;      // range boundaries are multiples of gran (1 = stream-K, KS = whole tiles)
  uint32_t upg_q, upg_r;  // (units / gran) = upg_q * gridDim.x + upg_r
  FastDiv dKS, dTT, dGrid;
  int M, N, KS, NT, TT;
  int y_bf16;
  // fused activation quantization (mq_linear, M <= 8; kernel template FUSED): the raw activations and a
  // zero-state control block {amax bits [16], arrived, finished}
  const uint16_t* A;
  int64_t lda;
  int a_bf16;
  uint32_t* fz_ctrl;
  FastDiv dRowChunks;   // K / 8: 16-byte chunks per activation row
#ifdef MQ_TRACE
  long long* trace;  // [grid][64] clock64 stamps (development builds only)
#endif
};

#ifdef MQ_TRACE
#define MQ_STAMP(slot) do { p.trace[(size_t)blockIdx.x * 128 + (slot)] = clock64(); } while (0)
#define MQ_ACC_DECL(v) long long v = 0
#define MQ_ACC_BEGIN(v) v -= clock64()
#define MQ_ACC_END(v) v += clock64()
#define MQ_ACC_OUT(cond, slot, v) do { if (cond) p.trace[(size_t)blockIdx.x * 128 + (slot)] = (v); } while (0)
#define MQ_STAMP_IF(cond, slot) do { if (cond) MQ_STAMP(slot); } while (0)
#else
#define MQ_STAMP(slot) do { } while (0)
#define MQ_ACC_DECL(v) do { } while (0)
#define MQ_ACC_BEGIN(v) do { } while (0)
#define MQ_ACC_END(v) do { } while (0)
#define MQ_ACC_OUT(cond, slot, v) do { } while (0)
#define MQ_STAMP_IF(cond, slot) do { } while (0)
#endif

// All index arithmetic is 32-bit unsigned: a 64-bit division costs a single-thread role ~400 cycles.
// first unit of CTA c's range: gran * floor((units / gran) * c / grid)
__device__ __forceinline__ uint32_t range_begin(const GemmParams& p, uint32_t c) {
  return p.gran * (p.upg_q * c + fdiv(p.upg_r * c, p.dGrid));
}
// the CTA whose range holds unit x
__device__ __forceinline__ int owner_of(const GemmParams& p, uint32_t x) {
  int c = (int)((float)(x / p.gran) * (float)gridDim.x / (float)(p.upg_q * gridDim.x + p.upg_r));
  c = max(0, min(c, (int)gridDim.x - 1));
  while (c + 1 < (int)gridDim.x && range_begin(p, (uint32_t)c + 1) <= x) ++c;
  while (c > 0 && range_begin(p, (uint32_t)c) > x) --c;
  return c;
}

// One P stage of a CTA's work: up to SK consecutive K-steps of one (n-tile, token-tile).
struct Stage {
  uint32_t u;         // index of the stage's first K-step in the CTA-independent unit sequence
  int nt, tt, ks, nks;
  bool first, last;   // first / last stage of this CTA's segment of the tile
};
// Walks a CTA's unit range [g, u_end) segment by segment (segment = this CTA's K-steps of one
// tile) and, inside a segment, in P stages of up to SK K-steps.
struct StageIter {
  uint32_t g, u_end;
  FastDiv dKS, dTT;
  int KS, TT, k1, ks, nt, tt;
  __device__ StageIter(uint32_t u_beg, uint32_t u_end_, const FastDiv& dKS_, const FastDiv& dTT_)
      : g(u_beg), u_end(u_end_), dKS(dKS_), dTT(dTT_), KS((int)dKS_.d), TT((int)dTT_.d), k1(0), ks(0), nt(0), tt(0) {}
  template <int SK>
  __device__ bool next(Stage& s) {
    s.first = false;
    if (ks >= k1) {
      if (g >= u_end) return false;
      const uint32_t tile = fdiv(g, dKS);
      ks = (int)(g - tile * (uint32_t)KS);
      k1 = (int)min((uint32_t)KS, (uint32_t)ks + (u_end - g));
      g += (uint32_t)(k1 - ks);
      nt = (int)fdiv(tile, dTT);
      tt = (int)(tile - (uint32_t)nt * (uint32_t)TT);
      s.first = true;
    }
    s.u = g - (uint32_t)(k1 - ks);
    s.nt = nt;
    s.tt = tt;
    s.ks = ks;
    s.nks = min(SK, k1 - ks);
    ks += s.nks;
    s.last = ks >= k1;
    return true;
  }
};

// number of P stages of the range [u_beg, u_end): closed form of StageIter
__device__ __forceinline__ int count_stages(uint32_t u_beg, uint32_t u_end, const FastDiv& dKS, uint32_t SK) {
  if (u_end <= u_beg) return 0;
  const uint32_t KS = dKS.d, n = u_end - u_beg;
  const uint32_t head = KS - (u_beg - fdiv(u_beg, dKS) * KS);
  if (n <= head) return (int)((n + SK - 1) / SK);
  const uint32_t rem = n - head, whole = fdiv(rem, dKS);
  return (int)((head + SK - 1) / SK + whole * ((KS + SK - 1) / SK) + (rem - whole * KS + SK - 1) / SK);
}

// 32 packed nibbles (16 B) -> 32 int8 = 16 x value.  Output element order inside the 32
// bytes: for each packed word, its even nibbles then its odd nibbles; identical for both
// MMA operands.
__device__ __forceinline__ void unpack16(const uint4& p, uint32_t* o) {
  const uint32_t HI = 0xF0F0F0F0u;
  o[0] = (p.x << 4) & HI;
  o[1] = p.x & HI;
  o[2] = (p.y << 4) & HI;
  o[3] = p.y & HI;
  o[4] = (p.z << 4) & HI;
  o[5] = p.z & HI;
  o[6] = (p.w << 4) & HI;
  o[7] = p.w & HI;
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, const uint32_t* v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory");
}
__device__ __forceinline__ int lds32(uint32_t addr) {
  int v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts32(uint32_t addr, int v) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// FUSED path: 8 consecutive fp16/bf16 activations (one 16-byte load) -> the two int8 words the unpack
// of their packed int4 form would give: evens [e0,e2,e4,e6] and odds [e1,e3,e5,e7], each byte = 16 x q.
// The arithmetic is mq_quantize_act's, operation for operation (Eq.1; A1-A3): exact conversion to
// fp32, quant1() = IEEE division by the token scale, round half to even, clamp to [-7, 7].
__device__ __forceinline__ void quant8_i8x16(const uint4& raw, float s, float inv_s, bool bf16, uint32_t& ev, uint32_t& od) {
  const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
  ev = 0;
  od = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    float f0, f1;
    if (bf16) {
      f0 = __uint_as_float(w[i] << 16);
      f1 = __uint_as_float(w[i] & 0xFFFF0000u);
    } else {
      const float2 t = __half22float2(*reinterpret_cast<const __half2*>(&w[i]));
      f0 = t.x;
      f1 = t.y;
    }
    const int q0 = quant1(f0, s, inv_s), q1 = quant1(f1, s, inv_s);
    ev |= ((uint32_t)(q0 & 0xF) << 4) << (8 * i);
    od |= ((uint32_t)(q1 & 0xF) << 4) << (8 * i);
  }
}

template <bool BF16>
__device__ __forceinline__ void store_y(void* Y, size_t o, float y) {
  if (BF16)
    reinterpret_cast<__nv_bfloat16*>(Y)[o] = __float2bfloat16_rn(y);
  else
    reinterpret_cast<__half*>(Y)[o] = __float2half_rn(y);
}

// FUSED (BT = 16 only): the activation quantizer runs inside this kernel (north_star (i)
// "optionally fused into the GEMM prologue"): the epilogue warps find the per-token absmax together with
// all other CTAs (atomic max + grid-wide arrival count, hidden behind the first weight stage's HBM
// latency), and the unpack groups quantize the fp16/bf16 tokens of their K-steps straight into the int8
// operand tile -- no packed activations, no second kernel.
template <int BT, bool FUSED, bool A8>
__global__ void __launch_bounds__(Cfg<BT, FUSED, A8>::NUM_THREADS, 1)
mq_gemm_kernel(const __grid_constant__ CUtensorMap tmap_a, const GemmParams p) {
  using C = Cfg<BT, FUSED, A8>;
  constexpr int SK = C::SK, UK = C::UK, IPS = C::IPS;
  extern __shared__ uint8_t smem_raw[];
  // Known addresses (KA): for the prefill tile the shared-memory window and the tensor-memory allocation are taken as
  // compile-time constants -- dynamic shared memory starts at 1024 (the first KB is the system's) and a 512-column
  // allocation can only start at column 0 -- so that every barrier address, descriptor and TMEM operand of the
  // MMA-issuing warp's loop is an immediate instead of 16 R2UR / UIADD3 per K-step (that warp's dependent
  // instruction chain paces prefill).  Both assumptions are checked at run time: a mismatch traps.
  constexpr bool KA = BT == 128 && C::TMEM_COLS == 512;
  const uint32_t smem_base_rt = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t smem_base = KA ? 1024u : smem_base_rt;
  if (KA && smem_base_rt != 1024u) __trap();

  const uint32_t sU = smem_base + C::OFF_U, sP = smem_base + C::OFF_P, sRP = smem_base + C::OFF_RP,
                 sBar = smem_base + C::OFF_BAR;
  auto bar = [&](int i) { return sBar + 8u * (uint32_t)i; };
  constexpr int B_FULL_P = 0, B_EMPTY_P = C::PSTAGES, B_FULL_U = 2 * C::PSTAGES, B_EMPTY_U = B_FULL_U + C::USTAGES,
                B_FULL_Q = B_EMPTY_U + C::USTAGES, B_EMPTY_Q = B_FULL_Q + C::NQ,
                B_FULL_RU = B_EMPTY_Q + C::NQ, B_EMPTY_RU = B_FULL_RU + C::RSTAGES,
                B_TFULL = B_EMPTY_RU + C::RSTAGES, B_A0E = B_TFULL + 2, B_A1E = B_A0E + C::ACC0_STAGES,
                B_SA = B_A1E + C::ACC1_STAGES;   // FUSED: token scales are in shared memory
  static_assert(B_SA + 1 == C::NUM_BARS, "barrier map");
  // small shared words: metadata rings, TMEM base, fix-up flags
  const uint32_t sMetaP = smem_base + C::OFF_META;              // [PSTAGES][SK]
  const uint32_t sMetaU = sMetaP + 4u * C::PSTAGES * SK;        // [USTAGES][UK]
  const uint32_t sMisc = sMetaU + 4u * C::USTAGES * UK;         // [0] tmem base, [1..5] fix-up, [6..7] acc_flag
  volatile int32_t* misc = reinterpret_cast<volatile int32_t*>(smem_raw + (sMisc - smem_u32(smem_raw)));
  volatile int32_t* pend = misc + 1;      // [2][4] partial tiles awaiting the fix-up: tile, c_lo, c_hi, lo_slot
  volatile int32_t* acc_flag = misc + 9;
  volatile float* sa_s = reinterpret_cast<volatile float*>(misc + 12);   // [16] FUSED: token scales
  float* sa_tile = reinterpret_cast<float*>((reinterpret_cast<uintptr_t>(const_cast<int32_t*>(misc) + 28) + 15) & ~(uintptr_t)15);   // [2][BT], BT >= 64, 16-byte aligned

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#ifdef MQ_TRACE
  if (threadIdx.x == 0) {
    unsigned long long gt;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
    p.trace[(size_t)blockIdx.x * 128 + 12] = (long long)gt;
    MQ_STAMP(0);
  }
#endif

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmap_a);
    for (int i = 0; i < C::PSTAGES; ++i) {
      mbar_init(bar(B_FULL_P + i), 2);          // TMA issue (expect_tx) + metadata published
      mbar_init(bar(B_EMPTY_P + i), 4 * IPS);   // one arrival per unpack warp per item
    }
    for (int i = 0; i < C::USTAGES; ++i) {
      mbar_init(bar(B_FULL_U + i), C::PAIR ? 8 : 4);   // PAIR: barriers 0, 1 serve stages {0, 1}, {2, 3}
      mbar_init(bar(B_EMPTY_U + i), 1);
    }
    for (int i = 0; i < C::NQ; ++i) {
      mbar_init(bar(B_FULL_Q + i), 1);
      mbar_init(bar(B_EMPTY_Q + i), 4);         // every warp of the owning unpack group
    }
    for (int i = 0; i < C::RSTAGES; ++i) {
      mbar_init(bar(B_FULL_RU + i), 4);
      mbar_init(bar(B_EMPTY_RU + i), 1);
    }
    for (int i = 0; i < 2; ++i) mbar_init(bar(B_TFULL + i), 2);
    for (int i = 0; i < C::ACC0_STAGES; ++i) mbar_init(bar(B_A0E + i), 4);
    for (int i = 0; i < C::ACC1_STAGES; ++i) mbar_init(bar(B_A1E + i), 4);
    mbar_init(bar(B_SA), 1);
    fence_mbar_init();
  }
  if (warp == 1) {
    tmem_alloc(sMisc, C::TMEM_COLS);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = KA ? 0u : (uint32_t)misc[0];
  if (KA && misc[0] != 0) __trap();
  MQ_STAMP_IF(threadIdx.x == 0, 1);
  // PDL: the next kernel in the stream may start its prologue as this grid's CTAs retire
  griddep_launch();

  const uint32_t u_beg = range_begin(p, blockIdx.x);
  const uint32_t u_end = blockIdx.x + 1 == gridDim.x ? p.units : range_begin(p, blockIdx.x + 1);
  const int n_stages = count_stages(u_beg, u_end, p.dKS, SK);
  const int n_items = n_stages * IPS;

  if (warp == 0) {
    // ===================== producer (TMA); all lanes run the loop, one elected lane issues =====================
    StageIter it(u_beg, u_end, p.dKS, p.dTT);
    Stage cur, nxt;
    // Residual metadata {quarter mask, first quarter} is fetched 32 K-steps at a time (lane L: unit
    // ub + L) and two batches ahead, so that the producer never waits on global memory per stage.
    auto load_batch = [&](uint32_t ub) {
      const uint32_t u = ub + (uint32_t)lane;
      int2 v = make_int2(0, 0);
      if (u < u_end && p.unit_meta) {   // unit_meta == NULL: dense-only launch (the naive pipeline's first kernel)
        const uint32_t tile = fdiv(u, p.dKS);
        v = __ldg(p.unit_meta + (size_t)fdiv(tile, p.dTT) * p.KS + (u - tile * (uint32_t)p.KS));
      }
      return v;
    };
    uint32_t ubA = u_beg;
    int2 umA = load_batch(ubA), umB = load_batch(ubA + 32);
    // PDL prologue: the packed weights are static, so the first ring-full of weight copies is issued
    // BEFORE waiting for the previous kernel (which produces the quantized activations).
    int pre = 0;
    {
      StageIter itp = it;
      Stage s;
      for (; pre < C::PSTAGES && itp.next<SK>(s); ++pre) {
        if (elect_one()) {
          MQ_STAMP_IF(pre == 0, 2);
          const uint32_t fb = bar(B_FULL_P + pre);
          mbar_arrive_expect_tx(fb, (uint32_t)s.nks * (TILE_BYTES + C::TOK_KSTEP));
          tma_load_1d(sP + pre * C::P_STAGE, p.base + ((size_t)s.nt * p.KS + s.ks) * TILE_BYTES,
                      (uint32_t)s.nks * TILE_BYTES, fb);
        }
        __syncwarp();
      }
    }
    griddep_wait();
    MQ_ACC_DECL(tp_e);
    bool have = it.next<SK>(cur);
    int ps = 0, si = 0;
    int qseq_g[C::G], rseq_g[C::G];   // residual quarters / cells handed to each unpack group so far
#pragma unroll
    for (int g2 = 0; g2 < C::G; ++g2) qseq_g[g2] = rseq_g[g2] = 0;
    auto pick = [&](const int* a, int g2) {   // a[g2] without dynamic register indexing
      int v = a[0];
#pragma unroll
      for (int i = 1; i < C::G; ++i) v = g2 == i ? a[i] : v;
      return v;
    };
    uint32_t pphase = 0;
    while (have) {
      const bool have_n = it.next<SK>(nxt);
      MQ_ACC_BEGIN(tp_e);
      mbar_wait(bar(B_EMPTY_P + ps), pphase ^ 1);
      MQ_ACC_END(tp_e);
      MQ_ACC_OUT(lane == 0, 72, tp_e);
      __syncwarp();
      const uint32_t dst = sP + ps * C::P_STAGE;
      if (elect_one()) {
        MQ_STAMP_IF(si < 16, 48 + si);
        MQ_STAMP_IF(si == n_stages - 1, 3);
        const uint32_t fb = bar(B_FULL_P + ps);
        if (si >= pre) {   // the prologue already issued the weights of the first `pre` stages
          mbar_arrive_expect_tx(fb, (uint32_t)cur.nks * (TILE_BYTES + C::TOK_KSTEP));
          tma_load_1d(dst, p.base + ((size_t)cur.nt * p.KS + cur.ks) * TILE_BYTES, (uint32_t)cur.nks * TILE_BYTES, fb);
        }
        for (int j = 0; j < cur.nks; ++j) {
          if constexpr (FUSED)   // raw activations: box {128 elements, 8 rows} of the 16-bit tensor map over A
            tma_load_2d(dst + C::P_W + j * C::TOK_KSTEP, &tmap_a, (cur.ks + j) * BK, 0, fb);
          else
            tma_load_2d(dst + C::P_W + j * C::TOK_KSTEP, &tmap_a, (cur.ks + j) * (A8 ? BK : BK / 2), cur.tt * BT, fb);
        }
      }
      // metadata words of the stage (lane j writes K-step j), then the second arrival publishes them.
      // The empty asm pins the first USE of the prefetched metadata behind the TMA issue above.
      asm volatile("" : "+r"(umA.x), "+r"(umA.y));
      if (cur.u - ubA >= 32) {          // rotate: batch B was requested >= 32 K-steps ago
        umA = umB;
        ubA += 32;
        umB = load_batch(ubA + 32);
      }
      int2 um;
      {
        const uint32_t rel = cur.u - ubA + (uint32_t)(lane < SK ? lane : 0);   // < 64
        um.x = __shfl_sync(0xffffffffu, umA.x, rel & 31);
        um.y = __shfl_sync(0xffffffffu, umA.y, rel & 31);
        if (cur.u - ubA + SK > 32) {     // warp-uniform: the stage straddles into batch B (loaded long ago)
          const int bx = __shfl_sync(0xffffffffu, umB.x, rel & 31), by = __shfl_sync(0xffffffffu, umB.y, rel & 31);
          if (rel >= 32) um = make_int2(bx, by);
        }
      }
      const int mask = lane < cur.nks ? (um.x & 0xF) : 0;
      const uint32_t nz = __ballot_sync(0xffffffffu, mask != 0);
      // the unpack group that will handle K-step `lane` of this stage: item index mod 2
      const int my_group = (si * IPS + (lane < SK ? lane : 0) / UK) & (C::G - 1);
      // quarters stored by the cells of the lower lanes of the same group (SK <= 4: plain loop)
      int qbefore = 0, cbefore = 0;   // ... and cells
#pragma unroll
      for (int j = 0; j < SK; ++j) {
        const int mj = __shfl_sync(0xffffffffu, mask, j);
        const int gj = __shfl_sync(0xffffffffu, my_group, j);
        if (j < lane && gj == my_group) {
          qbefore += __popc(mj);
          cbefore += mj != 0;
        }
      }
      if (lane < SK) {
        int word = 0;
        if (lane < cur.nks) {
          const int my_rseq = pick(rseq_g, my_group) + cbefore;
          word = META_VALID | mask | ((my_rseq & 0xFF) << 4) |
                 (((pick(qseq_g, my_group) + qbefore) & 0xFFFF) << 12);
          if (cur.first && lane == 0) word |= META_FIRST;
          if (cur.last && lane == cur.nks - 1) word |= META_LAST;
        }
        sts32(sMetaP + 4u * (uint32_t)(ps * SK + lane), word);
      }
      __syncwarp();
      if (elect_one()) mbar_arrive(bar(B_FULL_P + ps));
      // residual cells of the stage: each present quarter is one 2 KB bulk copy into the quarter ring
      uint32_t todo = nz;
      while (todo) {
        const int j = __ffs((int)todo) - 1;
        todo &= todo - 1;
        const int m = __shfl_sync(0xffffffffu, mask, j);
        const int gj = __shfl_sync(0xffffffffu, my_group, j);
        const uint8_t* rsrc = p.res + (size_t)__shfl_sync(0xffffffffu, um.y, j) * QUARTER_BYTES;
        const int q0 = pick(qseq_g, gj);
        for (int q = 0; q < __popc(m); ++q) {
          const int slot = gj * C::QG + (q0 + q) % C::QG;
          mbar_wait(bar(B_EMPTY_Q + slot), (((uint32_t)(q0 + q) / C::QG) & 1) ^ 1);
          __syncwarp();
          if (elect_one()) {
            const uint32_t rb = bar(B_FULL_Q + slot);
            mbar_arrive_expect_tx(rb, QUARTER_BYTES);
            tma_load_1d(sRP + slot * QUARTER_BYTES, rsrc + (size_t)q * QUARTER_BYTES, QUARTER_BYTES, rb);
          }
        }
#pragma unroll
        for (int g2 = 0; g2 < C::G; ++g2)
          if (gj == g2) {
            qseq_g[g2] += __popc(m);
            rseq_g[g2] += 1;
          }
      }
      if (++ps == C::PSTAGES) {
        ps = 0;
        pphase ^= 1;
      }
      ++si;
      cur = nxt;
      have = have_n;
    }
  } else if (warp == 1) {
    // ===================== MMA issuer: warp-uniform control, one elected lane issues =====================
    constexpr uint32_t IDESC = make_idesc_i8(BN, BT);
    int seg = 0;                 // index of the current segment (selects the accumulator stages)
    MQ_ACC_DECL(tw_u); MQ_ACC_DECL(tw_a0); MQ_ACC_DECL(tw_tot);
    MQ_ACC_BEGIN(tw_tot);
    uint32_t acc0_on = 0, acc1_on = 0;
    uint32_t d0 = 0, d1 = 0;
    int a0s = 0, a1s = 0;
    auto seg_first = [&]() {   // first K-step of a segment: claim the accumulator stages
      a0s = seg % C::ACC0_STAGES;
      a1s = seg % C::ACC1_STAGES;
      MQ_ACC_BEGIN(tw_a0);
      mbar_wait(bar(B_A0E + a0s), (((uint32_t)seg / C::ACC0_STAGES) & 1) ^ 1);
      MQ_ACC_END(tw_a0);
      tc_fence_after();
      d0 = tmem_base + (uint32_t)(a0s * BT);
      d1 = tmem_base + (uint32_t)(C::ACC1_COL0 + a1s * BT);
      acc0_on = 0;
      acc1_on = 0;
    };
    auto seg_last = [&]() {    // last K-step of a segment: hand the accumulators to the epilogue
      if (!acc1_on) {
        // keep the acc1 ring's phases in step: the epilogue releases it once per segment
        mbar_wait(bar(B_A1E + a1s), (((uint32_t)seg / C::ACC1_STAGES) & 1) ^ 1);
      }
      __syncwarp();
      if (elect_one()) {
        acc_flag[a0s] = (int32_t)acc1_on;
        mbar_arrive(bar(B_TFULL + a0s));   // release: publishes acc_flag to the epilogue warps
        tc_commit(bar(B_TFULL + a0s));     // completes the phase when the MMAs have finished
        MQ_STAMP(8);
      }
      ++seg;
    };
    auto mma_item = [&](const int us, const int item, const uint32_t uphase) {
      MQ_ACC_BEGIN(tw_u);
      mbar_wait(bar(B_FULL_U + us), uphase);
      MQ_ACC_END(tw_u);
      tc_fence_after();
      MQ_STAMP_IF(item == 0 && lane == 0, 7);
      MQ_STAMP_IF(item < 16 && lane == 0, 32 + item);
      if constexpr (UK > 1) {
        // Decode path: all base MMAs of the item (up to 4*UK) go out as ONE elected block, then the
        // item's residual cells follow (acc0 and acc1 are separate accumulators, so their MMAs may be
        // reordered; the token sub-tiles stay valid until EMPTY_U is committed).  A segment's FIRST
        // flag can only sit on an item's first K-step, LAST on its last valid one.  Issuing K-step by
        // K-step costs ~60 dependent instructions per K-step, which is the latency of a short
        // kernel's tail and, with residual cells in half of the items, of the steady state too.
        int mw[UK], nk = 0;
#pragma unroll
        for (int j = 0; j < UK; ++j) mw[j] = lds32(sMetaU + 4u * (uint32_t)(us * UK + j));
#pragma unroll
        for (int j = 0; j < UK; ++j)
          if (mw[j] & META_VALID) ++nk;
        if (nk > 0) {
          if (mw[0] & META_FIRST) seg_first();
          int last = 0;
#pragma unroll
          for (int j = 0; j < UK; ++j)
            if (j == nk - 1) last = mw[j] & META_LAST;
          const uint64_t dt0 = make_desc_sw128(sU + us * C::U_STAGE);
          __syncwarp();
          if (elect_one()) {
            const uint32_t at0 = tmem_base + (uint32_t)(C::A_COL0 + us * UK * A_COLS);
#pragma unroll
            for (int j = 0; j < UK; ++j)
              if (j < nk) {
#pragma unroll
                for (int k = 0; k < 4; ++k)
                  mma_i8_ts(d0, at0 + (uint32_t)(j * A_COLS + k * 8), dt0 + (uint64_t)(j * (C::U_SUB >> 4) + k * 2), IDESC,
                            (j == 0 && k == 0) ? acc0_on : 1u);
              }
          }
          acc0_on = 1;
#pragma unroll
          for (int j = 0; j < UK; ++j) {
            const int mask = j < nk ? (mw[j] & 0xF) : 0;
            if (mask) {
              if (!acc1_on) {
                // first residual MMA of the segment: the epilogue must have drained this acc1 stage
                mbar_wait(bar(B_A1E + a1s), (((uint32_t)seg / C::ACC1_STAGES) & 1) ^ 1);
                tc_fence_after();
              }
              const int rseq = (mw[j] >> 4) & 0xFF;
              const int rs = (item & (C::G - 1)) * C::RG + rseq % C::RG;
              mbar_wait(bar(B_FULL_RU + rs), ((uint32_t)rseq / C::RG) & 1);
              tc_fence_after();
              __syncwarp();
              if (elect_one()) {
                const uint32_t rt = tmem_base + (uint32_t)(C::R_COL0 + rs * A_COLS);
                const uint64_t dt = dt0 + (uint64_t)(j * (C::U_SUB >> 4));
                uint32_t on = acc1_on;
#pragma unroll
                for (int h = 0; h < 2; ++h)
                  if (mask & (3 << (2 * h))) {
#pragma unroll
                    for (int k = 2 * h; k < 2 * h + 2; ++k) {
                      mma_i8_ts(d1, rt + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), IDESC, on);
                      on = 1;
                    }
                  }
                tc_commit(bar(B_EMPTY_RU + rs));
              }
              acc1_on = 1;
            }
          }
          if (last) seg_last();
        }
        __syncwarp();
        if (elect_one()) tc_commit(bar(B_EMPTY_U + us));
        return;
      }
      if constexpr (UK == 1) {
        // Prefill: ONE elected block per K-step issues the base MMAs, the cell's MMAs and the commit that
        // hands the U stage back (this warp's dependent instructions per K-step pace the pipeline).
        const int m = lds32(sMetaU + 4u * (uint32_t)us);
        const int mask = (m & META_VALID) ? (m & 0xF) : 0;
        if ((m & META_VALID) && (m & META_FIRST)) seg_first();
        if (mask && !acc1_on) {
          // first residual MMA of the segment: the epilogue must have drained this acc1 stage
          mbar_wait(bar(B_A1E + a1s), (((uint32_t)seg / C::ACC1_STAGES) & 1) ^ 1);
          tc_fence_after();
        }
        const uint32_t at = tmem_base + (uint32_t)(C::A_COL0 + us * A_COLS);
        const uint32_t rt = tmem_base + (uint32_t)(C::R_COL0 + us * A_COLS);   // the cell rides in its U stage
        const uint64_t dt = make_desc_sw128(sU + us * C::U_STAGE);
        __syncwarp();
        if (elect_one()) {
          if (m & META_VALID) {
#pragma unroll
            for (int k = 0; k < 4; ++k) mma_i8_ts(d0, at + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), IDESC, k == 0 ? acc0_on : 1u);
            if (mask) {
              uint32_t on = acc1_on;
#pragma unroll
              for (int h = 0; h < 2; ++h)
                if (mask & (3 << (2 * h))) {
#pragma unroll
                  for (int k = 2 * h; k < 2 * h + 2; ++k) {
                    mma_i8_ts(d1, rt + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), IDESC, on);
                    on = 1;
                  }
                }
            }
          }
          tc_commit(bar(B_EMPTY_U + us));
        }
        if (m & META_VALID) {
          acc0_on = 1;
          if (mask) acc1_on = 1;
          if (m & META_LAST) seg_last();
        }
        return;
      }
    };
    if constexpr (C::PAIR) {
      // Prefill tile: one iteration = one P stage = the two K-steps in U stages {2 pr, 2 pr + 1}: one barrier wait,
      // one elected block with up to 8 base MMAs and the cells' MMAs, one commit.
      for (int item0 = 0; item0 < n_items; item0 += C::USTAGES) {
        const uint32_t uphase = ((uint32_t)item0 / C::USTAGES) & 1;
#pragma unroll
        for (int pr = 0; pr < 2; ++pr) {
          if (item0 + 2 * pr >= n_items) break;
          MQ_ACC_BEGIN(tw_u);
          mbar_wait(bar(B_FULL_U + pr), uphase);
          MQ_ACC_END(tw_u);
          tc_fence_after();
          const int m0 = lds32(sMetaU + 4u * (uint32_t)(2 * pr)), m1 = lds32(sMetaU + 4u * (uint32_t)(2 * pr + 1));
          const bool v1 = (m1 & META_VALID) != 0;            // (the first K-step of a P stage always exists)
          if (m0 & META_FIRST) seg_first();
          const int mask0 = m0 & 0xF, mask1 = v1 ? (m1 & 0xF) : 0;
          if ((mask0 | mask1) && !acc1_on) {
            // first residual MMA of the segment: the epilogue must have drained this acc1 stage
            mbar_wait(bar(B_A1E + a1s), (((uint32_t)seg / C::ACC1_STAGES) & 1) ^ 1);
            tc_fence_after();
          }
          __syncwarp();
          if (elect_one()) {
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              if (j == 1 && !v1) break;
              const int us = 2 * pr + j;
              const uint32_t at = tmem_base + (uint32_t)(C::A_COL0 + us * A_COLS);
              const uint64_t dt = make_desc_sw128(sU + us * C::U_STAGE);
#pragma unroll
              for (int k = 0; k < 4; ++k) mma_i8_ts(d0, at + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), IDESC, (j == 0 && k == 0) ? acc0_on : 1u);
            }
            uint32_t on = acc1_on;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              const int mask = j == 0 ? mask0 : mask1;
              if (!mask) continue;
              const int us = 2 * pr + j;
              const uint32_t rt = tmem_base + (uint32_t)(C::R_COL0 + us * A_COLS);   // the cell rides in its U stage
              const uint64_t dt = make_desc_sw128(sU + us * C::U_STAGE);
#pragma unroll
              for (int h = 0; h < 2; ++h)
                if (mask & (3 << (2 * h))) {
#pragma unroll
                  for (int k = 2 * h; k < 2 * h + 2; ++k) {
                    mma_i8_ts(d1, rt + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), IDESC, on);
                    on = 1;
                  }
                }
            }
            tc_commit(bar(B_EMPTY_U + pr));
          }
          acc0_on = 1;
          if (mask0 | mask1) acc1_on = 1;
          if ((v1 ? m1 : m0) & META_LAST) seg_last();
        }
      }
    } else if constexpr (UK == 1) {
      // Prefill: the U stages are visited in a fixed rotation and the loop is unrolled over them, so
      // that every barrier address, TMEM column and shared-memory descriptor of the hot path is a
      // constant offset (this warp's instruction count per K-step is what paces prefill).
      for (int item0 = 0; item0 < n_items; item0 += C::USTAGES) {
        const uint32_t uphase = ((uint32_t)item0 / C::USTAGES) & 1;
#pragma unroll
        for (int us = 0; us < C::USTAGES; ++us)
          if (item0 + us < n_items) mma_item(us, item0 + us, uphase);
      }
    } else {
      // Decode kernels are short: code size (cold instruction cache) matters more than the arithmetic.
      for (int item = 0; item < n_items; ++item)
        mma_item(item % C::USTAGES, item, ((uint32_t)item / C::USTAGES) & 1);
    }
    MQ_ACC_END(tw_tot);
    MQ_ACC_OUT(lane == 0, 64, tw_u); MQ_ACC_OUT(lane == 0, 65, tw_a0); MQ_ACC_OUT(lane == 0, 66, tw_tot);
  } else if (warp >= FIRST_UNPACK_WARP) {
    // ============ unpack groups: int4 -> int8 (x16); weights -> TMEM, tokens -> smem ============
    const int gi = (warp - FIRST_UNPACK_WARP) >> 2;               // group: takes items i = gi (mod 2)
    const int wq = warp & 3;                                      // TMEM lane quadrant of this warp
    const uint32_t row = (uint32_t)(wq * 32 + lane);              // output channel inside the tile
    const uint32_t gtid = (uint32_t)(((warp - FIRST_UNPACK_WARP) & 3) * 32 + lane);
    const uint32_t lane_addr = tmem_base + ((uint32_t)(wq * 32) << 16);
    const int rhalf = wq >> 1;                                    // row half of a residual cell
    bool sa_ready = false;                                        // FUSED: token scales observed
    MQ_ACC_DECL(tu_p); MQ_ACC_DECL(tu_eu); MQ_ACC_DECL(tu_tot); MQ_ACC_DECL(tu_work);
    MQ_ACC_BEGIN(tu_tot);
    for (int item = gi; item < n_items; item += C::G) {
      const int stage = item / IPS, sub = item - stage * IPS;
      const int ps = stage % C::PSTAGES, us = item % C::USTAGES;
      MQ_ACC_BEGIN(tu_p);
      mbar_wait(bar(B_FULL_P + ps), ((uint32_t)stage / C::PSTAGES) & 1);
      MQ_ACC_END(tu_p);
      MQ_STAMP_IF(item == 0 && gtid == 0, 4);
      int mw[UK];
#pragma unroll
      for (int j = 0; j < UK; ++j) mw[j] = lds32(sMetaP + 4u * (uint32_t)(ps * SK + sub * UK + j));
      const uint32_t pw = sP + ps * C::P_STAGE + sub * UK * TILE_BYTES;
      if constexpr (UK == 1) {
        // Prefill path: the packed operands are loaded into registers BEFORE waiting for the U stage,
        // so that the stage's turnaround (MMA done -> next item published) is the int4 -> int8
        // expansion (2 logic ops per 8 elements), the stores and the fences.  The cell's unpacked weights ride in the U stage's own residual columns
        // (R stage = U stage), so FULL_U / EMPTY_U cover them and no separate hand-off is needed.
        static_assert(UK != 1 || (BT * 4) % 128 == 0, "token chunks per thread");
        constexpr int TCH = BT * (A8 ? 8 : 4) / 128;   // 16-byte token chunks per thread and K-step
        const int m = mw[0];
        const bool valid = (m & META_VALID) != 0;
        const int mask = valid ? (m & 0xF) : 0;
        uint4 v4[4], t4[TCH];   // packed operands stay packed (32 registers) across the wait
        uint32_t landed = 0;
        if (valid) {
#pragma unroll
          for (int c = 0; c < 4; ++c) v4[c] = lds128(pw + c * (BN * 16) + row * 16);
          const uint32_t pt1 = sP + ps * C::P_STAGE + C::P_W + sub * C::TOK_KSTEP;
#pragma unroll
          for (int i = 0; i < TCH; ++i) t4[i] = lds128(pt1 + (gtid + 128u * i) * 16);
          // the loads must have landed before the P stage is handed back: the arrival depends on every loaded word
          landed = fold4(v4[0]) ^ fold4(v4[1]) ^ fold4(v4[2]) ^ fold4(v4[3]);
#pragma unroll
          for (int i = 0; i < TCH; ++i) landed ^= fold4(t4[i]);
          landed = zero_after(landed);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(B_EMPTY_P + ps) + landed);   // this warp's reads of the P stage are done
        MQ_ACC_BEGIN(tu_eu);
        mbar_wait(bar(B_EMPTY_U + (C::PAIR ? us >> 1 : us)), (((uint32_t)item / C::USTAGES) & 1) ^ 1);
        MQ_ACC_END(tu_eu);
        MQ_ACC_BEGIN(tu_work);
        tc_fence_after();
        if (valid) {
          {
            uint32_t o[32];
#pragma unroll
            for (int c = 0; c < 4; ++c) unpack16(v4[c], o + 8 * c);
            tmem_st32(lane_addr + (uint32_t)(C::A_COL0 + us * A_COLS), o);
          }
          if (mask) {
            // residual cell (about one item in five): expanded after the base columns are on their
            // way, so that its registers do not add to the hot path's pressure
            const int qseq0 = (m >> 12) & 0xFFFF;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              if (!(mask & (3 << (2 * h)))) continue;   // k-half without any block: never read by the MMA
              uint32_t ro[16];
#pragma unroll
              for (int z = 0; z < 16; ++z) ro[z] = 0;
              // EVERY warp of the group passes through every present quarter's barrier, in ring
              // order, whether or not the quarter holds its rows: a parity wait is only sound for a
              // waiter that has seen the slot's previous phase.
#pragma unroll
              for (int r = 0; r < 2; ++r) {
                const int q = 2 * h + r;
                if (!(mask & (1 << q))) continue;
                const int qs = (qseq0 + __popc(mask & ((1 << q) - 1))) & 0xFFFF;
                const int slot = gi * C::QG + qs % C::QG;
                mbar_wait(bar(B_FULL_Q + slot), ((uint32_t)qs / C::QG) & 1);
                uint32_t landed = 0;   // (the slot's hand-back depends on the loaded words: zero_after, mq_ptx.cuh)
                if (r == rhalf) {
                  const uint32_t rp = sRP + slot * QUARTER_BYTES;
                  const uint4 r0 = lds128(rp + (row & 63) * 16);
                  const uint4 r1 = lds128(rp + 1024 + (row & 63) * 16);
                  unpack16(r0, ro);
                  unpack16(r1, ro + 8);
                  landed = zero_after(fold4(r0) ^ fold4(r1));
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_EMPTY_Q + slot) + landed);
              }
              tmem_st16(lane_addr + (uint32_t)(C::R_COL0 + us * A_COLS + 16 * h), ro);
            }
          }
          const uint32_t ut1 = sU + us * C::U_STAGE;
#pragma unroll
          for (int i = 0; i < TCH; ++i) {
            if constexpr (A8) {
              // 16 int8 tokens elements: only the even / odd re-ordering the weights' expansion produces
              const uint32_t idx = gtid + 128u * i, t = idx >> 3, c = idx & 7;
              const uint32_t tw[4] = {__byte_perm(t4[i].x, t4[i].y, 0x6420), __byte_perm(t4[i].x, t4[i].y, 0x7531),
                                      __byte_perm(t4[i].z, t4[i].w, 0x6420), __byte_perm(t4[i].z, t4[i].w, 0x7531)};
              sts128(ut1 + t * 128 + ((c ^ (t & 7)) << 4), tw);
            } else {
              const uint32_t idx = gtid + 128u * i, t = idx >> 2, c = idx & 3;
              uint32_t tw[8];
              unpack16(t4[i], tw);
              sts128(ut1 + t * 128 + (((2 * c) ^ (t & 7)) << 4), tw);
              sts128(ut1 + t * 128 + (((2 * c + 1) ^ (t & 7)) << 4), tw + 4);
            }
          }
        }
        tmem_st_wait();
        tc_fence_before();
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
          MQ_STAMP_IF(item == 0 && gtid == 0, 5);
          MQ_STAMP_IF(gi == 0 && gtid == 0 && item < 32, 16 + item / 2);
          MQ_STAMP_IF(gi == 0 && gtid == 0, 6);
          if (wq == 0) sts32(sMetaU + 4u * (uint32_t)us, m);
          mbar_arrive(bar(B_FULL_U + (C::PAIR ? us >> 1 : us)));
        }
        MQ_ACC_END(tu_work);
        continue;
      }
      // the first K-step's packed weights are fetched before the U stage is known to be free
      uint4 v[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) v[c] = lds128(pw + c * (BN * 16) + row * 16);
      mbar_wait(bar(B_EMPTY_U + us), (((uint32_t)item / C::USTAGES) & 1) ^ 1);
      tc_fence_after();
      int nk = 0;
#pragma unroll
      for (int j = 0; j < UK; ++j) {
        if (mw[j] & META_VALID) {
          ++nk;
          uint32_t o[32];
#pragma unroll
          for (int c = 0; c < 4; ++c) unpack16(v[c], o + 8 * c);
          if (j + 1 < UK && (mw[j + 1] & META_VALID)) {
#pragma unroll
            for (int c = 0; c < 4; ++c) v[c] = lds128(pw + (j + 1) * TILE_BYTES + c * (BN * 16) + row * 16);
          }
          tmem_st32(lane_addr + (uint32_t)(C::A_COL0 + (us * UK + j) * A_COLS), o);
        }
      }
      // tokens: packed [UK][BT][64 B] -> UK sub-tiles [BT][128 B] K-major SWIZZLE_128B
      const uint32_t pt = sP + ps * C::P_STAGE + C::P_W + sub * UK * C::TOK_KSTEP, ut = sU + us * C::U_STAGE;
      if constexpr (FUSED) {
        // Units of 8 activations (one 16-byte piece of the stage's raw tile [UK][8 rows][256 B]) are
        // dealt round-robin to the group's 128 threads: M * 64 units per item.  A unit becomes the
        // two int8 words (even / odd elements) the packed form's expansion would give, i.e. 8 bytes
        // of a swizzled 16-byte chunk of the operand tile.
        static_assert(!FUSED || (BT == 16 && UK == 4), "fused activation quantization: BT = 16 only");
        if (!sa_ready) {
          mbar_wait(bar(B_SA), 0);
          sa_ready = true;
        }
        for (uint32_t u = gtid; u < (uint32_t)p.M * 64u; u += 128) {
          const uint32_t t = u >> 6, jj = (u >> 4) & 3, c8 = u & 15;
          if ((int)jj < nk) {
            const float s = sa_s[t], inv_s = quant_inv_scale(s);
            uint32_t ev, od;
            quant8_i8x16(lds128(pt + jj * C::TOK_KSTEP + t * (BK * 2) + c8 * 16), s, inv_s, p.a_bf16 != 0, ev, od);
            const uint32_t dst = ut + jj * C::U_SUB + t * 128 + ((((c8 >> 1)) ^ (t & 7)) << 4) + (c8 & 1) * 8;
            asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(dst), "r"(ev), "r"(od) : "memory");
          }
        }
      } else if constexpr (A8) {
#pragma unroll
        for (uint32_t idx = gtid; idx < (uint32_t)(UK * BT * 8); idx += 128) {
          const uint32_t jj = idx / (BT * 8), rem = idx % (BT * 8), t = rem >> 3, c = rem & 7;
          if ((int)jj < nk) {
            const uint4 tv = lds128(pt + idx * 16);
            const uint32_t tw[4] = {__byte_perm(tv.x, tv.y, 0x6420), __byte_perm(tv.x, tv.y, 0x7531),
                                    __byte_perm(tv.z, tv.w, 0x6420), __byte_perm(tv.z, tv.w, 0x7531)};
            sts128(ut + jj * C::U_SUB + t * 128 + ((c ^ (t & 7)) << 4), tw);
          }
        }
      } else {
#pragma unroll
        for (uint32_t idx = gtid; idx < (uint32_t)(UK * BT * 4); idx += 128) {
          const uint32_t jj = idx / (BT * 4), rem = idx % (BT * 4), t = rem >> 2, c = rem & 3;
          if ((int)jj < nk) {
            const uint4 tv = lds128(pt + idx * 16);
            uint32_t w8[8];
            unpack16(tv, w8);
            const uint32_t dst = ut + jj * C::U_SUB + t * 128;
            sts128(dst + (((2 * c) ^ (t & 7)) << 4), w8);
            sts128(dst + (((2 * c + 1) ^ (t & 7)) << 4), w8 + 4);
          }
        }
      }
      tmem_st_wait();
      tc_fence_before();
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) {
        MQ_STAMP_IF(item == 0 && gtid == 0, 5);
        MQ_STAMP_IF(gi == 0 && gtid == 0 && item < 32, 16 + item / 2);
        MQ_STAMP_IF(gi == 0 && gtid == 0, 6);
        if (wq == 0) {
#pragma unroll
          for (int j = 0; j < UK; ++j) sts32(sMetaU + 4u * (uint32_t)(us * UK + j), mw[j]);
        }
        mbar_arrive(bar(B_FULL_U + us));
        mbar_arrive(bar(B_EMPTY_P + ps));
      }
      // residual cells of this item's K-steps
#pragma unroll
      for (int j = 0; j < UK; ++j) {
        const int mask = (mw[j] & META_VALID) ? (mw[j] & 0xF) : 0;
        if (mask) {
          const int rseq = (mw[j] >> 4) & 0xFF, rs = gi * C::RG + rseq % C::RG;
          const int qseq0 = (mw[j] >> 12) & 0xFFFF;
          mbar_wait(bar(B_EMPTY_RU + rs), (((uint32_t)rseq / C::RG) & 1) ^ 1);
          tc_fence_after();
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            if (!(mask & (3 << (2 * h)))) continue;   // k-half without any block: never read by the MMA
            uint32_t ro[16];
#pragma unroll
            for (int z = 0; z < 16; ++z) ro[z] = 0;
            // the cell's present quarters sit in consecutive ring slots in ascending q; EVERY warp of
            // the group passes through every present quarter's barrier, in ring order, whether or not
            // the quarter holds its rows (a parity wait is only sound for a waiter that has seen the
            // slot's previous phase)
#pragma unroll
            for (int r = 0; r < 2; ++r) {
              const int q = 2 * h + r;
              if (!(mask & (1 << q))) continue;
              const int qs = (qseq0 + __popc(mask & ((1 << q) - 1))) & 0xFFFF;
              const int slot = gi * C::QG + qs % C::QG;
              mbar_wait(bar(B_FULL_Q + slot), ((uint32_t)qs / C::QG) & 1);
              uint32_t landed = 0;
              if (r == rhalf) {
                const uint32_t rp = sRP + slot * QUARTER_BYTES;
                const uint4 r0 = lds128(rp + (row & 63) * 16);
                const uint4 r1 = lds128(rp + 1024 + (row & 63) * 16);
                unpack16(r0, ro);
                unpack16(r1, ro + 8);
                landed = zero_after(fold4(r0) ^ fold4(r1));
              }
              __syncwarp();
              if (lane == 0) mbar_arrive(bar(B_EMPTY_Q + slot) + landed);
            }
            tmem_st16(lane_addr + (uint32_t)(C::R_COL0 + rs * A_COLS + 16 * h), ro);
          }
          tmem_st_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar(B_FULL_RU + rs));
        }
      }
    }
    MQ_ACC_END(tu_tot);
    MQ_ACC_OUT(gtid == 0 && gi == 0, 68, tu_p); MQ_ACC_OUT(gtid == 0 && gi == 0, 69, tu_eu);
    MQ_ACC_OUT(gtid == 0 && gi == 0, 70, tu_work); MQ_ACC_OUT(gtid == 0 && gi == 0, 71, tu_tot);
  } else {
    // ===================== epilogue warps (2..5) =====================
    griddep_wait();   // s_a, Y, the workspace: ordered after the previous kernel in the stream
    const int lq = warp & 3;  // TMEM lane quadrant this warp may access
    const int et = (warp - FIRST_EPI_WARP) * 32 + lane;  // 0..127 within the epilogue group
    const int n_loc = lq * 32 + lane;
    const uint32_t my_first_tile = fdiv(u_beg, p.dKS);
    constexpr int PART = BT * BN;  // int32 elements of one partial accumulator
    if constexpr (FUSED) {
      // ---- per-token absmax over the whole row, found together with all CTAs of the grid --------
      // fz_ctrl: [0..15] absmax as fp32 bits (non-negative floats order like unsigned integers),
      // [16] CTAs arrived, [17] CTAs finished; all zero between calls.  Every CTA looks at one
      // 16-byte chunk per epilogue thread (M * K / 8 chunks <= grid * 128 for the shapes this path
      // takes), warp-reduces, and issues one atomic max per warp and row.
      const uint32_t total = (uint32_t)p.M * p.dRowChunks.d;
      for (uint32_t eb = blockIdx.x * 128u + (uint32_t)(et & ~31); eb < total; eb += gridDim.x * 128u) {   // warp-uniform
        const uint32_t e = eb + (uint32_t)lane;
        float am = 0.f;
        uint32_t rowi = 0xffffffffu;
        if (e < total) {
          rowi = fdiv(e, p.dRowChunks);
          const uint4 v = __ldcg(reinterpret_cast<const uint4*>(p.A + (size_t)rowi * p.lda) + (e - rowi * p.dRowChunks.d));
          const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            float f0, f1;
            if (p.a_bf16) {
              f0 = __uint_as_float(w[i] << 16);
              f1 = __uint_as_float(w[i] & 0xFFFF0000u);
            } else {
              const float2 t2 = __half22float2(*reinterpret_cast<const __half2*>(&w[i]));
              f0 = t2.x;
              f1 = t2.y;
            }
            am = fmaxf(am, fmaxf(fabsf(f0), fabsf(f1)));
          }
        }
        // lanes of a warp hold consecutive chunks: at most two rows per warp
        const uint32_t row_lo = __shfl_sync(0xffffffffu, rowi, 0);
        float a_lo = rowi == row_lo ? am : 0.f, a_hi = (rowi != row_lo && rowi != 0xffffffffu) ? am : 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          a_lo = fmaxf(a_lo, __shfl_xor_sync(0xffffffffu, a_lo, o));
          a_hi = fmaxf(a_hi, __shfl_xor_sync(0xffffffffu, a_hi, o));
        }
        const uint32_t row_hi = __shfl_sync(0xffffffffu, rowi, 31);
        if (lane == 0 && row_lo != 0xffffffffu && a_lo > 0.f) atomicMax(p.fz_ctrl + row_lo, __float_as_uint(a_lo));
        if (lane == 0 && row_hi != 0xffffffffu && row_hi != row_lo && a_hi > 0.f) atomicMax(p.fz_ctrl + row_hi, __float_as_uint(a_hi));
      }
      __threadfence();
      named_bar_sync(1, 128);
      if (et == 0) {
        atomicAdd(p.fz_ctrl + 16, 1u);
        uint32_t spins = 0, seen;
        do {   // all CTAs are resident (grid <= SM count, one CTA per SM), so this terminates
          asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(p.fz_ctrl + 16) : "memory");
          if (++spins > (1u << 24)) __trap();
        } while (seen < gridDim.x);
      }
      named_bar_sync(1, 128);
      if (et < 16) {
        const float a = et < p.M ? __uint_as_float(__ldcg(p.fz_ctrl + et)) : 0.f;
        sa_s[et] = a == 0.f ? 1.0f : __fdiv_rn(a, 7.0f);   // Eq.1 with q_max = 7; all-zero row: s = 1 (A2)
      }
      named_bar_sync(1, 128);
      if (et == 0) mbar_arrive(bar(B_SA));   // release: the unpack groups may read the token scales
    }
    MQ_ACC_DECL(te_t); MQ_ACC_DECL(te_d);
    int seg = 0, npend = 0;      // npend: partial tiles published by this CTA (at most 2)
    constexpr bool kBothParts = BT <= 32;
    uint32_t g = u_beg;
    while (g < u_end) {
      const uint32_t tile = fdiv(g, p.dKS);
      const int k0 = (int)(g - tile * (uint32_t)p.KS);
      const int k1 = (int)min((uint32_t)p.KS, (uint32_t)k0 + (u_end - g));
      g += (uint32_t)(k1 - k0);
      const int nt = (int)fdiv(tile, p.dTT), tt = (int)(tile - (uint32_t)nt * (uint32_t)p.TT);
      const int a0s = seg % C::ACC0_STAGES, a1s = seg % C::ACC1_STAGES;
      const uint32_t aphase = ((uint32_t)seg / C::ACC0_STAGES) & 1;
      ++seg;
      const int n = nt * BN + n_loc;
      const int t_base = tt * BT;
      const int t_cnt = min(BT, p.M - t_base);
      const float swn = __ldg(p.sw + n) * C::ACC_INV, srn = __ldg(p.sr + n) * C::ACC_INV;  // accumulators are x256 (x16: A8)
      auto emit = [&](int t, float sat, int32_t a0, int32_t a1) {
        const float y = sat * ((float)a0 * swn + (float)a1 * srn);
        const size_t o = (size_t)(t_base + t) * p.ldy + n;
        if (p.y_bf16)
          store_y<true>(p.Y, o, y);
        else
          store_y<false>(p.Y, o, y);
        if (p.dbg0) p.dbg0[(size_t)(t_base + t) * p.N + n] = a0 >> C::ACC_SHIFT;
        if (p.dbg1) p.dbg1[(size_t)(t_base + t) * p.N + n] = a1 >> C::ACC_SHIFT;
      };

      // prefill fast drain (whole tile, all BT tokens, no parity hooks): the tile's token scales go to
      // shared memory BEFORE the accumulator wait (one scale per epilogue thread), so that no global load
      // sits between the accumulator's completion and its release
      const bool whole_k = (k0 == 0 && k1 == p.KS);
      const bool fast = BT >= 64 && !FUSED && whole_k && t_cnt == BT && !p.dbg0 && !p.dbg1;
      float* sat = sa_tile + (seg & 1) * BT;
      if (BT >= 64) {
        if (fast && et < BT) sat[et] = __ldg(p.sa + t_base + et);
        named_bar_sync(1, 128);   // every segment: also orders this buffer's readers (two segments ago) before its writers
      }
      MQ_ACC_BEGIN(te_t);
      mbar_wait(bar(B_TFULL + a0s), aphase);
      MQ_ACC_END(te_t);
      MQ_ACC_BEGIN(te_d);
      tc_fence_after();
      MQ_STAMP_IF(et == 0 && seg == 1, 9);
      const bool has_res = acc_flag[a0s] != 0;  // acc1 is undefined when no residual MMA was issued
      // small token tiles (kBothParts): partial tiles always carry both accumulators (zeros when
      // there was no residual MMA), which takes the flag round trip out of the fix-up's latency chain
      const uint32_t lane_off = (uint32_t)(lq * 32) << 16;
      const uint32_t t0addr = tmem_base + lane_off + (uint32_t)(a0s * BT);
      const uint32_t t1addr = tmem_base + lane_off + (uint32_t)(C::ACC1_COL0 + a1s * BT);
      const bool whole = (k0 == 0 && k1 == p.KS);
      const int slot = tile == my_first_tile ? 0 : 1;
      int32_t* part0 = p.ws_part + ((size_t)blockIdx.x * 2 + slot) * (2 * PART);
      int32_t* part1 = part0 + PART;

      if (BT >= 64 && fast) {
        // 8-token batches, two in flight: the TMEM loads of batch b+1 run under the arithmetic and the
        // stores of batch b
        uint16_t* yp = reinterpret_cast<uint16_t*>(p.Y) + (size_t)t_base * p.ldy + n;
        auto drain = [&](auto res_c, auto bf_c) {
          constexpr bool RES = decltype(res_c)::value, BF = decltype(bf_c)::value;
          uint32_t a[2][8], r[2][8];
#pragma unroll
          for (int i = 0; i < 8; ++i) r[0][i] = r[1][i] = 0;
          tmem_ld8(t0addr, a[0]);
          if (RES) tmem_ld8(t1addr, r[0]);
#pragma unroll
          for (int b = 0; b < BT / 8; ++b) {
            const int cur = b & 1;
            tmem_ld_wait8(a[cur], r[cur]);
            if (b + 1 < BT / 8) {
              tmem_ld8(t0addr + (b + 1) * 8, a[cur ^ 1]);
              if (RES) tmem_ld8(t1addr + (b + 1) * 8, r[cur ^ 1]);
            }
            const float4 s_lo = *reinterpret_cast<const float4*>(sat + b * 8);
            const float4 s_hi = *reinterpret_cast<const float4*>(sat + b * 8 + 4);
            const float sv[8] = {s_lo.x, s_lo.y, s_lo.z, s_lo.w, s_hi.x, s_hi.y, s_hi.z, s_hi.w};
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              float y = (float)(int32_t)a[cur][i] * swn;
              if (RES) y += (float)(int32_t)r[cur][i] * srn;   // same operation order as the general path
              y *= sv[i];
              *yp = BF ? __bfloat16_as_ushort(__float2bfloat16_rn(y)) : __half_as_ushort(__float2half_rn(y));
              yp += p.ldy;
            }
          }
        };
        if (has_res) {
          if (p.y_bf16) drain(std::true_type{}, std::true_type{}); else drain(std::true_type{}, std::false_type{});
        } else {
          if (p.y_bf16) drain(std::false_type{}, std::true_type{}); else drain(std::false_type{}, std::false_type{});
        }
      } else
      for (int c0 = 0; c0 < t_cnt; c0 += 16) {
        uint32_t v0[16], v1[16];
        float sav[16];   // token scales of the chunk, fetched up front (read-only path: one L2 round trip
                         // per chunk instead of one per token behind the stores)
        if (whole) {
#pragma unroll
          for (int i = 0; i < 16; ++i) sav[i] = c0 + i < t_cnt ? (FUSED ? sa_s[c0 + i] : __ldg(p.sa + t_base + c0 + i)) : 0.f;
        }
        tmem_ld16(t0addr + c0, v0);
        if (has_res) {
          tmem_ld16(t1addr + c0, v1);
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i) v1[i] = 0;
        }
        tmem_ld_wait();
        if (whole && !p.dbg0 && !p.dbg1 && c0 + 16 <= t_cnt) {
          // hot path (full chunk, no parity hooks): branch-free, one pointer bump per token
          uint16_t* yp = reinterpret_cast<uint16_t*>(p.Y) + (size_t)(t_base + c0) * p.ldy + n;
          if (p.y_bf16) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
              const float y = sav[i] * ((float)(int32_t)v0[i] * swn + (float)(int32_t)v1[i] * srn);
              *yp = __bfloat16_as_ushort(__float2bfloat16_rn(y));
              yp += p.ldy;
            }
          } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
              const float y = sav[i] * ((float)(int32_t)v0[i] * swn + (float)(int32_t)v1[i] * srn);
              *yp = __half_as_ushort(__float2half_rn(y));
              yp += p.ldy;
            }
          }
        } else if (whole) {
#pragma unroll
          for (int i = 0; i < 16; ++i)
            if (c0 + i < t_cnt) emit(c0 + i, sav[i], (int32_t)v0[i], (int32_t)v1[i]);
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i)
            if (c0 + i < t_cnt) {
              __stcg(part0 + (c0 + i) * BN + n_loc, (int32_t)v0[i]);
              if (kBothParts || has_res) __stcg(part1 + (c0 + i) * BN + n_loc, (int32_t)v1[i]);
            }
        }
      }
      // accumulator stages drained: hand them back to the MMA warp
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(bar(B_A1E + a1s));
        mbar_arrive(bar(B_A0E + a0s));
      }
      MQ_ACC_END(te_d);
      MQ_ACC_OUT(et == 0, 74, te_t); MQ_ACC_OUT(et == 0, 75, te_d);

      if (!whole) {
        // stream-K fix-up, part 1: publish this partial (release) and count the arrival.  Nothing
        // waits here; a CTA waits only after ALL of its partials are published (part 2), so the
        // contributors of different tiles cannot wait on each other in a cycle.
        if (!kBothParts && et == 0) p.ws_flag[blockIdx.x * 2 + slot] = has_res ? 1 : 0;
        __threadfence();
        named_bar_sync(1, 128);
        if (et == 0) {
          const int c_lo = owner_of(p, tile * (uint32_t)p.KS), c_hi = owner_of(p, (tile + 1) * (uint32_t)p.KS - 1);
          atomicAdd(p.ws_cnt + tile, 1);
          int32_t* pd = const_cast<int32_t*>(pend) + npend * 4;
          pd[0] = (int32_t)tile;
          pd[1] = c_lo;
          pd[2] = c_hi;
          pd[3] = (fdiv(range_begin(p, (uint32_t)c_lo), p.dKS) == tile) ? 0 : 1;  // slot of c_lo's partial
        }
        ++npend;
      }
      MQ_STAMP_IF(et == 0, 10);
    }

    // stream-K fix-up, part 2: the S contributors of a tile wait until all S partials are visible,
    // then EACH reduces and finishes 1/S of the tile (16-byte loads, all contributors in flight).
    // All CTAs of the grid are resident (grid <= SM count, one CTA per SM), so the wait terminates.
    if (npend) named_bar_sync(1, 128);   // pend[] written by thread et == 0
    for (int pi = 0; pi < npend; ++pi) {
      const uint32_t tile = (uint32_t)pend[pi * 4 + 0];
      const int c_lo = pend[pi * 4 + 1], c_hi = pend[pi * 4 + 2], lo_slot = pend[pi * 4 + 3];
      const int S = c_hi - c_lo + 1, r = (int)blockIdx.x - c_lo;
      const int nt = (int)fdiv(tile, p.dTT), tt = (int)(tile - (uint32_t)nt * (uint32_t)p.TT);
      const int t_base = tt * BT;
      const int t_cnt = min(BT, p.M - t_base);
      {
        uint32_t spins = 0;
        int seen;
        do {
          asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(p.ws_cnt + tile) : "memory");
          if (++spins > (1u << 24)) __trap();
        } while (seen < S);
      }
      // residual flags of the contributors (bit c - c_lo) for S <= 32; beyond that each flag is read in the loop
      // (a contributor without residual MMAs never wrote its part1 slot: it must not be added)
      uint32_t fm = 0xffffffffu;
      if (!kBothParts && S <= 32) {
        int f = 0;
        if (lane < S) f = __ldcg(p.ws_flag + (c_lo + lane) * 2 + (lane == 0 ? lo_slot : 0));
        fm = __ballot_sync(0xffffffffu, f != 0);
      }
      const int E4 = t_cnt * (BN / 4);                       // 16-byte units of one accumulator
      const int e_lo = (int)(((long long)E4 * r) / S), e_hi = (int)(((long long)E4 * (r + 1)) / S);
      const bool y_vec = ((reinterpret_cast<uintptr_t>(p.Y) | (uintptr_t)(p.ldy * 2)) & 7) == 0;
      for (int e = e_lo + et; e < e_hi; e += 128) {
        const int t = e / (BN / 4), n0 = (e - t * (BN / 4)) * 4;
        int4 s0 = make_int4(0, 0, 0, 0), s1 = make_int4(0, 0, 0, 0);
#pragma unroll 4
        for (int c = c_lo; c <= c_hi; ++c) {
          const int32_t* q0 = p.ws_part + ((size_t)c * 2 + (c == c_lo ? lo_slot : 0)) * (2 * PART) + t * BN + n0;
          const int4 a = __ldcg(reinterpret_cast<const int4*>(q0));
          int4 b = make_int4(0, 0, 0, 0);
          const bool has1 = kBothParts || (S <= 32 ? ((fm >> ((c - c_lo) & 31)) & 1u) != 0
                                                   : __ldcg(p.ws_flag + c * 2 + (c == c_lo ? lo_slot : 0)) != 0);
          if (has1) b = __ldcg(reinterpret_cast<const int4*>(q0 + PART));
          s0.x += a.x; s0.y += a.y; s0.z += a.z; s0.w += a.w;
          s1.x += b.x; s1.y += b.y; s1.z += b.z; s1.w += b.w;
        }
        const int n = nt * BN + n0;
        const float4 sw4 = *reinterpret_cast<const float4*>(p.sw + n), sr4 = *reinterpret_cast<const float4*>(p.sr + n);
        const float sat = (FUSED ? sa_s[t] : __ldg(p.sa + t_base + t)) * C::ACC_INV;    // accumulators are x256 (x16: A8)
        float y[4];
        y[0] = sat * ((float)s0.x * sw4.x + (float)s1.x * sr4.x);
        y[1] = sat * ((float)s0.y * sw4.y + (float)s1.y * sr4.y);
        y[2] = sat * ((float)s0.z * sw4.z + (float)s1.z * sr4.z);
        y[3] = sat * ((float)s0.w * sw4.w + (float)s1.w * sr4.w);
        const size_t o = (size_t)(t_base + t) * p.ldy + n;
        if (y_vec) {
          uint2 pk;
          if (p.y_bf16) {
            __nv_bfloat162 lo = __floats2bfloat162_rn(y[0], y[1]), hi = __floats2bfloat162_rn(y[2], y[3]);
            pk.x = *reinterpret_cast<uint32_t*>(&lo);
            pk.y = *reinterpret_cast<uint32_t*>(&hi);
          } else {
            __half2 lo = __floats2half2_rn(y[0], y[1]), hi = __floats2half2_rn(y[2], y[3]);
            pk.x = *reinterpret_cast<uint32_t*>(&lo);
            pk.y = *reinterpret_cast<uint32_t*>(&hi);
          }
          *reinterpret_cast<uint2*>(reinterpret_cast<uint16_t*>(p.Y) + o) = pk;
        } else {
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            if (p.y_bf16)
              store_y<true>(p.Y, o + i, y[i]);
            else
              store_y<false>(p.Y, o + i, y[i]);
          }
        }
        const size_t od = (size_t)(t_base + t) * p.N + n;
        if (p.dbg0) *reinterpret_cast<int4*>(p.dbg0 + od) = make_int4(s0.x >> C::ACC_SHIFT, s0.y >> C::ACC_SHIFT, s0.z >> C::ACC_SHIFT, s0.w >> C::ACC_SHIFT);
        if (p.dbg1) *reinterpret_cast<int4*>(p.dbg1 + od) = make_int4(s1.x >> C::ACC_SHIFT, s1.y >> C::ACC_SHIFT, s1.z >> C::ACC_SHIFT, s1.w >> C::ACC_SHIFT);
      }
      // the last contributor to finish returns the tile's counters to zero for the next call
      named_bar_sync(1, 128);
      if (et == 0) {
        const int old = atomicAdd(p.ws_done + tile, 1);
        if (old == S - 1) {
          p.ws_cnt[tile] = 0;
          p.ws_done[tile] = 0;
        }
      }
    }
    if constexpr (FUSED) {
      // the last CTA to finish returns the absmax control block to zero for the next call
      if (et == 0) {
        const uint32_t old = atomicAdd(p.fz_ctrl + 17, 1u);
        if (old == gridDim.x - 1) {
          for (int i = 0; i < 18; ++i) p.fz_ctrl[i] = 0;
        }
      }
    }
  }

  // teardown (single-lane regions re-converge first: bar.sync must be reached warp-convergent)
  __syncwarp();
  tc_fence_before();
  __syncthreads();
  MQ_STAMP_IF(threadIdx.x == 0, 11);
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, C::TMEM_COLS);
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  return (EncodeTiledFn)mq::tensor_map_encode_fn();
}

}  // namespace

void* mq::tensor_map_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)ptr;
    else
      cudaGetLastError();
  }
  return (void*)fn;
}

namespace {

size_t align256(size_t x) { return (x + 255) / 256 * 256; }

FastDiv make_fastdiv(uint32_t d) {
  FastDiv f;
  f.d = d;
  f.mul = 0;
  f.shr = 0;
  if (d > 1) {
    uint32_t l = 0;
    while ((1ull << l) < d) ++l;
    f.mul = (uint32_t)(((1ull << (31 + l)) / d) + 1);
    f.shr = l - 1;
  }
  return f;
}

struct Plan {
  int BT = 16, TT = 1, grid = 1, gran = 1;
  int64_t units = 0;   // K-steps of all tiles; the kernel indexes them with 32 bits
  size_t off_done = 0, off_flag = 0, off_part = 0, ws_bytes = 0;
};

Plan make_plan(const mq_weights* w, int64_t M) {
  Plan pl;
  const Options& o = options();
  const int NT = (int)(w->N / BN), KS = (int)(w->K / BK);
  int G = sm_count() > 0 ? sm_count() : 148;
  if (o.max_ctas > 0) G = (int)std::min<int64_t>(G, o.max_ctas);
  int bt;
  if (o.token_tile) {
    bt = (int)o.token_tile;
  } else if (M <= 32) {
    bt = M <= 16 ? 16 : 32;
  } else {
    // Mid-size M: the smallest token tile whose tile count still fits one wave (most CTAs busy with
    // whole tiles, no split-K fix-up); if even 128-token tiles need several waves, the tile that
    // wastes least (M <= 64: 64, else 128).
    bt = M <= 64 ? 64 : 128;
    for (int cand = 32; cand <= 128; cand *= 2)
      if ((int64_t)NT * ((M + cand - 1) / cand) <= G) {
        bt = cand;
        break;
      }
  }
  pl.BT = bt;
  pl.TT = (int)((M + bt - 1) / bt);
  const int64_t tiles = (int64_t)NT * pl.TT;
  pl.units = tiles * KS;
  // Decode (M <= 32) streams weights and needs every SM pulling: split K whenever whole tiles would not
  // balance.  Beyond that a partial tile costs BT x 128 x 8 bytes in the fix-up, so K is split only when
  // most SMs would otherwise idle.
  bool stream_k = M <= 32 ? tiles < 8LL * G
                          : (bt <= 32 ? tiles * 2 <= G && (tiles * 3 <= G || KS >= 64)   // cheap fix-up: long K pays
                                      : tiles * 2 <= G);
  if (o.split_k == 1) stream_k = false;
  if (o.split_k >= 2) stream_k = true;
  if (tiles > WS_MAX_TILES) stream_k = false;   // one counter per tile in the workspace prefix
  pl.gran = stream_k ? 1 : KS;
  pl.grid = (int)std::min<int64_t>(G, pl.units / pl.gran);
  // Few tiles: cut every tile into the same S parts (grid = tiles * S makes the stream-K ranges
  // tile-aligned), so that each CTA owns ONE partial segment and pays the fix-up latency once.
  if (stream_k && o.split_k == 0 && tiles * 2 <= G) {
    const int64_t S = std::min<int64_t>(G / tiles, KS);
    pl.grid = (int)(tiles * S);
  }
  if (stream_k) {
    // zero-state words (counters) live in the plan-independent prefix (mq_internal.h); flags and partial
    // tiles behind it are written before they are read
    pl.off_done = WS_OFF_DONE;
    pl.off_flag = WS_PREFIX;
    pl.off_part = pl.off_flag + align256((size_t)pl.grid * 2 * 4);
    pl.ws_bytes = pl.off_part + (size_t)pl.grid * 2 * 2 * bt * BN * 4;
  }
  return pl;
}

template <int BT, bool FUSED = false, bool A8 = false>
int launch(const CUtensorMap& tmap, const GemmParams& gp, int grid, cudaStream_t st) {
  using C = Cfg<BT, FUSED, A8>;
  // the attribute belongs to the (device, function) pair: set it again whenever the current device changes
  static int attr_dev = -1;
  int dev = -1;
  cudaGetDevice(&dev);
  if (dev != attr_dev) {
    if (cudaFuncSetAttribute(mq_gemm_kernel<BT, FUSED, A8>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES) !=
        cudaSuccess) {
      cudaGetLastError();
      return MQ_ERR_CUDA;
    }
    attr_dev = dev;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(C::NUM_THREADS);
  cfg.dynamicSmemBytes = C::SMEM_BYTES;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = options().pdl ? 1 : 0;
  if (cudaLaunchKernelEx(&cfg, mq_gemm_kernel<BT, FUSED, A8>, tmap, gp) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  return MQ_OK;
}

}  // namespace

#ifdef MQ_TRACE
static long long* g_trace = nullptr;
extern "C" void mq_debug_set_trace(long long* dev_buf) { g_trace = dev_buf; }
#endif

extern "C" size_t mq_gemm_workspace_bytes(const mq_weights* w, int64_t M) {
  if (!w || M <= 0) return 0;
  if (mq::check_device() != MQ_OK) return 0;
  // the larger of the two kernels' needs, so that a workspace sized once serves the call whichever kernel the
  // options in force at call time select
  const size_t d = M <= 32 ? mq::decode_workspace_bytes(w, M) : 0;
  return std::max(d, make_plan(w, M).ws_bytes);
}

namespace {

// mq_gemm proper; with fused_A != NULL the kernel quantizes the raw activations itself (mq_linear, M <= 8)
// and qA / sA are unused.
int gemm_impl(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
              int32_t* dbg0, int32_t* dbg1, void* workspace, size_t workspace_bytes, void* cuda_stream,
              const void* fused_A, mq_dtype a_dtype, int64_t lda, uint32_t* fz_ctrl, bool a8 = false,
              bool ignore_res = false) {
  const bool fused = fused_A != nullptr;
  if (a8 && (fused || (w && (long double)127 * 7 * 16 * (long double)w->K >= 2147483648.0L))) return MQ_ERR_ACC_OVERFLOW;
  if (!w) return MQ_ERR_INVALID_ARG;
  if (M < 0 || M > (1 << 30)) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (y_dtype != MQ_F16 && y_dtype != MQ_BF16) return MQ_ERR_INVALID_ARG;
  mq::set_launch_count(0);
  if (M == 0) return MQ_OK;
  if (!Y || ldy < w->N || ((uintptr_t)Y & 1)) return MQ_ERR_INVALID_ARG;
  if (!fused) {
    if (!qA || !sA) return MQ_ERR_INVALID_ARG;
    if (((uintptr_t)qA & 15) || ((uintptr_t)sA & 3)) return MQ_ERR_INVALID_ARG;
  }
  if (((uintptr_t)dbg0 & 15) || ((uintptr_t)dbg1 & 15)) return MQ_ERR_INVALID_ARG;
  int rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  EncodeTiledFn enc = get_encode_fn();
  if (!enc) return MQ_ERR_CUDA;

  // block-local residual scales (reading A4b) exist in the decode kernel only
  if (w->blockscale && (fused || a8 || !mq::decode_eligible(w, M))) return MQ_ERR_UNSUPPORTED_SHAPE;
  // decode shapes: the lean TMEM-free kernel (mq_decode.cu)
  if (!fused && !a8 && mq::decode_eligible(w, M))
    return mq::decode_gemm(w, qA, sA, M, Y, y_dtype, ldy, dbg0, dbg1, workspace, workspace_bytes, cuda_stream, ignore_res);
  // prefill shapes whose whole tiles fill the machine: the whole-tile kernel (mq_prefill.cu)
  if (!fused && a8 && mq::decode_a8_eligible(w, M))
    return mq::decode_gemm_a8(w, qA, sA, M, Y, y_dtype, ldy, dbg0, dbg1, cuda_stream, ignore_res);
  if (!fused && mq::prefill_eligible(w, M, a8))
    return mq::prefill_gemm(w, qA, sA, M, Y, y_dtype, ldy, dbg0, dbg1, cuda_stream, ignore_res, a8);

  const Plan pl = make_plan(w, M);
  if (pl.units >= (int64_t)1 << 31) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (pl.ws_bytes > 0) {
    if (!workspace || workspace_bytes < pl.ws_bytes) return MQ_ERR_WORKSPACE;
    if ((uintptr_t)workspace & 15) return MQ_ERR_INVALID_ARG;
  }

  // 2-D tensor map over the canonical packed activations: [M rows][K/2 bytes]
  CUtensorMap tmap;
  memset(&tmap, 0, sizeof(tmap));
  if (fused && pl.BT != 16) return MQ_ERR_INVALID_ARG;
  // (W4A8: int8 activations [M rows][K bytes], box {128 B, BT rows})
  const cuuint64_t row_bytes = a8 ? (cuuint64_t)w->K : (cuuint64_t)(w->K / 2);
  const cuuint64_t gdim[2] = {row_bytes, (cuuint64_t)M};
  const cuuint64_t gstride[1] = {row_bytes};
  const cuuint32_t box[2] = {(cuuint32_t)(a8 ? BK : BK / 2), (cuuint32_t)pl.BT};
  const cuuint32_t estr[2] = {1, 1};
  if (!fused && enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(qA), gdim, gstride, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return MQ_ERR_CUDA;
  if (fused) {
    // 2-D tensor map over the raw 16-bit activations [M rows][K elements], box {128 elements, 8 rows}
    const cuuint64_t fdim[2] = {(cuuint64_t)w->K, (cuuint64_t)M};
    const cuuint64_t fstride[1] = {(cuuint64_t)lda * 2};
    const cuuint32_t fbox[2] = {(cuuint32_t)BK, 8};
    if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, const_cast<void*>(fused_A), fdim, fstride, fbox, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return MQ_ERR_CUDA;
  }

  GemmParams gp;
  gp.base = w->d_base;
  gp.sw = w->d_sw;
  gp.sr = w->d_sr;
  gp.res = w->d_res;
  gp.unit_meta = ignore_res ? nullptr : (const int2*)w->d_unit_meta;
  gp.sa = sA;
  gp.Y = Y;
  gp.dbg0 = dbg0;
  gp.dbg1 = dbg1;
  gp.ldy = ldy;
  gp.M = (int)M;
  gp.N = (int)w->N;
  gp.KS = (int)(w->K / BK);
  gp.NT = (int)(w->N / BN);
  gp.TT = pl.TT;
  gp.units = (uint32_t)pl.units;
  gp.gran = (uint32_t)pl.gran;
  gp.upg_q = (uint32_t)((pl.units / pl.gran) / pl.grid);
  gp.upg_r = (uint32_t)((pl.units / pl.gran) % pl.grid);
  gp.dKS = make_fastdiv((uint32_t)gp.KS);
  gp.dTT = make_fastdiv((uint32_t)gp.TT);
  gp.dGrid = make_fastdiv((uint32_t)pl.grid);
  gp.y_bf16 = y_dtype == MQ_BF16;
  gp.A = (const uint16_t*)fused_A;
  gp.lda = lda;
  gp.a_bf16 = a_dtype == MQ_BF16;
  gp.fz_ctrl = fz_ctrl;
  gp.dRowChunks = make_fastdiv((uint32_t)(w->K / 8));
  uint8_t* ws = (uint8_t*)workspace;
  gp.ws_cnt = (int32_t*)(ws + WS_OFF_CNT);
  gp.ws_done = (int32_t*)(ws + pl.off_done);
  gp.ws_flag = (int32_t*)(ws + pl.off_flag);
  gp.ws_part = (int32_t*)(ws + pl.off_part);
#ifdef MQ_TRACE
  gp.trace = g_trace;
  if (!g_trace) return MQ_ERR_INVALID_ARG;
#endif

  cudaStream_t st = (cudaStream_t)cuda_stream;
  switch (pl.BT) {
    case 16:
      rc = fused ? launch<16, true>(tmap, gp, pl.grid, st)
                 : (a8 ? launch<16, false, true>(tmap, gp, pl.grid, st) : launch<16>(tmap, gp, pl.grid, st));
      break;
    case 32: rc = a8 ? launch<32, false, true>(tmap, gp, pl.grid, st) : launch<32>(tmap, gp, pl.grid, st); break;
    case 64: rc = a8 ? launch<64, false, true>(tmap, gp, pl.grid, st) : launch<64>(tmap, gp, pl.grid, st); break;
    case 128: rc = a8 ? launch<128, false, true>(tmap, gp, pl.grid, st) : launch<128>(tmap, gp, pl.grid, st); break;
    default: rc = MQ_ERR_INVALID_ARG;
  }
  if (rc == MQ_OK) mq::set_launch_count(1);
  return rc;
}

}  // namespace

extern "C" int mq_gemm(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype,
                       int64_t ldy, int32_t* dbg0, int32_t* dbg1, void* workspace, size_t workspace_bytes,
                       void* cuda_stream) {
  return gemm_impl(w, qA, sA, M, Y, y_dtype, ldy, dbg0, dbg1, workspace, workspace_bytes, cuda_stream, nullptr, MQ_F16, 0,
                   nullptr);
}

extern "C" int mq_gemm_a8(const mq_weights* w, const int8_t* qA8, const float* sA, int64_t M, void* Y, mq_dtype y_dtype,
                          int64_t ldy, int32_t* dbg0, int32_t* dbg1, void* workspace, size_t workspace_bytes,
                          void* cuda_stream) {
  return gemm_impl(w, qA8, sA, M, Y, y_dtype, ldy, dbg0, dbg1, workspace, workspace_bytes, cuda_stream, nullptr, MQ_F16, 0,
                   nullptr, true);
}

// ------------------------------------------------------------------------------------------------------
// The paper's NAIVE pipeline (Fig.3), for the fused-vs-naive ablation:
//   (i)   dense W4A4 GEMM: this library's kernel with the residual switched off, 16-bit Y0 = s_a s_w acc0
//   (ii)  a separate sparse-block GEMM that re-reads the quantized activations from HBM and writes a partial
//         output (acc1, int32 [M, N]), SIMT dp4a, one CTA per (n-tile, 16 tokens) walking the n-tile's cells
//   (iii) reduce-add: Y = round16(Y0 + s_a s_r acc1)
// Three launches and two extra passes over [M, N]; it also rounds twice.
namespace {

constexpr int NAIVE_TOK = 16;

__device__ __forceinline__ int dp4a_s8(uint32_t a, uint32_t b, int c) {
  int d;
  asm("dp4a.s32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}

__global__ void __launch_bounds__(128) naive_sparse_kernel(const uint8_t* __restrict__ res, const mq::CellMeta* __restrict__ cells,
                                                           const int32_t* __restrict__ cell_ptr, const uint8_t* __restrict__ qA,
                                                           int64_t M, int64_t K, int64_t N, int32_t* __restrict__ acc1, int cells_per_cta) {
  const int nt = blockIdx.x, row = threadIdx.x, rhalf = row >> 6;
  const int64_t m0 = (int64_t)blockIdx.y * NAIVE_TOK;
  const int mt = (int)min((int64_t)NAIVE_TOK, M - m0);
  int acc[NAIVE_TOK];
#pragma unroll
  for (int t = 0; t < NAIVE_TOK; ++t) acc[t] = 0;
  const uint32_t HI = 0xF0F0F0F0u;
  // the n-tile's cells are dealt to gridDim.z CTAs (cells_per_cta each); with more than one, the partial sums meet
  // in acc1 through int32 atomics (exact, so the result does not depend on the order)
  // (runs of cells_per_cta cells, strided by gridDim.z runs: every cell is visited whatever the cap on gridDim.z)
  const int c_end = cell_ptr[nt + 1];
  if (gridDim.z > 1 && cell_ptr[nt] + (int)blockIdx.z * cells_per_cta >= c_end) return;
  for (int c0 = cell_ptr[nt] + (int)blockIdx.z * cells_per_cta; c0 < c_end; c0 += (int)gridDim.z * cells_per_cta)
  for (int c = c0; c < min(c_end, c0 + cells_per_cta); ++c) {
    const int km = cells[c].kstep_mask, kstep = km & 0xFFFFFF, mask = (km >> 24) & 0xF;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int q = 2 * h + rhalf;
      if (!(mask & (1 << q))) continue;
      const uint8_t* qp = res + ((size_t)cells[c].qoff + (size_t)__popc(mask & ((1 << q) - 1))) * QUARTER_BYTES + (size_t)(row & 63) * 16;
      const uint4 w0 = *reinterpret_cast<const uint4*>(qp), w1 = *reinterpret_cast<const uint4*>(qp + 1024);
      const uint32_t ww[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
      const size_t koff = ((size_t)kstep * BK + (size_t)h * 64) / 2;   // byte offset of the 64 activations in a row of qA
#pragma unroll
      for (int t = 0; t < NAIVE_TOK; ++t) {
        if (t >= mt) break;
        const uint8_t* ap = qA + (size_t)(m0 + t) * (size_t)(K / 2) + koff;
        const uint4 a0 = __ldg(reinterpret_cast<const uint4*>(ap)), a1 = __ldg(reinterpret_cast<const uint4*>(ap + 16));
        const uint32_t aw[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
        int sacc = acc[t];
#pragma unroll
        for (int i = 0; i < 8; ++i) {   // both operands x16, even / odd nibbles pair up: sum is 256 x the dot product
          sacc = dp4a_s8((ww[i] << 4) & HI, (aw[i] << 4) & HI, sacc);
          sacc = dp4a_s8(ww[i] & HI, aw[i] & HI, sacc);
        }
        acc[t] = sacc;
      }
    }
  }
#pragma unroll
  for (int t = 0; t < NAIVE_TOK; ++t)
    if (t < mt) {
      int32_t* dst = acc1 + (size_t)(m0 + t) * (size_t)N + (size_t)nt * BN + row;
      if (gridDim.z > 1) {
        if (acc[t]) atomicAdd(dst, acc[t] >> 8);
      } else {
        *dst = acc[t] >> 8;
      }
    }
}

template <bool BF16>
__global__ void naive_add_kernel(void* __restrict__ Y, int64_t ldy, const int32_t* __restrict__ acc1, const float* __restrict__ sa,
                                 const float* __restrict__ sr, int64_t M, int64_t N) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= M * N) return;
  const int64_t m = idx / N, n = idx - m * N;
  const size_t o = (size_t)m * (size_t)ldy + (size_t)n;
  float y0;
  if (BF16)
    y0 = __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(Y)[o]);
  else
    y0 = __half2float(reinterpret_cast<const __half*>(Y)[o]);
  store_y<BF16>(Y, o, y0 + sa[m] * (sr[n] * (float)acc1[idx]));
}

}  // namespace

extern "C" size_t mq_gemm_naive_scratch_bytes(const mq_weights* w, int64_t M) {
  return (!w || M <= 0) ? 0 : (size_t)M * (size_t)w->N * sizeof(int32_t);
}

extern "C" int mq_gemm_naive(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype,
                             int64_t ldy, void* workspace, size_t workspace_bytes, int32_t* scratch, size_t scratch_bytes,
                             void* cuda_stream) {
  if (!w) return MQ_ERR_INVALID_ARG;
  if (w->blockscale) return MQ_ERR_UNSUPPORTED_SHAPE;   // block-local residual scales: mq_gemm only
  if (M > 0 && (!scratch || ((uintptr_t)scratch & 3))) return MQ_ERR_INVALID_ARG;
  if (M > 0 && scratch_bytes < mq_gemm_naive_scratch_bytes(w, M)) return MQ_ERR_WORKSPACE;
  const int rc = gemm_impl(w, qA, sA, M, Y, y_dtype, ldy, nullptr, nullptr, workspace, workspace_bytes, cuda_stream, nullptr,
                           MQ_F16, 0, nullptr, false, true);
  if (rc != MQ_OK || M == 0) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // few tokens: split an n-tile's cells over several CTAs so that the kernel is not a handful of long serial loops
  const int cells_per_cta = M <= 64 ? 2 : (M <= 512 ? 8 : 1 << 20);
  const unsigned gz = (unsigned)std::max(1, std::min(64, (w->max_cells_per_tile + cells_per_cta - 1) / cells_per_cta));
  const dim3 grid((unsigned)(w->N / BN), (unsigned)((M + NAIVE_TOK - 1) / NAIVE_TOK), gz);
  if (grid.y > 65535) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (gz > 1 && cudaMemsetAsync(scratch, 0, (size_t)M * (size_t)w->N * sizeof(int32_t), st) != cudaSuccess) return MQ_ERR_CUDA;
  naive_sparse_kernel<<<grid, 128, 0, st>>>(w->d_res, w->d_cell_meta, w->d_cell_ptr, (const uint8_t*)qA, M, w->K, w->N, scratch,
                                            gz > 1 ? cells_per_cta : 1 << 20);
  const int64_t total = M * w->N;
  const unsigned blocks = (unsigned)((total + 255) / 256);
  if (y_dtype == MQ_BF16)
    naive_add_kernel<true><<<blocks, 256, 0, st>>>(Y, ldy, scratch, sA, w->d_sr, M, w->N);
  else
    naive_add_kernel<false><<<blocks, 256, 0, st>>>(Y, ldy, scratch, sA, w->d_sr, M, w->N);
  if (cudaGetLastError() != cudaSuccess) return MQ_ERR_CUDA;
  mq::set_launch_count(3);
  return MQ_OK;
}

extern "C" size_t mq_linear_workspace_bytes(const mq_weights* w, int64_t M) {
  if (!w || M <= 0) return 0;
  size_t q = (mq_qact_bytes(M, w->K) + 255) / 256 * 256;
  size_t s = ((size_t)M * 4 + 255) / 256 * 256;
  return std::max(align256(mq_gemm_workspace_bytes(w, M)), mq::WS_PREFIX) + q + s;
}

extern "C" int mq_linear(const mq_weights* w, const void* A, mq_dtype a_dtype, int64_t M, int64_t lda, void* Y,
                         mq_dtype y_dtype, int64_t ldy, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!w) return MQ_ERR_INVALID_ARG;
  if (M == 0) return MQ_OK;
  if (M < 0) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (a_dtype != MQ_F16 && a_dtype != MQ_BF16) return MQ_ERR_INVALID_ARG;
  if (!A || lda < w->K || (lda % 8) != 0 || ((uintptr_t)A & 15)) return MQ_ERR_INVALID_ARG;
  if (!workspace || ((uintptr_t)workspace & 255)) return MQ_ERR_INVALID_ARG;
  const size_t need = mq_linear_workspace_bytes(w, M);
  if (workspace_bytes < need) return MQ_ERR_WORKSPACE;
  // zero-state regions first (the GEMM's counters, the fused path's control block), so that the
  // caller's one-time memset covers them; then the packed activations and their scales
  const size_t g = mq_gemm_workspace_bytes(w, M);
  const size_t g_al = std::max(align256(g), mq::WS_PREFIX);   // the prefix also carries the fused path's control block
  uint8_t* base = (uint8_t*)workspace;
  uint32_t* ctrl = (uint32_t*)(base + mq::WS_OFF_FZ);
  uint8_t* qa = base + g_al;
  float* sa = (float*)(qa + (mq_qact_bytes(M, w->K) + 255) / 256 * 256);
  if ((size_t)((uint8_t*)sa + (size_t)M * 4 - base) > workspace_bytes) return MQ_ERR_WORKSPACE;
  // Decode-sized calls (M <= 8): ONE kernel, the activation quantizer runs inside the GEMM.
  // Larger M: the quantizer as its own kernel (chained by programmatic dependent launch).
  const Options& o = options();
  if (o.fused_quant && M <= 8 && w->K >= 256 && (o.token_tile == 0 || o.token_tile == 16))
    return gemm_impl(w, nullptr, nullptr, M, Y, y_dtype, ldy, nullptr, nullptr, base, g_al, cuda_stream, A, a_dtype, lda, ctrl);
  int rc = mq_quantize_act(A, a_dtype, M, w->K, lda, qa, sa, cuda_stream);
  if (rc != MQ_OK) return rc;
  rc = mq_gemm(w, qa, sa, M, Y, y_dtype, ldy, nullptr, nullptr, base, g_al, cuda_stream);
  if (rc == MQ_OK) mq::set_launch_count(2);
  return rc;
}

extern "C" size_t mq_linear_host_staging_bytes(const mq_weights* w, int64_t M) {
  if (!w || M <= 0) return 0;
  return align256((size_t)M * (size_t)w->K * 2) + align256((size_t)M * (size_t)w->N * 2);
}

extern "C" int mq_linear_host(const mq_weights* w, const void* A_host, mq_dtype a_dtype, int64_t M, void* Y_host,
                              mq_dtype y_dtype, void* staging, size_t staging_bytes, void* workspace,
                              size_t workspace_bytes, void* cuda_stream) {
  if (!w) return MQ_ERR_INVALID_ARG;
  if (M == 0) return MQ_OK;
  if (M < 0) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (!A_host || !Y_host || !staging || ((uintptr_t)staging & 255)) return MQ_ERR_INVALID_ARG;
  if (staging_bytes < mq_linear_host_staging_bytes(w, M)) return MQ_ERR_WORKSPACE;
  int rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  uint8_t* a_dev = (uint8_t*)staging;
  uint8_t* y_dev = a_dev + align256((size_t)M * (size_t)w->K * 2);
  if (cudaMemcpyAsync(a_dev, A_host, (size_t)M * (size_t)w->K * 2, cudaMemcpyHostToDevice, st) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  rc = mq_linear(w, a_dev, a_dtype, M, w->K, y_dev, y_dtype, w->N, workspace, workspace_bytes, cuda_stream);
  if (rc != MQ_OK) return rc;
  if (cudaMemcpyAsync(Y_host, y_dev, (size_t)M * (size_t)w->N * 2, cudaMemcpyDeviceToHost, st) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  return MQ_OK;
}

// ------------------------------------------------------------------------------------------------------
// mq_linear_static: mq_linear for callers that cannot allocate device memory (code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc).  The workspace of mq_linear (the stream-K kernel's counters, flags
// and partial tiles, the packed activations and their scales) lives in a file-scope device array of a fixed size
// instead of a caller buffer.  Every GPU that loads the library holds the array until the process exits.
namespace {

constexpr size_t STATIC_WS_BYTES = (size_t)16 << 20;   // 16 MiB
static __device__ __align__(256) uint8_t g_static_ws[STATIC_WS_BYTES];

// In host code `g_static_ws` is only the host-side stand-in of the symbol, not a device address: the address a kernel
// may use comes from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int STATIC_WS_MAX_DEVICES = 64;
void* g_static_ws_addr[STATIC_WS_MAX_DEVICES] = {};
std::mutex g_static_ws_mutex;

int static_ws_address(void** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  if (dev < 0 || dev >= STATIC_WS_MAX_DEVICES) return MQ_ERR_UNSUPPORTED_DEVICE;
  std::lock_guard<std::mutex> lock(g_static_ws_mutex);
  if (!g_static_ws_addr[dev]) {
    void* ptr = nullptr;
    if (cudaGetSymbolAddress((void**)&ptr, g_static_ws) != cudaSuccess || !ptr) {
      cudaGetLastError();
      return MQ_ERR_CUDA;
    }
    g_static_ws_addr[dev] = ptr;
  }
  *out = g_static_ws_addr[dev];
  return MQ_OK;
}

}  // namespace

extern "C" size_t mq_linear_static_max_bytes(void) { return STATIC_WS_BYTES; }

extern "C" int mq_linear_static(const mq_weights* w, const void* A, mq_dtype a_dtype, int64_t M, int64_t lda, void* Y,
                                mq_dtype y_dtype, int64_t ldy, void* cuda_stream) {
  if (!w) return MQ_ERR_INVALID_ARG;
  if (M == 0) return MQ_OK;
  if (M < 0) return MQ_ERR_UNSUPPORTED_SHAPE;
  int rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  // the layer and token count decide the size: beyond the array the call is refused, nothing is allocated instead
  if (mq_linear_workspace_bytes(w, M) > STATIC_WS_BYTES) return MQ_ERR_STATIC_SCRATCH;
  void* ws = nullptr;
  rc = static_ws_address(&ws);
  if (rc != MQ_OK) return rc;
  // The array keeps the previous call's contents.  What must start at zero (the workspace's 16 KB prefix: the stream-K
  // kernel's arrival counters, the fused quantizer's control block) is cleared on the stream before every call, so
  // that a call is correct even after one that was aborted half-way; the rest is written before it is read.
  if (cudaMemsetAsync(ws, 0, mq::WS_PREFIX, (cudaStream_t)cuda_stream) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  return mq_linear(w, A, a_dtype, M, lda, Y, y_dtype, ldy, ws, STATIC_WS_BYTES, cuda_stream);
}
