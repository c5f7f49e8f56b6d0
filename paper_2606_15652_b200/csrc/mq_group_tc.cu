// mq_group_tc.cu -- per-GROUP activation scales (reading A5g) on the tcgen05 tensor path, group = 128 channels:
//   Y[m,n] = sum_g s_a[m,g] (s_w[n] acc0_g[m,n] + s_r[n] acc1_g[m,n])          Eq.2, Eq.4 P:106 per group
// (first half).  A group of 128 channels is exactly one K-step of the packed layout, so the integer sum
// of a group is what ONE K-step's MMAs leave in the accumulator: the accumulator is drained after every K-step.
//
// Whole 128 x 128 tiles are dealt to persistent CTAs as in mq_prefill.cu, but the operands are the other way round: the
// TOKENS are the A operand (expanded int4 -> int8 x16 in registers -> tcgen05.st into TENSOR MEMORY, TMEM lane = token),
// the WEIGHTS are the B operand (expanded into K-major SWIZZLE_128B shared memory); tcgen05.mma kind::i8; residual
// cells are operand-ring items of their own (their weights in a B buffer, the K-step's tokens re-used from tensor
// memory).  So an accumulator lane is a token and a column a channel, and an epilogue thread owns ONE token:
// the group scale s_a[t, g], the factor that changes every K-step, is a register (one 4-byte load per thread and
// K-step), and the channel scales, which do not change, are applied once per tile.  (The first version had channels
// in the lanes: every thread then needed the 64 group scales of its tokens from shared memory in every K-step, 64 KB
// per K-step through the shared-memory pipe, plus a block-wide barrier per K-step to publish them.)
//   * three accumulator buffers of 128 columns are taken in rotation by base items (a K-step) and residual items (a
//     cell) alike, in the MMA warp's order: the MMAs of the next two items run while the epilogue warps read the sums of
//     the current one (tcgen05.ld), convert them and add them to fp32 running sums held in registers;
//   * the running sums are kept in units of s_w: y = sum_g s_a acc0_g + (s_a rho) acc1_g, rho = s_r / s_w, and
//     Y = (s_w / 256) y at the end of the tile (the operands are x16): two instructions per base sum (I2F, FFMA).  A tile
//     with a channel whose s_w is 0 (or whose ratio is not finite) keeps units of 1 instead (a third instruction);
//   * eight epilogue warps (two per TMEM lane quadrant, 64 channels each) keep 64 fp32 sums per thread for the whole
//     tile and store them as 128 contiguous bytes of the token's Y row.
// Tensor memory (512 columns): accumulators 3 x 128 | A operand ring 4 x 32.  Roles (16 warps = 512 threads in four
// warp groups; the block starts with 128 registers per thread and setmaxnreg moves 32 per thread from the other groups
// to the epilogue: 160 there (64 sums + two batches of 32 columns in flight), 96 elsewhere; one CTA per SM):
//   warp 0 producer (TMA) | warp 1 MMA issuer | warps 2-3 weight unpack (rows 0..63 -> shared memory) |
//   warps 4-11 epilogue | warps 12-15 token unpack (one per TMEM lane quadrant: a token row each -> tensor memory, plus
//   the weight rows 64..127 and the residual cells -> shared memory, so that all six unpack warps carry about the same).
// Arithmetic per output: fp32, groups in ascending order, one rounding to the 16-bit output at the end (tolerance T2 of
// DESIGN.md section 4).
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <type_traits>
#include <cstring>

#include "mq_internal.h"
#include "mq_ptx.cuh"

namespace {

using namespace mq;
using namespace mq::ptx;

constexpr int GT_BT = 128;                        // tokens per tile (MMA M: the tokens are the A operand, TMEM lane = token)
constexpr int GT_UST = 4;                         // operand (U) stages
constexpr int GT_EWARPS = 8;                      // epilogue warps: lane quadrant = warp % 4, channel half = (warp - GT_WARP_E0) / 4
constexpr int GT_WWARPS = 2;                      // weight-unpack warps (weight rows 0..63 -> shared memory)
constexpr int GT_TWARPS = 4;                      // token-unpack warps (one per TMEM lane quadrant; also weight rows 64..127 and the cells)
// warp groups of four (setmaxnreg acts on whole warp groups): {producer, MMA, weight unpack x 2} | epilogue | epilogue | token unpack
constexpr int GT_WARP_W0 = 2, GT_WARP_E0 = GT_WARP_W0 + GT_WWARPS, GT_WARP_T0 = GT_WARP_E0 + GT_EWARPS;
constexpr int GT_WARPS = GT_WARP_T0 + GT_TWARPS;
constexpr int GT_REGS_EPI = 160, GT_REGS_REST = 96;   // registers per thread after the split: 256 x 160 + 256 x 96 = 64 K
static_assert(GT_WARP_E0 == 4 && GT_WARP_T0 == 12 && GT_WARPS == 16, "roles fill whole warp groups");
constexpr int GT_THREADS = 32 * GT_WARPS;         // 512: the largest block that still gets 128 registers per thread
constexpr int GT_A_COLS = BK / 4;                 // 32 TMEM columns hold 128 int8 per lane (one K-step)
constexpr int GT_NACC = 3;                        // accumulator buffers of 128 columns, taken in rotation by base and residual items alike
constexpr int GT_A_COL0 = 3 * GT_BT;
constexpr int GT_PST = 8;                         // packed (P) stages of one K-step
constexpr int GT_U_STAGE = BN * BK;               // int8 weight sub-tile of one K-step (16 KB), the B operand
constexpr int GT_TOK_KSTEP = GT_BT * (BK / 2);    // packed tokens of one K-step (8 KB)
constexpr int GT_P_STAGE = TILE_BYTES + GT_TOK_KSTEP;
constexpr int GT_OFF_U = 0;
constexpr int GT_OFF_P = GT_OFF_U + GT_UST * GT_U_STAGE;
constexpr int GT_OFF_BAR = GT_OFF_P + GT_PST * GT_P_STAGE;
// barriers: FULL_P[8] EMPTY_P[8] FULL_U[4] EMPTY_U[4] GFULL[2] GEMPTY[2] A1E
constexpr int GT_B_FULL_P = 0, GT_B_EMPTY_P = GT_PST, GT_B_FULL_U = 2 * GT_PST, GT_B_EMPTY_U = GT_B_FULL_U + GT_UST,
              GT_B_GFULL = GT_B_EMPTY_U + GT_UST, GT_B_GEMPTY = GT_B_GFULL + GT_NACC, GT_NUM_BARS = GT_B_GEMPTY + GT_NACC;
constexpr int GT_OFF_MISC = GT_OFF_BAR + GT_NUM_BARS * 8 + 8;     // [0] tmem base
// per-tile channel constants, double-buffered by tile parity: [2]{[{fin, rho, bscale, s_r}][128] floats, flag word}
constexpr int GT_OFF_TC = (GT_OFF_MISC + 16 + 15) / 16 * 16;
constexpr int GT_TC_BYTES = 4 * BN * 4 + 16;
// output staging, private to an epilogue warp: [32 tokens][64 B of 16-bit outputs + 16 B pad] (half of a thread's 64
// channels at a time), so that global memory sees 64-byte row pieces from neighbouring lanes instead of 32 separate rows
constexpr int GT_YS_ROW = 80;
constexpr int GT_YS_WARP = 32 * GT_YS_ROW;
constexpr int GT_OFF_YS = (GT_OFF_TC + 2 * GT_TC_BYTES + 15) / 16 * 16;
constexpr int GT_SMEM_BYTES = GT_OFF_YS + GT_EWARPS * GT_YS_WARP + 1024;  // + slack for the 1024-byte alignment
static_assert(GT_SMEM_BYTES <= 232448, "shared memory budget");
static_assert(GT_A_COL0 + GT_UST * GT_A_COLS == 512, "tensor memory budget");
static_assert(GT_OFF_P % 1024 == 0 && GT_P_STAGE % 1024 == 0 && GT_U_STAGE % 1024 == 0, "swizzle atoms need 1024-byte alignment");

struct GtParams {
  const uint8_t* base;
  const uint8_t* res;
  const int2* unit_meta;   // [NT * KS] {quarter mask, first quarter}; NULL = dense only
  const float* sw;
  const float* sr;
  const float* sa;         // [M][KS] group scales
  void* Y;
  int32_t* dbg0;           // [KS][M][N] per-group base sums, or NULL
  int32_t* dbg1;           // [KS][M][N] per-group residual sums, or NULL
  int64_t ldy;
  int M, N, KS, NT, TT;
  int tiles;
  int y_bf16;
#ifdef GT_TRACE
  long long* trace;
#endif
};

__device__ __forceinline__ void gt_unpack16(const uint4& p, uint32_t* o) {
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
__device__ __forceinline__ uint4 gt_lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void gt_sts128(uint32_t addr, const uint32_t* v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory");
}
// wait for the outstanding tcgen05.ld's; the registers of the batches being waited for are tied to the statement so
// that no use of them can be scheduled above it (see mq_ptx.cuh)
__device__ __forceinline__ void gt_ld_wait32(uint32_t* a, uint32_t* b) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+r"(a[0]), "+r"(a[1]), "+r"(a[2]), "+r"(a[3]), "+r"(a[4]), "+r"(a[5]), "+r"(a[6]), "+r"(a[7]), "+r"(a[8]), "+r"(a[9]),
                 "+r"(a[10]), "+r"(a[11]), "+r"(a[12]), "+r"(a[13]), "+r"(a[14]), "+r"(a[15]), "+r"(b[0]), "+r"(b[1]), "+r"(b[2]),
                 "+r"(b[3]), "+r"(b[4]), "+r"(b[5]), "+r"(b[6]), "+r"(b[7]), "+r"(b[8]), "+r"(b[9]), "+r"(b[10]), "+r"(b[11]),
                 "+r"(b[12]), "+r"(b[13]), "+r"(b[14]), "+r"(b[15])
               :
               : "memory");
}

#ifdef GT_TRACE   // development: per-role wait-time sums of CTA 0 into p.trace (long long [64])
#define GT_T0() const long long gt_c0 = clock64()
#define GT_ACC(slot) do { gt_acc[(slot) & 1] += clock64() - gt_c0; } while (0)   // two register accumulators per role
#else
#define GT_T0() do { } while (0)
#define GT_ACC(slot) do { } while (0)
#endif

__device__ __forceinline__ void gt_tie16(uint32_t* a) {
  asm volatile(""
               : "+r"(a[0]), "+r"(a[1]), "+r"(a[2]), "+r"(a[3]), "+r"(a[4]), "+r"(a[5]), "+r"(a[6]), "+r"(a[7]), "+r"(a[8]), "+r"(a[9]),
                 "+r"(a[10]), "+r"(a[11]), "+r"(a[12]), "+r"(a[13]), "+r"(a[14]), "+r"(a[15]));
}

template <bool DBG>
__global__ void __launch_bounds__(GT_THREADS, 1) mq_group_tc_kernel(const __grid_constant__ CUtensorMap tmap_a, const GtParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sU = smem_base + GT_OFF_U, sP = smem_base + GT_OFF_P, sBar = smem_base + GT_OFF_BAR, sMisc = smem_base + GT_OFF_MISC,
                 sTC = smem_base + GT_OFF_TC;
  auto bar = [&](int i) { return sBar + 8u * (uint32_t)i; };
  volatile int32_t* misc = reinterpret_cast<volatile int32_t*>(smem_raw + (sMisc - smem_u32(smem_raw)));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int KS = p.KS;
  const int tile0 = (int)blockIdx.x, tstride = (int)gridDim.x;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmap_a);
    for (int i = 0; i < GT_PST; ++i) {
      mbar_init(bar(GT_B_FULL_P + i), 1);            // the producer's arrival; the copies complete the transaction count
      mbar_init(bar(GT_B_EMPTY_P + i), GT_WWARPS + GT_TWARPS);   // every unpack warp has its part in registers
    }
    for (int i = 0; i < GT_UST; ++i) {
      mbar_init(bar(GT_B_FULL_U + i), GT_WWARPS + GT_TWARPS);
      mbar_init(bar(GT_B_EMPTY_U + i), 1);
    }
    for (int i = 0; i < GT_NACC; ++i) {
      mbar_init(bar(GT_B_GFULL + i), 1);             // tcgen05.commit after the item's MMAs
      mbar_init(bar(GT_B_GEMPTY + i), GT_EWARPS);    // every epilogue warp has read its part of the buffer
    }
    fence_mbar_init();
    for (int i = 0; i < 2; ++i) asm volatile("st.shared.u32 [%0], %1;" ::"r"(sTC + (uint32_t)(i * GT_TC_BYTES + 4 * BN * 4)), "r"(0u) : "memory");
  }
  if (warp == 1) {
    tmem_alloc(sMisc, 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = (uint32_t)misc[0];
  griddep_launch();
  // The block is launched with 128 registers per thread (512 threads: the whole register file).  The epilogue warp groups
  // take 160 (64 running sums + two batches of 32 accumulator columns in flight), the other two give theirs up: the
  // first statement of every role (inside the role's branch, so that the compiler knows which budget holds where).
#define GT_REGS_DEC() asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(GT_REGS_REST))
#define GT_REGS_INC() asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(GT_REGS_EPI))
#ifdef GT_TRACE
  const long long gt_start = clock64();
  long long gt_acc[2] = {0, 0}, gt_drain = 0, gt_tile = 0, gt_m1 = 0, gt_m2 = 0, gt_m3 = 0;
#endif

  // residual metadata: every role that needs it keeps the {quarter mask, first quarter} words of 32 consecutive K-steps
  // in its lanes (one coalesced load per chunk, requested one chunk ahead) and derives the item sequence from them
  auto load_chunk = [&](int T, int c0) -> int2 {
    int2 v = make_int2(0, 0);
    if (p.unit_meta && T < p.tiles && c0 + lane < KS) v = __ldg(p.unit_meta + (size_t)(T / p.TT) * KS + c0 + lane);
    return v;
  };
  auto next_chunk = [&](int& T, int& c0) {
    c0 += 32;
    if (c0 >= KS) {
      c0 = 0;
      T += tstride;
    }
  };

  // the unpack role, instantiated for the token warps (warp group 3) and the weight warps (in warp group 0)
  auto unpack_role = [&](auto trole_c) {
    constexpr bool trole = decltype(trole_c)::value;
    // ============ unpack warps: int4 -> int8 (x16).  Token warps (12-15, one per TMEM lane quadrant): token row -> TENSOR
    // MEMORY (the A operand), plus their share of the weight rows (64..127) and the residual cells -> swizzled shared
    // memory (the B operand).  Weight warps (2-3): weight rows 0..63 -> swizzled shared memory. ============
    // All six walk all items in order; item i uses operand stage i % 4 (A columns and B buffer alike).  A stage is
    // complete when all six warps have arrived (for a residual item the weight warps have nothing to do, but arrive in
    // order all the same).
    const int wq = warp & 3;                            // TMEM lane quadrant of a token warp
    const uint32_t row = (uint32_t)(wq * 32 + lane);    // token warps: token inside the tile = TMEM lane; also the channel whose cell rows it expands
    const uint32_t wrow = trole ? 64u + (row & 63u) : (uint32_t)((warp - GT_WARP_W0) * 32 + lane);   // weight row this thread expands
    const uint32_t wc0 = trole ? 2u * (row >> 6) : 0u;  // ... and its first 16-byte chunk (token warps: two chunks, weight warps: all four)
    const uint32_t tsw = (row >> 1) & 3u;               // the token tile arrives with SWIZZLE_64B: chunk c of row r at ((c ^ (r >> 1 & 3)) << 4)
    const uint32_t lane_base = tmem_base + ((uint32_t)(wq * 32) << 16) + (uint32_t)GT_A_COL0;
    const int rhalf = (int)(row >> 6);
    uint32_t item = 0, q = 0;   // items / K-steps so far (the K-step counter names the P stage)
    auto wait_stage = [&](uint32_t idx) {   // operand stage idx % 4 has been consumed by the MMAs of item idx - 4
      GT_T0();
      mbar_wait_parked(bar(GT_B_EMPTY_U + (int)(idx & 3)), ((idx >> 2) & 1) ^ 1);
      GT_ACC(7);
      tc_fence_after();
    };
    auto publish = [&](uint32_t idx) {   // this warp's part of the item is in place: tell the MMA warp
      if (trole) tmem_st_wait();
      tc_fence_before();
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(GT_B_FULL_U + (int)(idx & 3)));
    };
    // 16 packed bytes (chunk c of weight row r) -> 32 int8 at the row's 16-byte columns 2c, 2c + 1 of the K-major
    // SWIZZLE_128B operand buffer
    auto expand_to_smem = [&](uint32_t su, uint32_t r, uint32_t c, const uint4& v) {
      uint32_t tw[8];
      gt_unpack16(v, tw);
      gt_sts128(su + r * 128 + (((2 * c) ^ (r & 7)) << 4), tw);
      gt_sts128(su + r * 128 + (((2 * c + 1) ^ (r & 7)) << 4), tw + 4);
    };
    int pT = tile0, pc0 = 0;
    int2 um_next = load_chunk(pT, pc0);
    for (int T = tile0; T < p.tiles; T += tstride) {
      for (int c0 = 0; c0 < KS; c0 += 32) {
        const int2 um = um_next;
        next_chunk(pT, pc0);
        um_next = load_chunk(pT, pc0);
        const uint32_t bits = __ballot_sync(0xffffffffu, (um.x & 0xF) != 0);
        const int nk = min(32, KS - c0);
        for (int j = 0; j < nk; ++j) {
          const uint32_t idx = item + (uint32_t)j + (uint32_t)__popc(bits & ((1u << j) - 1));   // item number of K-step j's base item
          const bool has = (bits >> j) & 1;
          const uint32_t ps = (q + (uint32_t)j) % GT_PST;
          {
            GT_T0();
            mbar_wait_parked(bar(GT_B_FULL_P + ps), ((q + (uint32_t)j) / GT_PST) & 1);
            GT_ACC(6);
          }
          const uint32_t pw = sP + ps * GT_P_STAGE, pt = pw + TILE_BYTES;
          const uint32_t su = sU + (idx & 3) * GT_U_STAGE;
          if (trole) {
            // ---- base item: one token row -> TMEM, two chunks of a weight row -> shared memory ----
            uint4 v4[4], w2[2];
#pragma unroll
            for (int c = 0; c < 4; ++c) v4[c] = gt_lds128(pt + row * 64 + (((uint32_t)c ^ tsw) << 4));
#pragma unroll
            for (int c = 0; c < 2; ++c) w2[c] = gt_lds128(pw + (wc0 + (uint32_t)c) * (BN * 16) + wrow * 16);
            // the packed stage is in registers: back to the producer (the arrival depends on every loaded word, see zero_after)
            const uint32_t landed = zero_after(fold4(v4[0]) ^ fold4(v4[1]) ^ fold4(v4[2]) ^ fold4(v4[3]) ^ fold4(w2[0]) ^ fold4(w2[1]));
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(GT_B_EMPTY_P + ps) + landed);
            wait_stage(idx);
            uint32_t o[32];
#pragma unroll
            for (int c = 0; c < 4; ++c) gt_unpack16(v4[c], o + 8 * c);
            tmem_st32(lane_base + (uint32_t)((idx & 3) * GT_A_COLS), o);
#pragma unroll
            for (int c = 0; c < 2; ++c) expand_to_smem(su, wrow, wc0 + (uint32_t)c, w2[c]);
            publish(idx);
            if (has) {
              // ---- residual item: the cell's packed rows straight from global memory -> the next stage's B buffer; this
              //      thread = channel `row`; a k-half that holds a block is written for all 128 channels (zeros where the
              //      other row half has no block), a k-half without any block is never read by the MMA ----
              const uint32_t rmask = (uint32_t)__shfl_sync(0xffffffffu, um.x, j) & 0xF;
              const uint32_t qoff = (uint32_t)__shfl_sync(0xffffffffu, um.y, j);
              uint4 r4[2][2];
#pragma unroll
              for (int h = 0; h < 2; ++h) {
                const int qq = 2 * h + rhalf;
                r4[h][0] = make_uint4(0, 0, 0, 0);
                r4[h][1] = make_uint4(0, 0, 0, 0);
                if (rmask & (1u << qq)) {
                  const uint8_t* src = p.res + ((size_t)qoff + (size_t)__popc(rmask & ((1u << qq) - 1))) * QUARTER_BYTES + (size_t)(row & 63) * 16;
                  r4[h][0] = __ldg(reinterpret_cast<const uint4*>(src));
                  r4[h][1] = __ldg(reinterpret_cast<const uint4*>(src + 1024));
                }
              }
              wait_stage(idx + 1);
              const uint32_t su2 = sU + ((idx + 1) & 3) * GT_U_STAGE;
#pragma unroll
              for (int h = 0; h < 2; ++h) {
                if (!(rmask & (3u << (2 * h)))) continue;
                expand_to_smem(su2, row, (uint32_t)(2 * h), r4[h][0]);
                expand_to_smem(su2, row, (uint32_t)(2 * h + 1), r4[h][1]);
              }
              publish(idx + 1);
            }
          } else {
            // ---- base item: one weight row (0..63), four chunks -> shared memory ----
            uint4 v4[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) v4[c] = gt_lds128(pw + c * (BN * 16) + wrow * 16);
            const uint32_t landed = zero_after(fold4(v4[0]) ^ fold4(v4[1]) ^ fold4(v4[2]) ^ fold4(v4[3]));
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(GT_B_EMPTY_P + ps) + landed);
            wait_stage(idx);
#pragma unroll
            for (int c = 0; c < 4; ++c) expand_to_smem(su, wrow, (uint32_t)c, v4[c]);
            publish(idx);
            if (has) {   // nothing to expand for a residual item: keep the stage's arrival count in step
              wait_stage(idx + 1);
              publish(idx + 1);
            }
          }
        }
        item += (uint32_t)nk + (uint32_t)__popc(nk == 32 ? bits : (bits & ((1u << nk) - 1)));
        q += (uint32_t)nk;
      }
    }
  };

  if (warp < GT_WARP_E0) {
    GT_REGS_DEC();   // one instruction for the whole warp group
    if (warp == 0) {
      if (lane == 0) {
        // ===================== producer (one thread): one K-step per stage =====================
        griddep_wait();   // the packed tokens are the previous kernel's output
        uint32_t q = 0;
        for (int T = tile0; T < p.tiles; T += tstride) {
          const int nt = T / p.TT, tt = T - nt * p.TT;
          const uint8_t* wsrc = p.base + (size_t)nt * KS * TILE_BYTES;
          for (int ks = 0; ks < KS; ++ks, ++q) {
            const uint32_t ps = q % GT_PST;
            mbar_wait_parked(bar(GT_B_EMPTY_P + ps), ((q / GT_PST) & 1) ^ 1);
            const uint32_t fb = bar(GT_B_FULL_P + ps), dst = sP + ps * GT_P_STAGE;
            mbar_arrive_expect_tx(fb, TILE_BYTES + GT_TOK_KSTEP);
            tma_load_1d(dst, wsrc + (size_t)ks * TILE_BYTES, TILE_BYTES, fb);
            tma_load_2d(dst + TILE_BYTES, &tmap_a, ks * (BK / 2), tt * GT_BT, fb);
          }
        }
      }
    } else if (warp == 1) {
      // ===================== MMA issuer: warp-uniform control, one elected lane issues =====================
      constexpr uint32_t IDESC = make_idesc_i8(GT_BT, BN);   // M = 128 tokens (A, tensor memory), N = 128 channels (B, shared memory)
      uint32_t item = 0, kq = 0;   // operand-ring items and K-steps so far
    uint32_t ab = 0, aph = 0;    // accumulator buffer of the next item (item % 3) and the parity of its use count
    auto next_acc = [&]() {
      if (++ab == GT_NACC) {
        ab = 0;
        aph ^= 1;
      }
    };
      bool pre_ok = false;                 // the barrier of the item about to be processed was already seen complete
      // the operand stage of item i: FULL_U[i & 3], phase (i >> 2) & 1; the next item's barrier is polled once BEFORE this
      // item's MMAs are issued, so that the round trip hides under the tensor pipe's work
      auto acquire = [&]() {
        if (!pre_ok) {
          GT_T0();
          mbar_wait_parked(bar(GT_B_FULL_U + (int)(item & 3)), (item >> 2) & 1);
          GT_ACC(0);
        }
        tc_fence_after();
        pre_ok = mbar_try_wait(bar(GT_B_FULL_U + (int)((item + 1) & 3)), ((item + 1) >> 2) & 1);
      };
      int pT = tile0, pc0 = 0;
      int2 um_next = load_chunk(pT, pc0);
      for (int T = tile0; T < p.tiles; T += tstride) {
        for (int c0 = 0; c0 < KS; c0 += 32) {
          const int2 um = um_next;
          next_chunk(pT, pc0);
          um_next = load_chunk(pT, pc0);
          const uint32_t bits = __ballot_sync(0xffffffffu, (um.x & 0xF) != 0);
          const int nk = min(32, KS - c0);
          for (int j = 0; j < nk; ++j, ++kq) {
            const bool has = (bits >> j) & 1;
            const int us = (int)(item & 3);
            acquire();
            {
              GT_T0();
              mbar_wait(bar(GT_B_GEMPTY + (int)ab), aph ^ 1);   // the epilogue has read the sums this buffer held three items ago
              GT_ACC(1);
            }
            tc_fence_after();
            const uint32_t d0 = tmem_base + ab * (uint32_t)BN;
            const uint32_t at = tmem_base + (uint32_t)(GT_A_COL0 + us * GT_A_COLS);
            const uint64_t dt = make_desc_sw128(sU + us * GT_U_STAGE);
            if (elect_one()) {
  #pragma unroll
              for (int k = 0; k < 4; ++k) mma_i8_ts(d0, at + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), IDESC, k == 0 ? 0u : 1u);   // a fresh sum per group
              if (!has) tc_commit(bar(GT_B_EMPTY_U + us));
              tc_commit(bar(GT_B_GFULL + (int)ab));
            }
            __syncwarp();
            ++item;
            next_acc();
            if (has) {
              // residual cell of this K-step: its weights in the next stage's B buffer, the tokens of this K-step's
              // stage (the paper's re-use of the activation tile), second accumulator, also a fresh sum
              const uint32_t mask = (uint32_t)__shfl_sync(0xffffffffu, um.x, j) & 0xF;
              const int us2 = (int)(item & 3);
              acquire();
              mbar_wait(bar(GT_B_GEMPTY + (int)ab), aph ^ 1);
              tc_fence_after();
              const uint32_t d1 = tmem_base + ab * (uint32_t)BN;
              const uint64_t dt2 = make_desc_sw128(sU + us2 * GT_U_STAGE);
              if (elect_one()) {
                uint32_t on = 0;
  #pragma unroll
                for (int h = 0; h < 2; ++h)
                  if (mask & (3u << (2 * h))) {
  #pragma unroll
                    for (int k = 2 * h; k < 2 * h + 2; ++k) {
                      mma_i8_ts(d1, at + (uint32_t)(k * 8), dt2 + (uint64_t)(k * 2), IDESC, on);
                      on = 1;
                    }
                  }
                tc_commit(bar(GT_B_EMPTY_U + us2));
                tc_commit(bar(GT_B_EMPTY_U + us));
                tc_commit(bar(GT_B_GFULL + (int)ab));
              }
              __syncwarp();
              ++item;
              next_acc();
            }
          }
        }
      }
    } else {
      unpack_role(std::false_type{});   // weight warps
    }
  } else if (warp >= GT_WARP_T0) {
    GT_REGS_DEC();
    unpack_role(std::true_type{});      // token warps
  }
  else {
    // ===================== epilogue warps (4..11): drain every K-step's sums into fp32 running sums =====================
    // A thread owns ONE token (its TMEM lane) and 64 channels (columns): the group scale s_a[t, g] is a register, the
    // channel scales are applied once per tile.  Register budget (160 per thread after the split): 64 running sums + two
    // batches of 32 + two dozen scalars; which K-steps own a cell comes from the metadata words kept in the lanes.
    GT_REGS_INC();
    griddep_wait();   // the group scales and Y are ordered after the previous kernel in the stream
    const int half = (warp - GT_WARP_E0) >> 2;        // which 64 channels of the tile; TMEM lane quadrant = warp % 4
    const int et = (warp - GT_WARP_E0) * 32 + lane;   // 0..255 within the epilogue group
    const int trow = (warp & 3) * 32 + lane;          // this thread's token inside the tile
    // Values the K-step loop uses again and again are made opaque to the compiler (an empty asm that "modifies" them):
    // otherwise it re-derives them from %tid and the shared-memory window at every use (special-register reads, shifts,
    // uniform-register moves: a third of the loop's time went there) instead of keeping six registers.
    uint32_t acc0_addr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(half * 64);
    uint32_t b_gfull = bar(GT_B_GFULL), b_gempty = bar(GT_B_GEMPTY);
    uint32_t lane0 = lane == 0 ? 1u : 0u;
    asm volatile("" : "+r"(acc0_addr), "+r"(b_gfull), "+r"(b_gempty), "+r"(lane0));
    float y[64];
#pragma unroll
    for (int i = 0; i < 64; ++i) y[i] = 0.f;
    // group scales s_a[t, g] of this thread's token: one scalar per K-step, requested one K-step ahead
    // (a pointer advanced by one per K-step and recomputed once per tile: no integer division in the K-step loop)
    int fT = tile0, fks = 0;     // the K-step the next request is for
    // &s_a[token of this thread in tile fT][0].  Always a valid row: a token past M (ragged last tile; its accumulator
    // rows are zero and it is never stored) reads the last row, requests past the last tile re-read the last one
    const float* fp = p.sa;
    auto gather_tile = [&]() {
      if (fT < p.tiles) fp = p.sa + (size_t)min((fT % p.TT) * GT_BT + trow, p.M - 1) * KS;
    };
    gather_tile();
    auto gather_into = [&](float& v) {
      // (asm volatile: the request must be ISSUED here, ahead of its use; a plain __ldg may be sunk to the use)
      asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(fp + fks));
      if (++fks == KS) {
        fks = 0;
        fT += tstride;
        gather_tile();
      }
    };
    auto gather = [&]() -> float {
      float v;
      gather_into(v);
      return v;
    };
    float sa_nxt = gather();   // K-step 0
    // which K-steps own a cell: the metadata words of 32 consecutive K-steps in the lanes, as in the other roles
    int pT = tile0, pc0 = 0;
    int2 um_next = load_chunk(pT, pc0);
    uint32_t kq = 0, tile_no = 0;
    // The sums leave tensor memory in batches of 32 channels (two tcgen05.ld of 16 columns), two register buffers: while
    // one batch is scaled and added the next one is in flight -- across passes and K-steps too: the first batch of the
    // NEXT pass (the residual sums of this K-step, or the base sums of the tile's next K-step, whose MMAs finished long
    // ago) is requested before the arithmetic of this pass's last batch.  tcgen05.wait::ld waits for every outstanding
    // load of the thread, so there is exactly one batch outstanding at every wait.
    uint32_t a[2][32];
    auto issue = [&](uint32_t col, uint32_t* dst) {
      tmem_ld16(acc0_addr + col, dst);
      tmem_ld16(acc0_addr + col + 16u, dst + 16);
    };
    auto landed = [&](uint32_t* v) { gt_ld_wait32(v, v + 16); };
    // (an empty statement that "modifies" a batch: the arithmetic on it cannot be scheduled above it, hence not above the
    // loads just issued; otherwise the compiler sinks the loads below the arithmetic and every batch pays the full
    // tensor-memory latency)
    auto tie = [&](uint32_t* v) {
      gt_tie16(v);
      gt_tie16(v + 16);
    };
    // accumulator buffer of the item being drained (base and residual items take the three buffers in rotation, in the
    // MMA warp's order) and the parity of its use count
    uint32_t eb = 0, eph = 0;
    auto request_item = [&]() {   // first batch of the item in buffer eb -> a[0]
      GT_T0();
      mbar_wait(b_gfull + 8u * eb, eph);
      GT_ACC(3);
      tc_fence_after();
      issue(eb * (uint32_t)BN, a[0]);
    };
    // the channel scales of a tile are requested one tile ahead (threads 0..127 of the epilogue group: one channel each)
    float sw_nx = 0.f, sr_nx = 0.f;
    auto request_scales = [&](int Tn) {
      if (et < BN && Tn < p.tiles) {
        const int nn = (Tn / p.TT) * BN + et;
        asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(sw_nx) : "l"(p.sw + nn));
        asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(sr_nx) : "l"(p.sr + nn));
      }
    };
    request_scales(tile0);
    for (int T = tile0; T < p.tiles; T += tstride, ++tile_no) {
      const int n0 = (T / p.TT) * BN;
      // Per-tile channel constants in shared memory (double-buffered by tile parity, one barrier per tile).  The running
      // sums are kept in units of s_w: y = sum_g s_a acc0_g + (s_a rho) acc1_g with rho = s_r / s_w, times fin = s_w / 256
      // at the end: two instructions per base sum (I2F, FFMA).  A tile that holds a channel with s_w = 0 (or a ratio that
      // is not finite) keeps its sums in units of 1 and pays a third instruction (bscale = s_w, rho = s_r, fin = 1/256).
      const uint32_t tc = sTC + (tile_no & 1u) * (uint32_t)GT_TC_BYTES;
      const float sw_raw = sw_nx, sr_raw = sr_nx;
      request_scales(T + tstride);
      if (et < BN) {
        const float ratio = __fdiv_rn(sr_raw, sw_raw);
        const bool odd = sw_raw == 0.f || !(fabsf(ratio) <= 3.0e38f);
        asm volatile("st.shared.f32 [%0], %1;" ::"r"(tc + 4u * (uint32_t)et), "f"(sw_raw * 0.00390625f) : "memory");          // fin (regular tile)
        asm volatile("st.shared.f32 [%0], %1;" ::"r"(tc + 4u * (uint32_t)(BN + et)), "f"(odd ? 0.f : ratio) : "memory");      // rho (regular tile)
        asm volatile("st.shared.f32 [%0], %1;" ::"r"(tc + 4u * (uint32_t)(2 * BN + et)), "f"(sw_raw) : "memory");             // bscale (irregular tile)
        asm volatile("st.shared.f32 [%0], %1;" ::"r"(tc + 4u * (uint32_t)(3 * BN + et)), "f"(sr_raw) : "memory");             // rho (irregular tile)
        // [4 * BN]: the number (+ 1) of the last irregular tile that used this buffer, written by any thread that sees an
        // odd channel (zero at kernel start; never cleared: a stale number does not match)
        if (odd) asm volatile("st.shared.u32 [%0], %1;" ::"r"(tc + 4u * (uint32_t)(4 * BN)), "r"(tile_no + 1u) : "memory");
      }
      named_bar_sync(1, 32 * GT_EWARPS);   // the constants of this tile are visible; everybody has left tile T - 2 * stride
      uint32_t flag;
      asm volatile("ld.shared.u32 %0, [%1];" : "=r"(flag) : "r"(tc + 4u * (uint32_t)(4 * BN)));
      const bool slow = flag == tile_no + 1u;
      const uint32_t tc_half = tc + (uint32_t)(half * 64 * 4);
      request_item();   // (no load is left in flight across the tile's output stage)
      // (the K-step loops once per kind of tile, regular / irregular channel scales: no test per K-step)
      auto k_loops = [&](auto slow_c) {
      constexpr bool SLOW = decltype(slow_c)::value;
      for (int c0 = 0; c0 < KS; c0 += 32) {
        const int2 um = um_next;
        next_chunk(pT, pc0);
        um_next = load_chunk(pT, pc0);
        const uint32_t bits = __ballot_sync(0xffffffffu, (um.x & 0xF) != 0);
        const int nk = min(32, KS - c0);
      for (int j = 0; j < nk; ++j, ++kq) {
        const int ks = c0 + j;
        const bool has = (bits >> j) & 1;
        // s_a[this token, this K-step's group], requested one K-step ago; the next one is requested now, into the same
        // register (nothing may touch that register before the next K-step: a copy right behind the load would wait for it)
        const float sa = sa_nxt;
        gather_into(sa_nxt);
#ifdef GT_TRACE
        const long long gt_d0 = clock64();
#endif
        // y += s_a * sum (base, regular tile) | s_a * (bscale * sum) (base, irregular tile) | (s_a * rho) * sum (residual)
        auto add32 = [&](const uint32_t* v, int b, auto mode_c, int32_t* dbg) {
          constexpr int MODE = decltype(mode_c)::value;
#pragma unroll
          for (int i4 = 0; i4 < 8; ++i4) {
            float cs[4] = {0.f, 0.f, 0.f, 0.f};
            if (MODE != 0) {
              const uint4 c4 = gt_lds128(tc_half + (uint32_t)(((MODE == 1 ? 2 : (SLOW ? 3 : 1)) * BN) * 4) + (uint32_t)((b * 32 + i4 * 4) * 4));
              cs[0] = __uint_as_float(c4.x);
              cs[1] = __uint_as_float(c4.y);
              cs[2] = __uint_as_float(c4.z);
              cs[3] = __uint_as_float(c4.w);
            }
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
              const int i = 4 * i4 + ii;
              const float f = (float)(int32_t)v[i];
              if (MODE == 0) y[b * 32 + i] = fmaf(sa, f, y[b * 32 + i]);
              if (MODE == 1) y[b * 32 + i] = fmaf(sa, cs[ii] * f, y[b * 32 + i]);
              if (MODE == 2) y[b * 32 + i] = fmaf(sa * cs[ii], f, y[b * 32 + i]);
            }
          }
          if (DBG && dbg) {   // parity hooks: the per-group integer sums
            const int t = (T % p.TT) * GT_BT + trow;
            if (t < p.M) {
#pragma unroll
              for (int i = 0; i < 32; ++i) dbg[((size_t)ks * p.M + (size_t)t) * p.N + n0 + half * 64 + b * 32 + i] = (int32_t)v[i] >> 8;
            }
          }
        };
        auto hand_back = [&]() {   // this warp's part of the item's sums is in registers: the buffer goes back to the MMA warp
          tc_fence_before();
          __syncwarp();
          if (lane0) mbar_arrive(b_gempty + 8u * eb);
          if (++eb == GT_NACC) {
            eb = 0;
            eph ^= 1;
          }
        };
        // ---- base sums (a[0] was requested during the previous pass) ----
        landed(a[0]);
        issue(eb * (uint32_t)BN + 32u, a[1]);
        tie(a[0]);
        add32(a[0], 0, std::integral_constant<int, SLOW ? 1 : 0>{}, p.dbg0);
        landed(a[1]);
        hand_back();
        if (has || ks + 1 < KS) request_item();   // the K-step's residual item, or the next K-step's base item
        tie(a[1]);
        add32(a[1], 1, std::integral_constant<int, SLOW ? 1 : 0>{}, p.dbg0);
        // ---- residual sums of a K-step that owns a cell (a pass of its own: inside the base pass the compiler if-converts
        //      the cell test and EVERY element pays for it) ----
        if (has) {
          landed(a[0]);
          issue(eb * (uint32_t)BN + 32u, a[1]);
          tie(a[0]);
          add32(a[0], 0, std::integral_constant<int, 2>{}, p.dbg1);
          landed(a[1]);
          hand_back();
          if (ks + 1 < KS) request_item();
          tie(a[1]);
          add32(a[1], 1, std::integral_constant<int, 2>{}, p.dbg1);
        } else if (DBG && p.dbg1) {
          const int t = (T % p.TT) * GT_BT + trow;
          if (t < p.M) {
#pragma unroll 1
            for (int i = 0; i < 64; ++i) p.dbg1[((size_t)ks * p.M + (size_t)t) * p.N + n0 + half * 64 + i] = 0;
          }
        }
#ifdef GT_TRACE
        gt_drain += clock64() - gt_d0;
#endif
      }
      }
      };
      if (slow) k_loops(std::true_type{}); else k_loops(std::false_type{});
      // the tile's sums are complete: times the channel constant, one rounding to the 16-bit output.  A thread owns 64
      // consecutive channels of one token (128 contiguous bytes of Y).  32 channels at a time go through the warp's
      // staging rows, so that a store instruction writes 64-byte pieces of 8 rows (4 neighbouring lanes per row) instead
      // of 16 bytes of 32 rows; rows that are not 16-byte aligned take the direct 2-byte path
      {
#ifdef GT_TRACE
        const long long gt_t0 = clock64();
#endif
        const int t_w0 = (T % p.TT) * GT_BT + (warp & 3) * 32;   // first token of this warp
        const bool vec = ((p.ldy & 7) == 0) && ((reinterpret_cast<uintptr_t>(p.Y) & 15) == 0);   // rows 16-byte aligned
        const uint32_t ys = smem_base + (uint32_t)GT_OFF_YS + (uint32_t)((warp - GT_WARP_E0) * GT_YS_WARP);
        auto tile_out = [&](auto bf_c) {
          constexpr bool BF = decltype(bf_c)::value;
#pragma unroll
          for (int h = 0; h < 2; ++h) {   // channels 32 h .. 32 h + 31 of this thread's 64
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              uint32_t w4[4];
#pragma unroll
              for (int h4 = 0; h4 < 2; ++h4) {
                const int i0 = 32 * h + 8 * k + 4 * h4;
                float fin[4] = {0.00390625f, 0.00390625f, 0.00390625f, 0.00390625f};
                if (!slow) {
                  const uint4 c4 = gt_lds128(tc_half + (uint32_t)(i0 * 4));   // fin of four channels
                  fin[0] = __uint_as_float(c4.x);
                  fin[1] = __uint_as_float(c4.y);
                  fin[2] = __uint_as_float(c4.z);
                  fin[3] = __uint_as_float(c4.w);
                }
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const int i = i0 + 2 * e;
                  const float v0 = y[i] * fin[2 * e], v1 = y[i + 1] * fin[2 * e + 1];
                  if (BF) {   // one rounding each (round to nearest even), packed {v0 low, v1 high}
                    const __nv_bfloat162 pk = __floats2bfloat162_rn(v0, v1);
                    w4[h4 * 2 + e] = *reinterpret_cast<const uint32_t*>(&pk);
                  } else {
                    const __half2 pk = __floats2half2_rn(v0, v1);
                    w4[h4 * 2 + e] = *reinterpret_cast<const uint32_t*>(&pk);
                  }
                  y[i] = 0.f;
                  y[i + 1] = 0.f;
                }
              }
              if (vec) {
                gt_sts128(ys + (uint32_t)(lane * GT_YS_ROW + k * 16), w4);
              } else if (t_w0 + lane < p.M) {
                uint16_t* dst = reinterpret_cast<uint16_t*>(p.Y) + (size_t)(t_w0 + lane) * p.ldy + n0 + half * 64 + 32 * h + 8 * k;
#pragma unroll
                for (int q2 = 0; q2 < 4; ++q2) {
                  dst[2 * q2] = (uint16_t)(w4[q2] & 0xFFFF);
                  dst[2 * q2 + 1] = (uint16_t)(w4[q2] >> 16);
                }
              }
            }
            if (vec) {
              __syncwarp();
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                const int r = (lane >> 2) + 8 * i, c = lane & 3;   // row r of the warp's 32 tokens, 16-byte piece c of its 64 bytes
                const uint4 v = gt_lds128(ys + (uint32_t)(r * GT_YS_ROW + c * 16));
                if (t_w0 + r < p.M)
                  *reinterpret_cast<uint4*>(reinterpret_cast<uint8_t*>(p.Y) + ((size_t)(t_w0 + r) * p.ldy + n0 + half * 64 + 32 * h + 8 * c) * 2) = v;
              }
              __syncwarp();
            }
          }
        };
        if (p.y_bf16) tile_out(std::true_type{}); else tile_out(std::false_type{});
#ifdef GT_TRACE
        gt_tile += clock64() - gt_t0;
#endif
      }
    }
  }


#ifdef GT_TRACE
  if (blockIdx.x == 0 && lane == 0 && (warp == 1 || warp == GT_WARP_E0 || warp == GT_WARP_W0 || warp == GT_WARP_T0)) {
    p.trace[32 + warp] = clock64() - gt_start;
    const int base = warp == 1 ? 0 : (warp == GT_WARP_E0 ? 2 : (warp == GT_WARP_W0 ? 6 : 8));
    p.trace[base] = gt_acc[0];
    p.trace[base + 1] = gt_acc[1];
    if (warp == GT_WARP_E0) { p.trace[4] = gt_drain; p.trace[5] = gt_tile; p.trace[20] = gt_m1; p.trace[21] = gt_m2; p.trace[22] = gt_m3; }
  }
#endif
  // teardown (single-lane regions re-converge first: bar.sync must be reached warp-convergent)
  __syncwarp();
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

}  // namespace

namespace mq {

// group = 128 only (one group per K-step); small token counts stay on the mma.sync kernel (mq_group.cu)
bool group_tc_eligible(const mq_weights* w, int group, int64_t M) {
  const Options& o = options();
  return w && !w->blockscale && group == 128 && M >= 64 && o.group_tc != 0 && o.group_simt == 0;
}

int group_tc_gemm(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                  int32_t* dbg0, int32_t* dbg1, void* cuda_stream) {
  typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  EncodeTiledFn enc = (EncodeTiledFn)tensor_map_encode_fn();
  if (!enc) return MQ_ERR_CUDA;
  // 2-D tensor map over the canonical packed activations [M rows][K/2 bytes]: box = one K-step of one token tile
  // (128 rows of 64 bytes, 16-byte chunks XOR-swizzled by (row >> 1) & 3 so that a thread per row reads without bank
  // conflicts); rows past M read as zero
  CUtensorMap tmap;
  memset(&tmap, 0, sizeof(tmap));
  const cuuint64_t row_bytes = (cuuint64_t)(w->K / 2);
  const cuuint64_t gdim[2] = {row_bytes, (cuuint64_t)M};
  const cuuint64_t gstride[1] = {row_bytes};
  const cuuint32_t box[2] = {(cuuint32_t)(BK / 2), (cuuint32_t)GT_BT};
  const cuuint32_t estr[2] = {1, 1};
  if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(qA), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
          CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return MQ_ERR_CUDA;

  GtParams gp;
  gp.base = w->d_base;
  gp.res = w->d_res;
  gp.unit_meta = w->nnz > 0 ? (const int2*)w->d_unit_meta : nullptr;
  gp.sw = w->d_sw;
  gp.sr = w->d_sr;
  gp.sa = sA;
  gp.Y = Y;
  gp.dbg0 = dbg0;
  gp.dbg1 = dbg1;
  gp.ldy = ldy;
  gp.M = (int)M;
  gp.N = (int)w->N;
  gp.KS = (int)(w->K / BK);
  gp.NT = (int)(w->N / BN);
  gp.TT = (int)((M + GT_BT - 1) / GT_BT);
  const int64_t tiles = (int64_t)gp.NT * gp.TT;
  if (tiles >= ((int64_t)1 << 31) || M >= ((int64_t)1 << 31)) return MQ_ERR_UNSUPPORTED_SHAPE;
  gp.tiles = (int)tiles;
  gp.y_bf16 = y_dtype == MQ_BF16;
#ifdef GT_TRACE
  gp.trace = (long long*)dbg1;
  gp.dbg1 = nullptr;
  dbg1 = nullptr;
#endif

  const bool dbg = dbg0 || dbg1;   // the parity hooks are a separate instantiation
  auto kern = dbg ? mq_group_tc_kernel<true> : mq_group_tc_kernel<false>;
  static int attr_dev[2] = {-1, -1};   // the attribute belongs to the (device, function) pair
  int dev = -1;
  cudaGetDevice(&dev);
  if (dev != attr_dev[dbg]) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, GT_SMEM_BYTES) != cudaSuccess) {
      cudaGetLastError();
      return MQ_ERR_CUDA;
    }
    attr_dev[dbg] = dev;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)std::min<int64_t>(tiles, sm_count()));
  cfg.blockDim = dim3(GT_THREADS);
  cfg.dynamicSmemBytes = GT_SMEM_BYTES;
  cfg.stream = (cudaStream_t)cuda_stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = options().pdl ? 1 : 0;
  if (cudaLaunchKernelEx(&cfg, kern, tmap, gp) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  set_launch_count(1);
  return MQ_OK;
}

}  // namespace mq
