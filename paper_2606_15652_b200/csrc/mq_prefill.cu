// mq_prefill.cu -- the fused base + residual int4 GEMM for PREFILL shapes (M > 32 tokens, many whole tiles):
// Eq.4, ZipperEngine on the tensor-bound side of the roofline.
//
// Same arithmetic and the same building blocks as mq_gemm.cu (weights expanded int4 -> int8 x16 in registers and
// written to TENSOR MEMORY as the MMA's A operand, tokens expanded into K-major SWIZZLE_128B shared memory as its B
// operand, tcgen05.mma kind::i8, base and residual accumulators in TMEM, fp32 epilogue), re-cut around what this
// round's measurements showed (profiles/r2_probe_int8.md):
//   * the tensor pipe sustains 95 % of peak on 128 x 128 x 32 instructions if it is fed, but its queue is shallow:
//     every instruction the issuing warp executes between two MMAs is pipe idle time;
//   * a single-thread role pays ~7 cycles per instruction, so the TMA producer's loop must be a handful of
//     instructions per stage (in mq_gemm.cu it computes all residual bookkeeping: ~150 instructions per two K-steps,
//     and the unpack groups wait for it a quarter of the time);
//   * the base accumulator must be double-buffered (the MMA warp waited 15 % of the time for the epilogue).
// Tensor memory (512 columns): acc0 2 x 128 | acc1 128 | A operand ring 4 x 32.  There is no room left for a residual
// operand, so a residual cell is an ITEM OF ITS OWN in the operand ring: right after the base item of its K-step, its
// expanded weights take the next A stage and its MMAs re-use the token tile of the base item (the paper's re-use of the
// quantized activation tile), accumulating into acc1 (s_r != s_w).
//
// Work: whole output tiles (128 output channels x 128 tokens), tile T = nt * TT + tt, dealt round-robin to the
// persistent CTAs (concurrent CTAs share n-tiles: the weights stay in L2).  Roles (22 warps, one CTA per SM):
//   warp 0      producer (one thread): per P stage = two K-steps: one bulk copy of 16 KB packed weights, two tensor
//               copies of packed tokens [128 x 64 B], the two K-steps' residual metadata (prefetched one stage ahead)
//   warps 6-21  four unpack groups of four warps; items (base K-step, or residual cell) are dealt to them in rotation.
//               Base item: packed weights -> int8 x16 -> tcgen05.st; packed tokens -> int8 x16 -> swizzled smem.
//               Residual item: the cell's packed quarters straight from global memory (rare: ~6 % of the K-steps).
//   warp 1      MMA issuer: per item one barrier wait, one elected block, one commit
//   warps 2-5   epilogue: tcgen05.ld, y = s_a (s_w acc0 + s_r acc1), 16-bit stores; overlaps the next tile's K-loop
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <type_traits>

#include "mq_internal.h"
#include "mq_ptx.cuh"

namespace {

using namespace mq;
using namespace mq::ptx;

constexpr int PF_BT = 128;                       // tokens per tile (MMA N)
constexpr int PF_UST = 4;                        // operand (U) stages = unpack groups
constexpr int PF_PST = 8;                        // packed (P) stages of one K-step
constexpr int PF_WARPS = 6 + 4 * PF_UST;
constexpr int PF_THREADS = 32 * PF_WARPS;
constexpr int PF_A_COLS = BK / 4;                // 32 TMEM columns hold 128 int8 per lane (one K-step)
constexpr int PF_ACC1_COL = 2 * PF_BT;
constexpr int PF_A_COL0 = 3 * PF_BT;
constexpr int PF_U_STAGE = PF_BT * BK;           // int8 token sub-tile of one K-step (16 KB)
constexpr int PF_TOK_KSTEP = PF_BT * (BK / 2);   // packed tokens of one K-step (8 KB)
constexpr int PF_P_STAGE = TILE_BYTES + PF_TOK_KSTEP;           // 16 KB: packed weights | packed tokens
constexpr int PF_OFF_U = 0;
constexpr int PF_OFF_P = PF_OFF_U + PF_UST * PF_U_STAGE;
constexpr int PF_OFF_BAR = PF_OFF_P + PF_PST * PF_P_STAGE;
// barriers: FULL_P[8] EMPTY_P[8] FULL_U[4] EMPTY_U[4] TFULL[2] A0E[2] A1E
constexpr int PF_B_FULL_P = 0, PF_B_EMPTY_P = PF_PST, PF_B_FULL_U = 2 * PF_PST, PF_B_EMPTY_U = PF_B_FULL_U + PF_UST,
              PF_B_TFULL = PF_B_EMPTY_U + PF_UST, PF_B_A0E = PF_B_TFULL + 2, PF_B_A1E = PF_B_A0E + 2, PF_NUM_BARS = PF_B_A1E + 1;
constexpr int PF_OFF_MISC = PF_OFF_BAR + PF_NUM_BARS * 8 + 8;    // [0] tmem base, [1..2] residual flag of the acc0 buffer
constexpr int PF_OFF_SA = (PF_OFF_MISC + 16 + 15) / 16 * 16;     // [2][128] token scales of the tile being drained
constexpr int PF_SMEM_BYTES = PF_OFF_SA + 2 * PF_BT * 4 + 1024;  // + slack for the 1024-byte alignment
static_assert(PF_SMEM_BYTES <= 232448, "shared memory budget");
static_assert(PF_A_COL0 + PF_UST * PF_A_COLS == 512, "tensor memory budget");

struct PfParams {
  const uint8_t* base;
  const uint8_t* res;
  const int2* unit_meta;   // [NT * KS] {quarter mask, first quarter}; NULL = dense only
  const float* sw;
  const float* sr;
  const float* sa;
  void* Y;
  int32_t* dbg0;
  int32_t* dbg1;
  int64_t ldy;
  int M, N, KS, NT, TT;
  int tiles;
  int y_bf16;
};

__device__ __forceinline__ void pf_unpack16(const uint4& p, uint32_t* o) {
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
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ uint4 pf_lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void pf_sts128(uint32_t addr, const uint32_t* v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory");
}
__device__ __forceinline__ uint32_t pf_lds32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void pf_sts32(uint32_t addr, uint32_t v) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

#ifndef PF_EXP_NOW   // development experiments (timing only, wrong results): skip parts of the unpack
#define PF_EXP_NOW 0
#endif
#ifndef PF_EXP_NOT
#define PF_EXP_NOT 0
#endif
#ifndef PF_EXP_NOS
#define PF_EXP_NOS 0
#endif
#ifdef PF_TRACE   // development: clock stamps of CTA 0 into the dbg1 buffer (8 words per tile)
#define PF_STAMP(cond, it, slot) do { if (blockIdx.x == 0 && (cond)) reinterpret_cast<long long*>(p.dbg1)[(it) * 8 + (slot)] = clock64(); } while (0)
#define PF_ADD(cond, it, slot, v) do { if (blockIdx.x == 0 && (cond)) reinterpret_cast<long long*>(p.dbg1)[(it) * 8 + (slot)] += (v); } while (0)
#define PF_FINE(slot) do { if (blockIdx.x == 0 && warp == 6 && lane == 0 && it == 5) reinterpret_cast<long long*>(p.dbg1)[4096 + (n_mine & 127) * 8 + (slot)] = clock64(); } while (0)
#else
#define PF_FINE(slot) do { } while (0)
#define PF_STAMP(cond, it, slot) do { } while (0)
#define PF_ADD(cond, it, slot, v) do { } while (0)
#endif

__global__ void __launch_bounds__(PF_THREADS, 1) mq_prefill_kernel(const __grid_constant__ CUtensorMap tmap_a, const PfParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sU = smem_base + PF_OFF_U, sP = smem_base + PF_OFF_P, sBar = smem_base + PF_OFF_BAR,
                 sMisc = smem_base + PF_OFF_MISC;
  auto bar = [&](int i) { return sBar + 8u * (uint32_t)i; };
  volatile int32_t* misc = reinterpret_cast<volatile int32_t*>(smem_raw + (sMisc - smem_u32(smem_raw)));
  float* sa_tile = reinterpret_cast<float*>(smem_raw + (smem_base + PF_OFF_SA - smem_u32(smem_raw)));   // [2][128]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int KS = p.KS;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmap_a);
    for (int i = 0; i < PF_PST; ++i) {
      mbar_init(bar(PF_B_FULL_P + i), 1);            // the producer's arrival; the copies complete the transaction count
      mbar_init(bar(PF_B_EMPTY_P + i), 4);           // the four warps of the group that owns the K-step
    }
    for (int i = 0; i < PF_UST; ++i) {
      mbar_init(bar(PF_B_FULL_U + i), 4);
      mbar_init(bar(PF_B_EMPTY_U + i), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar(PF_B_TFULL + i), 2);             // the MMA thread's arrival (publishes the residual flag) + tcgen05.commit
      mbar_init(bar(PF_B_A0E + i), 4);
    }
    mbar_init(bar(PF_B_A1E), 4);
    fence_mbar_init();
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
#ifdef PF_TRACE
  if (threadIdx.x == 64) {
    long long gt;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(gt));
    reinterpret_cast<long long*>(p.dbg1)[2048 + blockIdx.x] = gt;
  }
#endif

  // residual metadata: every role that needs it keeps the {quarter mask, first quarter} words of 32 consecutive K-steps
  // in its lanes (one coalesced load per chunk, requested one chunk ahead) and derives the item sequence from them:
  // no shared-memory metadata, no round trip in anybody's chain
  auto load_chunk = [&](int T, int c0) -> int2 {
    int2 v = make_int2(0, 0);
    if (p.unit_meta && T < p.tiles && c0 + lane < KS) v = __ldg(p.unit_meta + (size_t)(T / p.TT) * KS + c0 + lane);
    return v;
  };
  auto next_chunk = [&](int& T, int& c0) {
    c0 += 32;
    if (c0 >= KS) {
      c0 = 0;
      T += (int)gridDim.x;
    }
  };

  if (warp == 0) {
    if (lane == 0) {
      // ===================== producer (one thread): one K-step per stage =====================
      griddep_wait();   // the packed tokens are the previous kernel's output
      uint32_t q = 0;
      for (int T = (int)blockIdx.x; T < p.tiles; T += (int)gridDim.x) {
        const int nt = T / p.TT, tt = T - nt * p.TT;
        const uint8_t* wsrc = p.base + (size_t)nt * KS * TILE_BYTES;
        for (int ks = 0; ks < KS; ++ks, ++q) {
          const uint32_t ps = q % PF_PST;
          mbar_wait(bar(PF_B_EMPTY_P + ps), ((q / PF_PST) & 1) ^ 1);
          const uint32_t fb = bar(PF_B_FULL_P + ps), dst = sP + ps * PF_P_STAGE;
          mbar_arrive_expect_tx(fb, TILE_BYTES + PF_TOK_KSTEP);
          tma_load_1d(dst, wsrc + (size_t)ks * TILE_BYTES, TILE_BYTES, fb);
          tma_load_2d(dst + TILE_BYTES, &tmap_a, ks * (BK / 2), tt * PF_BT, fb);
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer: warp-uniform control, one elected lane issues =====================
    constexpr uint32_t IDESC = make_idesc_i8(BN, PF_BT);
    uint32_t item = 0;
    bool pre_ok = false;   // the barrier of the item about to be processed was already seen complete
    // the operand stage of item i: FULL_U[i & 3], phase (i >> 2) & 1.  The next item's barrier is polled once BEFORE
    // this item's MMAs are issued, so that the round trip hides under the tensor pipe's work.
    auto acquire = [&]() {
      if (!pre_ok) mbar_wait(bar(PF_B_FULL_U + (int)(item & 3)), (item >> 2) & 1);
      tc_fence_after();
      pre_ok = mbar_try_wait(bar(PF_B_FULL_U + (int)((item + 1) & 3)), ((item + 1) >> 2) & 1);
    };
    int it = 0;
    int pT = (int)blockIdx.x, pc0 = 0;
    int2 um_next = load_chunk(pT, pc0);
    for (int T = (int)blockIdx.x; T < p.tiles; T += (int)gridDim.x, ++it) {
      const int buf = it & 1;
      PF_STAMP(lane == 0, it, 3);
      mbar_wait(bar(PF_B_A0E + buf), (((uint32_t)it >> 1) & 1) ^ 1);   // the epilogue has drained this base accumulator
      PF_STAMP(lane == 0, it, 4);
      tc_fence_after();
      const uint32_t d0 = tmem_base + (uint32_t)(buf * PF_BT), d1 = tmem_base + (uint32_t)PF_ACC1_COL;
      uint32_t acc0_on = 0, acc1_on = 0;
      for (int c0 = 0; c0 < KS; c0 += 32) {
        const int2 um = um_next;
        next_chunk(pT, pc0);
        um_next = load_chunk(pT, pc0);
        const uint32_t bits = __ballot_sync(0xffffffffu, (um.x & 0xF) != 0);
        const int nk = min(32, KS - c0);
        for (int j = 0; j < nk; ++j) {
          const bool has = (bits >> j) & 1;
          const int us = (int)(item & 3);
          acquire();
          const uint32_t at = tmem_base + (uint32_t)(PF_A_COL0 + us * PF_A_COLS);
          const uint64_t dt = make_desc_sw128(sU + us * PF_U_STAGE);
          if (elect_one()) {
#pragma unroll
            for (int k = 0; k < 4; ++k) mma_i8_ts(d0, at + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), IDESC, k == 0 ? acc0_on : 1u);
            if (!has) tc_commit(bar(PF_B_EMPTY_U + us));
          }
          __syncwarp();
          acc0_on = 1;
          ++item;
          if (has) {
            // residual cell of this K-step: its weights in the next stage's A columns, the tokens of this K-step's
            // stage (the paper's re-use of the activation tile), second accumulator
            const uint32_t mask = (uint32_t)__shfl_sync(0xffffffffu, um.x, j) & 0xF;
            const int us2 = (int)(item & 3);
            acquire();
            if (!acc1_on) {
              mbar_wait(bar(PF_B_A1E), ((uint32_t)it & 1) ^ 1);   // the epilogue has read the previous tile's acc1
              tc_fence_after();
            }
            const uint32_t at2 = tmem_base + (uint32_t)(PF_A_COL0 + us2 * PF_A_COLS);
            if (elect_one()) {
              uint32_t on = acc1_on;
#pragma unroll
              for (int h = 0; h < 2; ++h)
                if (mask & (3u << (2 * h))) {
#pragma unroll
                  for (int k = 2 * h; k < 2 * h + 2; ++k) {
                    mma_i8_ts(d1, at2 + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), IDESC, on);
                    on = 1;
                  }
                }
              tc_commit(bar(PF_B_EMPTY_U + us2));
              tc_commit(bar(PF_B_EMPTY_U + us));
            }
            __syncwarp();
            acc1_on = 1;
            ++item;
          }
        }
      }
      PF_STAMP(lane == 0, it, 5);
      if (elect_one()) {
        misc[1 + buf] = (int32_t)acc1_on;
        mbar_arrive(bar(PF_B_TFULL + buf));   // release: publishes the flag to the epilogue warps
        tc_commit(bar(PF_B_TFULL + buf));     // completes the phase when the MMAs have finished
      }
      __syncwarp();
    }
  } else if (warp >= 6) {
    // ============ unpack groups: int4 -> int8 (x16); weights -> TMEM, tokens -> swizzled shared memory ============
    const int g = (warp - 6) >> 2;                      // group = U stage = items g, g + 4, ...
    const int wq = warp & 3;                            // TMEM lane quadrant of this warp
    const uint32_t row = (uint32_t)(wq * 32 + lane);    // output channel inside the tile
    const uint32_t gtid = (uint32_t)(((warp - 6) & 3) * 32 + lane);
    const uint32_t lane_addr = tmem_base + ((uint32_t)(wq * 32) << 16) + (uint32_t)(PF_A_COL0 + g * PF_A_COLS);
    const uint32_t su = sU + g * PF_U_STAGE;
    const int rhalf = (int)(row >> 6);
    uint32_t item = 0, n_mine = 0, q = 0;   // items / own items / K-steps so far (the K-step counter names the P stage)
#ifdef PF_TRACE
    int it = -1;
#endif
    auto publish = [&]() {   // the item is in place: tell the MMA warp
      PF_FINE(4);
      tmem_st_wait();
      PF_FINE(5);
      tc_fence_before();
      fence_proxy_async_smem();
      __syncwarp();
      PF_FINE(6);
      if (lane == 0) mbar_arrive(bar(PF_B_FULL_U + g));
      PF_FINE(7);
      ++n_mine;
    };
    int pT = (int)blockIdx.x, pc0 = 0;
    int2 um_next = load_chunk(pT, pc0);
    for (int T = (int)blockIdx.x; T < p.tiles; T += (int)gridDim.x) {
#ifdef PF_TRACE
      ++it;
#endif
      for (int c0 = 0; c0 < KS; c0 += 32) {
        const int2 um = um_next;
        next_chunk(pT, pc0);
        um_next = load_chunk(pT, pc0);
        const uint32_t bits = __ballot_sync(0xffffffffu, (um.x & 0xF) != 0);
        const int nk = min(32, KS - c0);
        for (int j = 0; j < nk; ++j) {
          const uint32_t idx = item + (uint32_t)j + (uint32_t)__popc(bits & ((1u << j) - 1));   // item number of K-step j's base item
          const bool has = (bits >> j) & 1;
          if ((idx & 3) == (uint32_t)g) {
            // ---- base item ----
            const uint32_t ps = (q + (uint32_t)j) % PF_PST;
            PF_FINE(0);
            mbar_wait(bar(PF_B_FULL_P + ps), ((q + (uint32_t)j) / PF_PST) & 1);
            PF_FINE(1);
            uint4 v4[4], t4[4];
            const uint32_t pw = sP + ps * PF_P_STAGE, pt = pw + TILE_BYTES;
#pragma unroll
            for (int c = 0; c < 4; ++c) v4[c] = PF_EXP_NOW ? make_uint4(row, c, ps, g) : pf_lds128(pw + c * (BN * 16) + row * 16);
#pragma unroll
            for (int i = 0; i < 4; ++i) t4[i] = PF_EXP_NOT ? make_uint4(row, i, ps, g) : pf_lds128(pt + (gtid + 128u * i) * 16);
            PF_FINE(2);
            mbar_wait(bar(PF_B_EMPTY_U + g), (n_mine & 1) ^ 1);   // the poll runs under the loads' latency
            tc_fence_after();
            PF_FINE(3);
            {
              uint32_t o[32];
#pragma unroll
              for (int c = 0; c < 4; ++c) pf_unpack16(v4[c], o + 8 * c);
              tmem_st32(lane_addr, o);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const uint32_t ti = gtid + 128u * i, t = ti >> 2, c = ti & 3;
              uint32_t tw[8];
              pf_unpack16(t4[i], tw);
              if (!PF_EXP_NOS) {
                pf_sts128(su + t * 128 + (((2 * c) ^ (t & 7)) << 4), tw);
                pf_sts128(su + t * 128 + (((2 * c + 1) ^ (t & 7)) << 4), tw + 4);
              } else {
                asm volatile("" ::"r"(tw[0]), "r"(tw[1]), "r"(tw[2]), "r"(tw[3]), "r"(tw[4]), "r"(tw[5]), "r"(tw[6]), "r"(tw[7]));
              }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(PF_B_EMPTY_P + ps));   // the packed stage is in registers: back to the producer
            publish();
          }
          if (has && ((idx + 1) & 3) == (uint32_t)g) {
            // ---- residual item: the cell's packed rows straight from global memory ----
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
            mbar_wait(bar(PF_B_EMPTY_U + g), (n_mine & 1) ^ 1);
            tc_fence_after();
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              if (!(rmask & (3u << (2 * h)))) continue;   // k-half without any block: never read by the MMA
              uint32_t ro[16];
              pf_unpack16(r4[h][0], ro);
              pf_unpack16(r4[h][1], ro + 8);
              tmem_st16(lane_addr + (uint32_t)(16 * h), ro);
            }
            publish();
          }
        }
        item += (uint32_t)nk + (uint32_t)__popc(nk == 32 ? bits : (bits & ((1u << nk) - 1)));
        q += (uint32_t)nk;
      }
    }
  } else {
    // ===================== epilogue warps (2..5) =====================
    griddep_wait();   // s_a and Y are ordered after the previous kernel in the stream
    const int lq = warp & 3;                     // TMEM lane quadrant this warp may access
    const int et = (warp - 2) * 32 + lane;       // 0..127 within the epilogue group
    const int n_loc = lq * 32 + lane;
    const uint32_t lane_off = (uint32_t)(lq * 32) << 16;
    int it = 0;
    for (int T = (int)blockIdx.x; T < p.tiles; T += (int)gridDim.x, ++it) {
      const int nt = T / p.TT, tt = T - nt * p.TT, buf = it & 1;
      const int n = nt * BN + n_loc, t_base = tt * PF_BT;
      const int t_cnt = min(PF_BT, p.M - t_base);
      const float swn = __ldg(p.sw + n) * 0.00390625f, srn = __ldg(p.sr + n) * 0.00390625f;   // accumulators are x256
      float* sat = sa_tile + buf * PF_BT;
      sat[et] = et < t_cnt ? __ldg(p.sa + t_base + et) : 0.f;
      named_bar_sync(1, 128);   // also orders this buffer's readers (two tiles ago) before its writers
      PF_STAMP(et == 0, it, 0);
      mbar_wait(bar(PF_B_TFULL + buf), ((uint32_t)it >> 1) & 1);
      PF_STAMP(et == 0, it, 1);
      tc_fence_after();
      const bool has_res = misc[1 + buf] != 0;   // acc1 is undefined when no residual MMA was issued
      const uint32_t t0addr = tmem_base + lane_off + (uint32_t)(buf * PF_BT), t1addr = tmem_base + lane_off + (uint32_t)PF_ACC1_COL;
      uint16_t* yp0 = reinterpret_cast<uint16_t*>(p.Y) + (size_t)t_base * p.ldy + n;
      // 8-token batches, two in flight: the TMEM loads of batch b+1 run under the arithmetic and the stores of batch b.
      // FULL = whole token tile and no parity hooks: branch-free, one pointer bump per token.
      auto drain = [&](auto res_c, auto bf_c, auto full_c) {
        constexpr bool RES = decltype(res_c)::value, BF = decltype(bf_c)::value, FULL = decltype(full_c)::value;
        uint16_t* yp = yp0;
        uint32_t a[2][8], r[2][8];
#pragma unroll
        for (int i = 0; i < 8; ++i) r[0][i] = r[1][i] = 0;
        tmem_ld8(t0addr, a[0]);
        if (RES) tmem_ld8(t1addr, r[0]);
#pragma unroll
        for (int b = 0; b < PF_BT / 8; ++b) {
          const int cur = b & 1;
          tmem_ld_wait8(a[cur], r[cur]);
          if (b + 1 < PF_BT / 8) {
            tmem_ld8(t0addr + (b + 1) * 8, a[cur ^ 1]);
            if (RES) tmem_ld8(t1addr + (b + 1) * 8, r[cur ^ 1]);
          }
          const float4 s_lo = *reinterpret_cast<const float4*>(sat + b * 8);
          const float4 s_hi = *reinterpret_cast<const float4*>(sat + b * 8 + 4);
          const float sv[8] = {s_lo.x, s_lo.y, s_lo.z, s_lo.w, s_hi.x, s_hi.y, s_hi.z, s_hi.w};
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            float y = (float)(int32_t)a[cur][i] * swn;
            if (RES) y += (float)(int32_t)r[cur][i] * srn;
            y *= sv[i];
            const uint16_t h = BF ? __bfloat16_as_ushort(__float2bfloat16_rn(y)) : __half_as_ushort(__float2half_rn(y));
            if (FULL) {
              *yp = h;
            } else if (b * 8 + i < t_cnt) {
              *yp = h;
              const size_t di = (size_t)(t_base + b * 8 + i) * p.N + n;
              if (p.dbg0) p.dbg0[di] = (int32_t)a[cur][i] >> 8;
#ifndef PF_TRACE
              if (p.dbg1) p.dbg1[di] = RES ? ((int32_t)r[cur][i] >> 8) : 0;
#endif
            }
            yp += p.ldy;
          }
        }
      };
      auto drain2 = [&](auto res_c, auto bf_c) {
        if (t_cnt == PF_BT && !p.dbg0 && !p.dbg1) drain(res_c, bf_c, std::true_type{});
        else drain(res_c, bf_c, std::false_type{});
      };
      if (has_res) {
        if (p.y_bf16) drain2(std::true_type{}, std::true_type{}); else drain2(std::true_type{}, std::false_type{});
      } else {
        if (p.y_bf16) drain2(std::false_type{}, std::true_type{}); else drain2(std::false_type{}, std::false_type{});
      }
      PF_STAMP(et == 0, it, 2);
      // accumulators drained: hand them back to the MMA warp
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(bar(PF_B_A1E));
        mbar_arrive(bar(PF_B_A0E + buf));
      }
    }
  }

#ifdef PF_TRACE
  if (threadIdx.x == 64) {
    long long gt;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(gt));
    reinterpret_cast<long long*>(p.dbg1)[1024 + blockIdx.x] = gt;
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

// Whole-tile scheduling has no stream-K tail: take the shapes whose last round of tiles is mostly full.
bool prefill_eligible(const mq_weights* w, int64_t M) {
  const Options& o = options();
  if (!w || w->blockscale || o.prefill_path == 1) return false;
  if (o.token_tile || o.split_k >= 2 || o.max_ctas || o.fused_quant) return false;   // knobs of the stream-K kernel
  if (M < 64) return false;
  if (o.prefill_path == 2) return true;
  const int64_t tiles = (w->N / BN) * ((M + PF_BT - 1) / PF_BT);
  const int64_t sms = sm_count();
  const int64_t rounds = (tiles + sms - 1) / sms;
  return tiles * 100 >= rounds * sms * 88;
}

int prefill_gemm(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                 int32_t* dbg0, int32_t* dbg1, void* cuda_stream, bool ignore_res) {
  typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  EncodeTiledFn enc = (EncodeTiledFn)tensor_map_encode_fn();
  if (!enc) return MQ_ERR_CUDA;
  // 2-D tensor map over the canonical packed activations [M rows][K/2 bytes]: box = one K-step of one token tile;
  // rows past M read as zero
  CUtensorMap tmap;
  memset(&tmap, 0, sizeof(tmap));
  const cuuint64_t row_bytes = (cuuint64_t)(w->K / 2);
  const cuuint64_t gdim[2] = {row_bytes, (cuuint64_t)M};
  const cuuint64_t gstride[1] = {row_bytes};
  const cuuint32_t box[2] = {(cuuint32_t)(BK / 2), (cuuint32_t)PF_BT};
  const cuuint32_t estr[2] = {1, 1};
  if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(qA), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
          CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return MQ_ERR_CUDA;

  PfParams pp;
  pp.base = w->d_base;
  pp.res = w->d_res;
  pp.unit_meta = (ignore_res || w->n_quarters == 0) ? nullptr : (const int2*)w->d_unit_meta;
  pp.sw = w->d_sw;
  pp.sr = w->d_sr;
  pp.sa = sA;
  pp.Y = Y;
  pp.dbg0 = dbg0;
  pp.dbg1 = dbg1;
  pp.ldy = ldy;
  pp.M = (int)M;
  pp.N = (int)w->N;
  pp.KS = (int)(w->K / BK);
  pp.NT = (int)(w->N / BN);
  pp.TT = (int)((M + PF_BT - 1) / PF_BT);
  const int64_t tiles = (int64_t)pp.NT * pp.TT;
  if (tiles >= ((int64_t)1 << 31)) return MQ_ERR_UNSUPPORTED_SHAPE;
  pp.tiles = (int)tiles;
  pp.y_bf16 = y_dtype == MQ_BF16;

  static int attr_dev = -1;   // the attribute belongs to the (device, function) pair
  int dev = -1;
  cudaGetDevice(&dev);
  if (dev != attr_dev) {
    if (cudaFuncSetAttribute(mq_prefill_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, PF_SMEM_BYTES) != cudaSuccess) {
      cudaGetLastError();
      return MQ_ERR_CUDA;
    }
    attr_dev = dev;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)std::min<int64_t>(tiles, sm_count()));
  cfg.blockDim = dim3(PF_THREADS);
  cfg.dynamicSmemBytes = PF_SMEM_BYTES;
  cfg.stream = (cudaStream_t)cuda_stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = options().pdl ? 1 : 0;
  if (cudaLaunchKernelEx(&cfg, mq_prefill_kernel, tmap, pp) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  set_launch_count(1);
  return MQ_OK;
}

}  // namespace mq
