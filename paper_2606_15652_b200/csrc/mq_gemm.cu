// mq_gemm.cu -- the fused base + residual int4 GEMM (ZipperEngine; Eq.4).
//
// Orientation ("swap-AB"): the WEIGHT tile is the MMA's M operand (128 output channels),
// the TOKEN tile is the MMA's N operand (BT = 16..256 tokens), so the same kernel serves
// decode (M = 1..32 tokens) and prefill.  Accumulators live in TMEM as D[n, t]:
// lane = output channel, column = token; acc0 (base, scale s_w) and acc1 (residual, scale
// s_r) are separate column ranges because the scales differ (north_star (iii)).
//
// Warp roles (448 threads, one persistent CTA per SM):
//   warp 0      producer : TMA.  Per K-step one 8 KB 1-D bulk copy of the pre-tiled packed
//                          base-weight tile + one 2-D tensor copy of the packed token tile
//                          into the "packed" ring; for K-steps that own a residual cell
//                          (CSR row of this n-tile) also the cell's present 2 KB quarters.
//   warps 6-13  unpack   : int4 -> int8 (value x16: nibble moved to the high half of a byte,
//                          two logic ops per 8 elements) from the packed ring into the
//                          "unpacked" ring in the K-major SWIZZLE_128B layout tcgen05 reads.
//                          Both operands use the same within-16-byte element order, so
//                          dot products are unchanged; accumulators are 256 x the true value.
//   warp 1      MMA      : one thread issues tcgen05.mma kind::i8 (4 per K-step for the base,
//                          2 per present k-half of a residual cell, re-using the SAME
//                          unpacked token tile) and commits to the ring's empty barriers.
//   warps 2-5   epilogue : tcgen05.ld both accumulators, y = s_a * (s_w*acc0 + s_r*acc1) in
//                          fp32, bf16/fp16 store; or, with split-K, red.add of the int32
//                          partials into the workspace and the last-arriving CTA finishes.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <algorithm>

#include "mq_internal.h"
#include "mq_ptx.cuh"

namespace {

using namespace mq;
using namespace mq::ptx;

constexpr int NUM_UNPACK_WARPS = 8;
constexpr int FIRST_EPI_WARP = 2;
constexpr int FIRST_UNPACK_WARP = 6;
constexpr int NUM_THREADS = 32 * (FIRST_UNPACK_WARP + NUM_UNPACK_WARPS);  // 448
constexpr int RSTAGES = 2;
constexpr int U_W_BYTES = BN * BK;       // 16 KB unpacked weight tile
constexpr int RP_BYTES = 4 * QUARTER_BYTES;  // 8 KB packed residual cell slot

template <int BT>
struct Cfg {
  static constexpr int PSTAGES = BT <= 32 ? 8 : (BT == 64 ? 5 : (BT == 128 ? 4 : 3));
  static constexpr int USTAGES = BT <= 64 ? 4 : (BT == 128 ? 3 : 2);
  static constexpr int P_TOK = BT * (BK / 2);
  static constexpr int P_STAGE = TILE_BYTES + P_TOK;
  static constexpr int U_TOK = BT * BK;
  static constexpr int U_STAGE = U_W_BYTES + U_TOK;
  static constexpr int ACC_STAGES = BT <= 128 ? 2 : 1;
  static constexpr int TMEM_NEED = ACC_STAGES * 2 * BT;
  static constexpr int TMEM_COLS = TMEM_NEED <= 32 ? 32 : (TMEM_NEED <= 64 ? 64 : (TMEM_NEED <= 128 ? 128 : (TMEM_NEED <= 256 ? 256 : 512)));
  // shared memory map (offsets from a 1024-aligned base)
  static constexpr int OFF_U = 0;
  static constexpr int OFF_RU = OFF_U + USTAGES * U_STAGE;
  static constexpr int OFF_P = OFF_RU + RSTAGES * U_W_BYTES;
  static constexpr int OFF_RP = OFF_P + PSTAGES * P_STAGE;
  static constexpr int OFF_BAR = OFF_RP + RSTAGES * RP_BYTES;
  static constexpr int NUM_BARS = 2 * PSTAGES + 2 * USTAGES + 4 * RSTAGES + 4;
  static constexpr int OFF_META = OFF_BAR + NUM_BARS * 8;
  static constexpr int OFF_END = OFF_META + (PSTAGES + USTAGES + 8) * 4;
  static constexpr int SMEM_BYTES = OFF_END + 1024;  // slack for the 1024-byte alignment
};

struct GemmParams {
  const uint8_t* base;
  const float* sw;
  const float* sr;
  const uint8_t* res;
  const int32_t* cell_ptr;
  const CellMeta* cell_meta;
  const float* sa;
  void* Y;
  int32_t* dbg0;
  int32_t* dbg1;
  int32_t* ws_acc;   // split-K partials: [tile][2][BT][128]
  int32_t* ws_cnt;   // split-K arrival counters: [tile]
  int64_t ldy;
  int M, N, KS, NT, TT, S;
  int y_bf16;
};

struct Ring {
  int stage = 0;
  uint32_t phase = 0;
  template <int N>
  __device__ __forceinline__ void next() {
    if (++stage == N) {
      stage = 0;
      phase ^= 1;
    }
  }
};

// 32 packed nibbles (16 B) -> 32 int8 = 16 x value.  Output element order inside the 32
// bytes: for each packed word, its even nibbles then its odd nibbles; identical for both
// MMA operands.
__device__ __forceinline__ void unpack16(const uint4& p, uint4& o0, uint4& o1) {
  const uint32_t HI = 0xF0F0F0F0u;
  o0.x = (p.x << 4) & HI;
  o0.y = p.x & HI;
  o0.z = (p.y << 4) & HI;
  o0.w = p.y & HI;
  o1.x = (p.z << 4) & HI;
  o1.y = p.z & HI;
  o1.z = (p.w << 4) & HI;
  o1.w = p.w & HI;
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, const uint4& v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

__device__ __forceinline__ void split_range(int KS, int S, int s, int& k0, int& k1) {
  k0 = (int)(((int64_t)KS * s) / S);
  k1 = (int)(((int64_t)KS * (s + 1)) / S);
}

template <int BT>
__global__ void __launch_bounds__(NUM_THREADS, 1)
mq_gemm_kernel(const __grid_constant__ CUtensorMap tmap_a, const GemmParams p) {
  using C = Cfg<BT>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));

  const uint32_t sU = smem_base + C::OFF_U, sRU = smem_base + C::OFF_RU, sP = smem_base + C::OFF_P,
                 sRP = smem_base + C::OFF_RP, sBar = smem_base + C::OFF_BAR;
  auto bar = [&](int i) { return sBar + 8u * (uint32_t)i; };
  constexpr int B_FULL_P = 0, B_EMPTY_P = C::PSTAGES, B_FULL_U = 2 * C::PSTAGES, B_EMPTY_U = B_FULL_U + C::USTAGES,
                B_FULL_RP = B_EMPTY_U + C::USTAGES, B_EMPTY_RP = B_FULL_RP + RSTAGES, B_FULL_RU = B_EMPTY_RP + RSTAGES,
                B_EMPTY_RU = B_FULL_RU + RSTAGES, B_TFULL = B_EMPTY_RU + RSTAGES, B_TEMPTY = B_TFULL + 2;
  volatile int32_t* meta_p = reinterpret_cast<volatile int32_t*>(smem_gen + C::OFF_META);
  volatile int32_t* meta_u = meta_p + C::PSTAGES;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(meta_u + C::USTAGES);
  volatile int32_t* flag_slot = reinterpret_cast<volatile int32_t*>(tmem_slot + 1);
  volatile int32_t* acc_flag = flag_slot + 1;  // [2]: did this accumulator stage receive residual MMAs?

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmap_a);
    for (int i = 0; i < C::PSTAGES; ++i) {
      mbar_init(bar(B_FULL_P + i), 1);
      mbar_init(bar(B_EMPTY_P + i), NUM_UNPACK_WARPS);
    }
    for (int i = 0; i < C::USTAGES; ++i) {
      mbar_init(bar(B_FULL_U + i), NUM_UNPACK_WARPS);
      mbar_init(bar(B_EMPTY_U + i), 1);
    }
    for (int i = 0; i < RSTAGES; ++i) {
      mbar_init(bar(B_FULL_RP + i), 1);
      mbar_init(bar(B_EMPTY_RP + i), NUM_UNPACK_WARPS);
      mbar_init(bar(B_FULL_RU + i), NUM_UNPACK_WARPS);
      mbar_init(bar(B_EMPTY_RU + i), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar(B_TFULL + i), 2);
      mbar_init(bar(B_TEMPTY + i), 4);
    }
    fence_mbar_init();
  }
  if (warp == 1) {
    tmem_alloc(smem_u32((const void*)tmem_slot), C::TMEM_COLS);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  const int items = p.NT * p.TT * p.S;

  if (warp == 0) {
    // ===================== producer (TMA) =====================
    if (lane == 0) {
      Ring rp, rr;
      for (int item = blockIdx.x; item < items; item += gridDim.x) {
        const int s = item % p.S, nt = (item / p.S) % p.NT, tt = item / (p.S * p.NT);
        int k0, k1;
        split_range(p.KS, p.S, s, k0, k1);
        int ci = p.cell_ptr[nt];
        const int cend = p.cell_ptr[nt + 1];
        CellMeta cm{0x7FFFFFFF, 0};
        while (ci < cend) {
          cm = p.cell_meta[ci];
          if ((cm.kstep_mask & 0xFFFFFF) >= k0) break;
          ++ci;
        }
        int next_ks = ci < cend ? (cm.kstep_mask & 0xFFFFFF) : 0x7FFFFFFF;
        const uint8_t* wsrc = p.base + ((size_t)nt * p.KS + k0) * TILE_BYTES;
        for (int ks = k0; ks < k1; ++ks, wsrc += TILE_BYTES) {
          mbar_wait(bar(B_EMPTY_P + rp.stage), rp.phase ^ 1);
          const int mask = (ks == next_ks) ? ((cm.kstep_mask >> 24) & 0xF) : 0;
          meta_p[rp.stage] = mask;
          const uint32_t dst = sP + rp.stage * C::P_STAGE;
          mbar_arrive_expect_tx(bar(B_FULL_P + rp.stage), C::P_STAGE);
          tma_load_1d(dst, wsrc, TILE_BYTES, bar(B_FULL_P + rp.stage));
          tma_load_2d(dst + TILE_BYTES, &tmap_a, ks * (BK / 2), tt * BT, bar(B_FULL_P + rp.stage));
          if (mask) {
            mbar_wait(bar(B_EMPTY_RP + rr.stage), rr.phase ^ 1);
            mbar_arrive_expect_tx(bar(B_FULL_RP + rr.stage), (uint32_t)__popc(mask) * QUARTER_BYTES);
            const uint8_t* rsrc = p.res + (size_t)cm.qoff * QUARTER_BYTES;
            for (int q = 0; q < 4; ++q)
              if (mask & (1 << q)) {
                tma_load_1d(sRP + rr.stage * RP_BYTES + q * QUARTER_BYTES, rsrc, QUARTER_BYTES,
                            bar(B_FULL_RP + rr.stage));
                rsrc += QUARTER_BYTES;
              }
            rr.next<RSTAGES>();
            ++ci;
            if (ci < cend) {
              cm = p.cell_meta[ci];
              next_ks = cm.kstep_mask & 0xFFFFFF;
            } else {
              next_ks = 0x7FFFFFFF;
            }
          }
          rp.next<C::PSTAGES>();
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      constexpr uint32_t IDESC = make_idesc_i8(BN, BT);
      Ring ru, rr;
      int it = 0;
      for (int item = blockIdx.x; item < items; item += gridDim.x, ++it) {
        const int s = item % p.S;
        int k0, k1;
        split_range(p.KS, p.S, s, k0, k1);
        const int a = C::ACC_STAGES == 2 ? (it & 1) : 0;
        const uint32_t aphase = C::ACC_STAGES == 2 ? ((it >> 1) & 1) : (it & 1);
        mbar_wait(bar(B_TEMPTY + a), aphase ^ 1);
        tc_fence_after();
        const uint32_t d0 = tmem_base + (uint32_t)(a * 2 * BT), d1 = d0 + BT;
        uint32_t acc0_on = 0, acc1_on = 0;
        for (int ks = k0; ks < k1; ++ks) {
          mbar_wait(bar(B_FULL_U + ru.stage), ru.phase);
          tc_fence_after();
          const int mask = meta_u[ru.stage];
          const uint32_t uw = sU + ru.stage * C::U_STAGE, ut = uw + U_W_BYTES;
          const uint64_t dw = make_desc_sw128(uw), dt = make_desc_sw128(ut);
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            mma_i8_ss(d0, dw + (uint64_t)(k * 2), dt + (uint64_t)(k * 2), IDESC, acc0_on);
            acc0_on = 1;
          }
          if (mask) {
            mbar_wait(bar(B_FULL_RU + rr.stage), rr.phase);
            tc_fence_after();
            const uint64_t dr = make_desc_sw128(sRU + rr.stage * U_W_BYTES);
#pragma unroll
            for (int h = 0; h < 2; ++h)
              if (mask & (3 << (2 * h))) {
#pragma unroll
                for (int k = 2 * h; k < 2 * h + 2; ++k) {
                  mma_i8_ss(d1, dr + (uint64_t)(k * 2), dt + (uint64_t)(k * 2), IDESC, acc1_on);
                  acc1_on = 1;
                }
              }
            tc_commit(bar(B_EMPTY_RU + rr.stage));
            rr.next<RSTAGES>();
          }
          tc_commit(bar(B_EMPTY_U + ru.stage));
          ru.next<C::USTAGES>();
        }
        acc_flag[a] = (int32_t)acc1_on;
        mbar_arrive(bar(B_TFULL + a));   // release: publishes acc_flag to the epilogue warps
        tc_commit(bar(B_TFULL + a));     // completes the phase when the MMAs have finished
      }
    }
  } else if (warp >= FIRST_UNPACK_WARP) {
    // ===================== unpack warps: int4 -> int8 (x16), swizzled =====================
    const int uw_id = warp - FIRST_UNPACK_WARP;
    // row-major packed tile: lane -> (row8 = lane/4, 16-byte chunk j = lane%4)
    const uint32_t row8 = (uint32_t)lane >> 2, j = (uint32_t)lane & 3;
    const uint32_t src_lane = (uint32_t)lane * 16;
    const uint32_t dst_lane0 = row8 * 128 + (((2 * j) ^ row8) << 4);
    const uint32_t dst_lane1 = row8 * 128 + (((2 * j + 1) ^ row8) << 4);
    // residual quarter [64 rows][32 B]: lane -> (row = lane/2, c = lane%2)
    const uint32_t rrow8 = ((uint32_t)lane >> 1) & 7, rc = (uint32_t)lane & 1;
    Ring rp, ru, rrp, rru;
    for (int item = blockIdx.x; item < items; item += gridDim.x) {
      const int s = item % p.S;
      int k0, k1;
      split_range(p.KS, p.S, s, k0, k1);
      for (int ks = k0; ks < k1; ++ks) {
        mbar_wait(bar(B_FULL_P + rp.stage), rp.phase);
        const int mask = meta_p[rp.stage];
        mbar_wait(bar(B_EMPTY_U + ru.stage), ru.phase ^ 1);
        const uint32_t ps = sP + rp.stage * C::P_STAGE, us = sU + ru.stage * C::U_STAGE;
        // weights: 16 warp-chunks of 8 rows; tokens: BT/8 warp-chunks
        constexpr int NCH = 16 + BT / 8;
#pragma unroll 2
        for (int wc = uw_id; wc < NCH; wc += NUM_UNPACK_WARPS) {
          const uint4 v = lds128(ps + wc * 512 + src_lane);
          uint4 o0, o1;
          unpack16(v, o0, o1);
          sts128(us + wc * 1024 + dst_lane0, o0);
          sts128(us + wc * 1024 + dst_lane1, o1);
        }
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
          if (uw_id == 0) meta_u[ru.stage] = mask;
          mbar_arrive(bar(B_FULL_U + ru.stage));
          mbar_arrive(bar(B_EMPTY_P + rp.stage));
        }
        rp.next<C::PSTAGES>();
        ru.next<C::USTAGES>();
        if (mask) {
          mbar_wait(bar(B_FULL_RP + rrp.stage), rrp.phase);
          mbar_wait(bar(B_EMPTY_RU + rru.stage), rru.phase ^ 1);
          const uint32_t rps = sRP + rrp.stage * RP_BYTES, rus = sRU + rru.stage * U_W_BYTES;
#pragma unroll
          for (int pid = uw_id; pid < 16; pid += NUM_UNPACK_WARPS) {
            const int q = pid >> 2, wcq = pid & 3, h = q >> 1, r = q & 1;
            if (!(mask & (3 << (2 * h)))) continue;  // k-half without any block: never read
            uint4 o0 = make_uint4(0, 0, 0, 0), o1 = o0;
            if (mask & (1 << q)) {
              const uint4 v = lds128(rps + q * QUARTER_BYTES + wcq * 512 + src_lane);
              unpack16(v, o0, o1);
            }
            const uint32_t row = (uint32_t)(64 * r + 16 * wcq) + ((uint32_t)lane >> 1);
            const uint32_t ch = (uint32_t)(4 * h) + 2 * rc;
            sts128(rus + row * 128 + ((ch ^ rrow8) << 4), o0);
            sts128(rus + row * 128 + (((ch + 1) ^ rrow8) << 4), o1);
          }
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            mbar_arrive(bar(B_FULL_RU + rru.stage));
            mbar_arrive(bar(B_EMPTY_RP + rrp.stage));
          }
          rrp.next<RSTAGES>();
          rru.next<RSTAGES>();
        }
      }
    }
  } else {
    // ===================== epilogue warps (2..5) =====================
    const int lq = warp & 3;  // TMEM lane quadrant this warp may access
    const int et = (warp - FIRST_EPI_WARP) * 32 + lane;  // 0..127 within the epilogue group
    int it = 0;
    for (int item = blockIdx.x; item < items; item += gridDim.x, ++it) {
      const int s = item % p.S, nt = (item / p.S) % p.NT, tt = item / (p.S * p.NT);
      int k0, k1;
      split_range(p.KS, p.S, s, k0, k1);
      const int a = C::ACC_STAGES == 2 ? (it & 1) : 0;
      const uint32_t aphase = C::ACC_STAGES == 2 ? ((it >> 1) & 1) : (it & 1);
      const int n_loc = lq * 32 + lane;
      const int n = nt * BN + n_loc;
      const int t_base = tt * BT;
      const int t_cnt = min(BT, p.M - t_base);
      const float swn = p.sw[n] * 0.00390625f, srn = p.sr[n] * 0.00390625f;  // / 256: accumulators are x256

      mbar_wait(bar(B_TFULL + a), aphase);
      tc_fence_after();
      const bool has_res = acc_flag[a] != 0;  // acc1 is undefined when no residual MMA was issued
      const uint32_t t0addr = tmem_base + ((uint32_t)(lq * 32) << 16) + (uint32_t)(a * 2 * BT);
      const int tile_id = tt * p.NT + nt;
      int32_t* ws0 = p.ws_acc + (size_t)tile_id * (2 * BT * BN);
      int32_t* ws1 = ws0 + BT * BN;

      for (int c0 = 0; c0 < t_cnt; c0 += 16) {
        uint32_t v0[16], v1[16];
        tmem_ld16(t0addr + c0, v0);
        if (has_res) {
          tmem_ld16(t0addr + BT + c0, v1);
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i) v1[i] = 0;
        }
        tmem_ld_wait();
        if (p.S == 1) {
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            const int t = c0 + i;
            if (t < t_cnt) {
              const int32_t a0 = (int32_t)v0[i], a1 = (int32_t)v1[i];
              const float y = p.sa[t_base + t] * ((float)a0 * swn + (float)a1 * srn);
              const size_t o = (size_t)(t_base + t) * p.ldy + n;
              if (p.y_bf16)
                reinterpret_cast<__nv_bfloat16*>(p.Y)[o] = __float2bfloat16_rn(y);
              else
                reinterpret_cast<__half*>(p.Y)[o] = __float2half_rn(y);
              if (p.dbg0) p.dbg0[(size_t)(t_base + t) * p.N + n] = a0 >> 8;
              if (p.dbg1) p.dbg1[(size_t)(t_base + t) * p.N + n] = a1 >> 8;
            }
          }
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            const int t = c0 + i;
            if (t < t_cnt) {
              atomicAdd(ws0 + t * BN + n_loc, (int32_t)v0[i]);
              if (has_res) atomicAdd(ws1 + t * BN + n_loc, (int32_t)v1[i]);
            }
          }
        }
      }
      // accumulator stage drained: hand it back to the MMA warp
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_TEMPTY + a));

      if (p.S > 1) {
        // split-K: the last CTA to arrive for this tile sums are complete -> finish + clean up
        __threadfence();
        named_bar_sync(1, 128);
        if (et == 0) {
          const int old = atomicAdd(p.ws_cnt + tile_id, 1);
          *flag_slot = (old == p.S - 1);
        }
        named_bar_sync(1, 128);
        const bool last = *flag_slot != 0;
        named_bar_sync(1, 128);  // flag_slot may be rewritten by the next item
        if (last) {
          __threadfence();
          for (int t = 0; t < t_cnt; ++t) {
            const int32_t a0 = __ldcg(ws0 + t * BN + n_loc), a1 = __ldcg(ws1 + t * BN + n_loc);
            __stcg(ws0 + t * BN + n_loc, 0);
            __stcg(ws1 + t * BN + n_loc, 0);
            const float y = p.sa[t_base + t] * ((float)a0 * swn + (float)a1 * srn);
            const size_t o = (size_t)(t_base + t) * p.ldy + n;
            if (p.y_bf16)
              reinterpret_cast<__nv_bfloat16*>(p.Y)[o] = __float2bfloat16_rn(y);
            else
              reinterpret_cast<__half*>(p.Y)[o] = __float2half_rn(y);
            if (p.dbg0) p.dbg0[(size_t)(t_base + t) * p.N + n] = a0 >> 8;
            if (p.dbg1) p.dbg1[(size_t)(t_base + t) * p.N + n] = a1 >> 8;
          }
          if (et == 0) p.ws_cnt[tile_id] = 0;
        }
      }
    }
  }

  // teardown
  tc_fence_before();
  __syncthreads();
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
  return fn;
}

struct Plan {
  int BT = 16, TT = 1, S = 1, grid = 1;
  size_t ws_bytes = 0;
};

Plan make_plan(const mq_weights* w, int64_t M) {
  Plan pl;
  const Options& o = options();
  int bt;
  if (o.token_tile)
    bt = (int)o.token_tile;
  else
    bt = M <= 16 ? 16 : (M <= 32 ? 32 : (M <= 64 ? 64 : 128));
  pl.BT = bt;
  pl.TT = (int)((M + bt - 1) / bt);
  const int NT = (int)(w->N / BN), KS = (int)(w->K / BK);
  int G = sm_count() > 0 ? sm_count() : 148;
  if (o.max_ctas > 0) G = (int)std::min<int64_t>(G, o.max_ctas);
  const int64_t tiles = (int64_t)NT * pl.TT;
  int S = 1;
  if (o.split_k > 0) {
    S = (int)std::min<int64_t>(o.split_k, KS);
  } else if (M <= 128 && tiles < 4LL * G) {
    // decode: pick the split that fills the persistent grid best (>= 4 K-steps per split)
    double best = 0.0;
    for (int s = 1; s <= 16 && KS / s >= 4; ++s) {
      const int64_t items = tiles * s;
      const int64_t waves = (items + G - 1) / G;
      double eff = (double)items / (double)(waves * G) - 0.01 * (s - 1);
      if (eff > best + 1e-9) {
        best = eff;
        S = s;
      }
    }
  }
  pl.S = S;
  pl.grid = (int)std::min<int64_t>(G, tiles * S);
  pl.ws_bytes = S > 1 ? (size_t)tiles * (2 * (size_t)bt * BN) * 4 + (size_t)tiles * 4 : 0;
  return pl;
}

template <int BT>
int launch(const CUtensorMap& tmap, const GemmParams& gp, int grid, cudaStream_t st) {
  using C = Cfg<BT>;
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(mq_gemm_kernel<BT>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES) !=
        cudaSuccess) {
      cudaGetLastError();
      return MQ_ERR_CUDA;
    }
    attr_set = true;
  }
  mq_gemm_kernel<BT><<<grid, NUM_THREADS, C::SMEM_BYTES, st>>>(tmap, gp);
  return cudaGetLastError() == cudaSuccess ? MQ_OK : MQ_ERR_CUDA;
}

}  // namespace

extern "C" size_t mq_gemm_workspace_bytes(const mq_weights* w, int64_t M) {
  if (!w || M <= 0) return 0;
  if (mq::check_device() != MQ_OK) return 0;
  return make_plan(w, M).ws_bytes;
}

extern "C" int mq_gemm(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype,
                       int64_t ldy, int32_t* dbg0, int32_t* dbg1, void* workspace, size_t workspace_bytes,
                       void* cuda_stream) {
  if (!w) return MQ_ERR_INVALID_ARG;
  if (M < 0 || M > (1 << 30)) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (y_dtype != MQ_F16 && y_dtype != MQ_BF16) return MQ_ERR_INVALID_ARG;
  mq::set_launch_count(0);
  if (M == 0) return MQ_OK;
  if (!qA || !sA || !Y || ldy < w->N) return MQ_ERR_INVALID_ARG;
  if (((uintptr_t)qA & 15) || ((uintptr_t)Y & 1) || ((uintptr_t)sA & 3)) return MQ_ERR_INVALID_ARG;
  int rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  EncodeTiledFn enc = get_encode_fn();
  if (!enc) return MQ_ERR_CUDA;

  const Plan pl = make_plan(w, M);
  if (pl.ws_bytes > 0) {
    if (!workspace || workspace_bytes < pl.ws_bytes) return MQ_ERR_WORKSPACE;
    if ((uintptr_t)workspace & 15) return MQ_ERR_INVALID_ARG;
  }

  // 2-D tensor map over the canonical packed activations: [M rows][K/2 bytes]
  CUtensorMap tmap;
  const cuuint64_t gdim[2] = {(cuuint64_t)(w->K / 2), (cuuint64_t)M};
  const cuuint64_t gstride[1] = {(cuuint64_t)(w->K / 2)};
  const cuuint32_t box[2] = {(cuuint32_t)(BK / 2), (cuuint32_t)pl.BT};
  const cuuint32_t estr[2] = {1, 1};
  if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(qA), gdim, gstride, box, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return MQ_ERR_CUDA;

  GemmParams gp;
  gp.base = w->d_base;
  gp.sw = w->d_sw;
  gp.sr = w->d_sr;
  gp.res = w->d_res;
  gp.cell_ptr = w->d_cell_ptr;
  gp.cell_meta = w->d_cell_meta;
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
  gp.S = pl.S;
  gp.y_bf16 = y_dtype == MQ_BF16;
  const size_t tiles = (size_t)gp.NT * gp.TT;
  gp.ws_acc = (int32_t*)workspace;
  gp.ws_cnt = pl.S > 1 ? (int32_t*)workspace + tiles * (2 * (size_t)pl.BT * BN) : nullptr;

  cudaStream_t st = (cudaStream_t)cuda_stream;
  switch (pl.BT) {
    case 16: rc = launch<16>(tmap, gp, pl.grid, st); break;
    case 32: rc = launch<32>(tmap, gp, pl.grid, st); break;
    case 64: rc = launch<64>(tmap, gp, pl.grid, st); break;
    case 128: rc = launch<128>(tmap, gp, pl.grid, st); break;
    case 256: rc = launch<256>(tmap, gp, pl.grid, st); break;
    default: rc = MQ_ERR_INVALID_ARG;
  }
  if (rc == MQ_OK) mq::set_launch_count(1);
  return rc;
}

extern "C" size_t mq_linear_workspace_bytes(const mq_weights* w, int64_t M) {
  if (!w || M <= 0) return 0;
  size_t q = (mq_qact_bytes(M, w->K) + 255) / 256 * 256;
  size_t s = ((size_t)M * 4 + 255) / 256 * 256;
  return q + s + mq_gemm_workspace_bytes(w, M);
}

extern "C" int mq_linear(const mq_weights* w, const void* A, mq_dtype a_dtype, int64_t M, int64_t lda, void* Y,
                         mq_dtype y_dtype, int64_t ldy, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!w) return MQ_ERR_INVALID_ARG;
  if (M == 0) return MQ_OK;
  if (M < 0) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (!workspace || ((uintptr_t)workspace & 255)) return MQ_ERR_INVALID_ARG;
  const size_t need = mq_linear_workspace_bytes(w, M);
  if (workspace_bytes < need) return MQ_ERR_WORKSPACE;
  // the GEMM's zero-state region comes first so that the caller's one-time memset covers it
  const size_t g = mq_gemm_workspace_bytes(w, M);
  const size_t g_al = (g + 255) / 256 * 256;
  uint8_t* base = (uint8_t*)workspace;
  uint8_t* qa = base + g_al;
  float* sa = (float*)(qa + (mq_qact_bytes(M, w->K) + 255) / 256 * 256);
  if ((size_t)((uint8_t*)sa + (size_t)M * 4 - base) > workspace_bytes) return MQ_ERR_WORKSPACE;
  int rc = mq_quantize_act(A, a_dtype, M, w->K, lda, qa, sa, cuda_stream);
  if (rc != MQ_OK) return rc;
  rc = mq_gemm(w, qa, sa, M, Y, y_dtype, ldy, nullptr, nullptr, base, g, cuda_stream);
  if (rc == MQ_OK) mq::set_launch_count(2);
  return rc;
}
