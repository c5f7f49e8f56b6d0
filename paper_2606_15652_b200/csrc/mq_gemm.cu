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
// Warp roles (448 threads, one persistent CTA per SM):
//   warp 0      producer : TMA.  Per K-step one 8 KB 1-D bulk copy of the pre-tiled packed
//                          base-weight tile + one 2-D tensor copy of the packed token tile
//                          into the "packed" ring; for K-steps that own a residual cell also
//                          the cell's present 2 KB quarters.
//   warps 6-9, 10-13       two unpack groups, alternating K-steps: int4 -> int8 (value x16:
//                          nibble moved to the high half of a byte, two logic ops per 8
//                          elements).  Weights -> TMEM (A operand), tokens -> shared memory in
//                          the K-major SWIZZLE_128B layout (B operand).  Both operands use the
//                          same within-32-byte element order, so dot products are unchanged;
//                          accumulators are 256 x the true value.
//   warp 1      MMA      : one thread issues tcgen05.mma kind::i8 (4 per K-step for the base,
//                          2 per present k-half of a residual cell, re-using the SAME token
//                          tile) and commits to the rings' empty barriers.
//   warps 2-5   epilogue : tcgen05.ld both accumulators, y = s_a * (s_w*acc0 + s_r*acc1) in
//                          fp32, bf16/fp16 store.
//
// Work distribution ("stream-K"): the K-steps of all output tiles form one sequence that is
// cut into gridDim.x equal contiguous ranges, so every SM streams the same number of weight
// bytes whatever N is.  A tile whose K range is shared by several CTAs is finished by the
// last of them to arrive: each writes its int32 partial tile to a private workspace slot
// (plain coalesced stores, integer adds are exact so the result stays bit-identical).
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

constexpr int FIRST_EPI_WARP = 2;
constexpr int FIRST_UNPACK_WARP = 6;
constexpr int NUM_UNPACK_GROUPS = 2;
constexpr int NUM_THREADS = 32 * (FIRST_UNPACK_WARP + 4 * NUM_UNPACK_GROUPS);  // 448
constexpr int RSTAGES = 2;
constexpr int A_COLS = BK / 4;               // 32 TMEM columns hold 128 int8 per lane
constexpr int RP_BYTES = 4 * QUARTER_BYTES;  // 8 KB packed residual cell slot

template <int BT>
struct Cfg {
  static constexpr int PSTAGES = BT <= 32 ? 10 : (BT == 64 ? 8 : 6);
  static constexpr int ASTAGES = BT <= 64 ? 4 : 3;
  static constexpr int P_TOK = BT * (BK / 2);
  static constexpr int P_STAGE = TILE_BYTES + P_TOK;
  static constexpr int U_TOK = BT * BK;
  static constexpr int ACC_STAGES = BT <= 64 ? 2 : 1;
  static constexpr int ACC_COLS = ACC_STAGES * 2 * BT;
  static constexpr int A_COL0 = ACC_COLS;
  static constexpr int R_COL0 = A_COL0 + ASTAGES * A_COLS;
  static constexpr int TMEM_NEED = R_COL0 + RSTAGES * A_COLS;
  static constexpr int TMEM_COLS = TMEM_NEED <= 32 ? 32 : (TMEM_NEED <= 64 ? 64 : (TMEM_NEED <= 128 ? 128 : (TMEM_NEED <= 256 ? 256 : 512)));
  static_assert(TMEM_NEED <= 512, "tensor memory budget");
  // shared memory map (offsets from a 1024-aligned base)
  static constexpr int OFF_U = 0;
  static constexpr int OFF_P = OFF_U + ASTAGES * U_TOK;
  static constexpr int OFF_RP = OFF_P + PSTAGES * P_STAGE;
  static constexpr int OFF_BAR = OFF_RP + RSTAGES * RP_BYTES;
  static constexpr int NUM_BARS = 2 * PSTAGES + 2 * ASTAGES + 4 * RSTAGES + 4;
  static constexpr int OFF_META = OFF_BAR + NUM_BARS * 8;
  static constexpr int OFF_END = OFF_META + (PSTAGES + ASTAGES + 8) * 4;
  static constexpr int SMEM_BYTES = OFF_END + 1024;  // slack for the 1024-byte alignment
};

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
  int32_t* ws_cnt;    // [tiles] arrival counters (zero between calls)
  int32_t* ws_flag;   // [grid][2] did this partial receive residual MMAs?
  int32_t* ws_part;   // [grid][2 slots][2 accs][BT][128] int32 partial tiles
  int64_t ldy;
  long long units;    // NT*TT*KS
  int gran;           // range boundaries are multiples of gran (1 = stream-K, KS = whole tiles)
  int M, N, KS, NT, TT;
  int y_bf16;
#ifdef MQ_TRACE
  long long* trace;  // [grid][64] clock64 stamps (development builds only)
#endif
};

#ifdef MQ_TRACE
#define MQ_STAMP(slot) do { p.trace[(size_t)blockIdx.x * 64 + (slot)] = clock64(); } while (0)
#define MQ_STAMP_IF(cond, slot) do { if (cond) MQ_STAMP(slot); } while (0)
#else
#define MQ_STAMP(slot) do { } while (0)
#define MQ_STAMP_IF(cond, slot) do { } while (0)
#endif

// first unit of CTA c's range
__device__ __forceinline__ long long range_begin(const GemmParams& p, int c) {
  return (long long)p.gran * (((p.units / p.gran) * (long long)c) / (long long)gridDim.x);
}
// the CTA whose range holds unit x
__device__ __forceinline__ int owner_of(const GemmParams& p, long long x) {
  int c = (int)((x * (long long)gridDim.x) / p.units);
  while (c + 1 < (int)gridDim.x && range_begin(p, c + 1) <= x) ++c;
  while (c > 0 && range_begin(p, c) > x) --c;
  return c;
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

template <bool BF16>
__device__ __forceinline__ void store_y(void* Y, size_t o, float y) {
  if (BF16)
    reinterpret_cast<__nv_bfloat16*>(Y)[o] = __float2bfloat16_rn(y);
  else
    reinterpret_cast<__half*>(Y)[o] = __float2half_rn(y);
}

template <int BT>
__global__ void __launch_bounds__(NUM_THREADS, 1)
mq_gemm_kernel(const __grid_constant__ CUtensorMap tmap_a, const GemmParams p) {
  using C = Cfg<BT>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));

  const uint32_t sU = smem_base + C::OFF_U, sP = smem_base + C::OFF_P, sRP = smem_base + C::OFF_RP,
                 sBar = smem_base + C::OFF_BAR;
  auto bar = [&](int i) { return sBar + 8u * (uint32_t)i; };
  constexpr int B_FULL_P = 0, B_EMPTY_P = C::PSTAGES, B_FULL_U = 2 * C::PSTAGES, B_EMPTY_U = B_FULL_U + C::ASTAGES,
                B_FULL_RP = B_EMPTY_U + C::ASTAGES, B_EMPTY_RP = B_FULL_RP + RSTAGES, B_FULL_RU = B_EMPTY_RP + RSTAGES,
                B_EMPTY_RU = B_FULL_RU + RSTAGES, B_TFULL = B_EMPTY_RU + RSTAGES, B_TEMPTY = B_TFULL + 2;
  // meta words: bits 0-3 quarter mask, bits 8.. sequence number of the residual cell in this CTA
  volatile int32_t* meta_p = reinterpret_cast<volatile int32_t*>(smem_gen + C::OFF_META);
  volatile int32_t* meta_u = meta_p + C::PSTAGES;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(meta_u + C::ASTAGES);
  volatile int32_t* flag_slot = reinterpret_cast<volatile int32_t*>(tmem_slot + 1);
  volatile int32_t* acc_flag = flag_slot + 1;  // [2]: did this accumulator stage receive residual MMAs?

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#ifdef MQ_TRACE
  if (threadIdx.x == 0) {
    unsigned long long gt;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
    p.trace[(size_t)blockIdx.x * 64 + 12] = (long long)gt;
    MQ_STAMP(0);
  }
#endif

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmap_a);
    for (int i = 0; i < C::PSTAGES; ++i) {
      mbar_init(bar(B_FULL_P + i), 1);
      mbar_init(bar(B_EMPTY_P + i), 4);
    }
    for (int i = 0; i < C::ASTAGES; ++i) {
      mbar_init(bar(B_FULL_U + i), 4);
      mbar_init(bar(B_EMPTY_U + i), 1);
    }
    for (int i = 0; i < RSTAGES; ++i) {
      mbar_init(bar(B_FULL_RP + i), 1);
      mbar_init(bar(B_EMPTY_RP + i), 4);
      mbar_init(bar(B_FULL_RU + i), 4);
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
  MQ_STAMP_IF(threadIdx.x == 0, 1);

  const long long u_beg = range_begin(p, (int)blockIdx.x);
  const long long u_end = blockIdx.x + 1 == gridDim.x ? p.units : range_begin(p, (int)blockIdx.x + 1);
  const int n_units = (int)(u_end - u_beg);

  if (warp == 0) {
    // ===================== producer (TMA) =====================
    int ps = 0, rseq = 0;
    uint32_t pphase = 0;
    for (int i0 = 0; i0 < n_units; i0 += 32) {
      // each lane looks up one unit of the batch: tile = nt * TT + tt, unit = tile * KS + ks
      int2 um = make_int2(0, 0);
      int l_wi = 0, l_c0 = 0, l_c1 = 0;
      if (i0 + lane < n_units) {
        const long long u = u_beg + i0 + lane;
        const long long tile = u / p.KS;
        const int ks = (int)(u - tile * p.KS);
        l_wi = (int)(tile / p.TT) * p.KS + ks;     // index of the base tile and of unit_meta
        l_c0 = ks * (BK / 2);                      // tensor-map coordinates of the token tile
        l_c1 = (int)(tile % p.TT) * BT;
        um = __ldg(p.unit_meta + l_wi);
      }
      const int nb = min(32, n_units - i0);
      for (int j = 0; j < nb; ++j) {
        const int mask = __shfl_sync(0xffffffffu, um.x, j);
        const int qoff = __shfl_sync(0xffffffffu, um.y, j);
        const int wi = __shfl_sync(0xffffffffu, l_wi, j);
        const int c0 = __shfl_sync(0xffffffffu, l_c0, j);
        const int c1 = __shfl_sync(0xffffffffu, l_c1, j);
        if (lane == 0) {
          mbar_wait(bar(B_EMPTY_P + ps), pphase ^ 1);
          MQ_STAMP_IF(i0 + j == 0, 2);
          MQ_STAMP_IF(i0 + j < 16, 48 + i0 + j);
          MQ_STAMP_IF(i0 + j == n_units - 1, 3);
          meta_p[ps] = mask | (rseq << 8);
          const uint32_t dst = sP + ps * C::P_STAGE;
          mbar_arrive_expect_tx(bar(B_FULL_P + ps), C::P_STAGE);
          tma_load_1d(dst, p.base + (size_t)wi * TILE_BYTES, TILE_BYTES, bar(B_FULL_P + ps));
          tma_load_2d(dst + TILE_BYTES, &tmap_a, c0, c1, bar(B_FULL_P + ps));
          if (mask) {
            const int rs = rseq % RSTAGES;
            mbar_wait(bar(B_EMPTY_RP + rs), (((uint32_t)rseq / RSTAGES) & 1) ^ 1);
            mbar_arrive_expect_tx(bar(B_FULL_RP + rs), (uint32_t)__popc(mask) * QUARTER_BYTES);
            const uint8_t* rsrc = p.res + (size_t)qoff * QUARTER_BYTES;
            for (int q = 0; q < 4; ++q)
              if (mask & (1 << q)) {
                tma_load_1d(sRP + rs * RP_BYTES + q * QUARTER_BYTES, rsrc, QUARTER_BYTES, bar(B_FULL_RP + rs));
                rsrc += QUARTER_BYTES;
              }
          }
        }
        if (mask) ++rseq;
        if (++ps == C::PSTAGES) {
          ps = 0;
          pphase ^= 1;
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      constexpr uint32_t IDESC = make_idesc_i8(BN, BT);
      int as = 0, it = 0;
      uint32_t aphase_u = 0;
      long long g = u_beg;
      while (g < u_end) {
        const int k0 = (int)(g % p.KS);
        const int k1 = (int)min((long long)p.KS, k0 + (u_end - g));
        g += k1 - k0;
        const int a = C::ACC_STAGES == 2 ? (it & 1) : 0;
        const uint32_t aphase = C::ACC_STAGES == 2 ? ((it >> 1) & 1) : (it & 1);
        ++it;
        mbar_wait(bar(B_TEMPTY + a), aphase ^ 1);
        tc_fence_after();
        const uint32_t d0 = tmem_base + (uint32_t)(a * 2 * BT), d1 = d0 + BT;
        uint32_t acc0_on = 0, acc1_on = 0;
        for (int ks = k0; ks < k1; ++ks) {
          mbar_wait(bar(B_FULL_U + as), aphase_u);
          tc_fence_after();
#ifdef MQ_TRACE
          { const int ui = (int)(g - (k1 - k0) - u_beg) + (ks - k0); MQ_STAMP_IF(ui == 0, 7); MQ_STAMP_IF(ui < 16, 32 + ui); }
#endif
          const int meta = meta_u[as];
          const int mask = meta & 0xF;
          const uint32_t at = tmem_base + (uint32_t)(C::A_COL0 + as * A_COLS);
          const uint64_t dt = make_desc_sw128(sU + as * C::U_TOK);
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            mma_i8_ts(d0, at + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), IDESC, acc0_on);
            acc0_on = 1;
          }
          if (mask) {
            const int rseq = meta >> 8, rs = rseq % RSTAGES;
            mbar_wait(bar(B_FULL_RU + rs), ((uint32_t)rseq / RSTAGES) & 1);
            tc_fence_after();
            const uint32_t rt = tmem_base + (uint32_t)(C::R_COL0 + rs * A_COLS);
#pragma unroll
            for (int h = 0; h < 2; ++h)
              if (mask & (3 << (2 * h))) {
#pragma unroll
                for (int k = 2 * h; k < 2 * h + 2; ++k) {
                  mma_i8_ts(d1, rt + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), IDESC, acc1_on);
                  acc1_on = 1;
                }
              }
            tc_commit(bar(B_EMPTY_RU + rs));
          }
          tc_commit(bar(B_EMPTY_U + as));
          if (++as == C::ASTAGES) {
            as = 0;
            aphase_u ^= 1;
          }
        }
        acc_flag[a] = (int32_t)acc1_on;
        mbar_arrive(bar(B_TFULL + a));   // release: publishes acc_flag to the epilogue warps
        tc_commit(bar(B_TFULL + a));     // completes the phase when the MMAs have finished
        MQ_STAMP(8);
      }
    }
  } else if (warp >= FIRST_UNPACK_WARP) {
    // ============ unpack groups: int4 -> int8 (x16); weights -> TMEM, tokens -> smem ============
    const int gi = (warp - FIRST_UNPACK_WARP) >> 2;               // group: takes units i = gi (mod 2)
    const int wq = warp & 3;                                      // TMEM lane quadrant of this warp
    const uint32_t row = (uint32_t)(wq * 32 + lane);              // output channel inside the tile
    const uint32_t gtid = (uint32_t)(((warp - FIRST_UNPACK_WARP) & 3) * 32 + lane);
    const uint32_t lane_addr = tmem_base + ((uint32_t)(wq * 32) << 16);
    const int rhalf = wq >> 1;                                    // row half of a residual cell
    for (int i = gi; i < n_units; i += NUM_UNPACK_GROUPS) {
      const int ps = i % C::PSTAGES, as = i % C::ASTAGES;
      mbar_wait(bar(B_FULL_P + ps), (uint32_t)(i / C::PSTAGES) & 1);
      MQ_STAMP_IF(i == 0 && gtid == 0, 4);
      const int meta = meta_p[ps];
      const uint32_t pw = sP + ps * C::P_STAGE;
      uint4 v[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) v[c] = lds128(pw + c * (BN * 16) + row * 16);
      mbar_wait(bar(B_EMPTY_U + as), ((uint32_t)(i / C::ASTAGES) & 1) ^ 1);
      tc_fence_after();
      uint32_t o[32];
#pragma unroll
      for (int c = 0; c < 4; ++c) unpack16(v[c], o + 8 * c);
      tmem_st32(lane_addr + (uint32_t)(C::A_COL0 + as * A_COLS), o);
      // tokens: packed [BT][64 B] row-major -> [BT][128 B] K-major SWIZZLE_128B
      const uint32_t pt = pw + TILE_BYTES, ut = sU + as * C::U_TOK;
#pragma unroll
      for (uint32_t idx = gtid; idx < (uint32_t)(BT * 4); idx += 128) {
        const uint32_t t = idx >> 2, j = idx & 3;
        const uint4 tv = lds128(pt + idx * 16);
        uint32_t w8[8];
        unpack16(tv, w8);
        sts128(ut + t * 128 + (((2 * j) ^ (t & 7)) << 4), w8);
        sts128(ut + t * 128 + (((2 * j + 1) ^ (t & 7)) << 4), w8 + 4);
      }
      tmem_st_wait();
      tc_fence_before();
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) {
        MQ_STAMP_IF(i == 0 && gtid == 0, 5);
        MQ_STAMP_IF(gi == 0 && gtid == 0 && i < 32, 16 + i / 2);
        MQ_STAMP_IF(gi == 0 && gtid == 0, 6);
        if (wq == 0) meta_u[as] = meta;
        mbar_arrive(bar(B_FULL_U + as));
        mbar_arrive(bar(B_EMPTY_P + ps));
      }
      const int mask = meta & 0xF;
      if (mask) {
        const int rseq = meta >> 8, rs = rseq % RSTAGES;
        const uint32_t rphase = ((uint32_t)rseq / RSTAGES) & 1;
        mbar_wait(bar(B_FULL_RP + rs), rphase);
        mbar_wait(bar(B_EMPTY_RU + rs), rphase ^ 1);
        tc_fence_after();
        const uint32_t rp = sRP + rs * RP_BYTES;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          if (!(mask & (3 << (2 * h)))) continue;   // k-half without any block: never read by the MMA
          const int q = 2 * h + rhalf;
          uint32_t ro[16];
          if (mask & (1 << q)) {
            const uint4 r0 = lds128(rp + q * QUARTER_BYTES + (row & 63) * 16);
            const uint4 r1 = lds128(rp + q * QUARTER_BYTES + 1024 + (row & 63) * 16);
            unpack16(r0, ro);
            unpack16(r1, ro + 8);
          } else {
#pragma unroll
            for (int z = 0; z < 16; ++z) ro[z] = 0;
          }
          tmem_st16(lane_addr + (uint32_t)(C::R_COL0 + rs * A_COLS + 16 * h), ro);
        }
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(bar(B_FULL_RU + rs));
          mbar_arrive(bar(B_EMPTY_RP + rs));
        }
      }
    }
  } else {
    // ===================== epilogue warps (2..5) =====================
    const int lq = warp & 3;  // TMEM lane quadrant this warp may access
    const int et = (warp - FIRST_EPI_WARP) * 32 + lane;  // 0..127 within the epilogue group
    const int n_loc = lq * 32 + lane;
    const long long my_first_tile = u_beg / p.KS;
    constexpr int PART = BT * BN;  // int32 elements of one partial accumulator
    int it = 0;
    long long g = u_beg;
    while (g < u_end) {
      const long long tile = g / p.KS;
      const int k0 = (int)(g % p.KS);
      const int k1 = (int)min((long long)p.KS, k0 + (u_end - g));
      g += k1 - k0;
      const int nt = (int)(tile / p.TT), tt = (int)(tile % p.TT);
      const int a = C::ACC_STAGES == 2 ? (it & 1) : 0;
      const uint32_t aphase = C::ACC_STAGES == 2 ? ((it >> 1) & 1) : (it & 1);
      ++it;
      const int n = nt * BN + n_loc;
      const int t_base = tt * BT;
      const int t_cnt = min(BT, p.M - t_base);
      const float swn = p.sw[n] * 0.00390625f, srn = p.sr[n] * 0.00390625f;  // / 256: accumulators are x256
      auto emit = [&](int t, int32_t a0, int32_t a1) {
        const float y = p.sa[t_base + t] * ((float)a0 * swn + (float)a1 * srn);
        const size_t o = (size_t)(t_base + t) * p.ldy + n;
        if (p.y_bf16)
          store_y<true>(p.Y, o, y);
        else
          store_y<false>(p.Y, o, y);
        if (p.dbg0) p.dbg0[(size_t)(t_base + t) * p.N + n] = a0 >> 8;
        if (p.dbg1) p.dbg1[(size_t)(t_base + t) * p.N + n] = a1 >> 8;
      };

      mbar_wait(bar(B_TFULL + a), aphase);
      tc_fence_after();
      MQ_STAMP_IF(et == 0 && it == 1, 9);
      const bool has_res = acc_flag[a] != 0;  // acc1 is undefined when no residual MMA was issued
      const uint32_t t0addr = tmem_base + ((uint32_t)(lq * 32) << 16) + (uint32_t)(a * 2 * BT);
      const bool whole = (k0 == 0 && k1 == p.KS);
      const int slot = tile == my_first_tile ? 0 : 1;
      int32_t* part0 = p.ws_part + ((size_t)blockIdx.x * 2 + slot) * (2 * PART);
      int32_t* part1 = part0 + PART;

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
        if (whole) {
#pragma unroll
          for (int i = 0; i < 16; ++i)
            if (c0 + i < t_cnt) emit(c0 + i, (int32_t)v0[i], (int32_t)v1[i]);
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i)
            if (c0 + i < t_cnt) {
              __stcg(part0 + (c0 + i) * BN + n_loc, (int32_t)v0[i]);
              if (has_res) __stcg(part1 + (c0 + i) * BN + n_loc, (int32_t)v1[i]);
            }
        }
      }
      // accumulator stage drained: hand it back to the MMA warp
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_TEMPTY + a));

      if (!whole) {
        // stream-K fix-up: the last CTA to arrive for this tile sums all partials and finishes it
        if (et == 0) p.ws_flag[blockIdx.x * 2 + slot] = has_res ? 1 : 0;
        __threadfence();
        named_bar_sync(1, 128);
        if (et == 0) {
          const int c_lo = owner_of(p, tile * p.KS), c_hi = owner_of(p, (tile + 1) * p.KS - 1);
          const int old = atomicAdd(p.ws_cnt + tile, 1);
          flag_slot[0] = (old == c_hi - c_lo);
          flag_slot[3] = c_lo;
          flag_slot[4] = c_hi;
        }
        named_bar_sync(1, 128);
        const bool last = flag_slot[0] != 0;
        const int c_lo = flag_slot[3], c_hi = flag_slot[4];
        named_bar_sync(1, 128);  // flag_slot may be rewritten by the next segment
        if (last) {
          __threadfence();
          for (int c0 = 0; c0 < t_cnt; c0 += 16) {
            int32_t s0[16], s1[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) s0[i] = s1[i] = 0;
            for (int c = c_lo; c <= c_hi; ++c) {
              const int cs = (range_begin(p, c) / p.KS == tile) ? 0 : 1;
              const int32_t* q0 = p.ws_part + ((size_t)c * 2 + cs) * (2 * PART) + n_loc;
              const bool cres = __ldcg(p.ws_flag + c * 2 + cs) != 0;
#pragma unroll
              for (int i = 0; i < 16; ++i)
                if (c0 + i < t_cnt) s0[i] += __ldcg(q0 + (c0 + i) * BN);
              if (cres) {
#pragma unroll
                for (int i = 0; i < 16; ++i)
                  if (c0 + i < t_cnt) s1[i] += __ldcg(q0 + PART + (c0 + i) * BN);
              }
            }
#pragma unroll
            for (int i = 0; i < 16; ++i)
              if (c0 + i < t_cnt) emit(c0 + i, s0[i], s1[i]);
          }
          if (et == 0) p.ws_cnt[tile] = 0;
        }
      }
      MQ_STAMP_IF(et == 0, 10);
    }
  }

  // teardown (single-lane roles re-converge first: bar.sync must be reached warp-convergent)
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

size_t align256(size_t x) { return (x + 255) / 256 * 256; }

struct Plan {
  int BT = 16, TT = 1, grid = 1, gran = 1;
  long long units = 0;
  size_t off_flag = 0, off_part = 0, ws_bytes = 0;
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
  pl.units = tiles * KS;
  // stream-K (ranges cut at K-step granularity) unless there are enough tiles to balance whole ones
  bool stream_k = tiles < 8LL * G;
  if (o.split_k == 1) stream_k = false;
  if (o.split_k >= 2) stream_k = true;
  pl.gran = stream_k ? 1 : KS;
  pl.grid = (int)std::min<int64_t>(G, pl.units / pl.gran);
  if (stream_k) {
    pl.off_flag = align256((size_t)tiles * 4);
    pl.off_part = pl.off_flag + align256((size_t)pl.grid * 2 * 4);
    pl.ws_bytes = pl.off_part + (size_t)pl.grid * 2 * 2 * bt * BN * 4;
  }
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

#ifdef MQ_TRACE
static long long* g_trace = nullptr;
extern "C" void mq_debug_set_trace(long long* dev_buf) { g_trace = dev_buf; }
#endif

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
  gp.unit_meta = (const int2*)w->d_unit_meta;
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
  gp.units = pl.units;
  gp.gran = pl.gran;
  gp.y_bf16 = y_dtype == MQ_BF16;
  uint8_t* ws = (uint8_t*)workspace;
  gp.ws_cnt = (int32_t*)ws;
  gp.ws_flag = (int32_t*)(ws + pl.off_flag);
  gp.ws_part = (int32_t*)(ws + pl.off_part);
#ifdef MQ_TRACE
  gp.trace = g_trace;
  if (!g_trace) return MQ_ERR_INVALID_ARG;
#endif

  cudaStream_t st = (cudaStream_t)cuda_stream;
  switch (pl.BT) {
    case 16: rc = launch<16>(tmap, gp, pl.grid, st); break;
    case 32: rc = launch<32>(tmap, gp, pl.grid, st); break;
    case 64: rc = launch<64>(tmap, gp, pl.grid, st); break;
    case 128: rc = launch<128>(tmap, gp, pl.grid, st); break;
    default: rc = MQ_ERR_INVALID_ARG;
  }
  if (rc == MQ_OK) mq::set_launch_count(1);
  return rc;
}

extern "C" size_t mq_linear_workspace_bytes(const mq_weights* w, int64_t M) {
  if (!w || M <= 0) return 0;
  size_t q = (mq_qact_bytes(M, w->K) + 255) / 256 * 256;
  size_t s = ((size_t)M * 4 + 255) / 256 * 256;
  return q + s + align256(mq_gemm_workspace_bytes(w, M));
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
  const size_t g_al = align256(g);
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
