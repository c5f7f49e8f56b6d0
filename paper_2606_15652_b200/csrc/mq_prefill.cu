// mq_prefill.cu -- the fused base + residual int4 GEMM for PREFILL shapes (M >= 64 tokens, many whole tiles):
// Eq.4, ZipperEngine on the tensor-bound side of the roofline.
//
// Same arithmetic and the same building blocks as mq_gemm.cu (weights expanded int4 -> int8 x16 in registers and
// written to TENSOR MEMORY as the MMA's A operand, tokens expanded into K-major SWIZZLE_128B shared memory as its B
// operand, tcgen05.mma kind::i8, base and residual accumulators in TMEM, fp32 epilogue), re-cut around what this
// round's measurements showed (profiles/r2_probe_int8.md, r2_ncu_prefill_gate_up_m8192.md):
//   * the tensor pipe runs at half speed while other agents write shared and tensor memory, so bytes moved per MAC
//     are what counts: CTA PAIRS (tcgen05.mma.cta_group::2, M = 256) halve the token expansion and the pipe's
//     shared-memory operand reads per SM;
//   * nobody's chain may contain a shared-memory round trip it does not need: the residual metadata lives in lanes
//     (one coalesced load per 32 K-steps), every role derives the item sequence from it by itself, the MMA warp polls
//     the next item's barrier before it issues the current item's MMAs;
//   * the base accumulator is double-buffered: the epilogue of a tile overlaps the K-loop of the next.
// Tensor memory (512 columns): acc0 2 x 128 | acc1 128 | A operand ring 4 x 32.  There is no room left for a residual
// operand, so a residual cell is an ITEM OF ITS OWN in the operand ring: right after the base item of its K-step, its
// expanded weights take the next A stage and its MMAs re-use the token tile of the base item (the paper's re-use of the
// quantized activation tile), accumulating into acc1 (s_r != s_w).
//
// Work: whole output tiles (128 output channels x 128 tokens; PAIR: 256 x 128 per cluster, each CTA its own n-tile and
// 64 of the tokens), tile T = n * TT + tt, dealt round-robin to the persistent CTAs / clusters (concurrent ones share
// n-tiles: weights and tokens stay in L2).  Roles (22 warps, one CTA per SM):
//   warp 0      producer (one thread): per K-step one bulk copy of 8 KB packed weights and one tensor copy of packed
//               tokens [128 (64) x 64 B] into a ring of 8 (16) stages
//   warps 6-21  four unpack groups of four warps; item i (base K-step, or residual cell) belongs to group i mod 4 and
//               to operand stage i mod 4.  Base item: packed weights -> int8 x16 -> tcgen05.st; packed tokens -> int8
//               x16 -> swizzled shared memory.  Residual item: the cell's packed quarters straight from global memory.
//   warp 1      MMA issuer (PAIR: the leader CTA's; the peer's only derives the per-tile residual flag)
//   warps 2-5   epilogue: tcgen05.ld, y = s_a (s_w acc0 + s_r acc1), 16-bit stores
// PAIR synchronisation: the unpack groups and epilogue warps of both CTAs arrive on the LEADER's barriers (remote
// mbarrier.arrive through mapa), the leader's tcgen05.commit multicasts to the barrier of the same name in both CTAs.
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

// Waits of the roles that wait most of the time (producer, unpack groups, epilogue): parked by the hardware (try_wait with
// a suspend-time hint) instead of spinning.  A spinning warp issues a try_wait, a counter update, a compare and a
// branch every few dozen cycles, on the same schedulers and the same ALU pipe the unpack warps need: with the waits
// parked the kernel runs 10-15 % faster (M = 8192: o 1779 -> 1959, gate_up 2092 -> 2346, down 2107 -> 2428 TOPS).
// PF_EXP_SPIN (development) brings the spinning waits back; PF_EXP_PARK_MMA parks the MMA warp's waits as well.
#ifdef PF_EXP_SPIN
#define PF_WAIT_SLACK(b, p) mbar_wait((b), (p))
#else
#define PF_WAIT_SLACK(b, p) mbar_wait_parked((b), (p))
#endif

constexpr int PF_BT = 128;                       // tokens per tile (MMA N)
constexpr int PF_UST = 4;                        // operand (U) stages = unpack groups
constexpr int PF_WARPS = 6 + 4 * PF_UST;
constexpr int PF_THREADS = 32 * PF_WARPS;
constexpr int PF_A_COLS = BK / 4;                // 32 TMEM columns hold 128 int8 per lane (one K-step)
constexpr int PF_ACC1_COL = 2 * PF_BT;
constexpr int PF_A_COL0 = 3 * PF_BT;
// shared-memory layout (PAIR: a CTA holds half of the token tile, so its stages are smaller and the packed ring deeper:
// the ring must cover the copies' latency under load, ~3000 cycles)
template <bool PAIR>
struct PfL {
  static constexpr int TOKR = PAIR ? PF_BT / 2 : PF_BT;          // token rows this CTA expands
  static constexpr int PST = PAIR ? 16 : 8;                      // packed (P) stages of one K-step (a power of two)
  static constexpr int U_STAGE = TOKR * BK;                      // int8 token sub-tile of one K-step
  static constexpr int TOK_KSTEP = TOKR * (BK / 2);              // packed tokens of one K-step
  static constexpr int P_STAGE = TILE_BYTES + TOK_KSTEP;         // packed weights | packed tokens
  static constexpr int OFF_U = 0;
  static constexpr int OFF_P = OFF_U + PF_UST * U_STAGE;
  static constexpr int OFF_BAR = OFF_P + PST * P_STAGE;
  // barriers: FULL_P[PST] EMPTY_P[PST] FULL_U[4] EMPTY_U[4] TFULL[2] A0E[2] A1E
  static constexpr int B_FULL_P = 0, B_EMPTY_P = PST, B_FULL_U = 2 * PST, B_EMPTY_U = B_FULL_U + PF_UST, B_TFULL = B_EMPTY_U + PF_UST,
                       B_A0E = B_TFULL + 2, B_A1E = B_A0E + 2, NUM_BARS = B_A1E + 1;
  static constexpr int OFF_MISC = OFF_BAR + NUM_BARS * 8 + 8;    // [0] tmem base, [1..2] residual flag of the acc0 buffer
  static constexpr int OFF_SA = (OFF_MISC + 16 + 15) / 16 * 16;  // [2][128] token scales of the tile being drained
  static constexpr int SMEM_BYTES = OFF_SA + 2 * PF_BT * 4 + 1024;   // + slack for the 1024-byte alignment
  static_assert(SMEM_BYTES <= 232448, "shared memory budget");
  static_assert(OFF_P % 1024 == 0 && P_STAGE % 1024 == 0 && U_STAGE % 1024 == 0, "swizzle atoms need 1024-byte alignment");
};
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
// W4A8: the int8 tokens come straight from global memory in canonical element order, so the weights are expanded in
// canonical order too: word 2i = elements (0,1,2,3), word 2i + 1 = elements (4,5,6,7) of the i-th group of eight
__device__ __forceinline__ void pf_unpack16c(const uint4& p, uint32_t* o) {
  const uint32_t HI = 0xF0F0F0F0u;
  const uint32_t w[4] = {p.x, p.y, p.z, p.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const uint32_t ev = (w[i] << 4) & HI, od = w[i] & HI;   // elements 0,2,4,6 | 1,3,5,7
    o[2 * i] = __byte_perm(ev, od, 0x5140);
    o[2 * i + 1] = __byte_perm(ev, od, 0x7362);
  }
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

// ---- CTA pairs (cluster of two CTAs on one TPC, tcgen05 cta_group::2) ----
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of `addr` (a shared::cta address of this CTA's window) in the CTA of rank `rank`
__device__ __forceinline__ uint32_t mapa_rank(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  // (default semantics: release at CTA scope.  What the arrival orders is this CTA's own writes before this CTA's
  // own tensor core reads them, triggered by the leader's MMA after it has seen the arrival; a cluster-scope release
  // costs ~1200 cycles per arrival here)
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait_cl(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait_cl(uint32_t bar, uint32_t parity) {
  uint32_t spins = 0;
  while (!mbar_try_wait_cl(bar, parity))
    if (++spins > (1u << 26)) __trap();
}
__device__ __forceinline__ void tmem_alloc2(uint32_t dst_smem, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_relinquish2() {
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc2(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// D[tmem of both CTAs: 128 rows each] (+)= A[tmem of both CTAs] * B[shared memory of both CTAs: half of N each]
__device__ __forceinline__ void mma_i8_ts2(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::i8 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(d_tmem),
      "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// arrives on the barrier at the same offset in both CTAs when the pair's previously issued MMAs have completed
__device__ __forceinline__ void tc_commit2(uint32_t bar) {
  const uint16_t mask = 3;
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar), "h"(mask) : "memory");
}

#ifndef PF_CL_WAIT   // 1: the leader's waits on barriers with remote arrivals use cluster-scope acquire
#define PF_CL_WAIT 0
#endif
#ifndef PF_EXP_NOW   // development experiments (timing only, wrong results): skip parts of the unpack
#define PF_EXP_NOW 0
#endif
#ifndef PF_EXP_NOT
#define PF_EXP_NOT 0
#endif
#ifndef PF_EXP_NOS
#define PF_EXP_NOS 0
#endif
#ifndef PF_EXP_NOTMA   // the producer signals its stages without copying anything
#define PF_EXP_NOTMA 0
#endif
#ifdef PF_TRACE   // development: clock stamps of CTA 0 into the dbg1 buffer (8 words per tile)
#define PF_STAMP(cond, it, slot) do { if (blockIdx.x == 0 && (cond)) reinterpret_cast<long long*>(p.dbg1)[(it) * 8 + (slot)] = clock64(); } while (0)
#define PF_ADD(cond, it, slot, v) do { if (blockIdx.x == 0 && (cond)) reinterpret_cast<long long*>(p.dbg1)[(it) * 8 + (slot)] += (v); } while (0)
#define PF_FINE(slot) do { if (blockIdx.x <= 1 && warp == 6 && lane == 0 && it == 5) reinterpret_cast<long long*>(p.dbg1)[4096 + blockIdx.x * 1024 + (n_mine & 127) * 8 + (slot)] = clock64(); } while (0)
#else
#define PF_FINE(slot) do { } while (0)
#define PF_STAMP(cond, it, slot) do { } while (0)
#define PF_ADD(cond, it, slot, v) do { } while (0)
#endif

// PAIR: the two CTAs of a cluster (one TPC) work on one 256-channel x 128-token tile pair: each expands the weights of
// its own n-tile into its own tensor memory and HALF of the token tile (64 tokens) into its own shared memory; the
// leader (rank 0) issues tcgen05.mma.cta_group::2 (M = 256) for both.  Per SM that halves the token expansion and the
// tensor pipe's shared-memory operand reads.
// A8 (W4A8, single-CTA form only): the tokens are int8 [M][K]; a tensor copy puts the tile's 128 x 128 B of a K-step
// straight into the operand stage in the MMA's SWIZZLE_128B layout (issued by the unpack group that owns the item, as
// soon as the stage is free): no token pass through the CUDA cores at all.  Accumulators are x16 (weights only).
template <bool PAIR, bool A8 = false>
__global__ void __launch_bounds__(PF_THREADS, 1) mq_prefill_kernel(const __grid_constant__ CUtensorMap tmap_a, const PfParams p) {
  static_assert(!(PAIR && A8), "W4A8 runs in the single-CTA form");
  using L = PfL<PAIR>;
  constexpr int PF_PST = L::PST, PF_U_STAGE = L::U_STAGE, PF_P_STAGE = L::P_STAGE, PF_OFF_U = L::OFF_U, PF_OFF_P = L::OFF_P,
                PF_OFF_BAR = L::OFF_BAR, PF_OFF_MISC = L::OFF_MISC, PF_OFF_SA = L::OFF_SA, PF_B_FULL_P = L::B_FULL_P,
                PF_B_EMPTY_P = L::B_EMPTY_P, PF_B_FULL_U = L::B_FULL_U, PF_B_EMPTY_U = L::B_EMPTY_U, PF_B_TFULL = L::B_TFULL,
                PF_B_A0E = L::B_A0E, PF_B_A1E = L::B_A1E;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sU = smem_base + PF_OFF_U, sP = smem_base + PF_OFF_P, sBar = smem_base + PF_OFF_BAR,
                 sMisc = smem_base + PF_OFF_MISC;
  auto bar = [&](int i) { return sBar + 8u * (uint32_t)i; };
  volatile int32_t* misc = reinterpret_cast<volatile int32_t*>(smem_raw + (sMisc - smem_u32(smem_raw)));
  float* sa_tile = reinterpret_cast<float*>(smem_raw + (smem_base + PF_OFF_SA - smem_u32(smem_raw)));   // [2][128]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int KS = p.KS;
  const uint32_t rank = PAIR ? cluster_ctarank() : 0u;
  const bool leader = rank == 0;
  const int tile0 = PAIR ? (int)(blockIdx.x >> 1) : (int)blockIdx.x, tstride = PAIR ? (int)(gridDim.x >> 1) : (int)gridDim.x;
  constexpr int TOKR = L::TOKR;
  constexpr uint32_t TOK_BYTES = L::TOK_KSTEP;
  // n-tile of tile T for this CTA
  auto nt_of = [&](int T) { return PAIR ? 2 * (T / p.TT) + (int)rank : T / p.TT; };

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmap_a);
    for (int i = 0; i < PF_PST; ++i) {
      mbar_init(bar(PF_B_FULL_P + i), 1);            // the producer's arrival; the copies complete the transaction count
      mbar_init(bar(PF_B_EMPTY_P + i), 4);           // the four warps of the group that owns the K-step
    }
    for (int i = 0; i < PF_UST; ++i) {
      mbar_init(bar(PF_B_FULL_U + i), PAIR ? 8 : 4);   // (the leader's: four warps of the group in each CTA)
      mbar_init(bar(PF_B_EMPTY_U + i), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar(PF_B_TFULL + i), 2);             // the MMA thread's arrival (publishes the residual flag) + tcgen05.commit
      mbar_init(bar(PF_B_A0E + i), PAIR && leader ? 8 : 4);   // the leader's: the epilogue warps of both CTAs
    }
    mbar_init(bar(PF_B_A1E), PAIR ? 8 : 4);
    fence_mbar_init();
  }
  if (warp == 1) {
    if (PAIR) {
      tmem_alloc2(sMisc, 512);
      tmem_relinquish2();
    } else {
      tmem_alloc(sMisc, 512);
      tmem_relinquish();
    }
  }
  tc_fence_before();
  if (PAIR) cluster_sync_all();   // the peer's barriers are initialised before anybody arrives on them
  else __syncthreads();
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
  // (PAIR: .z = the quarter mask of the peer's n-tile; a K-step has a residual item when either n-tile has a cell)
  auto load_chunk = [&](int T, int c0) -> int3 {
    int3 v = make_int3(0, 0, 0);
    if (p.unit_meta && T < p.tiles && c0 + lane < KS) {
      const int2 own = __ldg(p.unit_meta + (size_t)nt_of(T) * KS + c0 + lane);
      v.x = own.x;
      v.y = own.y;
      if (PAIR) v.z = __ldg(p.unit_meta + (size_t)(nt_of(T) ^ 1) * KS + c0 + lane).x;
    }
    return v;
  };
  auto next_chunk = [&](int& T, int& c0) {
    c0 += 32;
    if (c0 >= KS) {
      c0 = 0;
      T += tstride;
    }
  };

  if (warp == 0) {
    if (lane == 0) {
      // ===================== producer (one thread): one K-step per stage =====================
      if (!A8) griddep_wait();   // the packed tokens are the previous kernel's output (A8: only static weights here)
      uint32_t q = 0;
      for (int T = tile0; T < p.tiles; T += tstride) {
        const int nt = nt_of(T), tt = T % p.TT;
        const uint8_t* wsrc = p.base + (size_t)nt * KS * TILE_BYTES;
        for (int ks = 0; ks < KS; ++ks, ++q) {
          const uint32_t ps = q % PF_PST;
          PF_WAIT_SLACK(bar(PF_B_EMPTY_P + ps), ((q / PF_PST) & 1) ^ 1);
          const uint32_t fb = bar(PF_B_FULL_P + ps), dst = sP + ps * PF_P_STAGE;
          if (PF_EXP_NOTMA) {
            mbar_arrive(fb);
            continue;
          }
          mbar_arrive_expect_tx(fb, TILE_BYTES + (A8 ? 0u : TOK_BYTES));
          tma_load_1d(dst, wsrc + (size_t)ks * TILE_BYTES, TILE_BYTES, fb);
          if (!A8) tma_load_2d(dst + TILE_BYTES, &tmap_a, ks * (BK / 2), tt * PF_BT + (int)rank * TOKR, fb);
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer: warp-uniform control, one elected lane issues =====================
    constexpr uint32_t IDESC = make_idesc_i8(PAIR ? 2 * BN : BN, PF_BT);
    int it = 0;
    int pT = tile0, pc0 = 0;
    int3 um_next = load_chunk(pT, pc0);
    if (PAIR && !leader) {
      // the peer's MMA warp issues nothing: it only derives, per tile, whether the pair accumulated a residual, and
      // publishes that flag to its own epilogue warps (the leader's commit completes the phase in both CTAs)
      for (int T = tile0; T < p.tiles; T += tstride, ++it) {
        const int buf = it & 1;
        mbar_wait(bar(PF_B_A0E + buf), (((uint32_t)it >> 1) & 1) ^ 1);   // (local copy: the flag word is free again)
        uint32_t any = 0;
        for (int c0 = 0; c0 < KS; c0 += 32) {
          const int3 um = um_next;
          next_chunk(pT, pc0);
          um_next = load_chunk(pT, pc0);
          any |= __ballot_sync(0xffffffffu, ((um.x | um.z) & 0xF) != 0);
        }
        if (lane == 0) {
          misc[1 + buf] = any != 0;
          mbar_arrive(bar(PF_B_TFULL + buf));
        }
        __syncwarp();
      }
    } else {
    uint32_t item = 0;
    bool pre_ok = false;   // the barrier of the item about to be processed was already seen complete
    // the operand stage of item i: FULL_U[i & 3], phase (i >> 2) & 1.  The next item's barrier is polled once BEFORE
    // this item's MMAs are issued, so that the round trip hides under the tensor pipe's work.
    // (PAIR: the barriers collect arrivals from both CTAs: cluster-scope acquire)
#ifdef PF_TRACE
    long long tr_wait = 0, tr_nwait = 0, tr_pollok = 0, tr_pollno = 0, tr_fence = 0, tr_issue = 0;
#endif
    auto wait_b = [&](uint32_t b, uint32_t par) {
      if (PAIR && PF_CL_WAIT) mbar_wait_cl(b, par);
#ifdef PF_EXP_PARK_MMA
      else mbar_wait_parked(b, par);
#else
      else mbar_wait(b, par);
#endif
    };
    auto acquire = [&]() {
#ifdef PF_TRACE
      if (!pre_ok) {
        const long long c0 = clock64();
        wait_b(bar(PF_B_FULL_U + (int)(item & 3)), (item >> 2) & 1);
        tr_wait += clock64() - c0;
        tr_nwait += 1;
      }
#else
      if (!pre_ok) wait_b(bar(PF_B_FULL_U + (int)(item & 3)), (item >> 2) & 1);
#endif
#ifdef PF_TRACE
      const long long cf0 = clock64();
#endif
      tc_fence_after();
#ifdef PF_TRACE
      const long long cf1 = clock64();
#endif
      const uint32_t nb = bar(PF_B_FULL_U + (int)((item + 1) & 3)), np = ((item + 1) >> 2) & 1;
      pre_ok = PAIR && PF_CL_WAIT ? mbar_try_wait_cl(nb, np) : mbar_try_wait(nb, np);
#ifdef PF_TRACE
      if (pre_ok) tr_pollok += clock64() - cf1;   // poll that found the phase complete
      else tr_pollno += clock64() - cf1;          // poll that did not
      tr_fence += cf1 - cf0;
#endif
    };
    auto mma = [&](uint32_t d, uint32_t a, uint64_t b, uint32_t on) {
      if (PAIR) mma_i8_ts2(d, a, b, IDESC, on);
      else mma_i8_ts(d, a, b, IDESC, on);
    };
    auto commit = [&](uint32_t b) {
      if (PAIR) tc_commit2(b);
      else tc_commit(b);
    };
    for (int T = tile0; T < p.tiles; T += tstride, ++it) {
      const int buf = it & 1;
      PF_STAMP(lane == 0, it, 3);
      wait_b(bar(PF_B_A0E + buf), (((uint32_t)it >> 1) & 1) ^ 1);   // the epilogue has drained this base accumulator
      PF_STAMP(lane == 0, it, 4);
      tc_fence_after();
      const uint32_t d0 = tmem_base + (uint32_t)(buf * PF_BT), d1 = tmem_base + (uint32_t)PF_ACC1_COL;
      uint32_t acc0_on = 0, acc1_on = 0;
      for (int c0 = 0; c0 < KS; c0 += 32) {
        const int3 um = um_next;
        next_chunk(pT, pc0);
        um_next = load_chunk(pT, pc0);
        const uint32_t bits = __ballot_sync(0xffffffffu, ((um.x | um.z) & 0xF) != 0);
        const int nk = min(32, KS - c0);
        for (int j = 0; j < nk; ++j) {
          const bool has = (bits >> j) & 1;
          const int us = (int)(item & 3);
          acquire();
          const uint32_t at = tmem_base + (uint32_t)(PF_A_COL0 + us * PF_A_COLS);
          const uint64_t dt = make_desc_sw128(sU + us * PF_U_STAGE);
#ifdef PF_TRACE
          const long long ci0 = clock64();
#endif
          if (elect_one()) {
#pragma unroll
            for (int k = 0; k < 4; ++k) mma(d0, at + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), k == 0 ? acc0_on : 1u);
            if (!has) commit(bar(PF_B_EMPTY_U + us));
          }
          __syncwarp();
#ifdef PF_TRACE
          tr_issue += clock64() - ci0;
#endif
          acc0_on = 1;
          ++item;
          if (has) {
            // residual cell of this K-step: its weights in the next stage's A columns, the tokens of this K-step's
            // stage (the paper's re-use of the activation tile), second accumulator
            const uint32_t mask = (uint32_t)__shfl_sync(0xffffffffu, um.x | um.z, j) & 0xF;
            const int us2 = (int)(item & 3);
            acquire();
            if (!acc1_on) {
              wait_b(bar(PF_B_A1E), ((uint32_t)it & 1) ^ 1);   // the epilogue has read the previous tile's acc1
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
                    mma(d1, at2 + (uint32_t)(k * 8), dt + (uint64_t)(k * 2), on);
                    on = 1;
                  }
                }
              commit(bar(PF_B_EMPTY_U + us2));
              commit(bar(PF_B_EMPTY_U + us));
            }
            __syncwarp();
            acc1_on = 1;
            ++item;
          }
        }
      }
#ifdef PF_TRACE
      if (blockIdx.x == 0 && lane == 0) {
        long long* tb = reinterpret_cast<long long*>(p.dbg1) + it * 8;
        tb[0] = tr_pollok; tb[1] = tr_pollno; tb[2] = tr_issue; tb[5] = tr_fence; tb[6] = tr_wait; tb[7] = tr_nwait;
      }
      tr_wait = tr_nwait = tr_pollok = tr_pollno = tr_fence = tr_issue = 0;
#endif
      if (elect_one()) {
        misc[1 + buf] = (int32_t)acc1_on;
        mbar_arrive(bar(PF_B_TFULL + buf));   // release: publishes the flag to the epilogue warps
        commit(bar(PF_B_TFULL + buf));        // completes the phase when the MMAs have finished
      }
      __syncwarp();
    }
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
    const uint32_t full_u_leader = PAIR ? mapa_rank(bar(PF_B_FULL_U + g), 0) : 0u;
    auto publish = [&]() {   // the item is in place: tell the MMA warp
      PF_FINE(4);
      tmem_st_wait();
      PF_FINE(5);
      tc_fence_before();
      fence_proxy_async_smem();
      __syncwarp();
      PF_FINE(6);
      if (lane == 0) {
        if (PAIR) mbar_arrive_cluster(full_u_leader);   // the leader's barrier collects both CTAs' groups
        else mbar_arrive(bar(PF_B_FULL_U + g));
      }
      PF_FINE(7);
      ++n_mine;
    };
    if (A8) griddep_wait();   // the int8 tokens this group requests are the previous kernel's output
    int pT = tile0, pc0 = 0;
    int3 um_next = load_chunk(pT, pc0);
    for (int T = tile0; T < p.tiles; T += tstride) {
#ifdef PF_TRACE
      ++it;
#endif
      for (int c0 = 0; c0 < KS; c0 += 32) {
        const int3 um = um_next;
        next_chunk(pT, pc0);
        um_next = load_chunk(pT, pc0);
        const uint32_t bits = __ballot_sync(0xffffffffu, ((um.x | um.z) & 0xF) != 0);
        const int nk = min(32, KS - c0);
        for (int j = 0; j < nk; ++j) {
          const uint32_t idx = item + (uint32_t)j + (uint32_t)__popc(bits & ((1u << j) - 1));   // item number of K-step j's base item
          const bool has = (bits >> j) & 1;
          if ((idx & 3) == (uint32_t)g) {
            // ---- base item ----
            const uint32_t ps = (q + (uint32_t)j) % PF_PST;
            PF_FINE(0);
            PF_WAIT_SLACK(bar(PF_B_FULL_P + ps), ((q + (uint32_t)j) / PF_PST) & 1);
            PF_FINE(1);
            constexpr int TL = PAIR ? 2 : 4;   // 16-byte token chunks per thread
            uint4 v4[4], t4[TL];
            const uint32_t pw = sP + ps * PF_P_STAGE, pt = pw + TILE_BYTES;
#pragma unroll
            for (int c = 0; c < 4; ++c) v4[c] = PF_EXP_NOW ? make_uint4(row, c, ps, g) : pf_lds128(pw + c * (BN * 16) + row * 16);
#pragma unroll
            for (int i = 0; i < TL; ++i)
              t4[i] = (A8 || PF_EXP_NOT) ? make_uint4(row, i, ps, g) : pf_lds128(pt + (gtid + 128u * i) * 16);
            PF_FINE(2);
            PF_WAIT_SLACK(bar(PF_B_EMPTY_U + g), (n_mine & 1) ^ 1);   // the poll runs under the loads' latency
            tc_fence_after();
            PF_FINE(3);
            if (A8 && gtid == 0) {   // the stage is free: request the K-step's int8 token tile straight into it
              mbar_expect_tx(bar(PF_B_FULL_U + g), (uint32_t)PF_U_STAGE);
              tma_load_2d(su, &tmap_a, (c0 + j) * BK, (T % p.TT) * PF_BT, bar(PF_B_FULL_U + g));
            }
            {
              uint32_t o[32];
#pragma unroll
              for (int c = 0; c < 4; ++c) {
                if (A8) pf_unpack16c(v4[c], o + 8 * c);
                else pf_unpack16(v4[c], o + 8 * c);
              }
              tmem_st32(lane_addr, o);
            }
#pragma unroll
            for (int i = 0; i < (A8 ? 0 : TL); ++i) {
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
            const uint32_t rmask = (uint32_t)__shfl_sync(0xffffffffu, um.x, j) & 0xF;   // this n-tile's quarters
            const uint32_t qoff = (uint32_t)__shfl_sync(0xffffffffu, um.y, j);
            // the k-halves the MMA reads: those with a quarter in either CTA's cell (this CTA's rows are zero elsewhere)
            const uint32_t umask = PAIR ? (rmask | ((uint32_t)__shfl_sync(0xffffffffu, um.z, j) & 0xF)) : rmask;
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
            PF_WAIT_SLACK(bar(PF_B_EMPTY_U + g), (n_mine & 1) ^ 1);
            tc_fence_after();
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              if (!(umask & (3u << (2 * h)))) continue;   // k-half without any block: never read by the MMA
              uint32_t ro[16];
              if (A8) {
                pf_unpack16c(r4[h][0], ro);
                pf_unpack16c(r4[h][1], ro + 8);
              } else {
                pf_unpack16(r4[h][0], ro);
                pf_unpack16(r4[h][1], ro + 8);
              }
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
    const uint32_t a1e_leader = PAIR ? mapa_rank(bar(PF_B_A1E), 0) : 0u;
    for (int T = tile0; T < p.tiles; T += tstride, ++it) {
      const int nt = nt_of(T), tt = T % p.TT, buf = it & 1;
      const int n = nt * BN + n_loc, t_base = tt * PF_BT;
      const int t_cnt = min(PF_BT, p.M - t_base);
      constexpr float ACC_INV = A8 ? 0.0625f : 0.00390625f;   // accumulators are x256 (both operands x16), A8: x16
      constexpr int ACC_SHIFT = A8 ? 4 : 8;
      const float swn = __ldg(p.sw + n) * ACC_INV, srn = __ldg(p.sr + n) * ACC_INV;
      float* sat = sa_tile + buf * PF_BT;
      sat[et] = et < t_cnt ? __ldg(p.sa + t_base + et) : 0.f;
      named_bar_sync(1, 128);   // also orders this buffer's readers (two tiles ago) before its writers
      PF_WAIT_SLACK(bar(PF_B_TFULL + buf), ((uint32_t)it >> 1) & 1);
      tc_fence_after();
      const bool has_res = misc[1 + buf] != 0;   // acc1 is undefined when no residual MMA was issued
      const uint32_t t0addr = tmem_base + lane_off + (uint32_t)(buf * PF_BT), t1addr = tmem_base + lane_off + (uint32_t)PF_ACC1_COL;
      uint16_t* yp0 = reinterpret_cast<uint16_t*>(p.Y) + (size_t)t_base * p.ldy + n;
      // 8-token batches, two in flight: the TMEM loads of batch b+1 run under the arithmetic and the stores of batch b.
      // FULL = whole token tile and no parity hooks: branch-free, one pointer bump per token.
      auto drain = [&](auto res_c, auto bf_c) {
        constexpr bool RES = decltype(res_c)::value, BF = decltype(bf_c)::value;
        uint16_t* yp = yp0;
        uint32_t a[2][8], r[2][8];
#pragma unroll
        for (int i = 0; i < 8; ++i) r[0][i] = r[1][i] = 0;
        auto emit8 = [&](const uint32_t* av, const uint32_t* rv, int b) {
          const float4 s_lo = *reinterpret_cast<const float4*>(sat + b * 8);
          const float4 s_hi = *reinterpret_cast<const float4*>(sat + b * 8 + 4);
          const float sv[8] = {s_lo.x, s_lo.y, s_lo.z, s_lo.w, s_hi.x, s_hi.y, s_hi.z, s_hi.w};
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            float y = (float)(int32_t)av[i] * swn;
            if (RES) y += (float)(int32_t)rv[i] * srn;
            y *= sv[i];
            *yp = BF ? __bfloat16_as_ushort(__float2bfloat16_rn(y)) : __half_as_ushort(__float2half_rn(y));
            yp += p.ldy;
          }
        };
        tmem_ld8(t0addr, a[0]);
        if (RES) tmem_ld8(t1addr, r[0]);
        // (a rolled loop of two batches: the fully unrolled form of all variants was 700 KB of code)
#pragma unroll 1
        for (int b = 0; b < PF_BT / 8; b += 2) {
          tmem_ld_wait8(a[0], r[0]);
          tmem_ld8(t0addr + (b + 1) * 8, a[1]);
          if (RES) tmem_ld8(t1addr + (b + 1) * 8, r[1]);
          emit8(a[0], r[0], b);
          tmem_ld_wait8(a[1], r[1]);
          if (b + 2 < PF_BT / 8) {
            tmem_ld8(t0addr + (b + 2) * 8, a[0]);
            if (RES) tmem_ld8(t1addr + (b + 2) * 8, r[0]);
          }
          emit8(a[1], r[1], b + 1);
        }
      };
      if (t_cnt == PF_BT && !p.dbg0 && !p.dbg1) {
        if (has_res) {
          if (p.y_bf16) drain(std::true_type{}, std::true_type{}); else drain(std::true_type{}, std::false_type{});
        } else {
          if (p.y_bf16) drain(std::false_type{}, std::true_type{}); else drain(std::false_type{}, std::false_type{});
        }
      } else {
        // ragged last token tile, or the parity hooks are on: one generic loop, same operation order
#pragma unroll 1
        for (int b = 0; b < PF_BT / 8; ++b) {
          if (b * 8 >= t_cnt) break;
          uint32_t a[8], r[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) r[i] = 0;
          tmem_ld8(t0addr + b * 8, a);
          if (has_res) tmem_ld8(t1addr + b * 8, r);
          tmem_ld_wait8(a, r);
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int t = b * 8 + i;
            if (t < t_cnt) {
              float y = (float)(int32_t)a[i] * swn;
              if (has_res) y += (float)(int32_t)r[i] * srn;
              y *= sat[t];
              yp0[(size_t)t * p.ldy] = p.y_bf16 ? __bfloat16_as_ushort(__float2bfloat16_rn(y)) : __half_as_ushort(__float2half_rn(y));
              const size_t di = (size_t)(t_base + t) * p.N + n;
              if (p.dbg0) p.dbg0[di] = (int32_t)a[i] >> ACC_SHIFT;
#ifndef PF_TRACE
              if (p.dbg1) p.dbg1[di] = has_res ? ((int32_t)r[i] >> ACC_SHIFT) : 0;
#endif
            }
          }
        }
      }
      // accumulators drained: hand them back to the MMA warp
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (PAIR) {
          mbar_arrive_cluster(a1e_leader);
          mbar_arrive_cluster(mapa_rank(bar(PF_B_A0E + buf), 0));
          if (!leader) mbar_arrive(bar(PF_B_A0E + buf));   // local copy: paces the peer's flag writer
        } else {
          mbar_arrive(bar(PF_B_A1E));
          mbar_arrive(bar(PF_B_A0E + buf));
        }
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
  if (PAIR) cluster_sync_all();   // neither CTA frees tensor memory (or exits) while the pair's MMAs or remote arrivals are in flight
  else __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    if (PAIR) tmem_dealloc2(tmem_base, 512);
    else tmem_dealloc(tmem_base, 512);
  }
}

}  // namespace

namespace mq {

// Whole-tile scheduling has no stream-K tail: take the shapes whose last round of tiles is mostly full.
// CTA pairs need an even number of n-tiles
static bool prefill_use_pairs(const mq_weights* w) {
  const int64_t pp = options().prefill_path;
  return pp != 2 && (w->N / BN) % 2 == 0 && sm_count() >= 2;
}

bool prefill_eligible(const mq_weights* w, int64_t M, bool a8) {
  const Options& o = options();
  if (!w || w->blockscale || o.prefill_path == 1) return false;
  if (o.token_tile || o.split_k >= 2 || o.max_ctas || o.fused_quant) return false;   // knobs of the stream-K kernel
  if (M < 64) return false;
  if (o.prefill_path >= 2) return true;
  const bool pairs = !a8 && prefill_use_pairs(w);
  const int64_t tiles = (w->N / BN) * ((M + PF_BT - 1) / PF_BT) / (pairs ? 2 : 1);
  const int64_t slots = pairs ? sm_count() / 2 : sm_count();
  const int64_t rounds = (tiles + slots - 1) / slots;
  // (W4A8: the token tile of an item is requested only when its operand stage is free, so a CTA needs a few tiles to
  // amortise that latency: measured crossover against the stream-K kernel between one and five rounds)
  if (a8 && tiles < 3 * slots) return false;
  return tiles * 100 >= rounds * slots * 50;
}

int prefill_gemm(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                 int32_t* dbg0, int32_t* dbg1, void* cuda_stream, bool ignore_res, bool a8) {
  typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  EncodeTiledFn enc = (EncodeTiledFn)tensor_map_encode_fn();
  if (!enc) return MQ_ERR_CUDA;
  // 2-D tensor map over the canonical packed activations [M rows][K/2 bytes]: box = one K-step of one token tile;
  // rows past M read as zero
  CUtensorMap tmap;
  memset(&tmap, 0, sizeof(tmap));
  // (W4A8: int8 activations [M rows][K bytes]; box = 128 B x 128 rows, written in the MMA's SWIZZLE_128B layout)
  const cuuint64_t row_bytes = a8 ? (cuuint64_t)w->K : (cuuint64_t)(w->K / 2);
  const cuuint64_t gdim[2] = {row_bytes, (cuuint64_t)M};
  const cuuint64_t gstride[1] = {row_bytes};
  const bool pairs = !a8 && prefill_use_pairs(w);
  const cuuint32_t box[2] = {(cuuint32_t)(a8 ? BK : BK / 2), (cuuint32_t)(pairs ? PF_BT / 2 : PF_BT)};
  const cuuint32_t estr[2] = {1, 1};
  if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(qA), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
          a8 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
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
  const int64_t tiles = (int64_t)pp.NT * pp.TT / (pairs ? 2 : 1);   // (pairs: 256-channel x 128-token tile pairs)
  if (tiles >= ((int64_t)1 << 31)) return MQ_ERR_UNSUPPORTED_SHAPE;
  pp.tiles = (int)tiles;
  pp.y_bf16 = y_dtype == MQ_BF16;

  auto kern = a8 ? mq_prefill_kernel<false, true> : (pairs ? mq_prefill_kernel<true> : mq_prefill_kernel<false>);
  const int smem_bytes = pairs ? PfL<true>::SMEM_BYTES : PfL<false>::SMEM_BYTES;
  static int attr_dev[3] = {-1, -1, -1};   // the attribute belongs to the (device, function) pair
  const int kidx = a8 ? 2 : (pairs ? 1 : 0);
  int dev = -1;
  cudaGetDevice(&dev);
  if (dev != attr_dev[kidx]) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes) != cudaSuccess) {
      cudaGetLastError();
      return MQ_ERR_CUDA;
    }
    attr_dev[kidx] = dev;
  }
  cudaLaunchConfig_t cfg = {};
  const int64_t slots = pairs ? sm_count() / 2 : sm_count();
  cfg.gridDim = dim3((unsigned)(std::min<int64_t>(tiles, slots) * (pairs ? 2 : 1)));
  cfg.blockDim = dim3(PF_THREADS);
  cfg.dynamicSmemBytes = smem_bytes;
  cfg.stream = (cudaStream_t)cuda_stream;
  cudaLaunchAttribute attr[2];
  int na = 0;
  if (pairs) {
    attr[na].id = cudaLaunchAttributeClusterDimension;
    attr[na].val.clusterDim.x = 2;
    attr[na].val.clusterDim.y = 1;
    attr[na].val.clusterDim.z = 1;
    ++na;
  }
  if (options().pdl) {
    attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
  }
  cfg.attrs = attr;
  cfg.numAttrs = na;
  if (cudaLaunchKernelEx(&cfg, kern, tmap, pp) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  set_launch_count(1);
  return MQ_OK;
}

}  // namespace mq
