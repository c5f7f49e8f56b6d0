// mq_decode.cu -- the fused base + residual int4 GEMM for DECODE shapes (M <= 32 tokens): Eq.4,
// ZipperEngine on the HBM-bound side of the roofline.
//
// With 1..32 tokens the op is a matrix-vector product: 4*M integer operations per weight byte, the weight
// stream from HBM is the only cost that matters and every microsecond of fixed latency shows (a whole
// projection is 9-60 MB = 1.4-9 us of HBM time).  Tensor memory buys nothing here.  What the
// timelines of the first versions showed (profiles/r2_decode_timeline.md):
//   * a single-thread role (TMA producer) pays ~500 cycles per loop iteration whatever it moves, so an
//     8 KB hand-off caps a CTA at ~29 GB/s: hand-offs must be 8-16 KB and cost ONE copy instruction;
//   * a K-split across CTAs costs 3.5 us of fix-up (stores, fence, ticket, second fence, reduction), more than
//     the whole HBM time of a small projection: the split must stay inside the CTA.
// Hence ROW SLABS: a CTA owns R = 16 / 32 / 64 / 128 output channels and ALL of K (N / R CTAs, R chosen so
// that they are resident together), and needs no workspace, no atomics and no inter-CTA reduction.
//
//   * warp 8 (producer, one thread): per STAGE of UK K-steps ONE tensor-map copy of the slab's packed
//     weights (the device layout [n-tile][K-step][4 chunks][128 rows][16 B] seen as a 3-D tensor: 16-byte
//     row pieces x chunks along K x n-tiles; 8-16 KB per copy) and ONE tensor-map copy of the stage's packed
//     tokens [UK][MT x 64 B, SWIZZLE_64B]; warp 9 (one thread): one bulk copy per selected residual piece of
//     the stage (CSR metadata: unit_meta; "prefetch sparse residual blocks") into a FIFO ring, in
//     parallel with the dense stream so that a residual block never delays it.  The weights are static, so the first
//     ring-full is requested BEFORE griddepcontrol.wait: it streams while the previous kernel in the stream is
//     still running (a CTA needs < half an SM, so both kernels are resident together);
//   * warps 0-7 (consumers): warp = (row tile rt of 16 channels, K group kw): the K-steps of a stage are dealt
//     to the 8 / RT K groups.  ldmatrix fetches the packed words, two logic operations expand 8 nibbles to
//     8 int8 = 16 x value (both operands in the same K slots, so the K permutation cancels and the
//     accumulators are 256 x the exact sums), mma.sync.m16n8k32.s8 accumulates; the residual pieces of a
//     K-step are multiplied by the SAME token fragments into a second accumulator set (the paper's re-use of
//     the quantized activation tile; separate because s_r != s_w);
//   * the K groups meet in shared memory (int32, exact), then the epilogue (Eq.2, Eq.4):
//     y = s_a (s_w acc0 + s_r acc1) in fp32, one rounding to bf16 / fp16, coalesced along the channels.
// Two more forms of the same kernel: BSC (block-local residual scales, reading A4b: a piece's integer sum is scaled
// and added in fp32 right after its MMAs) and GRP (per-group activation scales, group = 128 = one K-step, P:441:
// the K-step's sums are scaled by s_a[t, g] and added in fp32 right after its MMAs, 16 tokens at a time; serves
// mq_gemm_group for M <= 32), and A8 (W4A8: int8 tokens go into the MMA as they are, the weight nibbles are
// expanded in canonical order; serves mq_gemm_a8 at decode sizes).
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>

#include "mq_internal.h"
#include "mq_ptx.cuh"

namespace {

using namespace mq;
using namespace mq::ptx;

constexpr int DEC_CWARPS = 8;          // consumer warps
constexpr int DEC_THREADS = 32 * (DEC_CWARPS + 2);   // + warp 8: weight / token producer, warp 9: residual producer
constexpr int DEC_QSLOTS = 16;         // residual pieces in flight per CTA (a FIFO ring); >= the pieces of one stage
constexpr int DEC_MAX_KS = 512;        // K-steps whose metadata fits the shared-memory table (K <= 65536)

// BIG: one CTA per SM with a ring of ~200 KB, for long-K layers with few slabs (K >> N): the bytes in flight, not
// the CTA count, are then what keeps HBM busy (measured: 14336 x 4096 at 32 rows: 10.8 us with 64 KB per CTA in flight)
// BSC: block-local residual scales (reading A4b): every residual piece carries one scale per row; its integer sum is
// converted and added in fp32 right after its two MMAs (the scale changes along K, so the sums of different blocks
// cannot share an integer accumulator).
// GRP: per-group activation scales, group = 128 = one K-step (reading A5g; mq_gemm_group for M <= 32): the integer
// sums of a K-step are converted and added to fp32 running sums right after its MMAs,
//   y += s_a[t, g] * (s_w * acc0_g)  (+ s_a[t, g] * (s_r * acc1_g) for a K-step that owns residual pieces),
// in mq_group.cu's order; the K groups' fp32 partial sums meet in shared memory in ascending order (tolerance T2).
// A8 (W4A8): the tokens are int8 [M][K] in canonical order and go into the MMA as they are (128 bytes per token
// and K-step, SWIZZLE_128B); the weight nibbles are expanded into canonical order too (two byte permutes more per word);
// the accumulators are 16 x the sums.
template <int RT, int MT, bool BIG = false, bool BSC = false, bool GRP = false, bool A8 = false>
struct DCfg {
  static constexpr int R = 16 * RT;                     // output channels per CTA
  static constexpr int KW = DEC_CWARPS / RT;            // K groups (warps that share a row tile)
  static constexpr int UK = RT <= 2 ? 8 : (RT == 4 ? 4 : 2);   // K-steps per stage
  static constexpr int KPW = UK / KW;                   // K-steps per warp and stage
  static constexpr int NST = MT / 8;                    // 8-token MMA column groups
  static constexpr int CH_BYTES = R * 16;               // one 32-channel chunk of the slab
  static constexpr int W_BYTES = 4 * UK * CH_BYTES;     // packed weights of a stage (8 or 16 KB)
  static constexpr int T_KSTEP = MT * (A8 ? BK : BK / 2);   // tokens of one K-step (packed int4, A8: int8)
  static constexpr int T_BYTES = UK * T_KSTEP;
  static constexpr int P_ROWS = R < 64 ? R : 64;        // rows of a residual piece (one k-half of a quarter)
  static constexpr int P_BYTES = P_ROWS * 32;
  static constexpr int PS_BYTES = P_BYTES + (BSC ? P_ROWS * 4 : 0);   // ring slot: codes + (BSC) the rows' scales
  static constexpr int RING = (BIG ? 217088 : 106496) - DEC_QSLOTS * PS_BYTES;
  static constexpr int MAXST = BIG ? 12 : 6;
  static constexpr int STAGES = RING / (W_BYTES + T_BYTES) > MAXST ? MAXST : RING / (W_BYTES + T_BYTES);
  static constexpr int OFF_W = 0;
  static constexpr int OFF_T = OFF_W + STAGES * W_BYTES;
  static constexpr int OFF_Q = OFF_T + STAGES * T_BYTES;
  static constexpr int OFF_BAR = OFF_Q + DEC_QSLOTS * PS_BYTES;
  static constexpr int OFF_SMETA = OFF_BAR + 2 * STAGES * 8;     // [STAGES] {residual pieces of the stage in the slot | first ring slot << 8}
  static constexpr int OFF_SA = OFF_SMETA + STAGES * 4;          // [32] token scales
  static constexpr int OFF_NP = OFF_SA + 32 * 4;                 // [DEC_MAX_KS / 2] uint16 per stage {pieces | K-steps with pieces << 8}
  static constexpr int OFF_UM = (OFF_NP + DEC_MAX_KS + 15) / 16 * 16;   // [DEC_MAX_KS] per K-step {pieces of this slab | pieces
                                                                 // of the stage's earlier K-steps << 8, first quarter | full mask << 28}
  static constexpr int SMEM_BYTES = OFF_UM + DEC_MAX_KS * 8 + 1024;   // + slack for the 1024-byte alignment
  // the K groups' partial sums [KW][2 accumulators][MT][R] int32 re-use the ring once all stages are consumed
  static constexpr int RED_BYTES = KW * (BSC ? 3 : (GRP ? 1 : 2)) * MT * R * 4;
  static_assert(KPW >= 1 && KPW * KW == UK, "the K-steps of a stage are dealt evenly to the K groups");
  static_assert(STAGES >= 2, "ring depth");
  static_assert(T_KSTEP % 1024 == 0 || (!A8 && T_KSTEP % 512 == 0), "SWIZZLE_64B / _128B boxes need 512- / 1024-byte aligned destinations");
  static_assert(W_BYTES % 1024 == 0 && (STAGES * W_BYTES) % 1024 == 0, "token stages start 1024-byte aligned");
  static_assert(RED_BYTES <= OFF_Q, "the reduction buffer fits the ring");
  static_assert((BIG ? 1 : 2) * (SMEM_BYTES + 1024) <= 232448, "two CTAs per SM (one: BIG)");
};

struct DecParams {
  const uint8_t* res;
  const float* qscale;     // BSC: [n_quarters][64] block-local residual scale of every row of every stored quarter
  const int2* unit_meta;   // [NT * KS] {quarter mask, first quarter index}; NULL = dense only
  const float* sw;
  const float* sr;
  const float* sa;         // [M] token scales; GRP: [M][KS] group scales
  void* Y;
  int32_t* dbg0;           // [M][N] sums, or NULL; GRP: [KS][M][N] per-group sums
  int32_t* dbg1;
  int64_t ldy;
  int M, N, KS;
  int y_bf16;
#ifdef MQ_DEC_TRACE
  unsigned long long* trace;   // [grid][32] %globaltimer stamps (development builds only)
#endif
};

#ifdef MQ_DEC_TRACE
__device__ __forceinline__ unsigned long long gtimer() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
#define DEC_STAMP(cond, slot) do { if ((cond) && p.trace) p.trace[(size_t)blockIdx.x * 32 + (slot)] = gtimer(); } while (0)
#else
#define DEC_STAMP(cond, slot) do { } while (0)
#endif

__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const void* tmap, int c0, int c1, int c2, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst),
      "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void ldmatrix_x4(uint32_t* r, uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(addr));
}
__device__ __forceinline__ void mma_s8(int (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                       uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint2 lds_u64(uint32_t addr) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void sts_u64(uint32_t addr, uint32_t a, uint32_t b) {
  asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(addr), "r"(a), "r"(b) : "memory");
}

template <int RT, int MT, bool BIG, bool BSC, bool GRP = false, bool A8 = false>
__global__ void __launch_bounds__(DEC_THREADS, BIG ? 1 : 2)
mq_decode_kernel(const __grid_constant__ CUtensorMap tmap_w, const __grid_constant__ CUtensorMap tmap_a, const DecParams p) {
  using C = DCfg<RT, MT, BIG, BSC, GRP, A8>;
  static_assert(!(BSC && GRP) && !(A8 && (BSC || GRP)), "the variants are not combined");
  constexpr int R = C::R, KW = C::KW, UK = C::UK, KPW = C::KPW, NST = C::NST, STAGES = C::STAGES;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sb = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sW = sb + C::OFF_W, sT = sb + C::OFF_T, sQ = sb + C::OFF_Q, sBar = sb + C::OFF_BAR,
                 sSMeta = sb + C::OFF_SMETA, sSA = sb + C::OFF_SA, sNP = sb + C::OFF_NP,
                 sUM = sb + C::OFF_UM;
  auto full_bar = [&](int s) { return sBar + 8u * (uint32_t)s; };
  auto empty_bar = [&](int s) { return sBar + 8u * (uint32_t)(STAGES + s); };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = (int)blockIdx.x * R;             // first output channel of the slab
  const int nt = r0 / BN, row0 = r0 % BN;         // its n-tile and first row inside it
  const int KS = p.KS;
  const int n_stages = (KS + UK - 1) / UK;
  const int pre = min(STAGES, n_stages);
  // residual quarters (q = 2 * k-half + row-half) that hold rows of this slab
  const uint32_t relevant = R >= BN ? 0xFu : (0x5u << ((row0 >> 6) & 1));
  DEC_STAMP(threadIdx.x == 0, 0);

  if (warp == DEC_CWARPS) {
    if (lane == 0) {
      prefetch_tmap(&tmap_w);
      prefetch_tmap(&tmap_a);
      for (int s = 0; s < STAGES; ++s) {
        mbar_init(full_bar(s), 2);               // the two producers' arrivals; the copies complete the transaction count
        mbar_init(empty_bar(s), DEC_CWARPS);     // one arrival per consumer warp
      }
      fence_mbar_init();
      // the packed weights are static: the first ring-full is requested at once, before anything else
      for (int s = 0; s < pre; ++s) {
        mbar_expect_tx(full_bar(s), C::W_BYTES);
        tma_load_3d(sW + s * C::W_BYTES, &tmap_w, row0 * 2, 4 * UK * s, nt, full_bar(s));
      }
    }
  } else if (warp < DEC_CWARPS) {
    // the n-tile's residual metadata -> shared memory, one thread per stage: the K-steps' {pieces of this slab,
    // first quarter | full mask} and the stage's piece count, so that the single producer thread pays one load
    // per stage on its common path (no residual piece in the stage)
    for (int s = threadIdx.x; s < n_stages; s += 32 * DEC_CWARPS) {
      int np = 0, kmask = 0;
      for (int j = 0; j < UK; ++j) {
        const int ks = s * UK + j;
        if (ks < KS) {
          int2 v = make_int2(0, 0);
          if (p.unit_meta) v = __ldg(p.unit_meta + (size_t)nt * KS + ks);
          const uint32_t m = (uint32_t)v.x & relevant;
          sts_u64(sUM + 8u * (uint32_t)ks, m | ((uint32_t)np << 8), (uint32_t)v.y | ((uint32_t)v.x << 28));
          np += __popc(m);
          if (m) kmask |= 1 << j;
        }
      }
      asm volatile("st.shared.u16 [%0], %1;" ::"r"(sNP + 2u * (uint32_t)s), "r"(np | (kmask << 8)) : "memory");
    }
  }
  __syncthreads();
  // PDL: the next kernel in the stream may become resident beside this one and request its weights
  griddep_launch();
  DEC_STAMP(threadIdx.x == 0, 1);

  if (warp == DEC_CWARPS) {
    if (lane != 0) return;
    // ===================== producer of the weight / token stream (one thread) =====================
    // Every instruction of a single-thread role costs ~7 cycles: this loop is two copy instructions and a wait.
    DEC_STAMP(true, 2);
    griddep_wait();   // the packed tokens are the previous kernel's output
    DEC_STAMP(true, 3);
    for (int s = 0; s < n_stages; ++s) {
      const int slot = s % STAGES;
      const uint32_t fb = full_bar(slot);
      if (s >= STAGES) mbar_wait(empty_bar(slot), (((uint32_t)s / STAGES) & 1) ^ 1);   // the stage's slot is free
      if (s >= pre) {
        mbar_expect_tx(fb, C::W_BYTES);
        tma_load_3d(sW + slot * C::W_BYTES, &tmap_w, row0 * 2, 4 * UK * s, nt, fb);
      }
      mbar_arrive_expect_tx(fb, C::T_BYTES);
      tma_load_3d(sT + slot * C::T_BYTES, &tmap_a, 0, 0, UK * s, fb);
      DEC_STAMP(s == 0, 21);
      DEC_STAMP(s == n_stages - 1, 23);
    }
    return;
  }
  if (warp == DEC_CWARPS + 1) {
    if (lane != 0) return;
    // ===================== producer of the residual pieces (one thread, static data: no dependency wait) =====================
    // FIFO ring of residual pieces: q_issued / q_freed count pieces since the start; qcum[stage slot] = q_issued
    // after that stage, read back when the stage is known to be consumed
    int q_issued = 0, q_freed = 0, consumed = 0;
    int qcum[STAGES];
#pragma unroll
    for (int i = 0; i < STAGES; ++i) qcum[i] = 0;
    auto set_qcum = [&](int slot, int v) {
#pragma unroll
      for (int i = 0; i < STAGES; ++i)
        if (i == slot) qcum[i] = v;
    };
    auto get_qcum = [&](int slot) {
      int v = qcum[0];
#pragma unroll
      for (int i = 1; i < STAGES; ++i) v = i == slot ? qcum[i] : v;
      return v;
    };
    auto advance_to = [&](int target) {   // wait (in order) until `target` stages are known to be consumed
      while (consumed < target) {
        mbar_wait(empty_bar(consumed % STAGES), ((uint32_t)consumed / STAGES) & 1);
        q_freed = get_qcum(consumed % STAGES);
        ++consumed;
      }
    };
    for (int s = 0; s < n_stages; ++s) {
      const int slot = s % STAGES;
      const uint32_t fb = full_bar(slot);
      if (s >= STAGES) advance_to(s - STAGES + 1);   // the stage's slot (and its metadata word) is free
      uint32_t npk;   // {pieces | K-steps with pieces << 8}
      asm volatile("ld.shared.u16 %0, [%1];" : "=r"(npk) : "r"(sNP + 2u * (uint32_t)s));
      const int np = (int)(npk & 0xFF);
      while (q_issued + np - q_freed > DEC_QSLOTS) advance_to(consumed + 1);   // room in the piece ring
      sts_u32(sSMeta + 4u * (uint32_t)slot, (uint32_t)np | ((uint32_t)(q_issued % DEC_QSLOTS) << 8));
      if (np) {   // only the K-steps that own pieces are visited
        mbar_expect_tx(fb, (uint32_t)np * C::PS_BYTES);
        for (uint32_t km = npk >> 8; km; km &= km - 1) {
          const int ks = s * UK + __ffs((int)km) - 1;
          const uint2 um = lds_u64(sUM + 8u * (uint32_t)ks);
          const uint32_t full_mask = um.y >> 28, qoff = um.y & 0x0FFFFFFFu;
          for (uint32_t mm = um.x & 0xF; mm; mm &= mm - 1) {
            const int q = __ffs((int)mm) - 1;
            const size_t qidx = (size_t)qoff + (size_t)__popc(full_mask & ((1u << q) - 1));
            const uint8_t* src = p.res + qidx * QUARTER_BYTES + (size_t)(row0 & 63) * 16;
            const uint32_t dst = sQ + (uint32_t)(q_issued % DEC_QSLOTS) * C::PS_BYTES;
            if (BSC) tma_load_1d(dst + C::P_BYTES, p.qscale + qidx * 64 + (size_t)(row0 & 63), C::P_ROWS * 4, fb);
            if (C::P_ROWS == 64) {
              tma_load_1d(dst, src, QUARTER_BYTES, fb);
            } else {   // the slab's rows of the quarter's two 32-channel chunks
              tma_load_1d(dst, src, C::P_ROWS * 16, fb);
              tma_load_1d(dst + C::P_ROWS * 16, src + 1024, C::P_ROWS * 16, fb);
            }
            ++q_issued;
          }
        }
      }
      set_qcum(slot, q_issued);
      mbar_arrive(fb);   // releases the metadata word; the phase completes when both producers' bytes have landed
    }
    return;
  }

  // ===================== consumers: warp = (row tile rt, K group kw) =====================
  griddep_wait();   // s_a and Y are ordered after the previous kernel in the stream
  if (!GRP && threadIdx.x < 32) sts_u32(sSA + 4u * threadIdx.x, __float_as_uint((int)threadIdx.x < p.M ? __ldg(p.sa + threadIdx.x) : 0.f));
  constexpr uint32_t HI = 0xF0F0F0F0u;
  constexpr float ACC_INV = A8 ? 0.0625f : 0.00390625f;   // the accumulators are 256 x the sums (both operands x16); A8: 16 x
  constexpr int ACC_SHIFT = A8 ? 4 : 8;
  const int rt = warp % RT, kw = warp / RT;
  const int g = lane >> 2, tq = lane & 3;
  const int lrow = lane & 7, lmat = lane >> 3;   // ldmatrix: this lane supplies row lrow of matrix lmat
  // weights of a stage [4 UK chunks][R rows][16 B]: one ldmatrix.x4 = chunks {2a, 2a+1} x row sets {+0..7, +8..15}
  const uint32_t w_off = (uint32_t)((lmat >> 1) * C::CH_BYTES + (16 * rt + (lmat & 1) * 8 + lrow) * 16);
  // tokens of a K-step [MT rows][64 B], 16-byte chunks XOR-swizzled with (row >> 1) & 3 (SWIZZLE_64B): matrix m = chunk m
  const uint32_t t_off = (uint32_t)(lrow * 64 + ((lmat ^ ((lrow >> 1) & 3)) << 4));
  // residual piece [2 chunks][P_ROWS rows][16 B]: matrices {chunk 0, chunk 1} x row sets
  const uint32_t r_off = (uint32_t)((lmat >> 1) * (C::P_ROWS * 16) + (((16 * rt) & (C::P_ROWS - 1)) + (lmat & 1) * 8 + lrow) * 16);
  const int rhalf = ((row0 + 16 * rt) >> 6) & 1;   // row half (of the n-tile) this warp's channels lie in
  const int ctid = threadIdx.x;                    // 0..255

  // static channel scales of this thread's epilogue elements (e = ctid + 256 i: channel e % R = ctid % R)
  const float ep_sw = __ldg(p.sw + r0 + (ctid % R)) * ACC_INV, ep_sr = __ldg(p.sr + r0 + (ctid % R)) * ACC_INV;
  // base accumulator sets: with few token groups the K-steps alternate between two sets (independent MMA chains;
  // NST >= 4 already gives four independent chains per chunk); one residual set
  constexpr int NACC = NST >= 4 ? 1 : 2;
  int d0[GRP ? 1 : NACC][GRP ? 1 : NST][4], d1[GRP ? 1 : NST][4];   // (GRP: the sums of a K-step live inside its block below)
  // BSC: sum over the pieces of s_rb * acc1_piece; GRP: the running sums y (fp32, K order inside the warp's K-steps)
  float f1[(BSC || GRP) ? NST : 1][4];
#pragma unroll
  for (int st = 0; st < ((BSC || GRP) ? NST : 1); ++st)
#pragma unroll
    for (int i = 0; i < 4; ++i) f1[st][i] = 0.f;
  // GRP: channel scales of this thread's fragment rows (g, g + 8), with the 2^-8 of the x16 operands
  float g_sw[2] = {0.f, 0.f}, g_sr[2] = {0.f, 0.f};
  if (GRP) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      g_sw[h] = __ldg(p.sw + r0 + 16 * rt + g + 8 * h) * ACC_INV;
      g_sr[h] = __ldg(p.sr + r0 + 16 * rt + g + 8 * h) * ACC_INV;
    }
  }
#pragma unroll
  for (int st = 0; st < (GRP ? 1 : NST); ++st)
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      d1[st][i] = 0;
#pragma unroll
      for (int a = 0; a < (GRP ? 1 : NACC); ++a) d0[a][st][i] = 0;
    }

  for (int s = 0; s < n_stages; ++s) {
    const int slot = s % STAGES;
    mbar_wait(full_bar(slot), ((uint32_t)s / STAGES) & 1);
    DEC_STAMP(ctid == 0 && s == 0, 4);
    DEC_STAMP(ctid == 0 && s < 14, 8 + s);
    const uint32_t smeta = lds_u32(sSMeta + 4u * (uint32_t)slot);   // {pieces of the stage, first ring slot}
#pragma unroll
    for (int jj = 0; jj < KPW; ++jj) {
      const int j = kw + KW * jj;   // this warp's K-step of the stage
      if (GRP) {
        // ---- per-group scales: the K-step's sums are converted and added at once.  Two token column groups (16 tokens) at
        //      a time, so that the sums, the token fragments and the group scales of a pass fit the registers ----
        constexpr int SH = NST < 2 ? NST : 2;
        const int ks = s * UK + j;
        const int ksg = min(ks, KS - 1);   // (K-steps past K in the last stage hold zeros: sums 0, any valid scale will do)
        uint32_t wx[8];
        const uint32_t wj = sW + slot * C::W_BYTES + j * 4 * C::CH_BYTES + w_off;
        ldmatrix_x4(wx, wj);
        ldmatrix_x4(wx + 4, wj + 2 * C::CH_BYTES);
        uint32_t meta = 0;
        if (smeta & 0xFF) meta = lds_u32(sUM + 8u * (uint32_t)ksg);
        const uint32_t mask = ks < KS ? (meta & 0xF) : 0;
        const int slot0 = (int)((smeta >> 8) + ((meta >> 8) & 0xFF));
#pragma unroll
        for (int sh = 0; sh < NST; sh += SH) {
          float sav[SH][2];   // s_a[t, g] of this thread's tokens 8 st + 2 tq, + 1 (tokens past M: zero operands, any valid row)
#pragma unroll
          for (int st = 0; st < SH; ++st)
#pragma unroll
            for (int h = 0; h < 2; ++h) sav[st][h] = __ldg(p.sa + (size_t)min(8 * (sh + st) + 2 * tq + h, p.M - 1) * (size_t)KS + ksg);
          uint32_t bw[SH][4];
#pragma unroll
          for (int st = 0; st < SH; ++st) ldmatrix_x4(bw[st], sT + slot * C::T_BYTES + j * C::T_KSTEP + (sh + st) * 512 + t_off);
          int dg[SH][4];
#pragma unroll
          for (int st = 0; st < SH; ++st)
#pragma unroll
            for (int e = 0; e < 4; ++e) dg[st][e] = 0;
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            const uint32_t a0 = (wx[2 * c] << 4) & HI, a1 = (wx[2 * c + 1] << 4) & HI, a2 = wx[2 * c] & HI, a3 = wx[2 * c + 1] & HI;
#pragma unroll
            for (int st = 0; st < SH; ++st) mma_s8(dg[st], a0, a1, a2, a3, (bw[st][c] << 4) & HI, bw[st][c] & HI);
          }
#pragma unroll
          for (int st = 0; st < SH; ++st)
#pragma unroll
            for (int e = 0; e < 4; ++e) {   // y += s_a[t, g] * (s_w * acc0_g)
              f1[sh + st][e] = fmaf(sav[st][e & 1], g_sw[e >> 1] * (float)dg[st][e], f1[sh + st][e]);
              const int t = 8 * (sh + st) + 2 * tq + (e & 1);
              if (p.dbg0 && ks < KS && t < p.M) p.dbg0[((size_t)ks * p.M + t) * p.N + r0 + 16 * rt + g + (e >> 1) * 8] = dg[st][e] >> 8;
            }
          if (mask || p.dbg1) {
#pragma unroll
            for (int st = 0; st < SH; ++st)
#pragma unroll
              for (int e = 0; e < 4; ++e) dg[st][e] = 0;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const int q = 2 * h + rhalf;
              if ((mask >> q) & 1) {   // warp-uniform
                const int ps = (slot0 + __popc(mask & ((1u << q) - 1))) % DEC_QSLOTS;
                uint32_t rx[4];
                ldmatrix_x4(rx, sQ + ps * C::PS_BYTES + r_off);
#pragma unroll
                for (int c2 = 0; c2 < 2; ++c2) {
                  const int c = 2 * h + c2;
                  const uint32_t a0 = (rx[2 * c2] << 4) & HI, a1 = (rx[2 * c2 + 1] << 4) & HI, a2 = rx[2 * c2] & HI, a3 = rx[2 * c2 + 1] & HI;
#pragma unroll
                  for (int st = 0; st < SH; ++st) mma_s8(dg[st], a0, a1, a2, a3, (bw[st][c] << 4) & HI, bw[st][c] & HI);
                }
              }
            }
#pragma unroll
            for (int st = 0; st < SH; ++st)
#pragma unroll
              for (int e = 0; e < 4; ++e) {   // y += s_a[t, g] * (s_r * acc1_g)
                if (mask) f1[sh + st][e] = fmaf(sav[st][e & 1], g_sr[e >> 1] * (float)dg[st][e], f1[sh + st][e]);
                const int t = 8 * (sh + st) + 2 * tq + (e & 1);
                if (p.dbg1 && ks < KS && t < p.M) p.dbg1[((size_t)ks * p.M + t) * p.N + r0 + 16 * rt + g + (e >> 1) * 8] = dg[st][e] >> 8;
              }
          }
        }
        continue;
      }
      if (A8) {
        // ---- W4A8: int8 tokens as they are.  MMA k-slots 4 tq .. 4 tq + 3 carry the chunk's elements 8 tq .. 8 tq + 3, slots
        //      16 + 4 tq .. carry 8 tq + 4 .. 8 tq + 7: the thread's packed weight word (8 nibbles) in canonical order is its
        //      A fragment pair, 8 consecutive token bytes are its B fragment pair (one 8-byte load) ----
        auto canon = [&](uint32_t w, uint32_t& lo, uint32_t& hi) {
          const uint32_t ev = (w << 4) & HI, od = w & HI;   // elements 0,2,4,6 | 1,3,5,7 of the word, x16
          lo = __byte_perm(ev, od, 0x5140);
          hi = __byte_perm(ev, od, 0x7362);
        };
        // token row 8 st + g of the K-step [MT rows][128 B], 16-byte chunks XOR-swizzled with row & 7 (SWIZZLE_128B)
        const uint32_t tk = sT + slot * C::T_BYTES + j * C::T_KSTEP + (uint32_t)(g * 128 + (tq & 1) * 8);
        auto tok8 = [&](int st, int c) { return lds_u64(tk + (uint32_t)(st * 1024) + ((uint32_t)((2 * c + (tq >> 1)) ^ g) << 4)); };
        uint32_t wx[8];
        const uint32_t wj = sW + slot * C::W_BYTES + j * 4 * C::CH_BYTES + w_off;
        ldmatrix_x4(wx, wj);
        ldmatrix_x4(wx + 4, wj + 2 * C::CH_BYTES);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          uint32_t a0, a1, a2, a3;
          canon(wx[2 * c], a0, a2);
          canon(wx[2 * c + 1], a1, a3);
#pragma unroll
          for (int st = 0; st < NST; ++st) {
            const uint2 tb = tok8(st, c);
            mma_s8(d0[jj % NACC][st], a0, a1, a2, a3, tb.x, tb.y);
          }
        }
        uint32_t meta = 0;
        if (smeta & 0xFF) meta = lds_u32(sUM + 8u * (uint32_t)min(s * UK + j, KS - 1));
        const uint32_t mask = s * UK + j < KS ? (meta & 0xF) : 0;
        if (mask) {
          const int slot0 = (int)((smeta >> 8) + ((meta >> 8) & 0xFF));
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const int q = 2 * h + rhalf;
            if ((mask >> q) & 1) {   // warp-uniform
              const int ps = (slot0 + __popc(mask & ((1u << q) - 1))) % DEC_QSLOTS;
              uint32_t rx[4];
              ldmatrix_x4(rx, sQ + ps * C::PS_BYTES + r_off);
#pragma unroll
              for (int c2 = 0; c2 < 2; ++c2) {
                const int c = 2 * h + c2;
                uint32_t a0, a1, a2, a3;
                canon(rx[2 * c2], a0, a2);
                canon(rx[2 * c2 + 1], a1, a3);
#pragma unroll
                for (int st = 0; st < NST; ++st) {
                  const uint2 tb = tok8(st, c);
                  mma_s8(d1[st], a0, a1, a2, a3, tb.x, tb.y);
                }
              }
            }
          }
        }
        continue;
      }
      uint32_t bw[NST][4];
#pragma unroll
      for (int st = 0; st < NST; ++st) ldmatrix_x4(bw[st], sT + slot * C::T_BYTES + j * C::T_KSTEP + st * 512 + t_off);
      uint32_t wx[8];   // {row g, row g+8} of chunk 0, chunk 1 | chunk 2, chunk 3
      const uint32_t wj = sW + slot * C::W_BYTES + j * 4 * C::CH_BYTES + w_off;
      ldmatrix_x4(wx, wj);
      ldmatrix_x4(wx + 4, wj + 2 * C::CH_BYTES);
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const uint32_t a0 = (wx[2 * c] << 4) & HI, a1 = (wx[2 * c + 1] << 4) & HI, a2 = wx[2 * c] & HI, a3 = wx[2 * c + 1] & HI;
#pragma unroll
        for (int st = 0; st < NST; ++st) mma_s8(d0[jj % NACC][st], a0, a1, a2, a3, (bw[st][c] << 4) & HI, bw[st][c] & HI);
      }
      uint32_t meta = 0;   // {pieces of this K-step, pieces of the stage's earlier K-steps}
      if (smeta & 0xFF) meta = lds_u32(sUM + 8u * (uint32_t)min(s * UK + j, KS - 1));
      const uint32_t mask = s * UK + j < KS ? (meta & 0xF) : 0;
      if (mask) {   // residual cell of this K-step: same token fragments, second accumulator set
        const int slot0 = (int)((smeta >> 8) + ((meta >> 8) & 0xFF));
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int q = 2 * h + rhalf;
          if ((mask >> q) & 1) {   // warp-uniform
            const int ps = (slot0 + __popc(mask & ((1u << q) - 1))) % DEC_QSLOTS;
            uint32_t rx[4];
            ldmatrix_x4(rx, sQ + ps * C::PS_BYTES + r_off);
            int dp[BSC ? NST : 1][4];   // BSC: this piece's own integer sums
            if (BSC) {
#pragma unroll
              for (int st = 0; st < NST; ++st)
#pragma unroll
                for (int e = 0; e < 4; ++e) dp[st][e] = 0;
            }
#pragma unroll
            for (int c2 = 0; c2 < 2; ++c2) {
              const int c = 2 * h + c2;
              const uint32_t a0 = (rx[2 * c2] << 4) & HI, a1 = (rx[2 * c2 + 1] << 4) & HI, a2 = rx[2 * c2] & HI, a3 = rx[2 * c2 + 1] & HI;
#pragma unroll
              for (int st = 0; st < NST; ++st) mma_s8(BSC ? dp[st] : d1[st], a0, a1, a2, a3, (bw[st][c] << 4) & HI, bw[st][c] & HI);
            }
            if (BSC) {   // Eq.4 with a block-local scale: s_rb[row] * acc1_piece, added in fp32; d1 keeps the integer checksum
              const uint32_t sp = sQ + ps * C::PS_BYTES + C::P_BYTES + (uint32_t)(((16 * rt) & (C::P_ROWS - 1)) + g) * 4;
              const float s_lo = __uint_as_float(lds_u32(sp)) * ACC_INV, s_hi = __uint_as_float(lds_u32(sp + 32)) * ACC_INV;
#pragma unroll
              for (int st = 0; st < NST; ++st)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                  f1[st][e] += (float)dp[st][e] * (e < 2 ? s_lo : s_hi);
                  d1[st][e] += dp[st][e];
                }
            }
          }
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(empty_bar(slot));   // this warp's reads of the stage are done
  }
  DEC_STAMP(ctid == 0, 5);
#pragma unroll
  for (int st = 0; st < NST; ++st)
#pragma unroll
    for (int i = 0; i < 4; ++i)
      if (!GRP && NACC > 1) d0[0][GRP ? 0 : st][i] += d0[GRP ? 0 : NACC - 1][GRP ? 0 : st][i];

  // ---------------- the K groups meet in shared memory, then the epilogue ----------------
  // red[kw][acc][t][r]: the ring is free once every warp has passed its last stage
  named_bar_sync(1, 32 * DEC_CWARPS);
  int32_t* red = reinterpret_cast<int32_t*>(smem_raw + (sb - smem_u32(smem_raw)));
  {
#pragma unroll
    for (int st = 0; st < NST; ++st)
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int t = 8 * st + 2 * tq + (e & 1), r = 16 * rt + g + (e >> 1) * 8;
        constexpr int NA = BSC ? 3 : (GRP ? 1 : 2);
        if (GRP) {
          red[(kw * MT + t) * R + r] = __float_as_int(f1[st][e]);
        } else {
          red[((kw * NA + 0) * MT + t) * R + r] = d0[0][GRP ? 0 : st][e];
          red[((kw * NA + 1) * MT + t) * R + r] = d1[GRP ? 0 : st][e];
          if (BSC) red[((kw * NA + 2) * MT + t) * R + r] = __float_as_int(f1[st][e]);
        }
      }
  }
  named_bar_sync(1, 32 * DEC_CWARPS);
  DEC_STAMP(ctid == 0, 16);
  for (int e = ctid; e < p.M * R; e += 32 * DEC_CWARPS) {
    const int t = e / R, r = e - t * R;
    constexpr int NA = BSC ? 3 : (GRP ? 1 : 2);
    int a0 = 0, a1 = 0;
    float fs = 0.f;
#pragma unroll
    for (int k = 0; k < KW; ++k) {
      if (GRP) {
        fs += __int_as_float(red[(k * MT + t) * R + r]);   // K groups in ascending order
      } else {
        a0 += red[((k * NA + 0) * MT + t) * R + r];
        a1 += red[((k * NA + 1) * MT + t) * R + r];
        if (BSC) fs += __int_as_float(red[((k * NA + 2) * MT + t) * R + r]);   // K groups in ascending order
      }
    }
    const int n = r0 + r;
    const float y = GRP ? fs
                        : __uint_as_float(lds_u32(sSA + 4u * (uint32_t)t)) * (BSC ? (float)a0 * ep_sw + fs : (float)a0 * ep_sw + (float)a1 * ep_sr);
    const size_t o = (size_t)t * p.ldy + n;
    if (p.y_bf16)
      reinterpret_cast<__nv_bfloat16*>(p.Y)[o] = __float2bfloat16_rn(y);
    else
      reinterpret_cast<__half*>(p.Y)[o] = __float2half_rn(y);
    if (!GRP && p.dbg0) p.dbg0[(size_t)t * p.N + n] = a0 >> ACC_SHIFT;
    if (!GRP && p.dbg1) p.dbg1[(size_t)t * p.N + n] = a1 >> ACC_SHIFT;
  }
  DEC_STAMP(ctid == 0, 6);
}

}  // namespace

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

constexpr int rt_index(int rows) { return rows == 16 ? 0 : (rows == 32 ? 1 : (rows == 64 ? 2 : 3)); }

// rows per CTA: the smallest slab whose CTAs are all resident at once (two per SM), so that every CTA streams
// from the first microsecond and the CTAs are as short as possible
int pick_rows(const mq_weights* w, int64_t M) {
  const Options& o = options();
  if (o.decode_rows) return (int)o.decode_rows;
  const int sms = sm_count() > 0 ? sm_count() : 148;
  int rows = 16;
  while (rows < 128 && w->N / rows > 2LL * sms) rows *= 2;
  (void)M;
  return rows;
}

#ifdef MQ_DEC_TRACE
unsigned long long* g_dec_trace = nullptr;
#endif

template <int RT, int MT, bool BIG, bool BSC = false, bool GRP = false, bool A8 = false>
int dec_launch(const CUtensorMap& tmw, const CUtensorMap& tma, const DecParams& dp, int grid, cudaStream_t st) {
  using C = DCfg<RT, MT, BIG, BSC, GRP, A8>;
  // the attribute belongs to the (device, function) pair: set it whenever the current device changes
  static int attr_dev = -1;
  int dev = -1;
  cudaGetDevice(&dev);
  if (dev != attr_dev) {
    if (cudaFuncSetAttribute(mq_decode_kernel<RT, MT, BIG, BSC, GRP, A8>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES) != cudaSuccess) {
      cudaGetLastError();
      return MQ_ERR_CUDA;
    }
    attr_dev = dev;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(DEC_THREADS);
  cfg.dynamicSmemBytes = C::SMEM_BYTES;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = options().pdl ? 1 : 0;
  if (cudaLaunchKernelEx(&cfg, mq_decode_kernel<RT, MT, BIG, BSC, GRP, A8>, tmw, tma, dp) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  return MQ_OK;
}

template <int RT>
int dec_launch_mt(int MT, bool big, bool bsc, bool grp, bool a8, const CUtensorMap& tmw, const CUtensorMap& tma, const DecParams& dp, int grid, cudaStream_t st) {
  if (a8) {    // W4A8 (small ring only; 32 token columns of int8 fit the ring for slabs of 64 channels and more, see
               // decode_a8_eligible)
    switch (MT) {
      case 8: return dec_launch<RT, 8, false, false, false, true>(tmw, tma, dp, grid, st);
      case 16: return dec_launch<RT, 16, false, false, false, true>(tmw, tma, dp, grid, st);
      default:
        if constexpr (RT >= 4) return dec_launch<RT, 32, false, false, false, true>(tmw, tma, dp, grid, st);
        else return MQ_ERR_UNSUPPORTED_SHAPE;
    }
  }
  if (grp) {   // per-group activation scales (small ring only)
    switch (MT) {
      case 8: return dec_launch<RT, 8, false, false, true>(tmw, tma, dp, grid, st);
      case 16: return dec_launch<RT, 16, false, false, true>(tmw, tma, dp, grid, st);
      default: return dec_launch<RT, 32, false, false, true>(tmw, tma, dp, grid, st);
    }
  }
  if (bsc) {   // block-local residual scales (small ring only)
    switch (MT) {
      case 8: return dec_launch<RT, 8, false, true>(tmw, tma, dp, grid, st);
      case 16: return dec_launch<RT, 16, false, true>(tmw, tma, dp, grid, st);
      default: return dec_launch<RT, 32, false, true>(tmw, tma, dp, grid, st);
    }
  }
  if (big) {   // (rows <= 64 only: the deep ring is for layers with few slabs)
    if constexpr (RT <= 4) {
      switch (MT) {
        case 8: return dec_launch<RT, 8, true>(tmw, tma, dp, grid, st);
        case 16: return dec_launch<RT, 16, true>(tmw, tma, dp, grid, st);
        default: return dec_launch<RT, 32, true>(tmw, tma, dp, grid, st);
      }
    }
  }
  switch (MT) {
    case 8: return dec_launch<RT, 8, false>(tmw, tma, dp, grid, st);
    case 16: return dec_launch<RT, 16, false>(tmw, tma, dp, grid, st);
    default: return dec_launch<RT, 32, false>(tmw, tma, dp, grid, st);
  }
}

int uk_of_rows(int rows) { return rows <= 32 ? 8 : (rows == 64 ? 4 : 2); }

}  // namespace

#ifdef MQ_DEC_TRACE
extern "C" void mq_debug_set_dec_trace(unsigned long long* dev_buf) { g_dec_trace = dev_buf; }
#endif

namespace mq {

// The packed base [N/128][K/128][4 chunks][128 rows][16 B] as a 3-D tensor of 8-byte elements:
//   dim 0: 256 elements = the 128 rows x 16 B of one chunk (contiguous)
//   dim 1: 4 * KS chunks along K of one n-tile (stride 2048 B)
//   dim 2: N / 128 n-tiles (stride KS * 8192 B)
// One box {2 R elements, 4 UK chunks, 1} = the rows of a slab for UK K-steps, laid out [chunk][R rows][16 B]
// in shared memory; chunks beyond K are zero-filled (a last stage with fewer than UK K-steps).
int build_weight_tmaps(mq_weights* w) {
  w->tmap_ok = false;
  EncodeTiledFn enc = (EncodeTiledFn)tensor_map_encode_fn();
  if (!enc) return MQ_ERR_CUDA;
  const int64_t KS = w->K / BK, NT = w->N / BN;
  if (4 * KS > 0xFFFFFFFFLL) return MQ_OK;   // not eligible for the decode kernel; the tcgen05 kernel serves it
  const int rows[4] = {16, 32, 64, 128};
  for (int i = 0; i < 4; ++i) {
    memset(&w->tmap_base[i], 0, sizeof(CUtensorMap));
    const cuuint64_t gdim[3] = {256, (cuuint64_t)(4 * KS), (cuuint64_t)NT};
    const cuuint64_t gstride[2] = {2048, (cuuint64_t)KS * TILE_BYTES};
    const cuuint32_t box[3] = {(cuuint32_t)(2 * rows[i]), (cuuint32_t)(4 * uk_of_rows(rows[i])), 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    if (enc(&w->tmap_base[i], CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, w->d_base, gdim, gstride, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return MQ_ERR_CUDA;
  }
  w->tmap_ok = true;
  return MQ_OK;
}

bool decode_eligible(const mq_weights* w, int64_t M) {
  const Options& o = options();
  if (!w || M <= 0 || !w->tmap_ok) return false;
  // block-local residual scales exist in this kernel only: it serves every M (32 tokens per pass) whatever the knobs say
  if (w->blockscale) return w->K / BK <= DEC_MAX_KS;
  if (M > 32) return false;
  // the tcgen05 kernel's own knobs select that kernel (tests and ablations address it through them)
  if (o.decode_path == 1 || o.token_tile != 0 || o.split_k >= 2 || o.max_ctas != 0 || o.fused_quant) return false;
  return w->K / BK <= DEC_MAX_KS;
}

size_t decode_workspace_bytes(const mq_weights*, int64_t) { return 0; }

static int decode_gemm_pass(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                            int32_t* dbg0, int32_t* dbg1, void* cuda_stream, bool ignore_res, bool grp = false, bool a8 = false);

// W4A8 at decode sizes: the same kernel with int8 tokens (A8 form)
bool decode_a8_eligible(const mq_weights* w, int64_t M) {
  const Options& o = options();
  if (!w || !w->tmap_ok || w->blockscale || M <= 0 || M > 32) return false;
  if (o.decode_path == 1 || o.token_tile != 0 || o.split_k >= 2 || o.max_ctas != 0) return false;
  // 32 token columns: a stage of 8 K-steps x 32 tokens x 128 B leaves no ring depth; slabs of 64 channels and more have
  // stages of 2-4 K-steps.  (Forcing 64-channel slabs on the layers that get shorter ones leaves too few CTAs: measured
  // slower than the stream-K kernel.)
  if (M > 16 && pick_rows(w, M) < 64) return false;
  return w->K / BK <= DEC_MAX_KS;
}

int decode_gemm_a8(const mq_weights* w, const void* qA8, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                   int32_t* dbg0, int32_t* dbg1, void* cuda_stream, bool ignore_res) {
  const int rc = decode_gemm_pass(w, qA8, sA, M, Y, y_dtype, ldy, dbg0, dbg1, cuda_stream, ignore_res, false, true);
  if (rc == MQ_OK) set_launch_count(1);
  return rc;
}

// per-group activation scales (group = 128) at decode sizes: the same kernel, sums converted per K-step
bool decode_group_eligible(const mq_weights* w, int group, int64_t M) {
  const Options& o = options();
  if (!w || !w->tmap_ok || w->blockscale || group != 128 || M <= 0 || M > 32) return false;
  if (o.group_tc == 0 || o.group_simt != 0 || o.decode_path == 1) return false;
  return w->K / BK <= DEC_MAX_KS;
}

int decode_gemm_group(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                      int32_t* dbg0, int32_t* dbg1, void* cuda_stream) {
  const int rc = decode_gemm_pass(w, qA, sA, M, Y, y_dtype, ldy, dbg0, dbg1, cuda_stream, false, true);
  if (rc == MQ_OK) set_launch_count(1);
  return rc;
}

// M <= 32: one launch.  More tokens (block-local scales only): passes of 32 tokens, each streaming the weights again
// (from L2 when the layer fits) -- a first path for that reading at prefill sizes, not a fast one.
int decode_gemm(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                int32_t* dbg0, int32_t* dbg1, void*, size_t, void* cuda_stream, bool ignore_res) {
  int launches = 0;
  for (int64_t m0 = 0; m0 < M; m0 += 32) {
    const int64_t mc = std::min<int64_t>(32, M - m0);
    const int rc = decode_gemm_pass(w, (const uint8_t*)qA + (size_t)m0 * (size_t)(w->K / 2), sA + m0, mc,
                                    (uint8_t*)Y + (size_t)m0 * (size_t)ldy * 2, y_dtype, ldy, dbg0 ? dbg0 + (size_t)m0 * w->N : nullptr,
                                    dbg1 ? dbg1 + (size_t)m0 * w->N : nullptr, cuda_stream, ignore_res);
    if (rc != MQ_OK) return rc;
    ++launches;
  }
  set_launch_count(launches);
  return MQ_OK;
}

static int decode_gemm_pass(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                            int32_t* dbg0, int32_t* dbg1, void* cuda_stream, bool ignore_res, bool grp, bool a8) {
  const int rows = pick_rows(w, M);
  const int MT = M <= 8 ? 8 : (M <= 16 ? 16 : 32);
  // 3-D tensor map over the canonical packed activations [M rows][K/2 bytes]: {64 B of a K-step, M rows, KS K-steps};
  // box {64 B, MT rows, UK K-steps} -> shared memory [K-step][token][64 B]; rows beyond M and K-steps beyond K are
  // zero-filled; 16-byte chunks XOR-swizzled (SWIZZLE_64B) so that the fragment loads are conflict-free
  EncodeTiledFn enc = (EncodeTiledFn)tensor_map_encode_fn();
  if (!enc) return MQ_ERR_CUDA;
  CUtensorMap tmap;
  memset(&tmap, 0, sizeof(tmap));
  // (A8: int8 tokens [M rows][K bytes], 128 B per K-step, SWIZZLE_128B)
  const cuuint64_t kb = a8 ? (cuuint64_t)BK : (cuuint64_t)(BK / 2);   // token bytes per K-step
  const cuuint64_t gdim[3] = {kb, (cuuint64_t)M, (cuuint64_t)(w->K / BK)};
  const cuuint64_t gstride[2] = {(cuuint64_t)(w->K / BK) * kb, kb};
  const cuuint32_t box[3] = {(cuuint32_t)kb, (cuuint32_t)MT, (cuuint32_t)uk_of_rows(rows)};
  const cuuint32_t estr[3] = {1, 1, 1};
  if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(qA), gdim, gstride, box, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, a8 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return MQ_ERR_CUDA;

  DecParams dp;
  dp.res = w->d_res;
  dp.qscale = w->d_qscale;
  dp.unit_meta = (ignore_res || w->nnz == 0) ? nullptr : (const int2*)w->d_unit_meta;
  dp.sw = w->d_sw;
  dp.sr = w->d_sr;
  dp.sa = sA;
  dp.Y = Y;
  dp.dbg0 = dbg0;
  dp.dbg1 = dbg1;
  dp.ldy = ldy;
  dp.M = (int)M;
  dp.N = (int)w->N;
  dp.KS = (int)(w->K / BK);
  dp.y_bf16 = y_dtype == MQ_BF16;
#ifdef MQ_DEC_TRACE
  dp.trace = g_dec_trace;
#endif
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int grid = (int)(w->N / rows);
  // deep ring (one CTA per SM): the slabs fit one CTA per SM and each has more stages than the small ring holds
  const Options& o = options();
  const int sms = sm_count() > 0 ? sm_count() : 148;
  const bool big = !grp && !a8 && (o.decode_big == 1 || (o.decode_big == 0 && rows <= 64 && grid <= sms && (w->K / BK) / uk_of_rows(rows) > 8));
  const CUtensorMap& tmw = w->tmap_base[rt_index(rows)];
  int rc;
  switch (rows) {
    case 16: rc = dec_launch_mt<1>(MT, big, w->blockscale, grp, a8, tmw, tmap, dp, grid, st); break;
    case 32: rc = dec_launch_mt<2>(MT, big, w->blockscale, grp, a8, tmw, tmap, dp, grid, st); break;
    case 64: rc = dec_launch_mt<4>(MT, big, w->blockscale, grp, a8, tmw, tmap, dp, grid, st); break;
    default: rc = dec_launch_mt<8>(MT, big, w->blockscale, grp, a8, tmw, tmap, dp, grid, st); break;
  }
  return rc;
}

}  // namespace mq
