// mq_group.cu -- SURVEY 8(f)-3: scales that vary along K.  Per-GROUP activation quantization, the paper's stated
// activation granularity for the 4-bit setting ("For the 4-bit setting, we adopt per-group
// and per-channel symmetric quantization for activations and weights, respectively"; group size not given:
// DESIGN.md reading A5g makes it a parameter, 32 / 64 / 128 consecutive input channels).
//
//   mq_quantize_act_group : Eq.1 on every run of `group` channels of every token.  One 16-byte load
//                           (8 elements) per thread, a team of group/8 lanes finds the run's absmax with
//                           xor-shuffles, every thread packs its 8 codes into one 32-bit word.  HBM-bound:
//                           2 B read + 0.5 B + 4/group B written per element.
//   mq_gemm_group         : Eq.2 / Eq.4 per group:
//                             Y[m,n] = sum_g s_a[m,g] (s_w[n] acc0_g[m,n] + s_r[n] acc1_g[m,n])
//                           The integer partial sums cannot cross a group boundary, so the fused tcgen05 kernel's
//                           single int32 accumulator per output does not apply.  Two kernels.  The first one written is SIMT (option
//                           group_simt; kept as the ablation): one
//                           thread per output channel, dp4a over the packed nibbles of the same device layout
//                           (base tiles + residual quarters, mq_internal.h), exact int32 per (group, token,
//                           channel), rescaled and added in fp32 after every group.  The residual quarters of a
//                           K-step are consumed in the same pass as its base tile (the activations are read once:
//                           the paper's fusion), K is split over CTAs when there are few tiles.
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <algorithm>

#include "mq_internal.h"
#include "mq_ptx.cuh"

using namespace mq;

namespace {

constexpr int GT = 256;    // threads per CTA of the quantizer
constexpr int TOK = 16;    // tokens per CTA of the GEMM
constexpr int TARGET_CTAS = 296;   // 2 x 148 SMs
constexpr int SIMT_MAX_M = 0;      // largest M served by the dp4a kernel by default (0: option group_simt only; measured:
                                   // the tensor-core kernel is level at M = 1 and 1.3-4 x faster from M = 2)

template <bool BF16>
__device__ __forceinline__ void cvt8g(const uint4& v, float* f) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (BF16) {
      f[2 * i] = __uint_as_float(w[i] << 16);
      f[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    } else {
      const float2 t = __half22float2(*reinterpret_cast<const __half2*>(&w[i]));
      f[2 * i] = t.x;
      f[2 * i + 1] = t.y;
    }
  }
}

// LANES = group / 8 lanes share one scale.  total = M * K / 8 chunks, a multiple of LANES, and a row holds a
// multiple of LANES chunks, so a team never straddles a row, a warp or the end of the grid's valid range.
template <bool BF16, int LANES>
__global__ void __launch_bounds__(GT) quantize_group_kernel(const uint16_t* __restrict__ A, int64_t lda, int chunks_per_row,
                                                            int64_t total, uint32_t* __restrict__ qA, float* __restrict__ sA) {
  mq::ptx::griddep_launch();
  mq::ptx::griddep_wait();
  const int64_t c = (int64_t)blockIdx.x * GT + threadIdx.x;
  const bool live = c < total;
  float f[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) f[i] = 0.f;
  int64_t m = 0;
  int cr = 0;
  if (live) {
    m = c / chunks_per_row;
    cr = (int)(c - m * chunks_per_row);
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(A + m * lda) + cr);
    cvt8g<BF16>(v, f);
  }
  float amax = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) amax = fmaxf(amax, fabsf(f[i]));
#pragma unroll
  for (int o = LANES / 2; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xFFFFFFFFu, amax, o));
  if (!live) return;
  const float s = amax == 0.f ? 1.0f : __fdiv_rn(amax, 7.0f);   // A2, A3
  const float inv_s = mq::ptx::quant_inv_scale(s);
  uint32_t out = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) out |= (uint32_t)(mq::ptx::quant1(f[i], s, inv_s) & 0xF) << (4 * i);
  qA[c] = out;   // row m starts at word m * chunks_per_row: dense [M, K/2] bytes
  if ((cr & (LANES - 1)) == 0) sA[m * (chunks_per_row / LANES) + cr / LANES] = s;
}

__device__ __forceinline__ int dp4a(uint32_t a, uint32_t b, int c) {
  int d;
  asm("dp4a.s32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}

// dot product of 32 int4 pairs (16 bytes each side, canonical nibble order): both operands are expanded to
// 16 x value in the high nibble of each byte, so the dp4a sum is 256 x the dot product, exactly.
__device__ __forceinline__ int dot32(const uint4& w, const uint4& a) {
  constexpr uint32_t HI = 0xF0F0F0F0u;
  const uint32_t ww[4] = {w.x, w.y, w.z, w.w}, aw[4] = {a.x, a.y, a.z, a.w};
  int s = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    s = dp4a((ww[i] << 4) & HI, (aw[i] << 4) & HI, s);
    s = dp4a(ww[i] & HI, aw[i] & HI, s);
  }
  return s >> 8;   // a multiple of 256: the arithmetic shift is exact
}

template <bool BF16>
__device__ __forceinline__ void store_y16(void* Y, size_t o, float y) {
  if (BF16)
    reinterpret_cast<__nv_bfloat16*>(Y)[o] = __float2bfloat16_rn(y);
  else
    reinterpret_cast<__half*>(Y)[o] = __float2half_rn(y);
}

struct GParams {
  const uint8_t* base;
  const uint8_t* res;
  const int32_t* unit_meta;   // [N/BN][KS][2] {quarter mask, first quarter}
  const float* sw;
  const float* sr;
  const uint8_t* qA;          // [M, K/2]
  const float* sa;            // [M, K/GROUP]
  void* Y;
  float* partial;             // [splits][M][N] when splits > 1
  int32_t* dbg0;              // [K/GROUP][M][N] or NULL
  int32_t* dbg1;
  int64_t M, N, K, ldy;
  int KS, ks_per_split, splits;
};

// grid (N/BN, ceil(M/TOK), splits), 128 threads: thread = output channel of the n-tile.
template <int GROUP, bool BF16>
__global__ void __launch_bounds__(BN) gemm_group_kernel(const GParams p) {
  mq::ptx::griddep_launch();
  mq::ptx::griddep_wait();
  constexpr int CPG = GROUP / 32;   // 32-channel chunks per group
  constexpr int GPS = 4 / CPG;      // groups per K-step
  const int nt = blockIdx.x, row = threadIdx.x, rhalf = row >> 6;
  const int64_t n = (int64_t)nt * BN + row;
  const int64_t m0 = (int64_t)blockIdx.y * TOK;
  const int mt = (int)min((int64_t)TOK, p.M - m0);
  const int k0 = (int)blockIdx.z * p.ks_per_split, k1 = min(p.KS, k0 + p.ks_per_split);
  const int G = (int)(p.K / GROUP);
  const float sw = __ldg(p.sw + n), sr = __ldg(p.sr + n);
  float y[TOK];
#pragma unroll
  for (int t = 0; t < TOK; ++t) y[t] = 0.f;

  for (int ks = k0; ks < k1; ++ks) {
    const uint8_t* tile = p.base + ((size_t)nt * p.KS + ks) * TILE_BYTES + (size_t)row * 16;
    uint4 wb[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) wb[c] = __ldg(reinterpret_cast<const uint4*>(tile + c * (BN * 16)));
    // residual quarters of this K-step that cover this thread's row half: chunk c = 2 h + j
    uint4 wr[4];
    bool has[2] = {false, false};
    if (p.unit_meta) {
      const int2 um = __ldg(reinterpret_cast<const int2*>(p.unit_meta) + (size_t)nt * p.KS + ks);
      const int mask = um.x & 0xF;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int q = 2 * h + rhalf;
        if (mask & (1 << q)) {
          has[h] = true;
          const uint8_t* qp = p.res + ((size_t)um.y + (size_t)__popc(mask & ((1 << q) - 1))) * QUARTER_BYTES + (size_t)(row & 63) * 16;
          wr[2 * h] = __ldg(reinterpret_cast<const uint4*>(qp));
          wr[2 * h + 1] = __ldg(reinterpret_cast<const uint4*>(qp + 1024));
        }
      }
    }
#pragma unroll
    for (int t = 0; t < TOK; ++t) {
      if (t >= mt) break;
      const int64_t m = m0 + t;
      const uint4* ap = reinterpret_cast<const uint4*>(p.qA + (size_t)m * (size_t)(p.K / 2) + (size_t)ks * (BK / 2));
      int a0[4], a1[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const uint4 av = __ldg(ap + c);   // the same address in every thread: one broadcast transaction
        a0[c] = dot32(wb[c], av);
        a1[c] = has[c >> 1] ? dot32(wr[c], av) : 0;
      }
      float acc = y[t];
#pragma unroll
      for (int gi = 0; gi < GPS; ++gi) {
        int s0 = 0, s1 = 0;
#pragma unroll
        for (int j = 0; j < CPG; ++j) {
          s0 += a0[gi * CPG + j];
          s1 += a1[gi * CPG + j];
        }
        const int g = ks * GPS + gi;
        const float s = __ldg(p.sa + (size_t)m * G + g);
        acc += s * (sw * (float)s0 + sr * (float)s1);   // |s0|, |s1| <= 49 * 128: exact in fp32
        if (p.dbg0) p.dbg0[((size_t)g * p.M + m) * p.N + n] = s0;
        if (p.dbg1) p.dbg1[((size_t)g * p.M + m) * p.N + n] = s1;
      }
      y[t] = acc;
    }
  }
#pragma unroll
  for (int t = 0; t < TOK; ++t) {
    if (t >= mt) break;
    const int64_t m = m0 + t;
    if (p.splits == 1)
      store_y16<BF16>(p.Y, (size_t)m * p.ldy + n, y[t]);
    else
      p.partial[((size_t)blockIdx.z * p.M + m) * p.N + n] = y[t];
  }
}


// ---- tensor-core path (default for every M): legacy warp-level mma.sync m16n8k32 s8 -- a group boundary every 32..128 channels
// means the int32 sums must leave the accumulator after at most one K-step, which a TMEM-resident tcgen05
// accumulator makes expensive (a tcgen05.ld drain per group); warp-level fragments are already in registers.
// 8 warps, warp v = output channels 16 v .. 16 v + 15 of the n-tile, TOKC tokens per CTA in sub-tiles of 8.
// A fragment = weights, B fragment = tokens.  Both sides expand word j of a 16-byte chunk (8 nibbles) into
// {even nibbles, odd nibbles} x 16 in int8 and place them in the same K slots, so the K permutation cancels and
// the accumulator is 256 x the exact dot product.
constexpr int TOKC = 32;
constexpr int MMA_THREADS = 256;
// shared-memory ring (cp.async, 16-byte copies): per stage the K-step's base tile (8 KB, layout as in HBM), its present
// residual quarters (<= 8 KB, compacted as in HBM) and the CTA's TOKC x 64 B of activation codes (16-byte chunks
// XOR-swizzled by token pair so that the 8-token fragment loads hit 32 distinct banks)
constexpr int MMA_STAGES = 4;
constexpr int ST_BASE = 0, ST_RES = TILE_BYTES, ST_ACT = 2 * TILE_BYTES, STAGE_BYTES = 2 * TILE_BYTES + TOKC * 64;
constexpr int MMA_SMEM = MMA_STAGES * STAGE_BYTES;

__device__ __forceinline__ void mma_s8(int (&d)[4], const uint32_t a0, const uint32_t a1, const uint32_t a2, const uint32_t a3,
                                       const uint32_t b0, const uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}

template <int GROUP, bool BF16, bool DBG>
__global__ void __launch_bounds__(MMA_THREADS, 2) gemm_group_mma_kernel(const GParams p) {
  extern __shared__ __align__(128) uint8_t g_smem[];
  __shared__ int s_mask[MMA_STAGES];
  mq::ptx::griddep_launch();
  mq::ptx::griddep_wait();
  constexpr uint32_t HI = 0xF0F0F0F0u;
  constexpr int CPG = GROUP / 32, GPS = 4 / CPG, NST = TOKC / 8;
  const int tid = threadIdx.x;
  const int nt = blockIdx.x, warp = tid >> 5, lane = tid & 31, gq = lane >> 2, tq = lane & 3;
  const int rhalf = warp >> 2;
  const int r0 = warp * 16 + gq, r1 = r0 + 8;                  // rows of the n-tile this thread's accumulators hold
  const int64_t n0 = (int64_t)nt * BN + r0, n1 = n0 + 8;
  const int64_t m0 = (int64_t)blockIdx.y * TOKC;
  const int nst = (int)min((int64_t)NST, (p.M - m0 + 7) / 8);
  const int k0 = (int)blockIdx.z * p.ks_per_split, k1 = min(p.KS, k0 + p.ks_per_split);
  const int nk = max(0, k1 - k0);
  const int G = (int)(p.K / GROUP);
  // the accumulators are 256 x the sums: the scales take the 2^-8 (exact), which saves the shifts
  const float sw0 = __ldg(p.sw + n0) * 0.00390625f, sw1 = __ldg(p.sw + n1) * 0.00390625f;
  const float sr0 = __ldg(p.sr + n0) * 0.00390625f, sr1 = __ldg(p.sr + n1) * 0.00390625f;
  const float* sa_cta = p.sa + (size_t)m0 * G;      // token t of the CTA, group g: sa_cta[t * G + g]
  const int tq2G = 2 * tq * G;
  uint32_t okmask = 0;                              // bit 2 st + j: token m0 + 8 st + 2 tq + j exists
#pragma unroll
  for (int st = 0; st < NST; ++st)
#pragma unroll
    for (int j = 0; j < 2; ++j)
      if (m0 + 8 * st + 2 * tq + j < p.M) okmask |= 1u << (2 * st + j);
  const uint32_t smem0 = (uint32_t)__cvta_generic_to_shared(g_smem);
  const int2* umeta = p.unit_meta ? reinterpret_cast<const int2*>(p.unit_meta) + (size_t)nt * p.KS : nullptr;
  float y[NST][4];
#pragma unroll
  for (int st = 0; st < NST; ++st)
#pragma unroll
    for (int i = 0; i < 4; ++i) y[st][i] = 0.f;

  // one K-step into one stage; every thread issues its share and the caller commits the group
  auto issue = [&](int ks, int stage, int2 um) {
    const uint32_t sb = smem0 + stage * STAGE_BYTES;
    const uint8_t* src = p.base + ((size_t)nt * p.KS + ks) * TILE_BYTES;
#pragma unroll
    for (int i = 0; i < TILE_BYTES / 16 / MMA_THREADS; ++i) cp_async16(sb + ST_BASE + (tid + i * MMA_THREADS) * 16, src + (size_t)(tid + i * MMA_THREADS) * 16);
    const int mask = um.x & 0xF;
    const int nchunk = __popc(mask) * (QUARTER_BYTES / 16);
    const uint8_t* rsrc = p.res + (size_t)um.y * QUARTER_BYTES;
    for (int i = tid; i < nchunk; i += MMA_THREADS) cp_async16(sb + ST_RES + i * 16, rsrc + (size_t)i * 16);
    if (tid < TOKC * 4) {
      const int t = tid >> 2, c = tid & 3;
      if (m0 + t < p.M)
        cp_async16(sb + ST_ACT + t * 64 + ((c ^ (t >> 1)) & 3) * 16,
                   p.qA + (size_t)(m0 + t) * (size_t)(p.K / 2) + (size_t)ks * (BK / 2) + c * 16);
    }
    if (tid == 0) s_mask[stage] = mask;
  };
  auto meta = [&](int ks) { return umeta ? __ldg(umeta + ks) : make_int2(0, 0); };

#pragma unroll
  for (int i = 0; i < MMA_STAGES - 1; ++i) {
    if (i < nk) issue(k0 + i, i, meta(k0 + i));
    asm volatile("cp.async.commit_group;" ::: "memory");
  }
  int2 um_next = (MMA_STAGES - 1 < nk) ? meta(k0 + MMA_STAGES - 1) : make_int2(0, 0);

  for (int it = 0; it < nk; ++it) {
    const int ks = k0 + it, stage = it % MMA_STAGES;
    asm volatile("cp.async.wait_group %0;" ::"n"(MMA_STAGES - 2) : "memory");
    __syncthreads();   // K-step `it` has landed for every thread; the stage read at it - 1 is free
    {
      const int nx = it + MMA_STAGES - 1;
      if (nx < nk) issue(k0 + nx, nx % MMA_STAGES, um_next);
      asm volatile("cp.async.commit_group;" ::: "memory");
      if (nx + 1 < nk) um_next = meta(k0 + nx + 1);
    }
    const uint32_t sb = smem0 + stage * STAGE_BYTES;
    const int mask = s_mask[stage];
    uint32_t wa[4][4], ra[4][4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const uint32_t x0 = lds32(sb + ST_BASE + c * (BN * 16) + r0 * 16 + tq * 4);
      const uint32_t x1 = lds32(sb + ST_BASE + c * (BN * 16) + r1 * 16 + tq * 4);
      wa[c][0] = (x0 << 4) & HI;
      wa[c][1] = (x1 << 4) & HI;
      wa[c][2] = x0 & HI;
      wa[c][3] = x1 & HI;
    }
    bool has[2];   // warp-uniform: a quarter covers 64 rows = 4 whole warps
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int q = 2 * h + rhalf;
      has[h] = (mask >> q) & 1;
      if (has[h]) {
        const uint32_t qp = sb + ST_RES + __popc(mask & ((1 << q) - 1)) * QUARTER_BYTES + (r0 & 63) * 16 + tq * 4;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const uint32_t x0 = lds32(qp + j * 1024), x1 = lds32(qp + j * 1024 + 8 * 16);
          ra[2 * h + j][0] = (x0 << 4) & HI;
          ra[2 * h + j][1] = (x1 << 4) & HI;
          ra[2 * h + j][2] = x0 & HI;
          ra[2 * h + j][3] = x1 & HI;
        }
      }
    }
#pragma unroll
    for (int st = 0; st < NST; ++st) {
      if (st >= nst) break;
      const int tb = 8 * st + gq;                          // token (within the CTA) of this lane's B fragment
      const int64_t t0 = m0 + 8 * st + 2 * tq, t1 = t0 + 1;   // tokens of this lane's accumulators
      uint32_t bw[4] = {0, 0, 0, 0};
      if (m0 + tb < p.M) {
#pragma unroll
        for (int c = 0; c < 4; ++c) bw[c] = lds32(sb + ST_ACT + tb * 64 + ((c ^ (tb >> 1)) & 3) * 16 + tq * 4);
      }
#pragma unroll
      for (int gi = 0; gi < GPS; ++gi) {
        int d0[4] = {0, 0, 0, 0}, d1[4] = {0, 0, 0, 0};
#pragma unroll
        for (int j = 0; j < CPG; ++j) {
          const int c = gi * CPG + j;
          const uint32_t b0 = (bw[c] << 4) & HI, b1 = bw[c] & HI;
          mma_s8(d0, wa[c][0], wa[c][1], wa[c][2], wa[c][3], b0, b1);
          if (has[c >> 1]) mma_s8(d1, ra[c][0], ra[c][1], ra[c][2], ra[c][3], b0, b1);
        }
        const int g = ks * GPS + gi;
        const int i0 = st * 8 * G + tq2G + g;
        const float s_t0 = (okmask >> (2 * st)) & 1 ? __ldg(sa_cta + i0) : 0.f;
        const float s_t1 = (okmask >> (2 * st + 1)) & 1 ? __ldg(sa_cta + i0 + G) : 0.f;
        // accumulator i: (row r0, t0), (r0, t1), (r1, t0), (r1, t1); |d| <= 256 * 49 * 128 < 2^24: exact in fp32
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const float swv = i < 2 ? sw0 : sw1, srv = i < 2 ? sr0 : sr1, sav = (i & 1) ? s_t1 : s_t0;
          float term = swv * (float)d0[i];
          if (has[(gi * CPG) >> 1] || has[(gi * CPG + CPG - 1) >> 1]) term = fmaf(srv, (float)d1[i], term);
          y[st][i] = fmaf(sav, term, y[st][i]);
          if (DBG) {
            const int64_t t = (i & 1) ? t1 : t0, n = i < 2 ? n0 : n1;
            if (t < p.M) {
              if (p.dbg0) p.dbg0[((size_t)g * p.M + t) * p.N + n] = d0[i] >> 8;
              if (p.dbg1) p.dbg1[((size_t)g * p.M + t) * p.N + n] = d1[i] >> 8;
            }
          }
        }
      }
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll
  for (int st = 0; st < NST; ++st) {
    if (st >= nst) break;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int64_t t = m0 + 8 * st + 2 * tq + (i & 1), n = i < 2 ? n0 : n1;
      if (t >= p.M) continue;
      if (p.splits == 1)
        store_y16<BF16>(p.Y, (size_t)t * p.ldy + n, y[st][i]);
      else
        p.partial[((size_t)blockIdx.z * p.M + t) * p.N + n] = y[st][i];
    }
  }
}

// the K-splits meet here, in split order (deterministic)
template <bool BF16>
__global__ void __launch_bounds__(256) group_reduce_kernel(const float* __restrict__ partial, int splits, int64_t M, int64_t N,
                                                           void* __restrict__ Y, int64_t ldy) {
  mq::ptx::griddep_launch();
  mq::ptx::griddep_wait();
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= M * N) return;
  const int64_t m = idx / N, n = idx - m * N;
  float s = 0.f;
  for (int z = 0; z < splits; ++z) s += partial[(size_t)z * M * N + idx];
  store_y16<BF16>(Y, (size_t)m * ldy + n, s);
}

template <typename Kern>
void launch_mma(Kern kern, dim3 grid, cudaStream_t st, const GParams& p) {
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, MMA_SMEM);
  kern<<<grid, MMA_THREADS, MMA_SMEM, st>>>(p);
}

bool group_use_simt(int64_t M) { return M <= SIMT_MAX_M || mq::options().group_simt != 0; }

int group_splits(const mq_weights* w, int64_t M) {
  const int tok = group_use_simt(M) ? TOK : TOKC;
  const int64_t ctas = (w->N / BN) * ((M + tok - 1) / tok);
  const int64_t KS = w->K / BK;
  if (ctas >= TARGET_CTAS) return 1;
  // at least 4 K-steps per split: a CTA's ring must fill before it pays off
  return (int)std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(std::max<int64_t>(KS / 4, 1), 32), (TARGET_CTAS + ctas - 1) / ctas));
}

bool group_ok(int group) { return group == 32 || group == 64 || group == 128; }

}  // namespace

extern "C" int mq_quantize_act_group(const void* A, mq_dtype a_dtype, int64_t M, int64_t K, int64_t lda, int group, void* qA,
                                     float* sA, void* cuda_stream) {
  if (M < 0 || K <= 0 || !group_ok(group) || K % group != 0 || K > (int64_t)1 << 30) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (a_dtype != MQ_F16 && a_dtype != MQ_BF16) return MQ_ERR_INVALID_ARG;
  if (M == 0) {
    mq::set_launch_count(0);
    return MQ_OK;
  }
  if (!A || !qA || !sA || lda < K || lda % 8 != 0) return MQ_ERR_INVALID_ARG;
  if (((uintptr_t)A & 15) || ((uintptr_t)qA & 15) || ((uintptr_t)sA & 3)) return MQ_ERR_INVALID_ARG;
  const int rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  const int64_t total = M * (K / 8);
  const int64_t blocks = (total + GT - 1) / GT;
  if (blocks > 0x7FFFFFFF) return MQ_ERR_UNSUPPORTED_SHAPE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const uint16_t* a = (const uint16_t*)A;
  uint32_t* q = (uint32_t*)qA;
  const int cpr = (int)(K / 8);
#define MQ_LAUNCH_Q(BF, LN) quantize_group_kernel<BF, LN><<<(unsigned)blocks, GT, 0, st>>>(a, lda, cpr, total, q, sA)
  const bool bf = a_dtype == MQ_BF16;
  if (group == 32) {
    if (bf) MQ_LAUNCH_Q(true, 4); else MQ_LAUNCH_Q(false, 4);
  } else if (group == 64) {
    if (bf) MQ_LAUNCH_Q(true, 8); else MQ_LAUNCH_Q(false, 8);
  } else {
    if (bf) MQ_LAUNCH_Q(true, 16); else MQ_LAUNCH_Q(false, 16);
  }
#undef MQ_LAUNCH_Q
  if (cudaGetLastError() != cudaSuccess) return MQ_ERR_CUDA;
  mq::set_launch_count(1);
  return MQ_OK;
}

extern "C" size_t mq_gemm_group_workspace_bytes(const mq_weights* w, int64_t M) {
  if (!w || M <= 0) return 0;
  const int splits = group_splits(w, M);
  return splits == 1 ? 0 : (size_t)splits * (size_t)M * (size_t)w->N * sizeof(float);
}

extern "C" int mq_gemm_group(const mq_weights* w, const void* qA, const float* sA, int group, int64_t M, void* Y, mq_dtype y_dtype,
                             int64_t ldy, int32_t* dbg0, int32_t* dbg1, void* workspace, size_t workspace_bytes,
                             void* cuda_stream) {
  if (!w) return MQ_ERR_INVALID_ARG;
  if (w->blockscale) return MQ_ERR_UNSUPPORTED_SHAPE;   // block-local residual scales: mq_gemm only
  if (M < 0 || !group_ok(group)) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (y_dtype != MQ_F16 && y_dtype != MQ_BF16) return MQ_ERR_INVALID_ARG;
  if (M == 0) {
    mq::set_launch_count(0);
    return MQ_OK;
  }
  if (!qA || !sA || !Y || ldy < w->N) return MQ_ERR_INVALID_ARG;
  if (((uintptr_t)qA & 15) || ((uintptr_t)sA & 3) || ((uintptr_t)Y & 1) || ((uintptr_t)dbg0 & 3) || ((uintptr_t)dbg1 & 3))
    return MQ_ERR_INVALID_ARG;
  const bool simt = group_use_simt(M);
  const int64_t mtiles = simt ? (M + TOK - 1) / TOK : (M + TOKC - 1) / TOKC;
  const int rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  // group = 128, decode token counts: the row-slab decode kernel, sums converted per K-step
  if (mq::decode_group_eligible(w, group, M)) return mq::decode_gemm_group(w, qA, sA, M, Y, y_dtype, ldy, dbg0, dbg1, cuda_stream);
  // group = 128 (one group per K-step), prefill token counts: the tcgen05 kernel, accumulator drained per K-step
  if (mq::group_tc_eligible(w, group, M)) {
    if ((uintptr_t)qA & 15) return MQ_ERR_INVALID_ARG;
    return mq::group_tc_gemm(w, qA, sA, M, Y, y_dtype, ldy, dbg0, dbg1, cuda_stream);
  }
  if (mtiles > 65535) return MQ_ERR_UNSUPPORTED_SHAPE;
  const int splits = group_splits(w, M);
  const size_t need = mq_gemm_group_workspace_bytes(w, M);
  if (need && (!workspace || ((uintptr_t)workspace & 15))) return MQ_ERR_INVALID_ARG;
  if (workspace_bytes < need) return MQ_ERR_WORKSPACE;
  GParams p;
  p.base = w->d_base;
  p.res = w->d_res;
  p.unit_meta = w->nnz > 0 ? w->d_unit_meta : nullptr;
  p.sw = w->d_sw;
  p.sr = w->d_sr;
  p.qA = (const uint8_t*)qA;
  p.sa = sA;
  p.Y = Y;
  p.partial = (float*)workspace;
  p.dbg0 = dbg0;
  p.dbg1 = dbg1;
  p.M = M;
  p.N = w->N;
  p.K = w->K;
  p.ldy = ldy;
  p.KS = (int)(w->K / BK);
  p.ks_per_split = (p.KS + splits - 1) / splits;
  p.splits = splits;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const dim3 grid((unsigned)(w->N / BN), (unsigned)mtiles, (unsigned)splits);
  const bool bf = y_dtype == MQ_BF16;
#define MQ_LAUNCH_G(GR)                                                                  \
  do {                                                                                   \
    if (simt) {                                                                          \
      if (bf) gemm_group_kernel<GR, true><<<grid, BN, 0, st>>>(p);                       \
      else gemm_group_kernel<GR, false><<<grid, BN, 0, st>>>(p);                         \
    } else {                                                                             \
      if (dbg0 || dbg1) {                                                                \
        if (bf) launch_mma(gemm_group_mma_kernel<GR, true, true>, grid, st, p);          \
        else launch_mma(gemm_group_mma_kernel<GR, false, true>, grid, st, p);            \
      } else {                                                                           \
        if (bf) launch_mma(gemm_group_mma_kernel<GR, true, false>, grid, st, p);         \
        else launch_mma(gemm_group_mma_kernel<GR, false, false>, grid, st, p);           \
      }                                                                                  \
    }                                                                                    \
  } while (0)
  if (group == 32) MQ_LAUNCH_G(32);
  else if (group == 64) MQ_LAUNCH_G(64);
  else MQ_LAUNCH_G(128);
#undef MQ_LAUNCH_G
  int launches = 1;
  if (splits > 1) {
    const int64_t total = M * w->N;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    if (bf)
      group_reduce_kernel<true><<<blocks, 256, 0, st>>>(p.partial, splits, M, w->N, Y, ldy);
    else
      group_reduce_kernel<false><<<blocks, 256, 0, st>>>(p.partial, splits, M, w->N, Y, ldy);
    launches = 2;
  }
  if (cudaGetLastError() != cudaSuccess) return MQ_ERR_CUDA;
  mq::set_launch_count(launches);
  return MQ_OK;
}
