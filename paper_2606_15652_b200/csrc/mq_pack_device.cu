// mq_pack_device.cu -- Algorithm 1 entirely on the device: mq_pack_weights_device.
//
//   alg1_score_kernel   one CTA per block-row: base quantization per output channel (Eq.1), packed base
//                       nibbles written straight into the kernels' tiled layout, R = W - Q(W) (Alg.1 line 1), Q(R) per
//                       output channel (A4), and the Delta-Hessian gains S_B = [sum_B h R^2 - sum_B h (R - Q(R))^2]_+
//                        in fp64 WITHOUT contraction, rows then k ascending: the host packer's and the oracle's bits
//   alg1_select_kernel  TopK: an 8-pass radix select over the scores' bit patterns (non-negative doubles
//                       order like unsigned integers) finds the budget-th largest score T; a block is selected when its
//                       score is > T, or == T and it is among the lowest-indexed ties that fill the budget; zero scores
//                       are never selected.  Exactly the set "sort by (score descending, index ascending), keep
//                       the first budget" (A6, A7).
//   alg1_cells_kernel   the residual layout's metadata from the dense selection flags: quarter mask and first-quarter
//                       index of every (n-tile, K-step) (= unit_meta), the CSR over n-tiles (cell_ptr, cell_meta)
//   alg1_resq_kernel    Q(R) of the selected blocks, packed into the 2 KB quarters of the residual area
//
// No pass over N*K data runs on the host and nothing of that size crosses PCIe: the host reads back three counters and
// the small CSR arrays it keeps for mq_weights_export and the launchers.  Rows of any length: the residual row is kept
// in shared memory when it fits and recomputed from W otherwise.
#include <cuda_runtime.h>

#include <algorithm>
#include <new>

#include "mq_internal.h"

namespace {

using mq::BK;
using mq::BN;
using mq::CellMeta;
using mq::QUARTER_BYTES;
using mq::TILE_BYTES;

__device__ __forceinline__ int dev_quant1(float x, float s) {
  const int v = (int)rintf(__fdiv_rn(x, s));
  return v > 7 ? 7 : (v < -7 ? -7 : v);
}
__device__ __forceinline__ float dev_residual(float w, float s, int q) {   // Alg.1 line 1: one rounding to fp64, one to fp32
  return __double2float_rn(__dsub_rn((double)w, __dmul_rn((double)s, (double)q)));
}
__device__ __forceinline__ float dev_block_max(float v, float* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  __syncthreads();   // red[] may still be read from the previous call
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  float m = red[0];
  for (int i = 1; i < (int)(blockDim.x >> 5); ++i) m = fmaxf(m, red[i]);
  return m;
}

constexpr int ALG1_THREADS = 256;
constexpr int ALG1_MAX_OWN = 8;   // k-blocks per thread: K <= 8 * 256 * block

// IN_SMEM: the residual row lives in shared memory (K * 4 bytes); otherwise it is recomputed from W where needed
template <bool IN_SMEM>
__global__ void __launch_bounds__(ALG1_THREADS) alg1_score_kernel(const float* __restrict__ W, const float* __restrict__ h,
                                                                  int64_t K, int block, uint8_t* __restrict__ base,
                                                                  float* __restrict__ sw, float* __restrict__ sr,
                                                                  double* __restrict__ score) {
  extern __shared__ float Rrow[];   // the residual of the current row, [K] (IN_SMEM)
  __shared__ float red[ALG1_THREADS / 32];
  const int tid = threadIdx.x;
  const int64_t bn = blockIdx.x;
  const int nbk = (int)(K / block);
  double gain[ALG1_MAX_OWN], loss[ALG1_MAX_OWN];
#pragma unroll
  for (int i = 0; i < ALG1_MAX_OWN; ++i) gain[i] = loss[i] = 0.0;
  for (int r = 0; r < block; ++r) {
    const int64_t n = bn * block + r;
    const float* w = W + n * K;
    float amax = 0.f;
    for (int64_t k = tid; k < K; k += ALG1_THREADS) amax = fmaxf(amax, fabsf(w[k]));
    amax = dev_block_max(amax, red);
    const float s = amax == 0.f ? 1.0f : __fdiv_rn(amax, 7.0f);   // Eq.1, q_max = 7 (A1-A3)
    float rmax = 0.f;
    for (int64_t kp = tid; kp < K / 2; kp += ALG1_THREADS) {      // two consecutive k = one packed byte
      const int64_t k = 2 * kp;
      const float2 wv = *reinterpret_cast<const float2*>(w + k);
      const int q0 = dev_quant1(wv.x, s), q1 = dev_quant1(wv.y, s);
      const float r0 = dev_residual(wv.x, s, q0), r1 = dev_residual(wv.y, s, q1);
      if (IN_SMEM) {
        Rrow[k] = r0;
        Rrow[k + 1] = r1;
      }
      rmax = fmaxf(rmax, fmaxf(fabsf(r0), fabsf(r1)));
      const int64_t tile = (n / BN) * (K / BK) + k / BK;
      const size_t off = (size_t)tile * TILE_BYTES + (size_t)((k % BK) >> 5) * (BN * 16) + (size_t)(n % BN) * 16 + (size_t)((k & 31) >> 1);
      base[off] = (uint8_t)((q0 & 0xF) | ((q1 & 0xF) << 4));
    }
    rmax = dev_block_max(rmax, red);   // (its barriers also publish Rrow)
    const float srn = rmax == 0.f ? 1.0f : __fdiv_rn(rmax, 7.0f);   // Q(R): per output channel over all K (A4)
    if (tid == 0) {
      sw[n] = s;
      sr[n] = srn;
    }
#pragma unroll
    for (int i = 0; i < ALG1_MAX_OWN; ++i) {
      const int bk = tid + i * ALG1_THREADS;
      if (bk < nbk) {
        double a = gain[i], b = loss[i];
        for (int k = bk * block; k < (bk + 1) * block; ++k) {
          float rf;
          if (IN_SMEM) {
            rf = Rrow[k];
          } else {
            const float wv = w[k];
            rf = dev_residual(wv, s, dev_quant1(wv, s));
          }
          const double rr = (double)rf;
          const double e = __dsub_rn(rr, __dmul_rn((double)srn, (double)dev_quant1(rf, srn)));
          const double hk = h ? (double)h[k] : 1.0;
          a = __dadd_rn(a, __dmul_rn(hk, __dmul_rn(rr, rr)));   // P:156, no contraction: the host's bits
          b = __dadd_rn(b, __dmul_rn(hk, __dmul_rn(e, e)));
        }
        gain[i] = a;
        loss[i] = b;
      }
    }
    __syncthreads();   // Rrow is overwritten by the next row
  }
#pragma unroll
  for (int i = 0; i < ALG1_MAX_OWN; ++i) {
    const int bk = tid + i * ALG1_THREADS;
    if (bk < nbk) {
      const double d = __dsub_rn(gain[i], loss[i]);
      score[bn * nbk + bk] = d > 0.0 ? d : 0.0;
    }
  }
}

// ---- TopK: one CTA.  ctrl[0] = nnz (out) -----------------------------------------------------------------------
constexpr int SEL_THREADS = 1024;

__global__ void __launch_bounds__(SEL_THREADS) alg1_select_kernel(const unsigned long long* __restrict__ key, int64_t n,
                                                                  int64_t budget, uint8_t* __restrict__ flag,
                                                                  int64_t* __restrict__ ctrl) {
  __shared__ unsigned int hist[256];
  __shared__ unsigned long long s_prefix, s_remaining, s_npos;
  __shared__ int s_warp_ties[SEL_THREADS / 32];
  __shared__ unsigned long long s_tie_base;
  const int tid = threadIdx.x;
  // positive scores
  if (tid == 0) s_npos = 0;
  __syncthreads();
  unsigned long long cnt = 0;
  for (int64_t i = tid; i < n; i += SEL_THREADS) cnt += key[i] != 0ull;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
  if ((tid & 31) == 0 && cnt) atomicAdd(&s_npos, cnt);
  __syncthreads();
  const unsigned long long npos = s_npos;
  unsigned long long T = 0, take_ties = 0;   // select key > T, and the first take_ties keys == T
  if ((unsigned long long)budget < npos) {
    // the budget-th largest key, byte by byte from the top
    if (tid == 0) {
      s_prefix = 0;
      s_remaining = (unsigned long long)budget;
    }
    for (int pass = 7; pass >= 0; --pass) {
      if (tid < 256) hist[tid] = 0;
      __syncthreads();
      const unsigned long long prefix = s_prefix;
      for (int64_t i = tid; i < n; i += SEL_THREADS) {
        const unsigned long long k = key[i];
        if (k != 0ull && (pass == 7 || (k >> (8 * (pass + 1))) == prefix)) atomicAdd(&hist[(k >> (8 * pass)) & 255], 1u);
      }
      __syncthreads();
      if (tid == 0) {
        unsigned long long cum = 0, rem = s_remaining;
        int digit = 0;
        for (int b = 255; b >= 0; --b) {
          if (cum + hist[b] >= rem) {
            digit = b;
            rem -= cum;
            break;
          }
          cum += hist[b];
        }
        s_prefix = (prefix << 8) | (unsigned long long)digit;
        s_remaining = rem;
      }
      __syncthreads();
    }
    T = s_prefix;
    take_ties = s_remaining;   // how many of the keys equal to T belong to the top `budget`
  }
  // dense selection flags; ties in ascending index order
  if (tid == 0) s_tie_base = 0;
  __syncthreads();
  unsigned long long nsel = 0;
  for (int64_t i0 = 0; i0 < n; i0 += SEL_THREADS) {
    const int64_t i = i0 + tid;
    const unsigned long long k = i < n ? key[i] : 0ull;
    const bool tie = T != 0ull && k == T;
    const unsigned int bal = __ballot_sync(0xffffffffu, tie);
    if ((tid & 31) == 0) s_warp_ties[tid >> 5] = __popc(bal);
    __syncthreads();
    unsigned long long before = s_tie_base;
    for (int wv = 0; wv < (tid >> 5); ++wv) before += (unsigned long long)s_warp_ties[wv];
    before += (unsigned long long)__popc(bal & ((1u << (tid & 31)) - 1u));
    const bool sel = k != 0ull && (k > T || (tie && before < take_ties));
    if (i < n) flag[i] = sel ? 1 : 0;
    nsel += sel;
    __syncthreads();
    if (tid == 0) {
      unsigned long long t = 0;
      for (int wv = 0; wv < SEL_THREADS / 32; ++wv) t += (unsigned long long)s_warp_ties[wv];
      s_tie_base += t;
    }
    __syncthreads();
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) nsel += __shfl_xor_sync(0xffffffffu, nsel, o);
  if (tid == 0) s_npos = 0;
  __syncthreads();
  if ((tid & 31) == 0 && nsel) atomicAdd(&s_npos, nsel);
  __syncthreads();
  if (tid == 0) ctrl[0] = (int64_t)s_npos;
}

// ---- residual layout metadata from the dense selection flags: one CTA, chunked scan over the (n-tile, K-step) cells ------
// ctrl[1] = stored quarters, ctrl[2] = cells (out)
__global__ void __launch_bounds__(SEL_THREADS) alg1_cells_kernel(const uint8_t* __restrict__ flag, int NT, int KS, int block, int nbk,
                                                                 int2* __restrict__ unit_meta, int32_t* __restrict__ cell_ptr,
                                                                 CellMeta* __restrict__ cell_meta, int64_t* __restrict__ ctrl) {
  __shared__ int s_wq[SEL_THREADS / 32], s_wc[SEL_THREADS / 32];
  __shared__ long long s_qbase, s_cbase;
  const int tid = threadIdx.x;
  if (tid == 0) s_qbase = s_cbase = 0;
  __syncthreads();
  const int64_t ncell = (int64_t)NT * KS;
  for (int64_t c0 = 0; c0 < ncell; c0 += SEL_THREADS) {
    const int64_t c = c0 + tid;
    int mask = 0, t = 0, ks = 0;
    if (c < ncell) {
      t = (int)(c / KS);
      ks = (int)(c - (int64_t)t * KS);
      if (block == 128) {
        mask = flag[(int64_t)t * nbk + ks] ? 0xF : 0;
      } else {   // quarter q = 2 * (k-half) + (row-half): block (2 t + r, 2 ks + h)
#pragma unroll
        for (int q = 0; q < 4; ++q)
          if (flag[(int64_t)(2 * t + (q & 1)) * nbk + (2 * ks + (q >> 1))]) mask |= 1 << q;
      }
    }
    const int nq = __popc(mask), nc = mask != 0;
    // block-wide exclusive scans of nq and nc
    int wq = nq, wc = nc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int a = __shfl_up_sync(0xffffffffu, wq, o), b = __shfl_up_sync(0xffffffffu, wc, o);
      if ((tid & 31) >= o) {
        wq += a;
        wc += b;
      }
    }
    if ((tid & 31) == 31) {
      s_wq[tid >> 5] = wq;
      s_wc[tid >> 5] = wc;
    }
    __syncthreads();
    long long qoff = s_qbase + (wq - nq), cidx = s_cbase + (wc - nc);
    for (int wv = 0; wv < (tid >> 5); ++wv) {
      qoff += s_wq[wv];
      cidx += s_wc[wv];
    }
    if (c < ncell) {
      unit_meta[c] = make_int2(mask, mask ? (int)qoff : 0);
      if (ks == 0) cell_ptr[t] = (int32_t)cidx;
      if (mask) {
        CellMeta m;
        m.kstep_mask = ks | (mask << 24);
        m.qoff = (int32_t)qoff;
        cell_meta[cidx] = m;
      }
    }
    __syncthreads();
    if (tid == 0) {
      long long tq = 0, tc = 0;
      for (int wv = 0; wv < SEL_THREADS / 32; ++wv) {
        tq += s_wq[wv];
        tc += s_wc[wv];
      }
      s_qbase += tq;
      s_cbase += tc;
    }
    __syncthreads();
  }
  if (tid == 0) {
    cell_ptr[NT] = (int32_t)s_cbase;
    ctrl[1] = s_qbase;
    ctrl[2] = s_cbase;
  }
}

// ---- Q(R) of the selected blocks into the residual quarters: one CTA per (n-tile, K-step) -----------------------------
__global__ void __launch_bounds__(256) alg1_resq_kernel(const float* __restrict__ W, int64_t K, int block, int KS,
                                                        const float* __restrict__ sw, const float* __restrict__ sr,
                                                        const int2* __restrict__ unit_meta, uint8_t* __restrict__ res) {
  const int2 um = unit_meta[blockIdx.x];
  const int mask = um.x & 0xF;
  if (!mask) return;
  const int t = (int)(blockIdx.x / KS), ks = (int)(blockIdx.x - (unsigned)t * KS);
  int stored = 0;
  for (int q = 0; q < 4; ++q) {
    if (!(mask & (1 << q))) continue;
    // the quarter's 64 rows x 64 input channels in W
    const int64_t n0 = (int64_t)t * BN + (q & 1) * 64, k0 = (int64_t)ks * BK + (q >> 1) * 64;
    uint8_t* dst = res + ((size_t)um.y + (size_t)stored) * QUARTER_BYTES;
    for (int b = threadIdx.x; b < QUARTER_BYTES; b += blockDim.x) {
      // byte b of the quarter layout [2 chunks of 32 k][64 rows][16 B]: elements 2i | 2i+1 << 4
      const int chunk = b >> 10, row = (b & 1023) >> 4, c = chunk * 32 + 2 * (b & 15);
      const int64_t n = n0 + row;
      const float s = sw[n], srn = sr[n];
      const float2 wv = *reinterpret_cast<const float2*>(W + n * K + k0 + c);
      const int q0 = dev_quant1(dev_residual(wv.x, s, dev_quant1(wv.x, s)), srn);
      const int q1 = dev_quant1(dev_residual(wv.y, s, dev_quant1(wv.y, s)), srn);
      dst[b] = (uint8_t)((q0 & 0xF) | ((q1 & 0xF) << 4));
    }
    ++stored;
  }
}

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace

extern "C" int mq_pack_weights_device(const float* W_dev, int64_t N, int64_t K, const float* h_dev, int block, int64_t budget,
                                      mq_weights** out, void* cuda_stream) {
  if (!out) return MQ_ERR_INVALID_ARG;
  *out = nullptr;
  if (!W_dev || budget < 0) return MQ_ERR_INVALID_ARG;
  if (N <= 0 || K <= 0 || (block != 64 && block != 128) || N % BN != 0 || K % BK != 0 || K / BK >= (1 << 24))
    return MQ_ERR_UNSUPPORTED_SHAPE;
  if ((long double)49 * 256 * (long double)K >= 2147483648.0L) return MQ_ERR_ACC_OVERFLOW;
  if (((uintptr_t)W_dev & 7) || ((uintptr_t)h_dev & 3)) return MQ_ERR_INVALID_ARG;
  int rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  const int64_t NT = N / BN, KS = K / BK, nbn = N / block, nbk = K / block, nblocks = nbn * nbk;
  if (nbk > (int64_t)ALG1_MAX_OWN * ALG1_THREADS || NT * KS >= ((int64_t)1 << 31)) return MQ_ERR_UNSUPPORTED_SHAPE;
  cudaStream_t st = (cudaStream_t)cuda_stream;

  // the layer's single device allocation, sized for the whole budget (fewer blocks may have a positive score)
  const int64_t max_blocks = std::min<int64_t>(budget, nblocks);
  const int64_t max_quarters = max_blocks * (block == 128 ? 4 : 1);
  const int64_t max_cells = std::min<int64_t>(max_quarters, NT * KS);
  const size_t base_bytes = (size_t)N * (size_t)K / 2;
  size_t o_base = 0;
  size_t o_sw = align_up(o_base + base_bytes, 256);
  size_t o_sr = align_up(o_sw + (size_t)N * 4, 256);
  size_t o_res = align_up(o_sr + (size_t)N * 4, 256);
  size_t o_cptr = align_up(o_res + std::max<size_t>((size_t)max_quarters * QUARTER_BYTES, 16), 256);
  size_t o_cmeta = align_up(o_cptr + ((size_t)NT + 1) * 4, 256);
  size_t o_umeta = align_up(o_cmeta + std::max<size_t>((size_t)max_cells, 1) * sizeof(CellMeta), 256);
  size_t o_qscale = align_up(o_umeta + (size_t)NT * KS * 8, 256);
  size_t total = align_up(o_qscale + 16, 256);

  mq_weights* w = new (std::nothrow) mq_weights();
  if (!w) return MQ_ERR_OOM;
  void* blob = nullptr;
  double* d_score = nullptr;
  uint8_t* d_flag = nullptr;
  int64_t* d_ctrl = nullptr;
  auto fail = [&](int code) {
    (void)cudaGetLastError();
    cudaFree(blob);
    cudaFree(d_score);
    cudaFree(d_flag);
    cudaFree(d_ctrl);
    delete w;
    return code;
  };
  if (cudaMalloc(&blob, total) != cudaSuccess || cudaMalloc(&d_score, (size_t)nblocks * 8) != cudaSuccess ||
      cudaMalloc(&d_flag, (size_t)nblocks) != cudaSuccess || cudaMalloc(&d_ctrl, 64) != cudaSuccess)
    return fail(MQ_ERR_OOM);
  uint8_t* p = (uint8_t*)blob;
  float* d_sw = (float*)(p + o_sw);
  float* d_sr = (float*)(p + o_sr);

  // 1. base quantization, residual, scores
  const size_t smem = (size_t)K * sizeof(float);
  if (smem <= 200 * 1024) {
    if (cudaFuncSetAttribute(alg1_score_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
      return fail(MQ_ERR_CUDA);
    alg1_score_kernel<true><<<(unsigned)nbn, ALG1_THREADS, smem, st>>>(W_dev, h_dev, K, block, p + o_base, d_sw, d_sr, d_score);
  } else {
    alg1_score_kernel<false><<<(unsigned)nbn, ALG1_THREADS, 0, st>>>(W_dev, h_dev, K, block, p + o_base, d_sw, d_sr, d_score);
  }
  // 2. TopK -> dense flags; 3. cells, CSR, unit_meta; 4. Q(R) of the selected blocks
  alg1_select_kernel<<<1, SEL_THREADS, 0, st>>>((const unsigned long long*)d_score, nblocks, budget, d_flag, d_ctrl);
  alg1_cells_kernel<<<1, SEL_THREADS, 0, st>>>(d_flag, (int)NT, (int)KS, block, (int)nbk, (int2*)(p + o_umeta),
                                                (int32_t*)(p + o_cptr), (CellMeta*)(p + o_cmeta), d_ctrl);
  alg1_resq_kernel<<<(unsigned)(NT * KS), 256, 0, st>>>(W_dev, K, block, (int)KS, d_sw, d_sr, (const int2*)(p + o_umeta), p + o_res);
  int64_t ctrl[3] = {0, 0, 0};
  if (cudaGetLastError() != cudaSuccess || cudaMemcpyAsync(ctrl, d_ctrl, sizeof(ctrl), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess)
    return fail(MQ_ERR_CUDA);

  w->N = N;
  w->K = K;
  w->block = block;
  w->nnz = ctrl[0];
  w->n_quarters = ctrl[1];
  w->n_cells = ctrl[2];
  if (w->n_quarters > max_quarters || w->n_cells > max_cells) return fail(MQ_ERR_CUDA);
  // the small CSR arrays the host side keeps (export, launch planning)
  try {
    w->h_cell_ptr.assign((size_t)NT + 1, 0);
    w->h_cell_meta.resize((size_t)w->n_cells);
  } catch (const std::bad_alloc&) {
    return fail(MQ_ERR_OOM);
  }
  if (cudaMemcpyAsync(w->h_cell_ptr.data(), p + o_cptr, ((size_t)NT + 1) * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      (w->n_cells && cudaMemcpyAsync(w->h_cell_meta.data(), p + o_cmeta, (size_t)w->n_cells * sizeof(CellMeta), cudaMemcpyDeviceToHost,
                                     st) != cudaSuccess) ||
      cudaStreamSynchronize(st) != cudaSuccess)
    return fail(MQ_ERR_CUDA);
  for (int64_t t = 0; t < NT; ++t)
    w->max_cells_per_tile = std::max(w->max_cells_per_tile, (int)(w->h_cell_ptr[(size_t)t + 1] - w->h_cell_ptr[(size_t)t]));
  w->dev_blob = blob;
  w->dev_bytes = total;
  w->d_base = p + o_base;
  w->d_sw = d_sw;
  w->d_sr = d_sr;
  w->d_res = p + o_res;
  w->d_cell_ptr = (int32_t*)(p + o_cptr);
  w->d_cell_meta = (CellMeta*)(p + o_cmeta);
  w->d_unit_meta = (int32_t*)(p + o_umeta);
  w->d_qscale = (float*)(p + o_qscale);
  cudaFree(d_score);
  cudaFree(d_flag);
  cudaFree(d_ctrl);
  d_score = nullptr;
  d_flag = nullptr;
  d_ctrl = nullptr;
  if (mq::build_weight_tmaps(w) != MQ_OK) return fail(MQ_ERR_CUDA);
  *out = w;
  return MQ_OK;
}
