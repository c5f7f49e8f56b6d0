// mq_pack.cu -- host side of mq_pack_weights / mq_pack_prequantized / mq_weights_export.
//
// Algorithm 1 of the paper runs here on the host, once per layer (offline,
// SURVEY 8(a) row a0), followed by the re-tiling into the kernel's device layout
// (mq_internal.h).  This is the product's own implementation; it shares no code with
// oracle/.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <new>
#include <thread>

#include "mq_internal.h"

namespace {

using mq::BK;
using mq::BN;
using mq::CellMeta;
using mq::QUARTER_BYTES;
using mq::TILE_BYTES;

template <class F>
void parallel_for(int64_t n, F&& fn) {
  unsigned hw = std::thread::hardware_concurrency();
  int64_t nt = std::max<int64_t>(1, std::min<int64_t>(hw ? hw : 1, n));
  if (nt == 1) {
    for (int64_t i = 0; i < n; ++i) fn(i);
    return;
  }
  std::atomic<int64_t> next{0};
  std::vector<std::thread> th;
  th.reserve((size_t)nt);
  for (int64_t t = 0; t < nt; ++t)
    th.emplace_back([&] {
      for (;;) {
        int64_t i = next.fetch_add(1);
        if (i >= n) break;
        fn(i);
      }
    });
  for (auto& t : th) t.join();
}

// Eq.1 with q_max = 7 (A1): scale of one row.  All-zero row -> 1 (A2).
float row_scale(const float* x, int64_t L) {
  float amax = 0.f;
  for (int64_t i = 0; i < L; ++i) amax = std::max(amax, std::fabs(x[i]));
  if (amax == 0.f) return 1.0f;
  volatile float s = amax / 7.0f;  // one binary32 division (A3)
  return s;
}
// Eq.1: one element.  IEEE binary32 division, round half to even, clamp to [-7,7].
inline int quant1(float x, float s) {
  volatile float t = x / s;
  int v = (int)std::nearbyintf(t);
  return v > 7 ? 7 : (v < -7 ? -7 : v);
}

struct SelBlock {
  int32_t bn, bk;
  std::vector<int8_t> q;  // [block][block], row = n, col = k
  std::vector<float> srow;  // [block] block-local residual scale of every row (blockscale layers only)
};

struct HostLayer {
  int64_t N = 0, K = 0;
  int block = 0;
  std::vector<uint8_t> base;  // tiled, see mq_internal.h
  std::vector<float> sw, sr;
  std::vector<SelBlock> blocks;
  bool blockscale = false;   // reading A4b: the residual scale is per (selected block, row), not per output channel
};

inline size_t base_offset(int64_t n, int64_t k, int64_t K) {
  int64_t tile = (n / BN) * (K / BK) + k / BK;
  // inside a tile: [chunk c = (k % BK) / 32][row n % BN][16 bytes] (mq_internal.h)
  return (size_t)tile * TILE_BYTES + (size_t)((k % BK) >> 5) * (BN * 16) + (size_t)(n % BN) * 16 +
         (size_t)((k & 31) >> 1);
}

// byte of element (row, c) inside a 2 KB residual quarter: [chunk c / 32][row 0..63][16 bytes]
inline size_t quarter_offset(int row, int c) { return (size_t)(c >> 5) * 1024 + (size_t)row * 16 + (size_t)((c & 31) >> 1); }

inline void put_nibble(uint8_t* byte, int hi, int v) {
  uint8_t nib = (uint8_t)(v & 0xF);
  if (hi)
    *byte = (uint8_t)((*byte & 0x0F) | (nib << 4));
  else
    *byte = (uint8_t)((*byte & 0xF0) | nib);
}
inline int get_nibble(uint8_t byte, int hi) {
  int v = hi ? (byte >> 4) : (byte & 0xF);
  return v >= 8 ? v - 16 : v;
}

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

int shape_check(int64_t N, int64_t K, int block) {
  if (N <= 0 || K <= 0) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (block != 64 && block != 128) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (N % BN != 0 || K % BK != 0) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (K / BK >= (1 << 24)) return MQ_ERR_UNSUPPORTED_SHAPE;
  // the kernel accumulates 16*q_a * 16*q_w: |acc| <= 49 * 256 * K must fit int32
  if ((long double)49 * 256 * (long double)K >= 2147483648.0L) return MQ_ERR_ACC_OVERFLOW;
  return MQ_OK;
}

// Build cells from the selected blocks, upload everything.
int finalize(HostLayer& L, mq_weights** out, cudaStream_t stream) {
  const int64_t NT = L.N / BN, KS = L.K / BK;
  // cell key = tile * KS + kstep ; quarter masks
  struct Q {
    int64_t key;
    int q;
    const SelBlock* b;
    int sub_r, sub_h;  // which 64x64 part of the block (block = 128 only)
  };
  std::vector<Q> qs;
  qs.reserve(L.blocks.size() * (L.block == 128 ? 4 : 1));
  for (const SelBlock& b : L.blocks) {
    if (L.block == 64) {
      int64_t key = (int64_t)(b.bn >> 1) * KS + (b.bk >> 1);
      qs.push_back(Q{key, 2 * (b.bk & 1) + (b.bn & 1), &b, 0, 0});
    } else {
      int64_t key = (int64_t)b.bn * KS + b.bk;
      for (int h = 0; h < 2; ++h)
        for (int r = 0; r < 2; ++r) qs.push_back(Q{key, 2 * h + r, &b, r, h});
    }
  }
  std::sort(qs.begin(), qs.end(), [](const Q& a, const Q& b) { return a.key != b.key ? a.key < b.key : a.q < b.q; });
  for (size_t i = 1; i < qs.size(); ++i)
    if (qs[i].key == qs[i - 1].key && qs[i].q == qs[i - 1].q) return MQ_ERR_INVALID_ARG;  // duplicate block

  mq_weights* w = new (std::nothrow) mq_weights();
  if (!w) return MQ_ERR_OOM;
  w->N = L.N;
  w->K = L.K;
  w->block = L.block;
  w->nnz = (int64_t)L.blocks.size();
  w->n_quarters = (int64_t)qs.size();
  w->h_cell_ptr.assign((size_t)NT + 1, 0);

  std::vector<uint8_t> res((size_t)qs.size() * QUARTER_BYTES, 0);
  std::vector<float> qscale(L.blockscale ? qs.size() * 64 : 0, 1.0f);
  for (size_t i = 0; i < qs.size(); ++i) {
    const Q& e = qs[i];
    if (L.blockscale)
      for (int row = 0; row < 64; ++row) qscale[i * 64 + (size_t)row] = e.b->srow[(size_t)(e.sub_r * 64 + row)];
    if (i == 0 || qs[i - 1].key != e.key) {
      CellMeta m;
      m.kstep_mask = (int32_t)(e.key % KS);
      m.qoff = (int32_t)i;
      w->h_cell_meta.push_back(m);
      w->h_cell_ptr[(size_t)(e.key / KS) + 1] += 1;
    }
    w->h_cell_meta.back().kstep_mask |= (1 << e.q) << 24;
    uint8_t* dst = res.data() + i * QUARTER_BYTES;
    const int bs = L.block;
    for (int row = 0; row < 64; ++row)
      for (int c = 0; c < 64; ++c) {
        int v = e.b->q[(size_t)(e.sub_r * 64 + row) * bs + (size_t)(e.sub_h * 64 + c)];
        put_nibble(dst + quarter_offset(row, c), c & 1, v);
      }
  }
  w->n_cells = (int64_t)w->h_cell_meta.size();
  for (int64_t t = 0; t < NT; ++t) {
    w->max_cells_per_tile = std::max(w->max_cells_per_tile, (int)w->h_cell_ptr[(size_t)t + 1]);
    w->h_cell_ptr[(size_t)t + 1] += w->h_cell_ptr[(size_t)t];
  }

  // one device allocation
  size_t o_base = 0;
  size_t o_sw = align_up(o_base + L.base.size(), 256);
  size_t o_sr = align_up(o_sw + (size_t)L.N * 4, 256);
  size_t o_res = align_up(o_sr + (size_t)L.N * 4, 256);
  size_t o_cptr = align_up(o_res + std::max<size_t>(res.size(), 16), 256);
  size_t o_cmeta = align_up(o_cptr + ((size_t)NT + 1) * 4, 256);
  size_t o_umeta = align_up(o_cmeta + std::max<size_t>((size_t)w->n_cells, 1) * sizeof(CellMeta), 256);
  size_t o_qscale = align_up(o_umeta + (size_t)NT * KS * 8, 256);
  size_t total = align_up(o_qscale + std::max<size_t>(qscale.size() * 4, 16), 256);
  // dense per-(n-tile, K-step) lookup of the CSR cells: {quarter mask, first quarter index}
  std::vector<int32_t> umeta((size_t)NT * KS * 2, 0);
  for (int64_t t = 0; t < NT; ++t)
    for (int32_t c = w->h_cell_ptr[(size_t)t]; c < w->h_cell_ptr[(size_t)t + 1]; ++c) {
      const CellMeta& m = w->h_cell_meta[(size_t)c];
      const size_t u = (size_t)t * KS + (size_t)(m.kstep_mask & 0xFFFFFF);
      umeta[2 * u] = (m.kstep_mask >> 24) & 0xF;
      umeta[2 * u + 1] = m.qoff;
    }
  void* blob = nullptr;
  cudaError_t ce = cudaMalloc(&blob, total);
  if (ce != cudaSuccess) {
    cudaGetLastError();
    delete w;
    return ce == cudaErrorMemoryAllocation ? MQ_ERR_OOM : MQ_ERR_CUDA;
  }
  uint8_t* p = (uint8_t*)blob;
  bool ok = true;
  ok &= cudaMemcpyAsync(p + o_base, L.base.data(), L.base.size(), cudaMemcpyHostToDevice, stream) == cudaSuccess;
  ok &= cudaMemcpyAsync(p + o_sw, L.sw.data(), (size_t)L.N * 4, cudaMemcpyHostToDevice, stream) == cudaSuccess;
  ok &= cudaMemcpyAsync(p + o_sr, L.sr.data(), (size_t)L.N * 4, cudaMemcpyHostToDevice, stream) == cudaSuccess;
  if (!res.empty())
    ok &= cudaMemcpyAsync(p + o_res, res.data(), res.size(), cudaMemcpyHostToDevice, stream) == cudaSuccess;
  ok &= cudaMemcpyAsync(p + o_cptr, w->h_cell_ptr.data(), ((size_t)NT + 1) * 4, cudaMemcpyHostToDevice, stream) ==
        cudaSuccess;
  if (w->n_cells)
    ok &= cudaMemcpyAsync(p + o_cmeta, w->h_cell_meta.data(), (size_t)w->n_cells * sizeof(CellMeta),
                          cudaMemcpyHostToDevice, stream) == cudaSuccess;
  ok &= cudaMemcpyAsync(p + o_umeta, umeta.data(), umeta.size() * 4, cudaMemcpyHostToDevice, stream) == cudaSuccess;
  if (!qscale.empty())
    ok &= cudaMemcpyAsync(p + o_qscale, qscale.data(), qscale.size() * 4, cudaMemcpyHostToDevice, stream) == cudaSuccess;
  ok &= cudaStreamSynchronize(stream) == cudaSuccess;
  if (!ok) {
    cudaGetLastError();
    cudaFree(blob);
    delete w;
    return MQ_ERR_CUDA;
  }
  w->dev_blob = blob;
  w->dev_bytes = total;
  w->d_base = p + o_base;
  w->d_sw = (float*)(p + o_sw);
  w->d_sr = (float*)(p + o_sr);
  w->d_res = p + o_res;
  w->d_cell_ptr = (int32_t*)(p + o_cptr);
  w->d_cell_meta = (CellMeta*)(p + o_cmeta);
  w->d_unit_meta = (int32_t*)(p + o_umeta);
  w->blockscale = L.blockscale;
  w->d_qscale = (float*)(p + o_qscale);
  if (mq::build_weight_tmaps(w) != MQ_OK) {
    cudaFree(blob);
    delete w;
    return MQ_ERR_CUDA;
  }
  *out = w;
  return MQ_OK;
}

}  // namespace

namespace {
int pack_prequantized_impl(const int8_t* qW, const float* sW, int64_t N, int64_t K, int block, int64_t nnz,
                           const int32_t* blk_n, const int32_t* blk_k, const int8_t* qR, const float* sR, const float* sRb,
                           mq_weights** out, void* cuda_stream);
}

extern "C" int mq_pack_prequantized(const int8_t* qW, const float* sW, int64_t N, int64_t K, int block, int64_t nnz,
                                    const int32_t* blk_n, const int32_t* blk_k, const int8_t* qR, const float* sR,
                                    mq_weights** out, void* cuda_stream) {
  if (!sR) return MQ_ERR_INVALID_ARG;
  return pack_prequantized_impl(qW, sW, N, K, block, nnz, blk_n, blk_k, qR, sR, nullptr, out, cuda_stream);
}

extern "C" int mq_pack_prequantized_blockscale(const int8_t* qW, const float* sW, int64_t N, int64_t K, int block, int64_t nnz,
                                               const int32_t* blk_n, const int32_t* blk_k, const int8_t* qR, const float* sRb,
                                               mq_weights** out, void* cuda_stream) {
  if (nnz > 0 && !sRb) return MQ_ERR_INVALID_ARG;
  static const float one = 1.0f;
  return pack_prequantized_impl(qW, sW, N, K, block, nnz, blk_n, blk_k, qR, nullptr, nnz > 0 ? sRb : &one, out, cuda_stream);
}

namespace {
int pack_prequantized_impl(const int8_t* qW, const float* sW, int64_t N, int64_t K, int block, int64_t nnz,
                           const int32_t* blk_n, const int32_t* blk_k, const int8_t* qR, const float* sR, const float* sRb,
                           mq_weights** out, void* cuda_stream) {
  if (!out) return MQ_ERR_INVALID_ARG;
  *out = nullptr;
  if (!qW || !sW || nnz < 0) return MQ_ERR_INVALID_ARG;
  if (nnz > 0 && (!blk_n || !blk_k || !qR)) return MQ_ERR_INVALID_ARG;
  int rc = shape_check(N, K, block);
  if (rc != MQ_OK) return rc;
  rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  const int64_t nbn = N / block, nbk = K / block;
  for (int64_t e = 0; e < nnz; ++e)
    if (blk_n[e] < 0 || blk_n[e] >= nbn || blk_k[e] < 0 || blk_k[e] >= nbk) return MQ_ERR_INVALID_ARG;

  HostLayer L;
  L.N = N;
  L.K = K;
  L.block = block;
  try {
    L.base.assign((size_t)N * (size_t)K / 2, 0);
    L.sw.assign(sW, sW + N);
    if (sR)
      L.sr.assign(sR, sR + N);
    else
      L.sr.assign((size_t)N, 1.0f);
    L.blockscale = sRb != nullptr;
    L.blocks.resize((size_t)nnz);
  } catch (const std::bad_alloc&) {
    return MQ_ERR_OOM;
  }
  std::atomic<int> bad{0};
  parallel_for(N, [&](int64_t n) {
    const int8_t* row = qW + n * K;
    for (int64_t k = 0; k < K; ++k) {
      int v = row[k];
      if (v < -7 || v > 7) bad = 1;
      put_nibble(&L.base[base_offset(n, k, K)], (int)(k & 1), v);
    }
  });
  const size_t bsz = (size_t)block * block;
  for (int64_t e = 0; e < nnz; ++e) {
    SelBlock& b = L.blocks[(size_t)e];
    b.bn = blk_n[e];
    b.bk = blk_k[e];
    b.q.assign(qR + (size_t)e * bsz, qR + (size_t)(e + 1) * bsz);
    if (sRb) b.srow.assign(sRb + (size_t)e * block, sRb + (size_t)(e + 1) * block);
    for (int8_t v : b.q)
      if (v < -7 || v > 7) bad = 1;
  }
  if (bad) return MQ_ERR_INVALID_ARG;
  return finalize(L, out, (cudaStream_t)cuda_stream);
}
}  // namespace

// Algorithm 1, in the paper's order.
namespace {
int pack_weights_impl(const float* W, int64_t N, int64_t K, const float* h, int block, int64_t budget, bool blockscale,
                      mq_weights** out, void* cuda_stream);
}
extern "C" int mq_pack_weights(const float* W, int64_t N, int64_t K, const float* h, int block, int64_t budget,
                               mq_weights** out, void* cuda_stream) {
  return pack_weights_impl(W, N, K, h, block, budget, false, out, cuda_stream);
}
// Algorithm 1 with block-local residual scales (reading A4b): Q(R) of Eq.1 is applied to every (channel, k-block) run.
extern "C" int mq_pack_weights_blockscale(const float* W, int64_t N, int64_t K, const float* h, int block, int64_t budget,
                                          mq_weights** out, void* cuda_stream) {
  return pack_weights_impl(W, N, K, h, block, budget, true, out, cuda_stream);
}
namespace {
int pack_weights_impl(const float* W, int64_t N, int64_t K, const float* h, int block, int64_t budget, bool blockscale,
                      mq_weights** out, void* cuda_stream) {
  if (!out) return MQ_ERR_INVALID_ARG;
  *out = nullptr;
  if (!W || budget < 0) return MQ_ERR_INVALID_ARG;
  int rc = shape_check(N, K, block);
  if (rc != MQ_OK) return rc;
  rc = mq::check_device();
  if (rc != MQ_OK) return rc;

  const int64_t nbn = N / block, nbk = K / block, nblocks = nbn * nbk;
  HostLayer L;
  L.N = N;
  L.K = K;
  L.block = block;
  L.blockscale = blockscale;
  std::vector<double> score;
  try {
    L.base.assign((size_t)N * (size_t)K / 2, 0);
    L.sw.assign((size_t)N, 0.f);
    L.sr.assign((size_t)N, 0.f);
    score.assign((size_t)nblocks, 0.0);
  } catch (const std::bad_alloc&) {
    return MQ_ERR_OOM;
  }

  // One block-row (block output channels) at a time: base quantize, R, Q(R), score.
  parallel_for(nbn, [&](int64_t bn) {
    std::vector<float> R((size_t)K);
    std::vector<double> gain((size_t)nbk), loss((size_t)nbk);
    std::fill(gain.begin(), gain.end(), 0.0);
    std::fill(loss.begin(), loss.end(), 0.0);
    for (int64_t n = bn * block; n < (bn + 1) * block; ++n) {
      const float* w = W + n * K;
      const float s = row_scale(w, K);  // base: per output channel
      L.sw[(size_t)n] = s;
      for (int64_t k = 0; k < K; ++k) {
        int q = quant1(w[k], s);
        put_nibble(&L.base[base_offset(n, k, K)], (int)(k & 1), q);
        R[(size_t)k] = (float)((double)w[k] - (double)s * (double)q);  // Alg.1 line 1
      }
      const float sr_row = row_scale(R.data(), K);  // Q(R): per output channel over all K (A4)
      L.sr[(size_t)n] = blockscale ? 1.0f : sr_row;
      // P:156  S_B = [ sum h R^2 - sum h (R - Q(R))^2 ]_+ ; rows ascending, k ascending
      for (int64_t bk = 0; bk < nbk; ++bk) {
        // A4b: the scale of this row inside this block
        const float sr = blockscale ? row_scale(R.data() + bk * block, block) : sr_row;
        double a = gain[(size_t)bk], b = loss[(size_t)bk];
        for (int64_t k = bk * block; k < (bk + 1) * block; ++k) {
          double r = (double)R[(size_t)k];
          double e = r - (double)sr * (double)quant1(R[(size_t)k], sr);
          double hk = h ? (double)h[k] : 1.0;
          a += hk * (r * r);
          b += hk * (e * e);
        }
        gain[(size_t)bk] = a;
        loss[(size_t)bk] = b;
      }
    }
    for (int64_t bk = 0; bk < nbk; ++bk) {
      double d = gain[(size_t)bk] - loss[(size_t)bk];
      score[(size_t)(bn * nbk + bk)] = d > 0.0 ? d : 0.0;
    }
  });

  // TopK: positive scores only, ties -> lower index (A7).
  std::vector<int64_t> cand;
  for (int64_t b = 0; b < nblocks; ++b)
    if (score[(size_t)b] > 0.0) cand.push_back(b);
  int64_t nnz = std::min<int64_t>(budget, (int64_t)cand.size());
  auto better = [&](int64_t x, int64_t y) {
    if (score[(size_t)x] != score[(size_t)y]) return score[(size_t)x] > score[(size_t)y];
    return x < y;
  };
  std::partial_sort(cand.begin(), cand.begin() + nnz, cand.end(), better);
  cand.resize((size_t)nnz);

  // Q(R) on the selected blocks (recomputed from W, s_w, s_r: same arithmetic as above).
  L.blocks.resize((size_t)nnz);
  parallel_for(nnz, [&](int64_t e) {
    SelBlock& b = L.blocks[(size_t)e];
    b.bn = (int32_t)(cand[(size_t)e] / nbk);
    b.bk = (int32_t)(cand[(size_t)e] % nbk);
    b.q.resize((size_t)block * block);
    if (blockscale) b.srow.resize((size_t)block);
    std::vector<float> rr((size_t)block);
    for (int i = 0; i < block; ++i) {
      int64_t n = (int64_t)b.bn * block + i;
      const float s = L.sw[(size_t)n];
      for (int j = 0; j < block; ++j) {
        int64_t k = (int64_t)b.bk * block + j;
        float wv = W[n * K + k];
        int q = quant1(wv, s);
        rr[(size_t)j] = (float)((double)wv - (double)s * (double)q);
      }
      const float sr = blockscale ? row_scale(rr.data(), block) : L.sr[(size_t)n];
      if (blockscale) b.srow[(size_t)i] = sr;
      for (int j = 0; j < block; ++j) b.q[(size_t)i * block + j] = (int8_t)quant1(rr[(size_t)j], sr);
    }
  });
  return finalize(L, out, (cudaStream_t)cuda_stream);
}
}  // namespace

extern "C" int mq_weights_export(const mq_weights* w, int8_t* qW, float* sW, int64_t* nnz, int32_t* blk_n,
                                 int32_t* blk_k, int8_t* qR, float* sR) {
  if (!w) return MQ_ERR_INVALID_ARG;
  const int64_t N = w->N, K = w->K, NT = N / BN;
  if (nnz) *nnz = w->nnz;
  if (sW && cudaMemcpy(sW, w->d_sw, (size_t)N * 4, cudaMemcpyDeviceToHost) != cudaSuccess) return MQ_ERR_CUDA;
  if (sR && cudaMemcpy(sR, w->d_sr, (size_t)N * 4, cudaMemcpyDeviceToHost) != cudaSuccess) return MQ_ERR_CUDA;
  if (qW) {
    std::vector<uint8_t> base((size_t)N * K / 2);
    if (cudaMemcpy(base.data(), w->d_base, base.size(), cudaMemcpyDeviceToHost) != cudaSuccess) return MQ_ERR_CUDA;
    parallel_for(N, [&](int64_t n) {
      for (int64_t k = 0; k < K; ++k) qW[n * K + k] = (int8_t)get_nibble(base[base_offset(n, k, K)], (int)(k & 1));
    });
  }
  if (blk_n || blk_k || qR) {
    std::vector<uint8_t> res((size_t)w->n_quarters * QUARTER_BYTES);
    std::vector<int32_t> cptr((size_t)NT + 1);
    std::vector<CellMeta> meta((size_t)w->n_cells);
    if (!res.empty() && cudaMemcpy(res.data(), w->d_res, res.size(), cudaMemcpyDeviceToHost) != cudaSuccess)
      return MQ_ERR_CUDA;
    if (cudaMemcpy(cptr.data(), w->d_cell_ptr, cptr.size() * 4, cudaMemcpyDeviceToHost) != cudaSuccess)
      return MQ_ERR_CUDA;
    if (!meta.empty() &&
        cudaMemcpy(meta.data(), w->d_cell_meta, meta.size() * sizeof(CellMeta), cudaMemcpyDeviceToHost) != cudaSuccess)
      return MQ_ERR_CUDA;
    struct Out {
      int32_t bn, bk;
      int64_t qidx[4];  // quarter index in res for each (h,r) part; block=64 uses [0]
    };
    std::vector<Out> outs;
    for (int64_t t = 0; t < NT; ++t)
      for (int32_t c = cptr[(size_t)t]; c < cptr[(size_t)t + 1]; ++c) {
        const int ks = meta[(size_t)c].kstep_mask & 0xFFFFFF, mask = (meta[(size_t)c].kstep_mask >> 24) & 0xF;
        int64_t qi = meta[(size_t)c].qoff;
        if (w->block == 128) {
          Out o{(int32_t)t, (int32_t)ks, {qi, qi + 1, qi + 2, qi + 3}};
          outs.push_back(o);
        } else {
          for (int q = 0; q < 4; ++q)
            if (mask & (1 << q)) {
              Out o{(int32_t)(2 * t + (q & 1)), (int32_t)(2 * ks + (q >> 1)), {qi, 0, 0, 0}};
              outs.push_back(o);
              ++qi;
            }
        }
      }
    std::sort(outs.begin(), outs.end(), [](const Out& a, const Out& b) { return a.bn != b.bn ? a.bn < b.bn : a.bk < b.bk; });
    if ((int64_t)outs.size() != w->nnz) return MQ_ERR_CUDA;
    const int bs = w->block;
    for (size_t e = 0; e < outs.size(); ++e) {
      if (blk_n) blk_n[e] = outs[e].bn;
      if (blk_k) blk_k[e] = outs[e].bk;
      if (!qR) continue;
      int8_t* dst = qR + e * (size_t)bs * bs;
      const int parts = bs == 128 ? 4 : 1;
      for (int p = 0; p < parts; ++p) {
        const int h = p >> 1, r = p & 1;
        const uint8_t* src = res.data() + (size_t)outs[e].qidx[p] * QUARTER_BYTES;
        for (int row = 0; row < 64; ++row)
          for (int c = 0; c < 64; ++c)
            dst[(size_t)(r * 64 + row) * bs + (size_t)(h * 64 + c)] = (int8_t)get_nibble(src[quarter_offset(row, c)], c & 1);
      }
    }
  }
  return MQ_OK;
}

extern "C" int mq_weights_is_blockscale(const mq_weights* w) { return w && w->blockscale ? 1 : 0; }

// the block-local residual scales of a blockscale layer, [nnz][block], blocks in mq_weights_export's order
extern "C" int mq_weights_export_blockscale(const mq_weights* w, float* sRb) {
  if (!w || !sRb) return MQ_ERR_INVALID_ARG;
  if (!w->blockscale) return MQ_ERR_INVALID_ARG;
  const int64_t NT = w->N / BN;
  std::vector<float> qs((size_t)w->n_quarters * 64);
  if (!qs.empty() && cudaMemcpy(qs.data(), w->d_qscale, qs.size() * 4, cudaMemcpyDeviceToHost) != cudaSuccess) return MQ_ERR_CUDA;
  struct Out {
    int32_t bn, bk;
    int64_t q_r0, q_r1;   // a quarter holding rows 0..63 / 64..127 of the block (block = 64: q_r0 only)
  };
  std::vector<Out> outs;
  for (int64_t t = 0; t < NT; ++t)
    for (int32_t c = w->h_cell_ptr[(size_t)t]; c < w->h_cell_ptr[(size_t)t + 1]; ++c) {
      const CellMeta& m = w->h_cell_meta[(size_t)c];
      const int ks = m.kstep_mask & 0xFFFFFF, mask = (m.kstep_mask >> 24) & 0xF;
      int64_t qi = m.qoff;
      if (w->block == 128) {
        outs.push_back(Out{(int32_t)t, (int32_t)ks, qi, qi + 1});   // quarters q = 2h + r in ascending q: (h0,r0), (h0,r1), ...
      } else {
        for (int q = 0; q < 4; ++q)
          if (mask & (1 << q)) {
            outs.push_back(Out{(int32_t)(2 * t + (q & 1)), (int32_t)(2 * ks + (q >> 1)), qi, 0});
            ++qi;
          }
      }
    }
  std::sort(outs.begin(), outs.end(), [](const Out& a, const Out& b) { return a.bn != b.bn ? a.bn < b.bn : a.bk < b.bk; });
  if ((int64_t)outs.size() != w->nnz) return MQ_ERR_CUDA;
  const int bs = w->block;
  for (size_t e = 0; e < outs.size(); ++e) {
    for (int row = 0; row < 64; ++row) sRb[e * (size_t)bs + (size_t)row] = qs[(size_t)outs[e].q_r0 * 64 + (size_t)row];
    if (bs == 128)
      for (int row = 0; row < 64; ++row) sRb[e * (size_t)bs + 64 + (size_t)row] = qs[(size_t)outs[e].q_r1 * 64 + (size_t)row];
  }
  return MQ_OK;
}

extern "C" int mq_weights_clone(const mq_weights* w, mq_weights** out, void* cuda_stream) {
  if (!w || !out) return MQ_ERR_INVALID_ARG;
  *out = nullptr;
  mq_weights* c = new (std::nothrow) mq_weights(*w);
  if (!c) return MQ_ERR_OOM;
  void* blob = nullptr;
  cudaError_t ce = cudaMalloc(&blob, w->dev_bytes);
  if (ce != cudaSuccess) {
    cudaGetLastError();
    delete c;
    return ce == cudaErrorMemoryAllocation ? MQ_ERR_OOM : MQ_ERR_CUDA;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (cudaMemcpyAsync(blob, w->dev_blob, w->dev_bytes, cudaMemcpyDeviceToDevice, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(blob);
    delete c;
    return MQ_ERR_CUDA;
  }
  const ptrdiff_t d = (uint8_t*)blob - (uint8_t*)w->dev_blob;
  c->dev_blob = blob;
  c->d_base = w->d_base + d;
  c->d_sw = (float*)((uint8_t*)w->d_sw + d);
  c->d_sr = (float*)((uint8_t*)w->d_sr + d);
  c->d_res = w->d_res + d;
  c->d_cell_ptr = (int32_t*)((uint8_t*)w->d_cell_ptr + d);
  c->d_cell_meta = (CellMeta*)((uint8_t*)w->d_cell_meta + d);
  c->d_unit_meta = (int32_t*)((uint8_t*)w->d_unit_meta + d);
  c->d_qscale = (float*)((uint8_t*)w->d_qscale + d);
  if (mq::build_weight_tmaps(c) != MQ_OK) {
    cudaFree(blob);
    delete c;
    return MQ_ERR_CUDA;
  }
  *out = c;
  return MQ_OK;
}

extern "C" int mq_weights_info(const mq_weights* w, int64_t* N, int64_t* K, int* block, int64_t* nnz,
                               size_t* device_bytes) {
  if (!w) return MQ_ERR_INVALID_ARG;
  if (N) *N = w->N;
  if (K) *K = w->K;
  if (block) *block = w->block;
  if (nnz) *nnz = w->nnz;
  if (device_bytes) *device_bytes = w->dev_bytes;
  return MQ_OK;
}

extern "C" void mq_weights_free(mq_weights* w) {
  if (!w) return;
  if (w->dev_blob) cudaFree(w->dev_blob);
  delete w;
}
