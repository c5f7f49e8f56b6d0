// mq_oracle.cpp -- CPU ORACLE for the MosaicQuant / ZipperEngine hot path.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
// shares no code with paper_2606_15652_b200/ (no headers, helpers, tables or
// constants), and nothing under paper_2606_15652_b200/ may include or link it.
//
// It is a plain, slow, step-by-step transcription of what the path computes, in the
// paper's order and notation.  Citations are PAPER.md lines ("P:<line>") of
// /root/reference/PAPER.md; "A<n>" are the readings listed in DESIGN.md section 3.
//
//   O1 quantize_row      Eq.1  P:75-80   uniform symmetric quantizer, q_max = 7 (A1-A3); q_max = 127 for the
//                                        8-bit activations of the W4A8 variant (Table 1 W4A8 rows)
//   O2 activation        P:439-441       per-token dynamic quantization (A5), 4-bit or 8-bit
//   O3 base weight + R   Alg.1 line 1    P:124, per output channel (A9)
//   O4 residual Q(R)     Alg.1 / Eq.4    P:106,124, per output channel over all K (A4)
//   O4b (oracle/__init__.py) the same operator per (output channel, k-block) run: block-local scales (A4b)
//   O5 h_j               Alg.1 line 2
//   O6 Delta-score S_B
//   O7 TopK              P:124,160,378   (A6, A7)
//   O8 integer GEMM      Eq.2, Eq.4 P:106   exact, int64 accumulation
//   O9 output            Eq.2, Eq.4      binary64
//
// Pins: every function here is pinned by tests/test_oracle_pins.py against closed
// forms, brute force and invariants (none of which call back into this file's
// formulas); the only unpinned item is the whole path against values printed by the
// paper ("parity unpinned": the paper prints no worked numeric example).
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
// -ffp-contract=off: no FMA contraction, so fp32 divisions and roundings are the
// literal IEEE operations written below.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <algorithm>
#include <vector>

#if defined(_OPENMP)
#include <omp.h>
#endif

namespace {

// exact fp16 (IEEE binary16) -> fp32
float half_bits_to_float(uint16_t h) {
  uint32_t sign = (uint32_t)(h >> 15) << 31;
  uint32_t exp = (h >> 10) & 0x1F;
  uint32_t man = h & 0x3FF;
  uint32_t out;
  if (exp == 0) {
    if (man == 0) {
      out = sign;
    } else {  // subnormal: value = man * 2^-24
      float v = std::ldexp((float)man, -24);
      std::memcpy(&out, &v, 4);
      out |= sign;
    }
  } else if (exp == 31) {
    out = sign | 0x7F800000u | (man << 13);
  } else {
    out = sign | ((exp + 112) << 23) | (man << 13);
  }
  float f;
  std::memcpy(&f, &out, 4);
  return f;
}

// exact bf16 -> fp32
float bf16_bits_to_float(uint16_t b) {
  uint32_t out = (uint32_t)b << 16;
  float f;
  std::memcpy(&f, &out, 4);
  return f;
}

// O1 -- Eq.1: Q_X = round(X / s_X), s_X = max|X| / q_max; q_max = 2^(b-1) - 1: 7 for the 4-bit
// operands (A1), 127 for the 8-bit activations of W4A8.  One binary32 division for s, one
// binary32 division per element, round half to even (A3).  All-zero row: s = 1, q = 0 (A2).
void quantize_row(const float* x, int64_t L, int8_t* q, float* s_out, int qmax = 7) {
  float amax = 0.0f;
  for (int64_t i = 0; i < L; ++i) {
    float a = std::fabs(x[i]);
    if (a > amax) amax = a;
  }
  if (amax == 0.0f) {
    *s_out = 1.0f;
    for (int64_t i = 0; i < L; ++i) q[i] = 0;
    return;
  }
  volatile float s = amax / (float)qmax;
  for (int64_t i = 0; i < L; ++i) {
    volatile float t = x[i] / s;
    float r = std::nearbyintf(t);  // default rounding mode: round half to even
    int v = (int)r;
    if (v > qmax) v = qmax;
    if (v < -qmax) v = -qmax;
    q[i] = (int8_t)v;
  }
  *s_out = s;
}

}  // namespace

extern "C" {

int orc_num_threads() {
#if defined(_OPENMP)
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// O1 exposed for pins.
void orc_quantize_row(const float* x, int64_t L, int8_t* q, float* s) { quantize_row(x, L, q, s); }
void orc_quantize_row_bits(const float* x, int64_t L, int bits, int8_t* q, float* s) {
  quantize_row(x, L, q, s, bits == 8 ? 127 : 7);
}

// O1 on every row of a dense fp32 matrix [rows, L] (used for the block-local residual scales, O4b: the rows are
// the (channel, k-block) runs of R).
void orc_quantize_rows(const float* X, int64_t rows, int64_t L, int8_t* q /*[rows,L]*/, float* s /*[rows]*/) {
#pragma omp parallel for schedule(static)
  for (int64_t r = 0; r < rows; ++r) quantize_row(X + r * L, L, q + r * L, s + r);
}

// O2 -- per-token activation quantization ("per-token dynamic activation
// quantization"; A5).  A is fp16 (dtype 0) or bf16 (dtype 1) bits, row stride lda
// elements; each row is converted exactly to fp32 and quantized by O1 over all K.
void orc_quantize_act_bits(const uint16_t* A_bits, int dtype, int64_t M, int64_t K, int64_t lda, int bits,
                           int8_t* qa /*[M,K]*/, float* sa /*[M]*/);
void orc_quantize_act(const uint16_t* A_bits, int dtype, int64_t M, int64_t K, int64_t lda,
                      int8_t* qa /*[M,K]*/, float* sa /*[M]*/) {
  orc_quantize_act_bits(A_bits, dtype, M, K, lda, 4, qa, sa);
}
// O2 with the activation width as a parameter: 4 bits (W4A4) or 8 bits (W4A8)
void orc_quantize_act_bits(const uint16_t* A_bits, int dtype, int64_t M, int64_t K, int64_t lda, int bits,
                           int8_t* qa /*[M,K]*/, float* sa /*[M]*/) {
  const int qmax = bits == 8 ? 127 : 7;
#pragma omp parallel
  {
    std::vector<float> row((size_t)K);
#pragma omp for schedule(static)
    for (int64_t m = 0; m < M; ++m) {
      const uint16_t* src = A_bits + m * lda;
      for (int64_t k = 0; k < K; ++k)
        row[(size_t)k] = dtype == 0 ? half_bits_to_float(src[k]) : bf16_bits_to_float(src[k]);
      quantize_row(row.data(), K, qa + m * K, sa + m, qmax);
    }
  }
}

// O3 + O4 -- Alg.1 line 1: R = W - Q(W) with Q per output channel (A9),
// then Q(R) per output channel over all K, for the whole matrix, before any
// selection (A4).  The product s_w*q_w is exact in binary64 (24-bit x 4-bit).
void orc_decompose(const float* W /*[N,K]*/, int64_t N, int64_t K, int8_t* qw /*[N,K]*/, float* sw /*[N]*/,
                   float* R /*[N,K]*/, int8_t* qr /*[N,K]*/, float* sr /*[N]*/) {
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < N; ++n) {
    quantize_row(W + n * K, K, qw + n * K, sw + n);
    for (int64_t k = 0; k < K; ++k) {
      double d = (double)W[n * K + k] - (double)sw[n] * (double)qw[n * K + k];
      R[n * K + k] = (float)d;
    }
    quantize_row(R + n * K, K, qr + n * K, sr + n);
  }
}

// O5 -- h_j = (2/N) sum_n X[n,j]^2 (Alg.1 line 2 P:124), binary64, n ascending.
void orc_hessian_diag(const float* X /*[Ncal,K]*/, int64_t Ncal, int64_t K, double* h /*[K]*/) {
  for (int64_t k = 0; k < K; ++k) {
    double acc = 0.0;
    for (int64_t n = 0; n < Ncal; ++n) {
      double x = (double)X[n * K + k];
      acc += x * x;
    }
    h[k] = (2.0 / (double)Ncal) * acc;
  }
}

// O6 -- Delta-Hessian score:
//   A_B = sum_{(i,j) in B} h_j R_ij^2 ;  B_B = sum h_j (R_ij - Q(R)_ij)^2 ;
//   delta_B = A_B - B_B ;  S_B = [delta_B]_+ .
// Blocks are bs x bs, aligned (A8); block (bn,bk) has linear index bn*(K/bs)+bk.
// binary64, rows ascending then columns ascending.
void orc_scores(const float* R, const int8_t* qr, const float* sr, const float* h /*[K] fp32*/, int64_t N,
                int64_t K, int64_t bs, double* A_B, double* B_B, double* delta, double* S) {
  const int64_t nbn = N / bs, nbk = K / bs;
#pragma omp parallel for schedule(static)
  for (int64_t b = 0; b < nbn * nbk; ++b) {
    const int64_t bn = b / nbk, bk = b % nbk;
    double a = 0.0, bb = 0.0;
    for (int64_t i = bn * bs; i < (bn + 1) * bs; ++i) {
      for (int64_t j = bk * bs; j < (bk + 1) * bs; ++j) {
        double r = (double)R[i * K + j];
        double e = r - (double)sr[i] * (double)qr[i * K + j];
        double hj = (double)h[j];
        a += hj * (r * r);
        bb += hj * (e * e);
      }
    }
    A_B[b] = a;
    B_B[b] = bb;
    delta[b] = a - bb;
    S[b] = (a - bb) > 0.0 ? (a - bb) : 0.0;
  }
}

// O7 -- S = TopK({S_B}, K) (Alg.1), global over the layer (A6); blocks with
// S_B = 0 are omitted; ties -> lower linear block index first (A7).
// Returns nnz; sel[] holds the selected linear indices in selection order
// (score descending).
int64_t orc_select(const double* S, int64_t n_blocks, int64_t budget, int64_t* sel /*[min(budget,n_blocks)]*/) {
  std::vector<int64_t> cand;
  for (int64_t b = 0; b < n_blocks; ++b)
    if (S[b] > 0.0) cand.push_back(b);
  std::stable_sort(cand.begin(), cand.end(), [&](int64_t x, int64_t y) {
    if (S[x] != S[y]) return S[x] > S[y];
    return x < y;
  });
  int64_t nnz = std::min<int64_t>(budget, (int64_t)cand.size());
  if (nnz < 0) nnz = 0;
  for (int64_t i = 0; i < nnz; ++i) sel[i] = cand[(size_t)i];
  return nnz;
}

// O8 -- exact integer GEMM (Eq.2; Eq.4):
//   acc0[m,n] = sum_k q_a[m,k] q_w[n,k]
//   acc1[m,n] = sum_{(bn,bk) in S, n in bn} sum_{k in bk} q_a[m,k] q_r[n,k]
// int64 accumulation.  qr is the full-matrix Q(R) of O4; the block list is the mask M_S.
// Returns 0, or -1 if some |acc| >= 2^31.
int orc_gemm(const int8_t* qa /*[M,K]*/, int64_t M, int64_t K, const int8_t* qw /*[N,K]*/, int64_t N,
             const int8_t* qr /*[N,K]*/, int64_t bs, int64_t nnz, const int32_t* blk_n, const int32_t* blk_k,
             int64_t* acc0 /*[M,N]*/, int64_t* acc1 /*[M,N]*/) {
  int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
  for (int64_t m = 0; m < M; ++m) {
    for (int64_t n = 0; n < N; ++n) {
      int64_t a = 0;
      for (int64_t k = 0; k < K; ++k) a += (int64_t)qa[m * K + k] * (int64_t)qw[n * K + k];
      acc0[m * N + n] = a;
      acc1[m * N + n] = 0;
      if (a >= (1LL << 31) || a <= -(1LL << 31)) bad |= 1;
    }
    for (int64_t e = 0; e < nnz; ++e) {
      const int64_t n0 = (int64_t)blk_n[e] * bs, k0 = (int64_t)blk_k[e] * bs;
      for (int64_t n = n0; n < n0 + bs; ++n) {
        int64_t a = 0;
        for (int64_t k = k0; k < k0 + bs; ++k) a += (int64_t)qa[m * K + k] * (int64_t)qr[n * K + k];
        acc1[m * N + n] += a;
      }
    }
    for (int64_t n = 0; n < N; ++n) {
      int64_t a = acc1[m * N + n];
      if (a >= (1LL << 31) || a <= -(1LL << 31)) bad |= 1;
    }
  }
  return bad ? -1 : 0;
}

// O9 -- Y_exact[m,n] = s_a[m] * ( s_w[n]*acc0 + s_r[n]*acc1 ) in binary64 (Eq.2, Eq.4).
// Also returns the tolerance scale |s_a| * (|s_w acc0| + |s_r acc1|) used by the parity rule.
void orc_output(const int64_t* acc0, const int64_t* acc1, const float* sa, const float* sw, const float* sr,
                int64_t M, int64_t N, double* Y /*[M,N]*/, double* mag /*[M,N] or NULL*/) {
#pragma omp parallel for schedule(static)
  for (int64_t m = 0; m < M; ++m) {
    for (int64_t n = 0; n < N; ++n) {
      double t0 = (double)sw[n] * (double)acc0[m * N + n];
      double t1 = (double)sr[n] * (double)acc1[m * N + n];
      Y[m * N + n] = (double)sa[m] * (t0 + t1);
      if (mag) mag[m * N + n] = std::fabs((double)sa[m]) * (std::fabs(t0) + std::fabs(t1));
    }
  }
}

// Convenience for timing (bench.py cpu_baseline): the online part O2 + O8 + O9 in one call,
// exactly the three functions above in sequence.
int orc_forward(const uint16_t* A_bits, int dtype, int64_t M, int64_t K, const int8_t* qw, const float* sw,
                int64_t N, const int8_t* qr, const float* sr, int64_t bs, int64_t nnz, const int32_t* blk_n,
                const int32_t* blk_k, double* Y) {
  std::vector<int8_t> qa((size_t)(M * K));
  std::vector<float> sa((size_t)M);
  std::vector<int64_t> a0((size_t)(M * N)), a1((size_t)(M * N));
  orc_quantize_act(A_bits, dtype, M, K, K, qa.data(), sa.data());
  int rc = orc_gemm(qa.data(), M, K, qw, N, qr, bs, nnz, blk_n, blk_k, a0.data(), a1.data());
  orc_output(a0.data(), a1.data(), sa.data(), sw, sr, M, N, Y, nullptr);
  return rc;
}

}  // extern "C"
