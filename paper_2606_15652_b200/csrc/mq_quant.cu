// mq_quant.cu -- kernel (i): per-token int4 activation quantization (Eq.1; A1-A3, A5)
// plus the library's small runtime (status strings, options, device check).
//
// One CTA per token row.  The row (fp16/bf16) is read once with 128-bit loads and kept in
// registers (up to 32 elements per thread per pass -> K <= 8192 at 256 threads; longer rows
// re-read from L2), |max| is reduced with warp shuffles + one shared-memory step, then each
// thread divides, rounds half-to-even, clamps and packs 8 nibbles per 32-bit word.
// HBM-bound: 2 B read + 0.5 B written per element.
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <cstring>

#include "mq_internal.h"
#include "mq_ptx.cuh"

namespace mq {

Options& options() {
  static Options o;
  return o;
}
static int g_launches = 0;
void set_launch_count(int n) { g_launches = n; }
void add_launch_count(int n) { g_launches += n; }

static int g_dev_checked = -1;  // device ordinal for which the check passed
static int g_sms = 0;
int check_device() {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_UNSUPPORTED_DEVICE;
  }
  if (dev == g_dev_checked) return MQ_OK;
  int major = 0, minor = 0, sms = 0;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  if (major != 10 || minor != 0) return MQ_ERR_UNSUPPORTED_DEVICE;
  g_dev_checked = dev;
  g_sms = sms;
  return MQ_OK;
}
int sm_count() { return g_sms; }

}  // namespace mq

namespace {

constexpr int QT = 256;  // threads per row

template <bool BF16>
__device__ __forceinline__ void cvt8(const uint4& v, float* f) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (BF16) {
      f[2 * i] = __uint_as_float(w[i] << 16);
      f[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    } else {
      __half2 h = *reinterpret_cast<const __half2*>(&w[i]);
      float2 t = __half22float2(h);
      f[2 * i] = t.x;
      f[2 * i + 1] = t.y;
    }
  }
}

// 8-bit activations (W4A8): 8 elements -> 8 bytes, canonical order
__device__ __forceinline__ uint2 quant_bytes8(const float* f, float s, float inv_s) {
  uint32_t w[2] = {0, 0};
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int q = mq::ptx::quant1q<127>(f[i], s, inv_s);
    w[i >> 2] |= (uint32_t)(q & 0xFF) << (8 * (i & 3));
  }
  return make_uint2(w[0], w[1]);
}

__device__ __forceinline__ uint32_t quant_pack8(const float* f, float s, float inv_s) {
  uint32_t out = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int q = mq::ptx::quant1(f[i], s, inv_s);   // == clamp(rint(IEEE f / s)), see mq_ptx.cuh (A3)
    out |= (uint32_t)(q & 0xF) << (4 * i);
  }
  return out;
}

// CHUNKS = 16-byte chunks (8 elements) each thread keeps in registers per pass.
// QMAX = 7: packed int4 output (4 bytes per 8 elements); QMAX = 127: int8 output (8 bytes per 8 elements)
// QTT = threads per row: 256 for few rows (one row's latency chain is what counts), 128 for many rows (twice as many rows
// resident per SM: the kernel is bound by the load -> reduce -> store chain of a row, not by bandwidth, until enough
// rows are in flight)
template <bool BF16, int CHUNKS, int QMAX = 7, int QTT = QT>
__global__ void __launch_bounds__(QTT) mq_quantize_act_kernel(const uint16_t* __restrict__ A, int64_t lda, int K,
                                                             uint8_t* __restrict__ qA, float* __restrict__ sA) {
  // PDL: the next kernel (mq_gemm) may start its prologue and weight prefetch now; A may have been
  // written by the previous kernel, so wait for it before the first load.
  mq::ptx::griddep_launch();
  mq::ptx::griddep_wait();
  const int64_t m = blockIdx.x;
  const uint4* row = reinterpret_cast<const uint4*>(A + m * lda);
  uint32_t* qrow = reinterpret_cast<uint32_t*>(qA + m * (int64_t)(K / 2));
  uint2* qrow8 = reinterpret_cast<uint2*>(qA + m * (int64_t)K);
  const int nchunk = K / 8;
  __shared__ float red[QTT / 32];

  uint4 cache[CHUNKS];
  float amax = 0.f;
#pragma unroll
  for (int c = 0; c < CHUNKS; ++c) {
    int idx = threadIdx.x + c * QTT;
    if (idx < nchunk) {
      cache[c] = __ldg(row + idx);
      float f[8];
      cvt8<BF16>(cache[c], f);
#pragma unroll
      for (int i = 0; i < 8; ++i) amax = fmaxf(amax, fabsf(f[i]));
    }
  }
  for (int idx = threadIdx.x + CHUNKS * QTT; idx < nchunk; idx += QTT) {  // rows longer than the register cache
    uint4 v = __ldg(row + idx);
    float f[8];
    cvt8<BF16>(v, f);
#pragma unroll
    for (int i = 0; i < 8; ++i) amax = fmaxf(amax, fabsf(f[i]));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = amax;
  __syncthreads();
  amax = red[0];
#pragma unroll
  for (int i = 1; i < QTT / 32; ++i) amax = fmaxf(amax, red[i]);

  const float s = amax == 0.f ? 1.0f : __fdiv_rn(amax, (float)QMAX);  // A2 / Eq.1
  if (threadIdx.x == 0) sA[m] = s;
  const float inv_s = mq::ptx::quant_inv_scale(s);

#pragma unroll
  for (int c = 0; c < CHUNKS; ++c) {
    int idx = threadIdx.x + c * QTT;
    if (idx < nchunk) {
      float f[8];
      cvt8<BF16>(cache[c], f);
      if (QMAX == 7)
        qrow[idx] = quant_pack8(f, s, inv_s);
      else
        qrow8[idx] = quant_bytes8(f, s, inv_s);
    }
  }
  for (int idx = threadIdx.x + CHUNKS * QTT; idx < nchunk; idx += QTT) {
    uint4 v = __ldg(row + idx);
    float f[8];
    cvt8<BF16>(v, f);
    if (QMAX == 7)
      qrow[idx] = quant_pack8(f, s, inv_s);
    else
      qrow8[idx] = quant_bytes8(f, s, inv_s);
  }
}

__global__ void mq_unpack_act_kernel(const uint8_t* __restrict__ qA, int64_t total_bytes, int8_t* __restrict__ q) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= total_bytes) return;
  uint8_t b = qA[i];
  int lo = b & 0xF, hi = b >> 4;
  q[2 * i] = (int8_t)(lo >= 8 ? lo - 16 : lo);
  q[2 * i + 1] = (int8_t)(hi >= 8 ? hi - 16 : hi);
}

}  // namespace

extern "C" const char* mq_status_string(int status) {
  switch (status) {
    case MQ_OK: return "ok";
    case MQ_ERR_INVALID_ARG: return "invalid argument";
    case MQ_ERR_UNSUPPORTED_SHAPE: return "unsupported shape";
    case MQ_ERR_UNSUPPORTED_DEVICE: return "unsupported device (needs compute capability 10.0, sm_100a)";
    case MQ_ERR_CUDA: return "CUDA error";
    case MQ_ERR_OOM: return "out of memory";
    case MQ_ERR_ACC_OVERFLOW: return "K too large for the int32 accumulator";
    case MQ_ERR_WORKSPACE: return "workspace too small";
    case MQ_ERR_STATIC_SCRATCH: return "mq_linear_static: the call needs more scratch than the built-in 16 MiB array (use mq_linear with a workspace)";
    default: return "unknown status";
  }
}

extern "C" int mq_set_option(const char* name, int64_t value) {
  if (!name || value < 0) return MQ_ERR_INVALID_ARG;
  mq::Options& o = mq::options();
  if (!strcmp(name, "split_k")) {
    o.split_k = value;
  } else if (!strcmp(name, "token_tile")) {
    if (value != 0 && value != 16 && value != 32 && value != 64 && value != 128)
      return MQ_ERR_INVALID_ARG;
    o.token_tile = value;
  } else if (!strcmp(name, "max_ctas")) {
    o.max_ctas = value;
  } else if (!strcmp(name, "pdl")) {
    if (value > 1) return MQ_ERR_INVALID_ARG;
    o.pdl = value;
  } else if (!strcmp(name, "fused_quant")) {
    if (value > 1) return MQ_ERR_INVALID_ARG;
    o.fused_quant = value;
  } else if (!strcmp(name, "decode_path")) {
    if (value > 1) return MQ_ERR_INVALID_ARG;
    o.decode_path = value;
  } else if (!strcmp(name, "decode_big")) {
    if (value > 2) return MQ_ERR_INVALID_ARG;
    o.decode_big = value;
  } else if (!strcmp(name, "decode_rows")) {
    if (value != 0 && value != 16 && value != 32 && value != 64 && value != 128) return MQ_ERR_INVALID_ARG;
    o.decode_rows = value;
  } else if (!strcmp(name, "prefill_path")) {
    if (value > 3) return MQ_ERR_INVALID_ARG;
    o.prefill_path = value;
  } else if (!strcmp(name, "group_tc")) {
    if (value > 1) return MQ_ERR_INVALID_ARG;
    o.group_tc = value;
  } else if (!strcmp(name, "group_simt")) {
    if (value > 1) return MQ_ERR_INVALID_ARG;
    o.group_simt = value;
  } else {
    return MQ_ERR_INVALID_ARG;
  }
  return MQ_OK;
}

extern "C" int mq_last_launch_count(void) { return mq::g_launches; }

extern "C" size_t mq_qact_bytes(int64_t M, int64_t K) {
  if (M < 0 || K < 0) return 0;
  return (size_t)M * (size_t)K / 2;
}

namespace {

template <int QMAX>
int quantize_act_impl(const void* A, mq_dtype a_dtype, int64_t M, int64_t K, int64_t lda, void* qA, float* sA,
                      void* cuda_stream) {
  if (M < 0 || K <= 0 || K % mq::BK != 0 || K > (int64_t)1 << 30) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (a_dtype != MQ_F16 && a_dtype != MQ_BF16) return MQ_ERR_INVALID_ARG;
  mq::set_launch_count(0);
  if (M == 0) return MQ_OK;
  if (!A || !qA || !sA || lda < K) return MQ_ERR_INVALID_ARG;
  if (((uintptr_t)A & 15) || ((uintptr_t)qA & 15) || (lda % 8) != 0 || ((uintptr_t)sA & 3)) return MQ_ERR_INVALID_ARG;
  if (M > 2147483647LL) return MQ_ERR_UNSUPPORTED_SHAPE;
  int rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const uint16_t* a = (const uint16_t*)A;
  dim3 grid((unsigned)M), blk(QT);
  const int nchunk_per_thread = (int)((K / 8 + QT - 1) / QT);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = blk;
  cfg.dynamicSmemBytes = 0;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = mq::options().pdl ? 1 : 0;
  const int Ki = (int)K;
  uint8_t* q8 = (uint8_t*)qA;
  cudaError_t le;
  // the whole row stays in registers for K <= 16384 (one pass over global memory, all loads in flight)
  const bool bf = a_dtype == MQ_BF16;
  if (M >= 2048 && K / 8 <= 4 * 128) {   // many short rows: 128 threads per row (measured: +12 % at M = 8192, K = 4096;
                                          // longer rows lose occupancy to the register cache, fewer rows gain nothing)
    cfg.blockDim = dim3(128);
    const int cpt = (int)((K / 8 + 127) / 128);
#define MQ_Q128(CH)                                                                                                    \
  (bf ? cudaLaunchKernelEx(&cfg, mq_quantize_act_kernel<true, CH, QMAX, 128>, a, lda, Ki, q8, sA)                       \
      : cudaLaunchKernelEx(&cfg, mq_quantize_act_kernel<false, CH, QMAX, 128>, a, lda, Ki, q8, sA))
    le = cpt <= 4 ? MQ_Q128(4) : (cpt <= 8 ? MQ_Q128(8) : MQ_Q128(16));
#undef MQ_Q128
  } else if (bf) {
    if (nchunk_per_thread <= 2)
      le = cudaLaunchKernelEx(&cfg, mq_quantize_act_kernel<true, 2, QMAX>, a, lda, Ki, q8, sA);
    else if (nchunk_per_thread <= 4)
      le = cudaLaunchKernelEx(&cfg, mq_quantize_act_kernel<true, 4, QMAX>, a, lda, Ki, q8, sA);
    else
      le = cudaLaunchKernelEx(&cfg, mq_quantize_act_kernel<true, 8, QMAX>, a, lda, Ki, q8, sA);
  } else {
    if (nchunk_per_thread <= 2)
      le = cudaLaunchKernelEx(&cfg, mq_quantize_act_kernel<false, 2, QMAX>, a, lda, Ki, q8, sA);
    else if (nchunk_per_thread <= 4)
      le = cudaLaunchKernelEx(&cfg, mq_quantize_act_kernel<false, 4, QMAX>, a, lda, Ki, q8, sA);
    else
      le = cudaLaunchKernelEx(&cfg, mq_quantize_act_kernel<false, 8, QMAX>, a, lda, Ki, q8, sA);
  }
  if (le != cudaSuccess) {
    cudaGetLastError();
    return MQ_ERR_CUDA;
  }
  mq::set_launch_count(1);
  if (cudaGetLastError() != cudaSuccess) return MQ_ERR_CUDA;
  return MQ_OK;
}

}  // namespace

extern "C" int mq_quantize_act(const void* A, mq_dtype a_dtype, int64_t M, int64_t K, int64_t lda, void* qA, float* sA,
                               void* cuda_stream) {
  return quantize_act_impl<7>(A, a_dtype, M, K, lda, qA, sA, cuda_stream);
}

extern "C" int mq_quantize_act8(const void* A, mq_dtype a_dtype, int64_t M, int64_t K, int64_t lda, int8_t* qA8, float* sA,
                                void* cuda_stream) {
  return quantize_act_impl<127>(A, a_dtype, M, K, lda, qA8, sA, cuda_stream);
}

extern "C" int mq_unpack_act(const void* qA, int64_t M, int64_t K, int8_t* q, void* cuda_stream) {
  if (M < 0 || K <= 0 || K % 2 != 0) return MQ_ERR_UNSUPPORTED_SHAPE;
  if (M == 0) return MQ_OK;
  if (!qA || !q) return MQ_ERR_INVALID_ARG;
  int rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  int64_t total = M * K / 2;
  int64_t blocks = (total + 255) / 256;
  if (blocks > 2147483647LL) return MQ_ERR_UNSUPPORTED_SHAPE;
  mq_unpack_act_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>((const uint8_t*)qA, total, q);
  if (cudaGetLastError() != cudaSuccess) return MQ_ERR_CUDA;
  return MQ_OK;
}
