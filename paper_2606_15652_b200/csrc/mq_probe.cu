// mq_probe.cu -- measures what the tensor pipe itself can do: a pure tcgen05.mma kind::i8 issue loop (SURVEY 7.1
// step 0).  bench.py reports tensor-bound fractions against this number next to the 2 x bf16 proxy.
//
// Every CTA (one per SM) holds one A tile [128 rows][128 B] and one B tile [N rows][128 B] of int8 zeros in
// shared memory (K-major, SWIZZLE_128B), and one warp issues `iters` batches of 4 x (128 x N x 32) MMAs into a
// TMEM accumulator, committing to an mbarrier every batch group.  No loads, no epilogue: the time is the pipe's.
#include <cuda_runtime.h>

#include "mq_internal.h"
#include "mq_ptx.cuh"

namespace {

using namespace mq::ptx;

template <int N>
__global__ void __launch_bounds__(128, 1) probe_i8_kernel(int iters) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sb = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sA = sb, sB = sb + 128 * 128, sBar = sB + N * 128, sTm = sBar + 16;
  for (int i = threadIdx.x; i < (128 + N) * 128 / 16; i += blockDim.x)
    asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(sb + 16u * i), "r"(0) : "memory");
  const int warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) {
    mbar_init(sBar, 1);
    fence_mbar_init();
  }
  if (warp == 0) {
    tmem_alloc(sTm, 256);
    tmem_relinquish();
  }
  fence_proxy_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem) : "r"(sTm));
  if (warp == 1) {
    constexpr uint32_t IDESC = make_idesc_i8(128, N);
    const uint64_t da = make_desc_sw128(sA), db = make_desc_sw128(sB);
    uint32_t phase = 0;
    for (int it = 0; it < iters; ++it) {
      if (elect_one()) {
#pragma unroll
        for (int b = 0; b < 8; ++b)
#pragma unroll
          for (int k = 0; k < 4; ++k) mma_i8_ss(tmem, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), IDESC, 1u);
        tc_commit(sBar);
      }
      __syncwarp();
      mbar_wait(sBar, phase);
      phase ^= 1;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) {
    tc_fence_after();
    tmem_dealloc(tmem, 256);
  }
}

template <int N>
int run_probe(int iters, double* tops, cudaStream_t st) {
  const int smem = (128 + N) * 128 + 1024 + 64;
  if (cudaFuncSetAttribute(probe_i8_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return MQ_ERR_CUDA;
  const int sms = mq::sm_count();
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return MQ_ERR_CUDA;
  probe_i8_kernel<N><<<sms, 128, smem, st>>>(iters / 8 + 1);   // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0, st);
    probe_i8_kernel<N><<<sms, 128, smem, st>>>(iters);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) {
      cudaGetLastError();
      cudaEventDestroy(e0);
      cudaEventDestroy(e1);
      return MQ_ERR_CUDA;
    }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    best = ms < best ? ms : best;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  const double ops = 2.0 * 128.0 * N * 32.0 * 32.0 * (double)iters * (double)sms;   // 32 MMAs per iteration
  *tops = ops / ((double)best * 1e-3) / 1e12;
  return MQ_OK;
}

}  // namespace

// Dense INT8 tensor-pipe throughput of the current device in TOPS: tcgen05.mma.cta_group::1.kind::i8, 128 x n x 32 per
// instruction (n = 128 or 256), operands in shared memory, `iters` x 32 instructions per SM.  Host-synchronous.
extern "C" int mq_probe_int8_peak(int n, int iters, double* tops_out, void* cuda_stream) {
  if (!tops_out || iters <= 0 || (n != 128 && n != 256)) return MQ_ERR_INVALID_ARG;
  const int rc = mq::check_device();
  if (rc != MQ_OK) return rc;
  return n == 128 ? run_probe<128>(iters, tops_out, (cudaStream_t)cuda_stream) : run_probe<256>(iters, tops_out, (cudaStream_t)cuda_stream);
}
