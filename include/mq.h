/* mq.h -- C ABI of libmq.so: the B200 (sm_100a) hot path of MosaicQuant / ZipperEngine.
 *
 * What the library computes (citations are lines of the paper text, "P:<line>" =
 * /root/reference/PAPER.md, and readings "A<n>" of DESIGN.md section 3):
 *
 *   Y = A * W^T for one bias-free linear layer, with
 *     A  [M,K]  activations, quantized per token to int4      (Eq.1; A5)
 *     W  [N,K]  weights = dense int4 base  Q(W)  per output channel (A9)
 *               + sparse int4 residual Q(R), R = W - Q(W), kept only on the top-K
 *                 blocks of the Delta-Hessian score          (Eq.4; Alg.1)
 *     Y[m,n] = s_a[m] * ( s_w[n] * acc0[m,n] + s_r[n] * acc1[m,n] )      (Eq.2; Eq.4)
 *     acc0 = sum_k q_a[m,k] q_w[n,k]                (dense 4-bit component)
 *     acc1 = sum over selected blocks containing n of sum_{k in block} q_a[m,k] q_r[n,k]
 *   with the residual blocks' MMAs issued inside the dense K-loop of ONE kernel
 *   (ZipperEngine, section 4.2, Fig.3).
 *
 * Conventions: every function returns an mq_status (0 = MQ_OK, negative = error);
 * nothing throws, aborts or prints.  "_dev" pointers are CUDA device pointers, "_host"
 * pointers are host pointers.  All device work is enqueued on `cuda_stream` (a
 * cudaStream_t passed as void*; NULL = the legacy default stream) and the online calls
 * (mq_quantize_act, mq_gemm, mq_linear) neither allocate nor synchronise with the host.
 * The caller owns every buffer it passes in; the library owns only what an
 * mq_weights* refers to.  There is no CPU fallback: on a machine without a
 * compute-capability-10.0 device the compute calls return MQ_ERR_UNSUPPORTED_DEVICE.
 */
#ifndef MQ_H_
#define MQ_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  MQ_OK = 0,
  MQ_ERR_INVALID_ARG = -1,        /* NULL pointer, bad enum, misaligned pointer, bad block list */
  MQ_ERR_UNSUPPORTED_SHAPE = -2,  /* N % 128, K % 128, block not in {64,128}, M < 0 ...        */
  MQ_ERR_UNSUPPORTED_DEVICE = -3, /* current device is not compute capability 10.0             */
  MQ_ERR_CUDA = -4,               /* a CUDA runtime / driver call failed                       */
  MQ_ERR_OOM = -5,                /* host or device allocation failed                          */
  MQ_ERR_ACC_OVERFLOW = -6,       /* K so large that the int32 accumulator could overflow      */
  MQ_ERR_WORKSPACE = -7,          /* workspace smaller than mq_gemm_workspace_bytes()          */
  MQ_ERR_STATIC_SCRATCH = -8      /* mq_linear_static: the call needs more than mq_linear_static_max_bytes() */
} mq_status;

typedef enum { MQ_F16 = 0, MQ_BF16 = 1 } mq_dtype;

/* Opaque packed layer: immutable after packing, safe to share between streams. */
typedef struct mq_weights mq_weights;

/* Static string for a status code; never NULL, never freed. */
const char* mq_status_string(int status);

/* ------------------------------------------------------------------------------------
 * (1) Activation quantization -- Eq.1, per token (A5), q_max = 7 (A1).
 *
 * Row m of A (fp16 or bf16, `lda_elems` elements between rows, 16-byte aligned rows) is
 * converted exactly to fp32; amax = max|a|; s = amax / 7 (one IEEE binary32 division);
 * q_k = clamp(rint(a_k / s), -7, 7) with an IEEE binary32 division and round-half-even
 * (A3); an all-zero row gives s = 1, q = 0 (A2).
 *
 * Output layout (canonical, part of the ABI):
 *   qA_dev : uint8 [M, K/2] row-major, row stride K/2 bytes; byte i of row m holds
 *            element 2i in bits 0-3 and element 2i+1 in bits 4-7, two's-complement
 *            nibbles.  mq_qact_bytes(M,K) = M*K/2.  Must be 16-byte aligned.
 *   sA_dev : float [M].
 * Requires K % 128 == 0, M >= 0 (M == 0 is a no-op).
 */
size_t mq_qact_bytes(int64_t M, int64_t K);
int mq_quantize_act(const void* A_dev, mq_dtype a_dtype, int64_t M, int64_t K, int64_t lda_elems,
                    void* qA_dev, float* sA_dev, void* cuda_stream);
/* Test aid: expands qA to one int8 per element, q_dev [M,K] row-major. */
int mq_unpack_act(const void* qA_dev, int64_t M, int64_t K, int8_t* q_dev, void* cuda_stream);

/* ------------------------------------------------------------------------------------
 * (2) Weight packing -- Algorithm 1 on the host, then the device layout.
 *
 * mq_pack_weights: W_host [N,K] fp32 row-major ([out,in], A9).  Steps, in the paper's
 * order: base quantize per output channel (Eq.1); R = W - s_w q_w (Alg.1 line 1);
 * Q(R) per output channel over all K, before selection (A4); Delta-Hessian score
 * S_B = [sum_B h_k R^2 - sum_B h_k (R - Q(R))^2]_+  over aligned block x block
 * blocks (A8), h_host [K] fp32 or NULL = all ones; global top-`budget_blocks` by score,
 * ties to the lower linear block index bn*(K/block)+bk, zero-score blocks never selected
 * (A6, A7).  The result is uploaded in the kernel's tiled layout (DESIGN.md
 * section 5).  Host inputs are copied; they may be freed on return.  The call
 * synchronises `cuda_stream` before returning.
 *
 * mq_pack_prequantized: layout only; the caller supplies the decomposition.
 *   qW [N,K] int8 in [-7,7]; sW [N]; nnz selected blocks with coordinates
 *   (blk_n[e], blk_k[e]) in units of `block`, no duplicates; qR [nnz][block][block]
 *   int8 in [-7,7] (row = n, col = k); sR [N] (A4: per output channel).
 *
 * Requires N % 128 == 0, K % 128 == 0, block in {64,128}, 49*256*K < 2^31.
 */
int mq_pack_weights(const float* W_host, int64_t N, int64_t K, const float* h_host, int block,
                    int64_t budget_blocks, mq_weights** out, void* cuda_stream);

/* Algorithm 1 with DEVICE inputs: W_dev [N,K] fp32 row-major and h_dev [K] (or NULL) are device
 * pointers (rows 8-byte aligned).  Base quantization, residual, Q(R) and the Delta-Hessian block scores (P:119-125,
 * P:156) run on the GPU, one CTA per block-row, with mq_pack_weights' arithmetic operation for operation (binary32
 * division + round-half-even for Eq.1; the score sums in fp64, uncontracted, rows then k ascending), so the selected
 * set, the integers and the scales are bit-identical to mq_pack_weights'.  The top-K over the N*K/block^2 scores and
 * the layout run on the host.  Same requirements and errors as mq_pack_weights, plus K <= 51200 (one residual row in
 * shared memory).  Synchronises `cuda_stream`. */
int mq_pack_weights_device(const float* W_dev, int64_t N, int64_t K, const float* h_dev, int block,
                           int64_t budget_blocks, mq_weights** out, void* cuda_stream);
int mq_pack_prequantized(const int8_t* qW_host, const float* sW_host, int64_t N, int64_t K, int block,
                         int64_t nnz, const int32_t* blk_n_host, const int32_t* blk_k_host,
                         const int8_t* qR_host, const float* sR_host, mq_weights** out,
                         void* cuda_stream);
/* Block-local residual scales (second half; north_star "residual block list with block coordinates and
 * per-block scales"; reading A4b).  Eq.1 is applied to R = W - Q(W) inside every block separately: for
 * block (bn, bk) and output channel n of bn, s_rb[n, bk] = max_{k in bk} |R[n, k]| / 7, q_rb = round(R / s_rb), computed
 * for EVERY block before selection (so that a block's gain does not depend on the selected set: Theorem 4.1, P:352,
 * P:368); scores, top-K and tie rule as mq_pack_weights.  The layer computes
 *     Y[m,n] = s_a[m] * ( s_w[n] * acc0[m,n] + sum_{selected blocks B containing n} s_rb[n, B] * acc1_B[m,n] )    (Eq.4)
 * with acc1_B the exact integer dot product over the block's 64 / 128 input channels; the block terms are added in
 * fp32 in ascending K.  mq_pack_prequantized_blockscale takes sRb_host [nnz][block] (scale of every row of every
 * selected block) instead of sR.  Handles made by these two calls are served by mq_gemm / mq_linear only (any M; the
 * decode kernel runs them, 32 tokens per pass beyond M = 32; parity hook dbg_acc_res = the integer sum of the block
 * accumulators); mq_gemm_a8 / mq_gemm_group / mq_gemm_naive return MQ_ERR_UNSUPPORTED_SHAPE for them, and K <= 65536.
 * mq_weights_export returns sR = all ones for them; mq_weights_export_blockscale returns sRb [nnz][block] in the same
 * block order; mq_weights_is_blockscale tells the two kinds of handle apart. */
int mq_pack_weights_blockscale(const float* W_host, int64_t N, int64_t K, const float* h_host, int block,
                               int64_t budget_blocks, mq_weights** out, void* cuda_stream);
int mq_pack_prequantized_blockscale(const int8_t* qW_host, const float* sW_host, int64_t N, int64_t K, int block,
                                    int64_t nnz, const int32_t* blk_n_host, const int32_t* blk_k_host,
                                    const int8_t* qR_host, const float* sRb_host, mq_weights** out, void* cuda_stream);
int mq_weights_export_blockscale(const mq_weights* w, float* sRb_host);
int mq_weights_is_blockscale(const mq_weights* w);
/* Reads the device layout back and returns the canonical arrays (any pointer may be
 * NULL = skipped).  Blocks are returned sorted by (blk_n, blk_k).  Host call; syncs. */
int mq_weights_export(const mq_weights* w, int8_t* qW_host, float* sW_host, int64_t* nnz,
                      int32_t* blk_n_host, int32_t* blk_k_host, int8_t* qR_host, float* sR_host);
/* Device-to-device copy of a packed layer into a fresh allocation (benchmarks rotate several
 * copies so that every timed call reads its weights from HBM, not from L2).  Syncs the stream. */
int mq_weights_clone(const mq_weights* w, mq_weights** out, void* cuda_stream);
int mq_weights_info(const mq_weights* w, int64_t* N, int64_t* K, int* block, int64_t* nnz,
                    size_t* device_bytes);
void mq_weights_free(mq_weights* w);

/* ------------------------------------------------------------------------------------
 * (3) Fused base + residual GEMM -- ZipperEngine (Eq.4).
 *
 *   qA_dev, sA_dev : output of mq_quantize_act for the same M and this layer's K
 *                    (row stride K/2 bytes).
 *   Y_dev          : [M,N] fp16/bf16 row-major, `ldy_elems` elements between rows.
 *   dbg_acc_base_dev / dbg_acc_res_dev : optional int32 [M,N] row-major (stride N), 16-byte
 *                    aligned; when non-NULL they receive acc0 / acc1 exactly (parity hooks).
 *   workspace_dev  : at least mq_gemm_workspace_bytes(w, M) bytes, 16-byte aligned.  Contract: its first
 *                    16384 bytes must be ZERO before the first call that uses it (cudaMemset once); they
 *                    hold the per-tile arrival counters of the split-K fix-up at positions that do not
 *                    depend on the layer shape, M or the options, and every call returns them to zero.
 *                    Everything behind those 16 KB (int32 partial tiles, flags) is written before it is
 *                    read and needs no initial content.  One workspace of the largest size may therefore
 *                    be shared by calls of different layers, M and options, as long as those calls do not
 *                    run concurrently (same stream, or otherwise ordered); concurrent calls need distinct
 *                    workspaces.  An asynchronous fault inside a call leaves the counters undefined:
 *                    zero the prefix again before re-use.
 * M == 0 is a no-op.
 */
size_t mq_gemm_workspace_bytes(const mq_weights* w, int64_t M);
int mq_gemm(const mq_weights* w, const void* qA_dev, const float* sA_dev, int64_t M, void* Y_dev,
            mq_dtype y_dtype, int64_t ldy_elems, int32_t* dbg_acc_base_dev, int32_t* dbg_acc_res_dev,
            void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* ------------------------------------------------------------------------------------
 * (3b) W4A8 variant -- the paper's other reported precision ("per-token ... activation quantization",
 * Table 1 W4A8 rows): per-token int8 activations (Eq.1 with q_max = 127) against the same packed int4
 * base + residual weights.  mq_quantize_act8 writes qA8_dev int8 [M, K] row-major (canonical order,
 * 16-byte aligned) and sA_dev float [M]; mq_gemm_a8 is mq_gemm on those (same arguments, workspace,
 * parity hooks and tolerances; acc0 / acc1 are the exact integer dot products of the int8 activations).
 * Requires 127*7*16*K < 2^31. */
int mq_quantize_act8(const void* A_dev, mq_dtype a_dtype, int64_t M, int64_t K, int64_t lda_elems,
                     int8_t* qA8_dev, float* sA_dev, void* cuda_stream);
int mq_gemm_a8(const mq_weights* w, const int8_t* qA8_dev, const float* sA_dev, int64_t M, void* Y_dev,
               mq_dtype y_dtype, int64_t ldy_elems, int32_t* dbg_acc_base_dev, int32_t* dbg_acc_res_dev,
               void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* (3c) The paper's NAIVE pipeline, for the fused-vs-naive ablation (Fig.3), NOT a
 * fast path: (i) mq_gemm with the residual switched off writes Y0 = s_a s_w acc0 as 16-bit Y, (ii) a separate
 * sparse-block GEMM re-reads qA_dev and writes the partial output acc1 (int32 [M, N] dense, exact) into scratch_dev,
 * (iii) a reduce-add kernel forms Y = round(Y0 + s_a s_r acc1).  Three launches; Y is rounded twice, so it agrees with
 * mq_gemm's only to about one unit in the last place of the larger of |Y0|, |Y|.  scratch_dev: at least
 * mq_gemm_naive_scratch_bytes(w, M) bytes, 4-byte aligned; it holds acc1 when the call returns (parity hook).
 * Other arguments, requirements and errors as mq_gemm; M <= 16 * 65535. */
size_t mq_gemm_naive_scratch_bytes(const mq_weights* w, int64_t M);
int mq_gemm_naive(const mq_weights* w, const void* qA_dev, const float* sA_dev, int64_t M, void* Y_dev,
                  mq_dtype y_dtype, int64_t ldy_elems, void* workspace_dev, size_t workspace_bytes,
                  int32_t* scratch_dev, size_t scratch_bytes, void* cuda_stream);

/* ------------------------------------------------------------------------------------
 * (3d) Scales that vary along K: per-GROUP activation quantization, the paper's stated activation
 * granularity for the 4-bit setting ("For the 4-bit setting, we adopt per-group and per-channel symmetric
 * quantization for activations and weights, respectively"; the group size is not given: reading A5g, `group` in
 * {32, 64, 128} consecutive input channels, K % group == 0).
 *
 * mq_quantize_act_group: Eq.1 on every run of `group` channels of every token.  A_dev fp16/bf16 [M, K]
 * (16-byte aligned, lda_elems % 8 == 0) -> qA_dev packed int4 [M, K/2] bytes in the canonical nibble order (byte i
 * of a row = elements 2i | 2i+1 << 4; mq_qact_bytes(M, K) bytes, 16-byte aligned; mq_unpack_act reads it) and
 * sA_dev float [M, K/group].  One launch, stream-ordered, no allocation.
 *
 * mq_gemm_group: Y[m,n] = sum_g s_a[m,g] (s_w[n] acc0_g[m,n] + s_r[n] acc1_g[m,n]) (Eq.2 P:82 and Eq.4 P:106 per
 * group), acc0_g / acc1_g the exact integer dot products of group g's activation codes with the base / selected
 * residual codes; the group terms are added in fp32 in ascending g (K-split partial sums in ascending split), then
 * rounded once to y_dtype.  Parity hooks: dbg_acc_base_g_dev / dbg_acc_res_g_dev int32 [K/group][M][N] or NULL.
 * workspace_dev: mq_gemm_group_workspace_bytes(w, M) bytes (may be 0), 16-byte aligned, no initial content
 * required.  Kernels: group = 128 and M >= 64 run on the tcgen05 tensor path (mq_group_tc.cu: whole 128 x 128 tiles, the
 * TMEM accumulator double-buffered and drained after every K-step = group into fp32 running sums; one launch, no
 * workspace); group = 128 and M <= 32 run in the row-slab decode kernel (mq_decode.cu, the sums of a K-step converted
 * and added right after its MMAs; one launch, no workspace); option "group_tc" = 0 switches both off; every other
 * case runs the warp-level mma.sync kernel on a cp.async shared-memory ring (one or two launches; M <= 16 * 65535).
 * Errors as mq_gemm. */
int mq_quantize_act_group(const void* A_dev, mq_dtype a_dtype, int64_t M, int64_t K, int64_t lda_elems, int group,
                          void* qA_dev, float* sA_dev, void* cuda_stream);
size_t mq_gemm_group_workspace_bytes(const mq_weights* w, int64_t M);
int mq_gemm_group(const mq_weights* w, const void* qA_dev, const float* sA_dev, int group, int64_t M, void* Y_dev,
                  mq_dtype y_dtype, int64_t ldy_elems, int32_t* dbg_acc_base_g_dev, int32_t* dbg_acc_res_g_dev,
                  void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* One linear layer from raw activations: A_dev fp16/bf16 [M, K] (rows 16-byte aligned, lda_elems % 8 == 0).
 * Default: mq_quantize_act into the workspace followed by mq_gemm on the same stream (two launches
 * chained by programmatic dependent launch).  With option "fused_quant" = 1 and M <= 8 the quantizer runs
 * inside the GEMM kernel (north_star (i) "optionally fused into the GEMM prologue"): one
 * launch, bit-identical Y; the per-token absmax is found with a grid-wide atomic max, the tokens of each
 * K-step are quantized from a TMA-staged raw tile.  Workspace: mq_linear_workspace_bytes(w, M), 256-byte aligned,
 * same contract as mq_gemm's (first 16384 bytes zero before the first use: the GEMM's counters and the fused
 * path's absmax control block, which every call returns to zero; the packed activations live behind them). */
size_t mq_linear_workspace_bytes(const mq_weights* w, int64_t M);
int mq_linear(const mq_weights* w, const void* A_dev, mq_dtype a_dtype, int64_t M, int64_t lda_elems,
              void* Y_dev, mq_dtype y_dtype, int64_t ldy_elems, void* workspace_dev,
              size_t workspace_bytes, void* cuda_stream);

/* mq_linear WITHOUT A CALLER WORKSPACE, for callers that cannot allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc).  Same operation, arguments, kernels and results as mq_linear
 * (bit-identical Y); the workspace (the stream-K kernel's counters, flags and partial tiles, the packed activations and
 * their scales) is a file-scope `static __device__` array inside the library of mq_linear_static_max_bytes() =
 * 16 MiB, which every GPU that loads the library holds until the process exits.  The call itself allocates nothing
 * (no cudaMalloc / cudaFree / allocating library routine): it looks the array's device address up (once per device,
 * cudaGetSymbolAddress with that device current), clears the workspace's 16384-byte zero-state prefix with
 * cudaMemsetAsync on `cuda_stream`, and runs mq_linear on the array.
 * Limit: the call is refused with MQ_ERR_STATIC_SCRATCH when mq_linear_workspace_bytes(w, M) >
 * mq_linear_static_max_bytes() (e.g. K = 4096: up to M ~ 8000 tokens on the whole-tile kernels, decode sizes always
 * fit); use mq_linear with a workspace of your own then.
 * Sharing: ALL calls on a device use the same array, and it keeps the last call's contents.  Calls that may overlap
 * on the GPU (different streams, or graph branches without an edge between them) race on it and produce garbage;
 * calls on one stream, or otherwise ordered, are safe.  At most 64 devices per process. */
size_t mq_linear_static_max_bytes(void);
int mq_linear_static(const mq_weights* w, const void* A_dev, mq_dtype a_dtype, int64_t M, int64_t lda_elems,
                     void* Y_dev, mq_dtype y_dtype, int64_t ldy_elems, void* cuda_stream);

/* The same layer with HOST buffers (end-to-end entry): A_host fp16/bf16 [M, K] dense (row stride K) is
 * copied to the device, mq_linear runs, and Y [M, N] dense is copied back to Y_host, all enqueued on
 * `cuda_stream`; the caller synchronises the stream before reading Y_host.  Host buffers should be pinned
 * (page-locked) for the copies to be asynchronous; pageable memory works but blocks.  staging_dev: device
 * scratch of at least mq_linear_host_staging_bytes(w, M) bytes (A and Y images), 256-byte aligned;
 * workspace_dev as for mq_linear. */
size_t mq_linear_host_staging_bytes(const mq_weights* w, int64_t M);
int mq_linear_host(const mq_weights* w, const void* A_host, mq_dtype a_dtype, int64_t M, void* Y_host,
                   mq_dtype y_dtype, void* staging_dev, size_t staging_bytes, void* workspace_dev,
                   size_t workspace_bytes, void* cuda_stream);

/* Concurrency and co-residency.  The decode kernel (M <= 32) and the whole-tile prefill kernels (M >= 64) contain no
 * wait of one CTA for another (CTA pairs are clusters, co-scheduled by the hardware), so calls on different streams may
 * overlap freely.  The stream-K kernel (the remaining shapes, small-M mq_gemm_a8, option-selected paths) splits the K range of
 * a tile over S CTAs that WAIT for each other's partial tiles: its grid (<= the device's SM count, one CTA per SM) must
 * be co-resident.  That holds when the call has the GPU to itself; it does not hold under an MPS active-thread
 * percentage or a green context that exposes fewer SMs than cudaDevAttrMultiProcessorCount, or while another
 * long-running kernel holds SMs (including a second stream-K call on another stream): the waiting CTAs then run into
 * the kernel's watchdog (__trap, which poisons the context) instead of hanging.  In such environments set option
 * "split_k" = 1 (whole tiles per CTA, nothing waits) and leave "fused_quant" at 0. */

/* Tuning / ablation knobs.  They are PROCESS-WIDE globals read at call time without locking: set them while no
 * other thread is inside a library call (benchmarks and tests do; a serving process leaves the defaults).  The
 * compute calls themselves keep no other mutable state and may be issued from several threads on distinct
 * streams and workspaces; mq_last_launch_count is a diagnostic of the calling process, not synchronised.
 *   "split_k"   : 0 = automatic, 1 = whole output tiles per CTA, >= 2 = stream-K (the K-steps of
 *                 all tiles cut into equal per-CTA ranges, shared tiles finished by the last arriver)
 *   "token_tile": 0 = automatic, else 16/32/64/128
 *   "max_ctas"  : 0 = all SMs, else cap on the persistent grid
 *   "fused_quant": 0 (default) / 1: see mq_linear
 *   "group_simt": 0 (default) = mq_gemm_group uses its tensor-core (mma.sync) kernel; 1 = its dp4a kernel (ablation)
 *   "group_tc"  : 1 (default) = mq_gemm_group with group = 128 runs the tcgen05 kernel for M >= 64 and the decode kernel
 *                 for M <= 32; 0 = the mma.sync kernel for every M
 *   "decode_path": 0 (default) = mq_gemm with M <= 32 runs the lean decode kernel (row slabs: a CTA owns 16..128
 *                 output channels and all of K; TMA ring + mma.sync straight from the packed tiles, no tensor
 *                 memory, no workspace); 1 = the tcgen05 kernel for every M.  Setting "token_tile", "split_k" >= 2,
 *                 "max_ctas" or "fused_quant" also selects the tcgen05 kernel.  mq_gemm_a8 with M <= 16 (M <= 32 on
 *                 layers whose slabs are 64 channels or taller) and mq_gemm_group with group = 128 and M <= 32 run
 *                 forms of the same kernel.
 *   "decode_rows": 0 = automatic, else 16 / 32 / 64 / 128 output channels per CTA of the decode kernel
 *   "decode_big": 0 = automatic, 1 = deep shared-memory ring (one CTA per SM; rows <= 64), 2 = small ring (two per SM)
 *   "prefill_path": 0 (default) = mq_gemm with M >= 64 runs the whole-tile tcgen05 kernel (128 x 128 output tiles dealt
 *                 round-robin to persistent CTAs, no workspace; CTA pairs with tcgen05.mma.cta_group::2 when the layer
 *                 has an even number of 128-channel tiles) when the last round of tiles is at least half full, else
 *                 the stream-K tcgen05 kernel; mq_gemm_a8 runs the whole-tile kernel's W4A8 form (single CTAs, int8
 *                 token tiles by TMA straight into the MMA operand stage) from three rounds of tiles per CTA upwards
 *                 (and, for M <= 32, the decode kernel's W4A8 form: see "decode_path");
 *                 1 = never; 2 = for every M >= 64, one CTA per tile; 3 = for every M >= 64, CTA pairs where possible.
 *                 The stream-K knobs above ("token_tile", "split_k" >= 2, "max_ctas") also select the stream-K kernel.
 *   "pdl"       : 1 (default) = kernels are launched as programmatic dependents of their predecessor
 *                 in the stream (prologue and weight prefetch overlap its tail); 0 = plain launches
 * Returns MQ_ERR_INVALID_ARG for an unknown name or value. */
int mq_set_option(const char* name, int64_t value);
/* Number of kernels the last mq_gemm / mq_linear / mq_quantize_act call launched. */
int mq_last_launch_count(void);

/* Diagnostic: the dense INT8 tensor-pipe throughput of the current device in TOPS, measured with
 * a pure issue loop of tcgen05.mma.cta_group::1.kind::i8 instructions of shape 128 x n x 32 (n = 128 or 256; operands
 * resident in shared memory, no loads, no epilogue), `iters` x 32 instructions on every SM.  This is the denominator
 * the north star's "INT8 tensor-core roofline" refers to on this machine.  Host-synchronous; errors as the other calls. */
int mq_probe_int8_peak(int n, int iters, double* tops_out, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* MQ_H_ */
