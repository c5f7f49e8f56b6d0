// mq_internal.h -- shared declarations of libmq.so's translation units (not installed).
//
// Device layout of a packed layer.  BN = 128 output channels per
// weight tile, BK = 128 input channels per K-step.
//
//   base   : uint8 [N/BN][K/BK][4 chunks][BN rows][16 bytes]   one 8 KB tile per (n-tile, K-step),
//            contiguous, so the kernel fetches it with ONE 1-D bulk copy (TMA).  Chunk c of a
//            row holds its 32 input channels 32c .. 32c+31 (one tcgen05.mma K slice) in the
//            canonical nibble order (byte i = elements 2i | 2i+1<<4); rows are 16 bytes apart
//            so that "one thread per output channel" reads shared memory without bank conflicts.
//   sw, sr : float [N]  base / residual scale per output channel (A4).
//   residual "cells": one cell per (n-tile, K-step) that holds >= 1 selected block,
//            CSR over n-tiles (cell_ptr[N/BN + 1]), sorted by K-step inside a tile.
//            A cell is split into four quarters q = 2*h + r  (h = k-half, r = row-half),
//            each 64 rows x 64 k = 2 KB packed [2 chunks of 32 k][64 rows][16 bytes].  Only present quarters
//            are stored, in ascending q, contiguously (res_data).
//              block = 64 : a selected block (bn,bk) is quarter (h = bk&1, r = bn&1) of
//                           cell (bn>>1, bk>>1)
//              block = 128: a selected block is a whole cell (mask 0xF)
//   cell_meta : int2 {kstep | mask << 24, first quarter index into res_data (2 KB units)}
//   unit_meta : int2 [N/BN][K/BK] {mask, first quarter index}: the same cells indexed densely by
//            (n-tile, K-step), so that the producer warp fetches the metadata of 32 consecutive
//            K-steps with one coalesced load (mask 0 = the K-step has no residual cell)
#pragma once

#include <cuda.h>

#include <cstddef>
#include <cstdint>
#include <vector>

#include "../../include/mq.h"

namespace mq {

constexpr int BN = 128;           // output channels per tile (MMA M)
constexpr int BK = 128;           // input channels per K-step
constexpr int TILE_BYTES = BN * BK / 2;   // 8192
constexpr int QUARTER_BYTES = 64 * 64 / 2;  // 2048

struct CellMeta {
  int32_t kstep_mask;  // bits 0-23: K-step index; bits 24-27: quarter-present mask
  int32_t qoff;        // index of the cell's first stored quarter (2 KB units)
};

}  // namespace mq

struct mq_weights {
  int64_t N = 0, K = 0;
  int block = 0;
  int64_t nnz = 0;         // selected blocks
  int64_t n_cells = 0;
  int64_t n_quarters = 0;
  // device buffers (one allocation, sub-pointers)
  void* dev_blob = nullptr;
  size_t dev_bytes = 0;
  uint8_t* d_base = nullptr;
  float* d_sw = nullptr;
  float* d_sr = nullptr;
  uint8_t* d_res = nullptr;
  int32_t* d_cell_ptr = nullptr;       // [N/BN + 1]
  mq::CellMeta* d_cell_meta = nullptr; // [n_cells]
  int32_t* d_unit_meta = nullptr;      // [N/BN][K/BK][2] dense index of the cells: {quarter mask, first quarter}
  // block-local residual scales (reading A4b; mq_pack_*_blockscale): one scale per row of every stored quarter,
  // float [n_quarters][64]; d_sr is then unused (all ones)
  bool blockscale = false;
  float* d_qscale = nullptr;
  // host copies of the small metadata (used by the launcher and by export)
  std::vector<int32_t> h_cell_ptr;
  std::vector<mq::CellMeta> h_cell_meta;
  int max_cells_per_tile = 0;
  // TMA descriptors over d_base for the decode kernel's row slabs of 16 / 32 / 64 / 128 output channels
  // (mq_decode.cu; built by mq::build_weight_tmaps when the handle is created or cloned)
  CUtensorMap tmap_base[4];
  bool tmap_ok = false;
};

namespace mq {

// options (mq_set_option)
struct Options {
  int64_t split_k = 0;
  int64_t token_tile = 0;
  int64_t max_ctas = 0;
  int64_t fused_quant = 0;   // mq_linear with M <= 8: quantize the activations inside the GEMM kernel (slower than
                             // the PDL-chained two-kernel path on B200; off by default)
  int64_t group_tc = 1;      // mq_gemm_group, group = 128, M >= 64: 1 = the tcgen05 kernel (mq_group_tc.cu); 0 = the mma.sync kernel
  int64_t group_simt = 0;    // mq_gemm_group: 1 = the dp4a kernel (ablation); 0 = the mma.sync kernel
  int64_t pdl = 1;   // launch kernels as programmatic dependents of their predecessor in the stream
  int64_t decode_path = 0;      // 0 = automatic (M <= 32 runs the lean mma.sync decode kernel), 1 = off (tcgen05 kernel)
  int64_t decode_big = 0;       // decode kernel ring: 0 = automatic, 1 = deep (one CTA per SM), 2 = small (two per SM)
  int64_t decode_rows = 0;      // 0 = automatic, else 16 / 32 / 64 / 128 output channels per CTA of the decode kernel
  int64_t prefill_path = 0;     // 0 = automatic (whole-tile kernel where its last round is mostly full), 1 = off, 2 = always
};
Options& options();
void set_launch_count(int n);
void add_launch_count(int n);

int check_device();  // MQ_OK or MQ_ERR_UNSUPPORTED_DEVICE / MQ_ERR_CUDA
int sm_count();

// Workspace contract shared by the GEMM kernels: the first WS_PREFIX bytes hold every word that must be ZERO
// between calls (per-tile arrival counters, the fused quantizer's control block) at positions that do not
// depend on the launch plan; every call returns them to zero.  Everything behind the prefix (partial tiles,
// flags, packed activations) is written before it is read and needs no initial content.
constexpr size_t WS_PREFIX = 16384;
constexpr int WS_MAX_TILES = 1536;                       // counters per array
constexpr size_t WS_OFF_CNT = 0;                         // int32 [WS_MAX_TILES]
constexpr size_t WS_OFF_DONE = WS_MAX_TILES * 4;         // int32 [WS_MAX_TILES]
constexpr size_t WS_OFF_FZ = 2 * WS_MAX_TILES * 4;       // uint32 [32] fused-quantizer control block

// the lean decode kernel (mq_decode.cu): M <= 32, per-token W4A4
bool decode_eligible(const mq_weights* w, int64_t M);
size_t decode_workspace_bytes(const mq_weights* w, int64_t M);
int decode_gemm(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype,
                int64_t ldy, int32_t* dbg0, int32_t* dbg1, void* workspace, size_t workspace_bytes,
                void* cuda_stream, bool ignore_res);
// the whole-tile prefill kernel (mq_prefill.cu): M >= 64, per-token W4A4, needs no workspace
bool prefill_eligible(const mq_weights* w, int64_t M, bool a8 = false);
int prefill_gemm(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype,
                 int64_t ldy, int32_t* dbg0, int32_t* dbg1, void* cuda_stream, bool ignore_res, bool a8 = false);
// per-group activation scales, group = 128, on the tcgen05 path (mq_group_tc.cu): M >= 64, no workspace
// W4A8 at decode sizes (M <= 32): the decode kernel's A8 form (mq_decode.cu)
bool decode_a8_eligible(const mq_weights* w, int64_t M);
int decode_gemm_a8(const mq_weights* w, const void* qA8, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                   int32_t* dbg0, int32_t* dbg1, void* cuda_stream, bool ignore_res);
// per-group activation scales at decode sizes (group = 128, M <= 32): the decode kernel's GRP form (mq_decode.cu)
bool decode_group_eligible(const mq_weights* w, int group, int64_t M);
int decode_gemm_group(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                      int32_t* dbg0, int32_t* dbg1, void* cuda_stream);
bool group_tc_eligible(const mq_weights* w, int group, int64_t M);
int group_tc_gemm(const mq_weights* w, const void* qA, const float* sA, int64_t M, void* Y, mq_dtype y_dtype, int64_t ldy,
                  int32_t* dbg0, int32_t* dbg1, void* cuda_stream);
int build_weight_tmaps(mq_weights* w);   // MQ_OK or MQ_ERR_CUDA
// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time libcuda dependency); NULL if absent
void* tensor_map_encode_fn();

}  // namespace mq
