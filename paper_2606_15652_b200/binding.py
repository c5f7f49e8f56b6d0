"""Thin ctypes binding of libmq.so (include/mq.h).  Argument marshalling only: every step of
the path runs in the library's CUDA kernels.  PyTorch supplies device memory and streams.

There is no fallback: if the shared library is missing or the device is not a B200
(compute capability 10.0) the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Tuple

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmq.so")

MQ_F16, MQ_BF16 = 0, 1

EXPORTS = [
    "mq_status_string", "mq_qact_bytes", "mq_quantize_act", "mq_unpack_act", "mq_pack_weights", "mq_pack_weights_device",
    "mq_pack_prequantized", "mq_weights_export", "mq_weights_clone", "mq_weights_info", "mq_weights_free",
    "mq_gemm_workspace_bytes", "mq_gemm", "mq_linear_workspace_bytes", "mq_linear", "mq_linear_host_staging_bytes",
    "mq_linear_host", "mq_quantize_act8", "mq_gemm_a8", "mq_gemm_naive", "mq_gemm_naive_scratch_bytes", "mq_set_option",
    "mq_last_launch_count", "mq_quantize_act_group", "mq_gemm_group_workspace_bytes", "mq_gemm_group",
    "mq_probe_int8_peak", "mq_pack_weights_blockscale", "mq_pack_prequantized_blockscale", "mq_weights_export_blockscale",
    "mq_weights_is_blockscale", "mq_linear_static_max_bytes", "mq_linear_static",
]

_lib = None


class MqError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: mq_status {status} ({status_string(status)})")


def lib() -> C.CDLL:
    """Load libmq.so (built in-tree by paper_2606_15652_b200.build).  Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} not found: build it with `python -m paper_2606_15652_b200.build` "
            "(there is no CPU or PyTorch fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32, sz = C.c_void_p, C.c_int64, C.c_int, C.c_size_t
    L.mq_status_string.restype = C.c_char_p
    L.mq_status_string.argtypes = [i32]
    L.mq_qact_bytes.restype = sz
    L.mq_qact_bytes.argtypes = [i64, i64]
    L.mq_quantize_act.restype = i32
    L.mq_quantize_act.argtypes = [vp, i32, i64, i64, i64, vp, vp, vp]
    L.mq_unpack_act.restype = i32
    L.mq_unpack_act.argtypes = [vp, i64, i64, vp, vp]
    L.mq_pack_weights.restype = i32
    L.mq_pack_weights.argtypes = [vp, i64, i64, vp, i32, i64, C.POINTER(vp), vp]
    L.mq_pack_weights_device.restype = i32
    L.mq_pack_weights_device.argtypes = [vp, i64, i64, vp, i32, i64, C.POINTER(vp), vp]
    L.mq_pack_weights_blockscale.restype = i32
    L.mq_pack_weights_blockscale.argtypes = [vp, i64, i64, vp, i32, i64, C.POINTER(vp), vp]
    L.mq_pack_prequantized_blockscale.restype = i32
    L.mq_pack_prequantized_blockscale.argtypes = [vp, vp, i64, i64, i32, i64, vp, vp, vp, vp, C.POINTER(vp), vp]
    L.mq_weights_export_blockscale.restype = i32
    L.mq_weights_export_blockscale.argtypes = [vp, vp]
    L.mq_weights_is_blockscale.restype = i32
    L.mq_weights_is_blockscale.argtypes = [vp]
    L.mq_pack_prequantized.restype = i32
    L.mq_pack_prequantized.argtypes = [vp, vp, i64, i64, i32, i64, vp, vp, vp, vp, C.POINTER(vp), vp]
    L.mq_weights_export.restype = i32
    L.mq_weights_export.argtypes = [vp, vp, vp, C.POINTER(i64), vp, vp, vp, vp]
    L.mq_weights_clone.restype = i32
    L.mq_weights_clone.argtypes = [vp, C.POINTER(vp), vp]
    L.mq_weights_info.restype = i32
    L.mq_weights_info.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(i32), C.POINTER(i64), C.POINTER(sz)]
    L.mq_weights_free.restype = None
    L.mq_weights_free.argtypes = [vp]
    L.mq_gemm_workspace_bytes.restype = sz
    L.mq_gemm_workspace_bytes.argtypes = [vp, i64]
    L.mq_gemm.restype = i32
    L.mq_gemm.argtypes = [vp, vp, vp, i64, vp, i32, i64, vp, vp, vp, sz, vp]
    L.mq_linear_workspace_bytes.restype = sz
    L.mq_linear_workspace_bytes.argtypes = [vp, i64]
    L.mq_linear.restype = i32
    L.mq_linear.argtypes = [vp, vp, i32, i64, i64, vp, i32, i64, vp, sz, vp]
    L.mq_linear_static_max_bytes.restype = sz
    L.mq_linear_static_max_bytes.argtypes = []
    L.mq_linear_static.restype = i32
    L.mq_linear_static.argtypes = [vp, vp, i32, i64, i64, vp, i32, i64, vp]
    L.mq_linear_host_staging_bytes.restype = sz
    L.mq_linear_host_staging_bytes.argtypes = [vp, i64]
    L.mq_linear_host.restype = i32
    L.mq_linear_host.argtypes = [vp, vp, i32, i64, vp, i32, vp, sz, vp, sz, vp]
    L.mq_quantize_act8.restype = i32
    L.mq_quantize_act8.argtypes = [vp, i32, i64, i64, i64, vp, vp, vp]
    L.mq_gemm_a8.restype = i32
    L.mq_gemm_a8.argtypes = [vp, vp, vp, i64, vp, i32, i64, vp, vp, vp, sz, vp]
    L.mq_gemm_naive_scratch_bytes.restype = sz
    L.mq_gemm_naive_scratch_bytes.argtypes = [vp, i64]
    L.mq_gemm_naive.restype = i32
    L.mq_gemm_naive.argtypes = [vp, vp, vp, i64, vp, i32, i64, vp, sz, vp, sz, vp]
    L.mq_quantize_act_group.restype = i32
    L.mq_quantize_act_group.argtypes = [vp, i32, i64, i64, i64, i32, vp, vp, vp]
    L.mq_gemm_group_workspace_bytes.restype = sz
    L.mq_gemm_group_workspace_bytes.argtypes = [vp, i64]
    L.mq_gemm_group.restype = i32
    L.mq_gemm_group.argtypes = [vp, vp, vp, i32, i64, vp, i32, i64, vp, vp, vp, sz, vp]
    L.mq_set_option.restype = i32
    L.mq_set_option.argtypes = [C.c_char_p, i64]
    L.mq_last_launch_count.restype = i32
    L.mq_last_launch_count.argtypes = []
    L.mq_probe_int8_peak.restype = i32
    L.mq_probe_int8_peak.argtypes = [i32, i32, C.POINTER(C.c_double), vp]
    _lib = L
    return L


def status_string(status: int) -> str:
    return lib().mq_status_string(int(status)).decode()


def _check(status: int, where: str) -> None:
    if status != 0:
        raise MqError(status, where)


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _dtype_code(dt: torch.dtype) -> int:
    if dt == torch.float16:
        return MQ_F16
    if dt == torch.bfloat16:
        return MQ_BF16
    raise TypeError(f"mq: unsupported dtype {dt}")


def _np_ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def mq_set_option(name: str, value: int) -> None:
    _check(lib().mq_set_option(name.encode(), int(value)), f"mq_set_option({name})")


def mq_last_launch_count() -> int:
    return int(lib().mq_last_launch_count())


def mq_probe_int8_peak(n: int = 256, iters: int = 2000) -> float:
    """Measured dense INT8 tensor-pipe throughput (TOPS) of the current device: a pure tcgen05.mma kind::i8 issue loop."""
    out = C.c_double()
    _check(lib().mq_probe_int8_peak(int(n), int(iters), C.byref(out), _stream()), "mq_probe_int8_peak")
    return float(out.value)


def mq_qact_bytes(M: int, K: int) -> int:
    return int(lib().mq_qact_bytes(M, K))


def mq_quantize_act(A: torch.Tensor, qA: Optional[torch.Tensor] = None,
                    sA: Optional[torch.Tensor] = None) -> Tuple[torch.Tensor, torch.Tensor]:
    """A [M,K] fp16/bf16 CUDA tensor (last dim contiguous) -> (qA uint8 [M,K/2], sA fp32 [M])."""
    assert A.is_cuda and A.dim() == 2 and A.stride(1) == 1
    M, K = A.shape
    if qA is None:
        qA = torch.empty((M, K // 2), dtype=torch.uint8, device=A.device)
    if sA is None:
        sA = torch.empty((M,), dtype=torch.float32, device=A.device)
    lda = A.stride(0) if M > 1 else K
    _check(lib().mq_quantize_act(A.data_ptr(), _dtype_code(A.dtype), M, K, lda, qA.data_ptr(), sA.data_ptr(),
                                 _stream()), "mq_quantize_act")
    return qA, sA


def mq_unpack_act(qA: torch.Tensor, M: int, K: int) -> torch.Tensor:
    q = torch.empty((M, K), dtype=torch.int8, device=qA.device)
    _check(lib().mq_unpack_act(qA.data_ptr(), M, K, q.data_ptr(), _stream()), "mq_unpack_act")
    return q


class Weights:
    """Owner of an mq_weights* handle."""

    def __init__(self, handle: int):
        self._h = C.c_void_p(handle)

    @property
    def handle(self) -> C.c_void_p:
        if not self._h:
            raise ValueError("mq_weights already freed")
        return self._h

    def info(self):
        N, K, nnz = C.c_int64(), C.c_int64(), C.c_int64()
        blk = C.c_int()
        nbytes = C.c_size_t()
        _check(lib().mq_weights_info(self.handle, C.byref(N), C.byref(K), C.byref(blk), C.byref(nnz),
                                     C.byref(nbytes)), "mq_weights_info")
        return dict(N=N.value, K=K.value, block=blk.value, nnz=nnz.value, device_bytes=nbytes.value)

    def export(self):
        """Canonical host arrays read back from the device layout (mq_weights_export)."""
        i = self.info()
        N, K, bs, nnz = i["N"], i["K"], i["block"], i["nnz"]
        qW = np.empty((N, K), np.int8)
        sW = np.empty(N, np.float32)
        sR = np.empty(N, np.float32)
        bn = np.empty(max(nnz, 1), np.int32)
        bk = np.empty(max(nnz, 1), np.int32)
        qR = np.empty((max(nnz, 1), bs, bs), np.int8)
        n = C.c_int64()
        _check(lib().mq_weights_export(self.handle, _np_ptr(qW), _np_ptr(sW), C.byref(n), _np_ptr(bn), _np_ptr(bk),
                                       _np_ptr(qR), _np_ptr(sR)), "mq_weights_export")
        return dict(qW=qW, sW=sW, sR=sR, blk_n=bn[:nnz], blk_k=bk[:nnz], qR=qR[:nnz], nnz=int(n.value))

    def is_blockscale(self) -> bool:
        return bool(lib().mq_weights_is_blockscale(self.handle))

    def export_blockscale(self) -> np.ndarray:
        """Block-local residual scales fp32 [nnz, block], blocks in export()'s order (mq_weights_export_blockscale)."""
        i = self.info()
        out = np.empty((max(i["nnz"], 1), i["block"]), np.float32)
        _check(lib().mq_weights_export_blockscale(self.handle, _np_ptr(out)), "mq_weights_export_blockscale")
        return out[:i["nnz"]]

    def clone(self) -> "Weights":
        out = C.c_void_p()
        _check(lib().mq_weights_clone(self.handle, C.byref(out), _stream()), "mq_weights_clone")
        return Weights(out.value)

    def free(self) -> None:
        if self._h:
            lib().mq_weights_free(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def mq_pack_weights(W: np.ndarray, h: Optional[np.ndarray], block: int, budget_blocks: int) -> Weights:
    """Algorithm 1 on the host + device layout.  W fp32 [N,K] (numpy), h fp32 [K] or None."""
    W = np.ascontiguousarray(W, dtype=np.float32)
    N, K = W.shape
    h32 = None if h is None else np.ascontiguousarray(h, dtype=np.float32)
    out = C.c_void_p()
    _check(lib().mq_pack_weights(_np_ptr(W), N, K, _np_ptr(h32), block, int(budget_blocks), C.byref(out), _stream()),
           "mq_pack_weights")
    return Weights(out.value)


def mq_pack_weights_blockscale(W: np.ndarray, h: Optional[np.ndarray], block: int, budget_blocks: int) -> Weights:
    """Algorithm 1 with block-local residual scales (reading A4b) on the host + device layout."""
    W = np.ascontiguousarray(W, dtype=np.float32)
    N, K = W.shape
    h32 = None if h is None else np.ascontiguousarray(h, dtype=np.float32)
    out = C.c_void_p()
    _check(lib().mq_pack_weights_blockscale(_np_ptr(W), N, K, _np_ptr(h32), block, int(budget_blocks), C.byref(out), _stream()),
           "mq_pack_weights_blockscale")
    return Weights(out.value)


def mq_pack_prequantized_blockscale(qW: np.ndarray, sW: np.ndarray, block: int, blk_n: np.ndarray, blk_k: np.ndarray,
                                    qR: np.ndarray, sRb: np.ndarray) -> Weights:
    qW = np.ascontiguousarray(qW, np.int8)
    N, K = qW.shape
    sW = np.ascontiguousarray(sW, np.float32)
    sRb = np.ascontiguousarray(sRb, np.float32)
    blk_n = np.ascontiguousarray(blk_n, np.int32)
    blk_k = np.ascontiguousarray(blk_k, np.int32)
    qR = np.ascontiguousarray(qR, np.int8)
    nnz = int(blk_n.shape[0])
    out = C.c_void_p()
    _check(lib().mq_pack_prequantized_blockscale(_np_ptr(qW), _np_ptr(sW), N, K, block, nnz, _np_ptr(blk_n) if nnz else None,
                                                 _np_ptr(blk_k) if nnz else None, _np_ptr(qR) if nnz else None,
                                                 _np_ptr(sRb) if nnz else None, C.byref(out), _stream()),
           "mq_pack_prequantized_blockscale")
    return Weights(out.value)


def mq_pack_weights_device(W: torch.Tensor, h: Optional[torch.Tensor], block: int, budget_blocks: int) -> Weights:
    """Algorithm 1 with the O(N*K) part on the GPU.  W fp32 [N,K] CUDA tensor (contiguous), h fp32 [K] CUDA tensor or None."""
    assert W.is_cuda and W.dtype == torch.float32 and W.is_contiguous()
    N, K = W.shape
    assert h is None or (h.is_cuda and h.dtype == torch.float32 and h.is_contiguous() and h.numel() == K)
    out = C.c_void_p()
    _check(lib().mq_pack_weights_device(W.data_ptr(), N, K, h.data_ptr() if h is not None else None, block,
                                        int(budget_blocks), C.byref(out), _stream()), "mq_pack_weights_device")
    return Weights(out.value)


def mq_pack_prequantized(qW: np.ndarray, sW: np.ndarray, block: int, blk_n: np.ndarray, blk_k: np.ndarray,
                         qR: np.ndarray, sR: np.ndarray) -> Weights:
    qW = np.ascontiguousarray(qW, np.int8)
    N, K = qW.shape
    sW = np.ascontiguousarray(sW, np.float32)
    sR = np.ascontiguousarray(sR, np.float32)
    blk_n = np.ascontiguousarray(blk_n, np.int32)
    blk_k = np.ascontiguousarray(blk_k, np.int32)
    qR = np.ascontiguousarray(qR, np.int8)
    nnz = int(blk_n.shape[0])
    out = C.c_void_p()
    _check(lib().mq_pack_prequantized(_np_ptr(qW), _np_ptr(sW), N, K, block, nnz, _np_ptr(blk_n) if nnz else None,
                                      _np_ptr(blk_k) if nnz else None, _np_ptr(qR) if nnz else None, _np_ptr(sR),
                                      C.byref(out), _stream()), "mq_pack_prequantized")
    return Weights(out.value)


def mq_gemm_workspace_bytes(w: Weights, M: int) -> int:
    return int(lib().mq_gemm_workspace_bytes(w.handle, M))


def mq_linear_workspace_bytes(w: Weights, M: int) -> int:
    return int(lib().mq_linear_workspace_bytes(w.handle, M))


def new_workspace(nbytes: int, device="cuda") -> Optional[torch.Tensor]:
    """A zeroed workspace (the zero-state contract of mq_gemm)."""
    if nbytes == 0:
        return None
    return torch.zeros(((nbytes + 255) // 256 * 256,), dtype=torch.uint8, device=device)


def mq_gemm(w: Weights, qA: torch.Tensor, sA: torch.Tensor, M: int, Y: Optional[torch.Tensor] = None,
            out_dtype: torch.dtype = torch.bfloat16, dbg: bool = False, workspace: Optional[torch.Tensor] = None):
    """Y [M,N] = fused base + residual GEMM.  Returns Y, or (Y, acc_base, acc_res) when dbg."""
    info = w.info()
    N = info["N"]
    if Y is None:
        Y = torch.empty((M, N), dtype=out_dtype, device=qA.device)
    need = mq_gemm_workspace_bytes(w, M)
    if need and workspace is None:
        workspace = new_workspace(need, qA.device)
    d0 = torch.empty((M, N), dtype=torch.int32, device=qA.device) if dbg else None
    d1 = torch.empty((M, N), dtype=torch.int32, device=qA.device) if dbg else None
    ldy = Y.stride(0) if M > 1 else N
    _check(lib().mq_gemm(w.handle, qA.data_ptr(), sA.data_ptr(), M, Y.data_ptr(), _dtype_code(Y.dtype), ldy,
                         d0.data_ptr() if dbg else None, d1.data_ptr() if dbg else None,
                         workspace.data_ptr() if workspace is not None else None,
                         workspace.numel() if workspace is not None else 0, _stream()), "mq_gemm")
    return (Y, d0, d1) if dbg else Y


def mq_linear(w: Weights, A: torch.Tensor, Y: Optional[torch.Tensor] = None, out_dtype: torch.dtype = torch.bfloat16,
              workspace: Optional[torch.Tensor] = None) -> torch.Tensor:
    info = w.info()
    M, K = A.shape
    N = info["N"]
    if Y is None:
        Y = torch.empty((M, N), dtype=out_dtype, device=A.device)
    if workspace is None:
        workspace = new_workspace(mq_linear_workspace_bytes(w, M), A.device)
    lda = A.stride(0) if M > 1 else K
    ldy = Y.stride(0) if M > 1 else N
    _check(lib().mq_linear(w.handle, A.data_ptr(), _dtype_code(A.dtype), M, lda, Y.data_ptr(), _dtype_code(Y.dtype),
                           ldy, workspace.data_ptr(), workspace.numel(), _stream()), "mq_linear")
    return Y


def mq_linear_static_max_bytes() -> int:
    return int(lib().mq_linear_static_max_bytes())


def mq_linear_static(w: Weights, A: torch.Tensor, Y: torch.Tensor) -> torch.Tensor:
    """mq_linear on the library's built-in scratch array: the call allocates nothing (the caller passes A and Y)."""
    M, K = A.shape
    N = Y.shape[1]
    lda = A.stride(0) if M > 1 else K
    ldy = Y.stride(0) if M > 1 else N
    _check(lib().mq_linear_static(w.handle, A.data_ptr(), _dtype_code(A.dtype), M, lda, Y.data_ptr(), _dtype_code(Y.dtype),
                                  ldy, _stream()), "mq_linear_static")
    return Y


def mq_linear_host_staging_bytes(w: Weights, M: int) -> int:
    return int(lib().mq_linear_host_staging_bytes(w.handle, M))


def mq_linear_host(w: Weights, A_host: torch.Tensor, Y_host: torch.Tensor, staging: torch.Tensor,
                   workspace: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """End-to-end entry with HOST tensors (pinned for asynchronous copies): enqueues H2D copy, mq_linear and
    D2H copy on `stream` (default: the current stream); the caller synchronises that stream before reading Y_host.
    Independent calls given different streams (and their own staging and workspace) overlap one call's copies with
    another's kernels."""
    M, K = A_host.shape
    assert A_host.is_contiguous() and Y_host.is_contiguous() and not A_host.is_cuda and not Y_host.is_cuda
    st = _stream() if stream is None else stream.cuda_stream
    _check(lib().mq_linear_host(w.handle, A_host.data_ptr(), _dtype_code(A_host.dtype), M, Y_host.data_ptr(),
                                _dtype_code(Y_host.dtype), staging.data_ptr(), staging.numel(), workspace.data_ptr(),
                                workspace.numel(), st), "mq_linear_host")
    return Y_host


def mq_quantize_act8(A: torch.Tensor) -> Tuple[torch.Tensor, torch.Tensor]:
    """W4A8: per-token int8 activations (q_max = 127).  Returns (qA8 int8 [M,K], sA float32 [M])."""
    M, K = A.shape
    q8 = torch.empty((M, K), dtype=torch.int8, device=A.device)
    sA = torch.empty((M,), dtype=torch.float32, device=A.device)
    lda = A.stride(0) if M > 1 else K
    _check(lib().mq_quantize_act8(A.data_ptr(), _dtype_code(A.dtype), M, K, lda, q8.data_ptr(), sA.data_ptr(), _stream()),
           "mq_quantize_act8")
    return q8, sA


def mq_gemm_a8(w: Weights, qA8: torch.Tensor, sA: torch.Tensor, M: int, Y: Optional[torch.Tensor] = None,
               out_dtype: torch.dtype = torch.bfloat16, dbg: bool = False, workspace: Optional[torch.Tensor] = None):
    """W4A8 fused base + residual GEMM (int8 activations).  Same contract as mq_gemm."""
    N = w.info()["N"]
    if Y is None:
        Y = torch.empty((M, N), dtype=out_dtype, device=qA8.device)
    need = mq_gemm_workspace_bytes(w, M)
    if need and workspace is None:
        workspace = new_workspace(need, qA8.device)
    d0 = torch.empty((M, N), dtype=torch.int32, device=qA8.device) if dbg else None
    d1 = torch.empty((M, N), dtype=torch.int32, device=qA8.device) if dbg else None
    ldy = Y.stride(0) if M > 1 else N
    _check(lib().mq_gemm_a8(w.handle, qA8.data_ptr(), sA.data_ptr(), M, Y.data_ptr(), _dtype_code(Y.dtype), ldy,
                            d0.data_ptr() if dbg else None, d1.data_ptr() if dbg else None,
                            workspace.data_ptr() if workspace is not None else None,
                            workspace.numel() if workspace is not None else 0, _stream()), "mq_gemm_a8")
    return (Y, d0, d1) if dbg else Y


def mq_gemm_naive_scratch_bytes(w: Weights, M: int) -> int:
    return int(lib().mq_gemm_naive_scratch_bytes(w.handle, M))


def mq_gemm_naive(w: Weights, qA: torch.Tensor, sA: torch.Tensor, M: int, Y: Optional[torch.Tensor] = None,
                  out_dtype: torch.dtype = torch.bfloat16, workspace: Optional[torch.Tensor] = None,
                  scratch: Optional[torch.Tensor] = None):
    """The paper's naive 3-kernel pipeline (dense GEMM, sparse-block GEMM, reduce-add): ablation only.
    Returns (Y, acc1) with acc1 the sparse kernel's int32 partial output [M, N]."""
    N = w.info()["N"]
    if Y is None:
        Y = torch.empty((M, N), dtype=out_dtype, device=qA.device)
    need = mq_gemm_workspace_bytes(w, M)
    if need and workspace is None:
        workspace = new_workspace(need, qA.device)
    if scratch is None:
        scratch = torch.empty((M, N), dtype=torch.int32, device=qA.device)
    ldy = Y.stride(0) if M > 1 else N
    _check(lib().mq_gemm_naive(w.handle, qA.data_ptr(), sA.data_ptr(), M, Y.data_ptr(), _dtype_code(Y.dtype), ldy,
                               workspace.data_ptr() if workspace is not None else None,
                               workspace.numel() if workspace is not None else 0,
                               scratch.data_ptr(), scratch.numel() * 4, _stream()), "mq_gemm_naive")
    return Y, scratch


def mq_quantize_act_group(A: torch.Tensor, group: int) -> Tuple[torch.Tensor, torch.Tensor]:
    """Per-group int4 activations.  Returns (qA uint8 [M,K/2], sA float32 [M,K/group])."""
    assert A.is_cuda and A.dim() == 2 and A.stride(1) == 1
    M, K = A.shape
    qA = torch.empty((M, K // 2), dtype=torch.uint8, device=A.device)
    sA = torch.empty((M, max(K // max(group, 1), 1)), dtype=torch.float32, device=A.device)
    lda = A.stride(0) if M > 1 else K
    _check(lib().mq_quantize_act_group(A.data_ptr(), _dtype_code(A.dtype), M, K, lda, group, qA.data_ptr(), sA.data_ptr(),
                                       _stream()), "mq_quantize_act_group")
    return qA, sA


def mq_gemm_group_workspace_bytes(w: Weights, M: int) -> int:
    return int(lib().mq_gemm_group_workspace_bytes(w.handle, M))


def mq_gemm_group(w: Weights, qA: torch.Tensor, sA: torch.Tensor, group: int, M: int, Y: Optional[torch.Tensor] = None,
                  out_dtype: torch.dtype = torch.bfloat16, dbg: bool = False, workspace: Optional[torch.Tensor] = None):
    """Base + residual GEMM with per-group activation scales.  dbg: also returns the per-group integer
    accumulators int32 [K/group, M, N] (base, residual)."""
    inf = w.info()
    N, K = inf["N"], inf["K"]
    if Y is None:
        Y = torch.empty((M, N), dtype=out_dtype, device=qA.device)
    need = mq_gemm_group_workspace_bytes(w, M)
    if need and workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=qA.device)
    G = K // group
    d0 = torch.empty((G, M, N), dtype=torch.int32, device=qA.device) if dbg else None
    d1 = torch.empty((G, M, N), dtype=torch.int32, device=qA.device) if dbg else None
    ldy = Y.stride(0) if M > 1 else N
    _check(lib().mq_gemm_group(w.handle, qA.data_ptr(), sA.data_ptr(), group, M, Y.data_ptr(), _dtype_code(Y.dtype), ldy,
                               d0.data_ptr() if dbg else None, d1.data_ptr() if dbg else None,
                               workspace.data_ptr() if workspace is not None else None,
                               workspace.numel() if workspace is not None else 0, _stream()), "mq_gemm_group")
    return (Y, d0, d1) if dbg else Y
