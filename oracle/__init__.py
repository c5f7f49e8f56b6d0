"""numpy front-end of the CPU oracle (oracle/mq_oracle.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  It imports nothing from
paper_2606_15652_b200 and that package imports nothing from here.

Function names follow the O-steps of the .cpp header (PAPER.md citations there).
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_select.restype = C.c_int64
        _lib.orc_gemm.restype = C.c_int
        _lib.orc_forward.restype = C.c_int
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def quantize_row(x: np.ndarray, bits: int = 4) -> Tuple[np.ndarray, np.float32]:
    """O1 (Eq.1); bits = 4 (q_max 7) or 8 (q_max 127: the W4A8 activations)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    q = np.empty(x.shape[0], dtype=np.int8)
    s = np.empty(1, dtype=np.float32)
    lib().orc_quantize_row_bits(_p(x), C.c_int64(x.shape[0]), C.c_int(bits), _p(q), _p(s))
    return q, s[0]


def _bits16(A) -> Tuple[np.ndarray, int]:
    """fp16 numpy array, or (uint16 bf16 bits, 'bf16') tuple -> (uint16 bits, dtype code)."""
    if isinstance(A, tuple):
        bits, kind = A
        assert kind == "bf16" and bits.dtype == np.uint16
        return np.ascontiguousarray(bits), 1
    assert A.dtype == np.float16
    return np.ascontiguousarray(A).view(np.uint16), 0


def quantize_act(A, bits: int = 4) -> Tuple[np.ndarray, np.ndarray]:
    """O2: per-token int4 (or int8, W4A8) quantization of fp16 (np.float16) or bf16 ((bits,'bf16')) activations."""
    b16, code = _bits16(A)
    M, K = b16.shape
    qa = np.empty((M, K), dtype=np.int8)
    sa = np.empty(M, dtype=np.float32)
    lib().orc_quantize_act_bits(_p(b16), C.c_int(code), C.c_int64(M), C.c_int64(K), C.c_int64(K), C.c_int(bits), _p(qa), _p(sa))
    return qa, sa


@dataclass
class Decomp:
    qw: np.ndarray  # int8 [N,K]
    sw: np.ndarray  # fp32 [N]
    R: np.ndarray   # fp32 [N,K]
    qr: np.ndarray  # int8 [N,K]  (whole matrix, before selection)
    sr: np.ndarray  # fp32 [N]


def decompose(W: np.ndarray) -> Decomp:
    """O3 + O4 (Alg.1 line 1; Eq.4)."""
    W = np.ascontiguousarray(W, dtype=np.float32)
    N, K = W.shape
    d = Decomp(np.empty((N, K), np.int8), np.empty(N, np.float32), np.empty((N, K), np.float32),
               np.empty((N, K), np.int8), np.empty(N, np.float32))
    lib().orc_decompose(_p(W), C.c_int64(N), C.c_int64(K), _p(d.qw), _p(d.sw), _p(d.R), _p(d.qr), _p(d.sr))
    return d


def hessian_diag(X: np.ndarray) -> np.ndarray:
    """O5: binary64 h[K]."""
    X = np.ascontiguousarray(X, dtype=np.float32)
    h = np.empty(X.shape[1], dtype=np.float64)
    lib().orc_hessian_diag(_p(X), C.c_int64(X.shape[0]), C.c_int64(X.shape[1]), _p(h))
    return h


@dataclass
class Scores:
    A_B: np.ndarray
    B_B: np.ndarray
    delta: np.ndarray
    S: np.ndarray


def scores(d: Decomp, h: np.ndarray, bs: int) -> Scores:
    """O6: h is taken as fp32 (the ABI's h_host type) and promoted."""
    h32 = np.ascontiguousarray(h, dtype=np.float32)
    N, K = d.R.shape
    nb = (N // bs) * (K // bs)
    s = Scores(*(np.empty(nb, np.float64) for _ in range(4)))
    lib().orc_scores(_p(d.R), _p(d.qr), _p(d.sr), _p(h32), C.c_int64(N), C.c_int64(K), C.c_int64(bs),
                     _p(s.A_B), _p(s.B_B), _p(s.delta), _p(s.S))
    return s


def select(S: np.ndarray, budget: int) -> np.ndarray:
    """O7: selected linear block indices, score descending."""
    S = np.ascontiguousarray(S, dtype=np.float64)
    sel = np.empty(max(1, min(int(budget), S.shape[0])), dtype=np.int64)
    nnz = lib().orc_select(_p(S), C.c_int64(S.shape[0]), C.c_int64(int(budget)), _p(sel))
    return sel[:nnz].copy()


def gemm(qa: np.ndarray, qw: np.ndarray, qr: np.ndarray, bs: int, blk_n: np.ndarray, blk_k: np.ndarray):
    """O8 (Eq.2, Eq.4): int64 acc0, acc1."""
    qa = np.ascontiguousarray(qa, np.int8)
    qw = np.ascontiguousarray(qw, np.int8)
    qr = np.ascontiguousarray(qr, np.int8)
    bn = np.ascontiguousarray(blk_n, np.int32)
    bk = np.ascontiguousarray(blk_k, np.int32)
    M, K = qa.shape
    N = qw.shape[0]
    acc0 = np.empty((M, N), np.int64)
    acc1 = np.empty((M, N), np.int64)
    rc = lib().orc_gemm(_p(qa), C.c_int64(M), C.c_int64(K), _p(qw), C.c_int64(N), _p(qr), C.c_int64(bs),
                        C.c_int64(bn.shape[0]), _p(bn), _p(bk), _p(acc0), _p(acc1))
    if rc != 0:
        raise OverflowError("accumulator exceeds int32 range")
    return acc0, acc1


def output(acc0, acc1, sa, sw, sr, want_mag: bool = False):
    """O9: binary64 Y_exact (and the parity rule's magnitude term)."""
    M, N = acc0.shape
    Y = np.empty((M, N), np.float64)
    mag = np.empty((M, N), np.float64) if want_mag else None
    lib().orc_output(_p(np.ascontiguousarray(acc0, np.int64)), _p(np.ascontiguousarray(acc1, np.int64)),
                     _p(np.ascontiguousarray(sa, np.float32)), _p(np.ascontiguousarray(sw, np.float32)),
                     _p(np.ascontiguousarray(sr, np.float32)), C.c_int64(M), C.c_int64(N), _p(Y),
                     _p(mag) if want_mag else None)
    return (Y, mag) if want_mag else Y


@dataclass
class PackedLayer:
    """Algorithm 1's outputs for one layer: everything mq_pack_prequantized needs."""
    N: int
    K: int
    bs: int
    d: Decomp
    sc: Optional[Scores]
    blk_n: np.ndarray  # int32 [nnz]
    blk_k: np.ndarray  # int32 [nnz]

    @property
    def nnz(self) -> int:
        return int(self.blk_n.shape[0])

    def qr_blocks(self) -> np.ndarray:
        """Q(R) gathered on the selected blocks: int8 [nnz, bs, bs] (row = n, col = k)."""
        out = np.empty((self.nnz, self.bs, self.bs), np.int8)
        for e in range(self.nnz):
            n0, k0 = int(self.blk_n[e]) * self.bs, int(self.blk_k[e]) * self.bs
            out[e] = self.d.qr[n0:n0 + self.bs, k0:k0 + self.bs]
        return out


def algorithm1(W: np.ndarray, h: Optional[np.ndarray], bs: int, budget: int) -> PackedLayer:
    """Algorithm 1: O3, O4, O6, O7 in order.  h None = all ones."""
    N, K = W.shape
    d = decompose(W)
    if h is None:
        h = np.ones(K, np.float32)
    sc = scores(d, h, bs)
    sel = select(sc.S, budget)
    nbk = K // bs
    return PackedLayer(N, K, bs, d, sc, (sel // nbk).astype(np.int32), (sel % nbk).astype(np.int32))


def forward(A, L: PackedLayer):
    """O2 + O8 + O9 for one layer; returns dict with qa, sa, acc0, acc1, Y, mag."""
    qa, sa = quantize_act(A)
    acc0, acc1 = gemm(qa, L.d.qw, L.d.qr, L.bs, L.blk_n, L.blk_k)
    Y, mag = output(acc0, acc1, sa, L.d.sw, L.d.sr, want_mag=True)
    return dict(qa=qa, sa=sa, acc0=acc0, acc1=acc1, Y=Y, mag=mag)


def forward_timed(A, L: PackedLayer) -> np.ndarray:
    """The same three steps through one C call (no Python between them) -- what bench.py times."""
    bits, code = _bits16(A)
    M, K = bits.shape
    Y = np.empty((M, L.N), np.float64)
    lib().orc_forward(_p(bits), C.c_int(code), C.c_int64(M), C.c_int64(K), _p(L.d.qw), _p(L.d.sw), C.c_int64(L.N),
                      _p(L.d.qr), _p(L.d.sr), C.c_int64(L.bs), C.c_int64(L.nnz), _p(L.blk_n), _p(L.blk_k), _p(Y))
    return Y


def round_to_bf16(Y: np.ndarray) -> np.ndarray:
    """RNE binary64 -> bf16, returned as float64 values (Y_ref of O9).  Double rounding via
    fp32 is avoided: round the binary64 value directly to 8 significant bits."""
    Y = np.asarray(Y, np.float64)
    out = np.zeros_like(Y)
    nz = Y != 0
    m, e = np.frexp(Y[nz])          # Y = m * 2^e, 0.5 <= |m| < 1
    scaled = m * 256.0              # 8 significant bits
    r = np.rint(scaled)             # RNE
    out[nz] = np.ldexp(r, e - 8)
    return out


# ------------------------------------------------------------------------------------------------
# per-group activation quantization -- the paper's stated activation granularity for
# the 4-bit setting ("For the 4-bit setting, we adopt per-group and per-channel
# symmetric quantization for activations and weights, respectively").  The paper gives no group size
# (reading A5g): `group` is a parameter, consecutive input channels, K % group == 0.
# Plain numpy on top of O1; no blocking beyond the definition.
def quantize_act_group(A, group: int, bits: int = 4) -> Tuple[np.ndarray, np.ndarray]:
    """O2g: Eq.1 applied to every run of `group` consecutive input channels of every token:
    row (m, g) of the [M*K/group, group] view of A is one quantization unit.  Returns the codes
    int8 [M, K] and the scales fp32 [M, K/group]."""
    b16, code = _bits16(A)
    M, K = b16.shape
    assert group > 0 and K % group == 0
    view = b16.reshape(M * (K // group), group)
    qa, sa = quantize_act(view.view(np.float16) if code == 0 else (view, "bf16"), bits=bits)
    return qa.reshape(M, K), sa.reshape(M, K // group)


def residual_mask(N: int, K: int, bs: int, blk_n: np.ndarray, blk_k: np.ndarray) -> np.ndarray:
    """The block mask M of Eq.4 as a 0/1 int8 matrix [N, K]."""
    mask = np.zeros((N, K), np.int8)
    for bn, bk in zip(np.asarray(blk_n).tolist(), np.asarray(blk_k).tolist()):
        mask[bn * bs:(bn + 1) * bs, bk * bs:(bk + 1) * bs] = 1
    return mask


def forward_group(A, L: PackedLayer, group: int, cols: Optional[np.ndarray] = None, rows: Optional[np.ndarray] = None):
    """O2g + O8g + O9g.  With a scale that changes along K the scaled product of Eq.2 holds per group:
        Y[m, n] = sum_g s_a[m, g] * ( s_w[n] * acc0_g[m, n] + s_r[n] * acc1_g[m, n] )          (binary64)
        acc0_g[m, n] = sum_{k in group g} q_a[m, k] q_w[n, k]                                   (integers)
        acc1_g[m, n] = sum_{k in group g} q_a[m, k] (M (.) q_r)[n, k]                           (Eq.4's sparse term)
    `cols` / `rows` restrict the output channels / tokens (full-size cases).  Returns qa, sa, the per-group
    integer accumulators [G, M, N], their sums over g (acc0, acc1), Y and the tolerance magnitude
    mag = sum_g s_a (|s_w acc0_g| + |s_r acc1_g|)."""
    qa, sa = quantize_act_group(A, group)
    if rows is not None:
        qa, sa = qa[rows], sa[rows]
    qw, qr, sw, sr = L.d.qw, L.d.qr * residual_mask(L.N, L.K, L.bs, L.blk_n, L.blk_k), L.d.sw, L.d.sr
    if cols is not None:
        qw, qr, sw, sr = qw[cols], qr[cols], sw[cols], sr[cols]
    M, K = qa.shape
    G = K // group
    N = qw.shape[0]
    acc0_g = np.empty((G, M, N), np.int64)
    acc1_g = np.empty((G, M, N), np.int64)
    Y = np.zeros((M, N), np.float64)
    mag = np.zeros((M, N), np.float64)
    sw64, sr64 = sw.astype(np.float64)[None, :], sr.astype(np.float64)[None, :]
    for g in range(G):
        ks = slice(g * group, (g + 1) * group)
        a = qa[:, ks].astype(np.int64)
        acc0_g[g] = a @ qw[:, ks].astype(np.int64).T
        acc1_g[g] = a @ qr[:, ks].astype(np.int64).T
        s = sa[:, g].astype(np.float64)[:, None]
        Y += s * (sw64 * acc0_g[g] + sr64 * acc1_g[g])
        mag += s * (np.abs(sw64 * acc0_g[g]) + np.abs(sr64 * acc1_g[g]))
    return dict(qa=qa, sa=sa, acc0_g=acc0_g, acc1_g=acc1_g, acc0=acc0_g.sum(0), acc1=acc1_g.sum(0), Y=Y, mag=mag)


# ------------------------------------------------------------------------------------------------
# SURVEY 8(f)-3, second half: PER-BLOCK-LOCAL residual scales (north_star: "residual block list with block
# coordinates and per-block scales").  DESIGN.md reading A4b: the quantizer of Eq.1 is applied to R inside every
# block separately: for block B = (bn, bk) and output channel n in bn,
#     s_rb[n, bk] = max_{k in bk} |R[n, k]| / 7 ,   q_rb[n, k] = round(R[n, k] / s_rb[n, bk])      (O1 on the run)
# computed for EVERY block before selection, so that the gain of a block does not depend on which other blocks are
# selected (Theorem 4.1 needs B_B independent of S) -- exactly as in reading A4, with a finer scale.
# Plain numpy on top of O1; no blocking beyond the definition.
@dataclass
class DecompBlockLocal:
    qw: np.ndarray   # int8 [N,K]
    sw: np.ndarray   # fp32 [N]
    R: np.ndarray    # fp32 [N,K]
    qr: np.ndarray   # int8 [N,K]   block-local codes, whole matrix, before selection
    srb: np.ndarray  # fp32 [N, K/bs] block-local residual scales


def decompose_blocklocal(W: np.ndarray, bs: int) -> DecompBlockLocal:
    """O3 + O4b: base quantization and R as in O3 (Alg.1 line 1); Q(R) per (channel, k-block) run."""
    d = decompose(W)
    N, K = d.R.shape
    assert K % bs == 0 and N % bs == 0
    runs = np.ascontiguousarray(d.R.reshape(N * (K // bs), bs))
    q = np.empty(runs.shape, np.int8)
    s = np.empty(runs.shape[0], np.float32)
    lib().orc_quantize_rows(_p(runs), C.c_int64(runs.shape[0]), C.c_int64(bs), _p(q), _p(s))
    return DecompBlockLocal(d.qw, d.sw, d.R, q.reshape(N, K), s.reshape(N, K // bs))


def scores_blocklocal(d: DecompBlockLocal, h: np.ndarray, bs: int) -> Scores:
    """O6 with the block-local Q(R): A_B = sum_B h_k R^2, B_B = sum_B h_k (R - s_rb q_rb)^2, binary64."""
    N, K = d.R.shape
    h64 = np.ascontiguousarray(h, np.float32).astype(np.float64)
    R = d.R.astype(np.float64)
    E = R - np.repeat(d.srb.astype(np.float64), bs, axis=1) * d.qr.astype(np.float64)
    nbn, nbk = N // bs, K // bs
    A = (h64[None, :] * R * R).reshape(nbn, bs, nbk, bs).sum(axis=(1, 3)).reshape(-1)
    B = (h64[None, :] * E * E).reshape(nbn, bs, nbk, bs).sum(axis=(1, 3)).reshape(-1)
    delta = A - B
    return Scores(A, B, delta, np.maximum(delta, 0.0))


@dataclass
class PackedLayerBlockLocal:
    N: int
    K: int
    bs: int
    d: DecompBlockLocal
    sc: Optional[Scores]
    blk_n: np.ndarray
    blk_k: np.ndarray

    @property
    def nnz(self) -> int:
        return int(self.blk_n.shape[0])

    def qr_blocks(self) -> np.ndarray:
        out = np.empty((self.nnz, self.bs, self.bs), np.int8)
        for e in range(self.nnz):
            n0, k0 = int(self.blk_n[e]) * self.bs, int(self.blk_k[e]) * self.bs
            out[e] = self.d.qr[n0:n0 + self.bs, k0:k0 + self.bs]
        return out

    def sr_blocks(self) -> np.ndarray:
        """fp32 [nnz, bs]: the scale of every row of every selected block."""
        out = np.empty((self.nnz, self.bs), np.float32)
        for e in range(self.nnz):
            n0 = int(self.blk_n[e]) * self.bs
            out[e] = self.d.srb[n0:n0 + self.bs, int(self.blk_k[e])]
        return out


def algorithm1_blocklocal(W: np.ndarray, h: Optional[np.ndarray], bs: int, budget: int) -> PackedLayerBlockLocal:
    """Algorithm 1 with block-local residual scales: O3, O4b, O6, O7."""
    N, K = W.shape
    d = decompose_blocklocal(W, bs)
    if h is None:
        h = np.ones(K, np.float32)
    sc = scores_blocklocal(d, h, bs)
    sel = select(sc.S, budget)
    nbk = K // bs
    return PackedLayerBlockLocal(N, K, bs, d, sc, (sel // nbk).astype(np.int32), (sel % nbk).astype(np.int32))


def forward_blocklocal(A, L: PackedLayerBlockLocal, rows: Optional[np.ndarray] = None):
    """O2 + O8b + O9b.  With a residual scale that changes from block to block the sparse term of Eq.4 is a sum
    of per-block scaled integer products:
        Y[m, n] = s_a[m] * ( s_w[n] * acc0[m, n] + sum_{(bn, bk) in S, n in bn} s_rb[n, bk] * acc1_B[m, n] )     (binary64)
        acc1_B[m, n] = sum_{k in bk} q_a[m, k] q_rb[n, k]                                                     (integers)
    Returns qa, sa, acc0, acc1sum (= sum over the selected blocks of acc1_B: an integer checksum of the sparse term,
    what the CUDA parity hook returns), Y, and the tolerance magnitude mag = |s_a| (|s_w acc0| + sum_B |s_rb acc1_B|)."""
    qa, sa = quantize_act(A)
    if rows is not None:
        qa, sa = qa[rows], sa[rows]
    M, K = qa.shape
    N, bs = L.N, L.bs
    a64 = qa.astype(np.int64)
    acc0 = a64 @ L.d.qw.astype(np.int64).T
    acc1sum = np.zeros((M, N), np.int64)
    sparse = np.zeros((M, N), np.float64)
    smag = np.zeros((M, N), np.float64)
    for bn, bk in zip(L.blk_n.tolist(), L.blk_k.tolist()):
        ns, ks = slice(bn * bs, (bn + 1) * bs), slice(bk * bs, (bk + 1) * bs)
        accB = a64[:, ks] @ L.d.qr[ns, ks].astype(np.int64).T            # [M, bs]
        sB = L.d.srb[ns, bk].astype(np.float64)[None, :]
        acc1sum[:, ns] += accB
        sparse[:, ns] += sB * accB
        smag[:, ns] += np.abs(sB * accB)
    sa64, sw64 = sa.astype(np.float64)[:, None], L.d.sw.astype(np.float64)[None, :]
    Y = sa64 * (sw64 * acc0 + sparse)
    mag = np.abs(sa64) * (np.abs(sw64 * acc0) + smag)
    return dict(qa=qa, sa=sa, acc0=acc0, acc1sum=acc1sum, Y=Y, mag=mag)
