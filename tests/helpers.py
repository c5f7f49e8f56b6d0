"""Shared helpers of the parity tests: build a seeded case with the ORACLE, run the CUDA path
through the C ABI, compare.  The oracle and the CUDA path meet only here (and in smoke/bench).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np

import oracle
import synth

# Tolerance on Y (tolerance T1 -- not a reading of the paper).  north_star: "within max relative error 2e-3
# (fp32 epilogue, bf16 output rounding)".  fp16 output: exactly that bound.  bf16 output: a bf16
# has 8 significant bits, so even the CORRECTLY ROUNDED result is up to 2^-8 = 3.9e-3 away (first
# GPU run: exact -5.13993 -> nearest bf16 -5.125, 2.9e-3); the bound used is therefore the
# tightest one any implementation can meet: half a bf16 ulp of the exact value.  Both carry an
# absolute term for the fp32 epilogue (cancellation between the base and residual terms).
Y_RTOL = 2e-3
Y_MAG_TOL = 1e-6


def y_tolerance(Y_exact: np.ndarray, mag: np.ndarray, out_dtype: str) -> np.ndarray:
    if out_dtype == "f16":
        return Y_RTOL * np.abs(Y_exact) + Y_MAG_TOL * mag
    _, e = np.frexp(Y_exact)                      # |Y| in [2^(e-1), 2^e)
    half_ulp = np.where(Y_exact == 0, 0.0, np.ldexp(1.0, e - 1 - 7 - 1))   # ulp = 2^(e-1) * 2^-7
    return half_ulp + Y_MAG_TOL * mag


@dataclass
class Case:
    M: int
    K: int
    N: int
    bs: int
    W: np.ndarray
    h: Optional[np.ndarray]
    A16: np.ndarray          # np.float16, or uint16 bf16 bits
    a_dtype: str             # "f16" | "bf16"
    L: "oracle.PackedLayer"


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """RNE fp32 -> bf16 bit patterns (uint16); inputs are finite."""
    u = np.ascontiguousarray(x, np.float32).view(np.uint32).astype(np.uint64)
    r = (u + 0x7FFF + ((u >> 16) & 1)) >> 16
    return r.astype(np.uint16)


def make_case(seed: int, M: int, K: int, N: int, bs: int = 64, rho: Optional[float] = 0.05,
              budget: Optional[int] = None, a_dtype: str = "f16", calib_tokens: int = 64,
              n_outlier_ch: Optional[int] = None) -> Case:
    W = synth.gen_weight(seed, N, K)
    if a_dtype == "f16":
        A16 = synth.gen_act(seed, M, K, n_outlier_ch=n_outlier_ch)
    else:
        A16 = f32_to_bf16_bits(synth.gen_act(seed, M, K, n_outlier_ch=n_outlier_ch, dtype="f32"))
    X = synth.gen_calib(seed, K, calib_tokens, n_outlier_ch=n_outlier_ch)
    h = oracle.hessian_diag(X).astype(np.float32)
    if budget is None:
        budget = synth.budget_from_density(rho, N, K, bs)
    L = oracle.algorithm1(W, h, bs, budget)
    return Case(M, K, N, bs, W, h, A16, a_dtype, L)


def oracle_act(case: Case, bits: int = 4):
    return oracle.quantize_act(case.A16 if case.a_dtype == "f16" else (case.A16, "bf16"), bits=bits)


def oracle_forward(case: Case, rows: Optional[np.ndarray] = None, bits: int = 4):
    """O2 + O8 + O9 (optionally on a subset of token rows); bits = activation width (4: W4A4, 8: W4A8)."""
    qa, sa = oracle_act(case, bits)
    if rows is not None:
        qa, sa = qa[rows], sa[rows]
    acc0, acc1 = oracle.gemm(qa, case.L.d.qw, case.L.d.qr, case.L.bs, case.L.blk_n, case.L.blk_k)
    Y, mag = oracle.output(acc0, acc1, sa, case.L.d.sw, case.L.d.sr, want_mag=True)
    return dict(qa=qa, sa=sa, acc0=acc0, acc1=acc1, Y=Y, mag=mag)


# ---------------------------------------------------------------------------------- CUDA side
def to_device_act(case: Case):
    import torch
    if case.a_dtype == "f16":
        return torch.from_numpy(case.A16).cuda()
    return torch.from_numpy(case.A16.view(np.int16)).cuda().view(torch.bfloat16)


def pack_from_oracle(case: Case):
    """mq_pack_prequantized on the oracle's decomposition (isolates GEMM parity from selection)."""
    import paper_2606_15652_b200 as mq
    L = case.L
    return mq.mq_pack_prequantized(L.d.qw, L.d.sw, L.bs, L.blk_n, L.blk_k, L.qr_blocks(), L.d.sr)


def run_cuda(case: Case, w=None, out_dtype="bf16", workspace=None, bits: int = 4, rows: Optional[np.ndarray] = None):
    """The CUDA path through the C ABI.  `rows`: bring back only these token rows (full-size cases: the arrays returned
    are then already row-sampled, see assert_parity's `sampled`)."""
    import torch
    import paper_2606_15652_b200 as mq
    if w is None:
        w = pack_from_oracle(case)
    A = to_device_act(case)
    odt = torch.bfloat16 if out_dtype == "bf16" else torch.float16
    ridx = None if rows is None else torch.from_numpy(np.asarray(rows, np.int64)).cuda()
    pick = (lambda t: t) if ridx is None else (lambda t: t.index_select(0, ridx))
    if bits == 8:
        q, sA = mq.mq_quantize_act8(A)
        Y, d0, d1 = mq.mq_gemm_a8(w, q, sA, case.M, out_dtype=odt, dbg=True, workspace=workspace)
    else:
        qA, sA = mq.mq_quantize_act(A)
        Y, d0, d1 = mq.mq_gemm(w, qA, sA, case.M, out_dtype=odt, dbg=True, workspace=workspace)
        q = mq.mq_unpack_act(qA, case.M, case.K)
    torch.cuda.synchronize()
    return dict(qa=pick(q).cpu().numpy(), sa=pick(sA).cpu().numpy(), acc0=pick(d0).cpu().numpy(), acc1=pick(d1).cpu().numpy(),
                Y=pick(Y).float().cpu().numpy().astype(np.float64), w=w, out_dtype=out_dtype, sampled=rows is not None)


def assert_parity(got: dict, want: dict, rows: Optional[np.ndarray] = None, what: str = ""):
    if got.get("sampled"):
        rows = None          # run_cuda(rows=...) already returned the sampled rows only
    g = {k: (v[rows] if rows is not None and isinstance(v, np.ndarray) else v) for k, v in got.items()}
    assert np.array_equal(g["sa"].view(np.uint32), want["sa"].view(np.uint32)), f"{what}: activation scales differ"
    assert np.array_equal(g["qa"], want["qa"]), f"{what}: activation ints differ"
    assert np.array_equal(g["acc0"].astype(np.int64), want["acc0"]), f"{what}: base accumulator not bit-exact"
    assert np.array_equal(g["acc1"].astype(np.int64), want["acc1"]), f"{what}: residual accumulator not bit-exact"
    err = np.abs(g["Y"] - want["Y"])
    tol = y_tolerance(want["Y"], want["mag"], got.get("out_dtype", "bf16"))
    assert (tol <= 2.0 ** -8 * np.abs(want["Y"]) + Y_MAG_TOL * want["mag"] + 1e-300).all()
    bad = err > tol
    assert not bad.any(), f"{what}: Y out of tolerance at {int(bad.sum())} of {bad.size} (max excess {float((err - tol).max()):.3e})"
