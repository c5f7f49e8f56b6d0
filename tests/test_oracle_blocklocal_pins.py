"""Pins for the block-local residual-scale oracle (oracle.decompose_blocklocal / scores_blocklocal /
algorithm1_blocklocal / forward_blocklocal; reading A4b; north_star "per-block scales"; Eq.1 P:77 applied to R
inside every block, Alg.1, Eq.4).  Each function is checked against something other than itself:
a hand-worked block, the degenerate partition that reduces to the per-channel reading A4, exact rational arithmetic,
brute-force loops with Python integers, and Theorem 4.1 by enumeration.  CPU only.
"""
from fractions import Fraction
from itertools import combinations

import numpy as np
import pytest

import oracle
import synth


def test_o4b_hand_worked_block():
    # tests/golden/o4b_hand_block.txt: a 2 x 4 residual with blocks of 2 columns, worked by hand:
    #   row 0: runs (0.7, -0.35) -> s = 0.1,  q = (7, -4) [3.5 -> 4: tie to even];  (0.0, 0.0) -> s = 1, q = (0, 0)   (A2)
    #   row 1: runs (-1.4, 0.3) -> s = 0.2, q = (-7, 2) [1.5 -> 2];                 (0.07, 0.07) -> s = 0.01, q = (7, 7)
    rows = [l.split() for l in open(__file__.replace("test_oracle_blocklocal_pins.py", "golden/o4b_hand_block.txt"))
            if l.strip() and not l.startswith("#")]
    R = np.array([[float(v) for v in r[:4]] for r in rows], np.float64)
    want_q = np.array([[int(v) for v in r[4:8]] for r in rows], np.int8)
    # exact binary scales: use dyadic multiples so that amax / 7 is exact in binary32
    R = R * np.array([[0.875 / 0.7]]).astype(np.float64)          # 0.7 -> 0.875 = 7 * 2^-3, 1.4 -> 1.75, 0.07 -> 0.0875
    W = np.zeros((2, 4), np.float32)
    runs = np.ascontiguousarray(R.astype(np.float32).reshape(4, 2))
    q = np.empty((4, 2), np.int8)
    s = np.empty(4, np.float32)
    import ctypes as C
    oracle.lib().orc_quantize_rows(runs.ctypes.data_as(C.c_void_p), C.c_int64(4), C.c_int64(2), q.ctypes.data_as(C.c_void_p),
                                   s.ctypes.data_as(C.c_void_p))
    assert q.reshape(2, 4).tolist() == want_q.tolist()
    assert s.tolist() == [0.125, 1.0, 0.25, np.float32(0.0875 / 7)]
    del W


def _case(seed=0, N=256, K=256, M=16):
    W = synth.gen_weight(seed, N, K)
    A = synth.gen_act(seed, M, K, n_outlier_ch=2)
    h = oracle.hessian_diag(A.astype(np.float32)).astype(np.float32)
    return W, A, h


def test_o4b_one_block_per_row_is_the_per_channel_reading():
    """bs = K = N: the only k-block of a row is the whole row, so s_rb == s_r and the codes, scores, selection and Y are
    those of the A4 path (oracle.decompose / algorithm1 / forward), bit for bit."""
    W, A, h = _case(3, 128, 128, 8)
    d4, db = oracle.decompose(W), oracle.decompose_blocklocal(W, 128)
    assert np.array_equal(db.qr, d4.qr) and np.array_equal(db.srb[:, 0].view(np.uint32), d4.sr.view(np.uint32))
    L4, Lb = oracle.algorithm1(W, h, 128, 1), oracle.algorithm1_blocklocal(W, h, 128, 1)
    assert np.allclose(Lb.sc.delta, L4.sc.delta, rtol=1e-12) and Lb.blk_n.tolist() == L4.blk_n.tolist()
    f4, fb = oracle.forward(A, L4), oracle.forward_blocklocal(A, Lb)
    assert np.array_equal(fb["acc0"], f4["acc0"]) and np.array_equal(fb["acc1sum"], f4["acc1"])
    assert np.allclose(fb["Y"], f4["Y"], rtol=1e-14, atol=0)


def test_o4b_runs_are_quantized_independently_and_bounds():
    W, A, h = _case(5)
    bs = 64
    d = oracle.decompose_blocklocal(W, bs)
    N, K = W.shape
    rng = np.random.default_rng(0)
    for _ in range(40):                                              # each run equals O1 on that run alone
        n, b = int(rng.integers(N)), int(rng.integers(K // bs))
        q, s = oracle.quantize_row(d.R[n, b * bs:(b + 1) * bs])
        assert np.array_equal(q, d.qr[n, b * bs:(b + 1) * bs]) and s == d.srb[n, b]
    srep = np.repeat(d.srb.astype(np.float64), bs, axis=1)
    err = np.abs(d.R.astype(np.float64) - srep * d.qr)
    assert (err <= srep / 2 * (1 + 2 ** -20)).all()                   # no clipping inside a block
    d4 = oracle.decompose(W)
    assert (d.srb <= d4.sr[:, None]).all() and (d.srb < d4.sr[:, None]).any()   # a block's absmax never exceeds its row's
    assert np.abs(d.qr).max() == 7


def test_o6b_scores_closed_form_identity_and_theorem_4_1():
    """delta_B >= 0 before clipping; L(S) = L(0) - sum_{B in S} delta_B with L evaluated directly from
    P:344 with the block-local codes; top-K minimises L over all subsets of size <= 2 (Theorem 4.1)."""
    W, A, h = _case(0)
    bs = 64
    L = oracle.algorithm1_blocklocal(W, h, bs, 2)
    d, sc = L.d, L.sc
    assert (sc.delta >= 0).all()
    h64 = h.astype(np.float64)
    E0 = d.R.astype(np.float64)
    Eq = E0 - np.repeat(d.srb.astype(np.float64), bs, axis=1) * d.qr
    nbk = W.shape[1] // bs

    def loss(blocks):
        E = E0.copy()
        for b in blocks:
            bn, bk = divmod(b, nbk)
            E[bn * bs:(bn + 1) * bs, bk * bs:(bk + 1) * bs] = Eq[bn * bs:(bn + 1) * bs, bk * bs:(bk + 1) * bs]
        return float((h64[None, :] * E * E).sum())
    L0 = loss([])
    nb = sc.delta.shape[0]
    for b in range(nb):
        assert abs((L0 - loss([b])) - sc.delta[b]) <= 1e-10 * L0
    best = min((loss(list(c)), c) for r in (1, 2) for c in combinations(range(nb), r))
    sel = sorted((L.blk_n * nbk + L.blk_k).tolist())
    assert sorted(best[1]) == sel
    # a closed-form block: constant residual r on a block with h = 1 -> s = r / 7, q = 7, reconstruction exact: delta = bs^2 r^2
    Wc = np.zeros((64, 64), np.float32)
    Wc[:] = 0.875                                                      # s_w = 0.125, q_w = 7, R = 0 ...
    Wc[0, 0] = 0.875 + 0.0625                                          # ... except one entry: s_w = (0.9375)/7, R != 0
    dc = oracle.decompose_blocklocal(Wc, 64)
    scc = oracle.scores_blocklocal(dc, np.ones(64, np.float32), 64)
    Rc = dc.R.astype(np.float64)
    Ec = Rc - np.repeat(dc.srb.astype(np.float64), 64, axis=1) * dc.qr
    assert abs(scc.delta[0] - ((Rc ** 2).sum() - (Ec ** 2).sum())) <= 1e-18


def test_o8b_o9b_brute_force_exact_rationals():
    """Y by brute force: Python integers for the block sums, exact rationals for the scaled sum; plus budget 0 (dense
    W4A4) and linearity of the sparse term over disjoint block sets."""
    N, K, M, bs = 128, 256, 3, 64
    W, A, h = _case(7, N, K, M)
    L = oracle.algorithm1_blocklocal(W, h, bs, 3)
    assert L.nnz == 3
    f = oracle.forward_blocklocal(A, L)
    qa, sa = oracle.quantize_act(A)
    sel = set(zip(L.blk_n.tolist(), L.blk_k.tolist()))
    rng = np.random.default_rng(1)
    cols = sorted(set(rng.integers(0, N, size=6).tolist()) | {int(L.blk_n[0]) * bs + 1})
    for m in range(M):
        for n in cols:
            a0 = sum(int(qa[m, k]) * int(L.d.qw[n, k]) for k in range(K))
            assert a0 == f["acc0"][m, n]
            y = Fraction(float(L.d.sw[n])) * a0
            a1sum = 0
            for bk in range(K // bs):
                if (n // bs, bk) in sel:
                    aB = sum(int(qa[m, k]) * int(L.d.qr[n, k]) for k in range(bk * bs, (bk + 1) * bs))
                    a1sum += aB
                    y += Fraction(float(L.d.srb[n, bk])) * aB
            y *= Fraction(float(sa[m]))
            assert a1sum == f["acc1sum"][m, n]
            assert abs(Fraction(f["Y"][m, n]) - y) <= abs(y) * Fraction(1, 10 ** 13) + Fraction(1, 10 ** 300)
    L0 = oracle.PackedLayerBlockLocal(N, K, bs, L.d, None, L.blk_n[:0], L.blk_k[:0])
    f0 = oracle.forward_blocklocal(A, L0)
    dense = sa.astype(np.float64)[:, None] * (L.d.sw.astype(np.float64)[None, :] * f0["acc0"])
    assert not f0["acc1sum"].any() and np.array_equal(f0["Y"], dense)
    La = oracle.PackedLayerBlockLocal(N, K, bs, L.d, None, L.blk_n[:1], L.blk_k[:1])
    Lb = oracle.PackedLayerBlockLocal(N, K, bs, L.d, None, L.blk_n[1:], L.blk_k[1:])
    fa, fb = oracle.forward_blocklocal(A, La), oracle.forward_blocklocal(A, Lb)
    assert np.array_equal(fa["acc1sum"] + fb["acc1sum"], f["acc1sum"])
    assert np.allclose((fa["Y"] - f0["Y"]) + (fb["Y"] - f0["Y"]), f["Y"] - f0["Y"], rtol=1e-9, atol=1e-12)


def test_block_local_scales_never_lose_to_per_channel_scales():
    """With every block selected the two-level reconstruction error of the block-local reading is <= the per-channel
    one's bound s_r / 2 everywhere, and strictly smaller in total (the finer scale is why north_star asks for it)."""
    W, A, h = _case(9)
    bs = 64
    db, d4 = oracle.decompose_blocklocal(W, bs), oracle.decompose(W)
    Eb = np.abs(db.R.astype(np.float64) - np.repeat(db.srb.astype(np.float64), bs, axis=1) * db.qr)
    E4 = np.abs(d4.R.astype(np.float64) - d4.sr.astype(np.float64)[:, None] * d4.qr)
    assert (Eb <= d4.sr.astype(np.float64)[:, None] / 2 * (1 + 2 ** -20)).all()
    assert (Eb ** 2).sum() < (E4 ** 2).sum()
