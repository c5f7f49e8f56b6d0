"""Pins for the per-group oracle (oracle.quantize_act_group / oracle.forward_group, PAPER.md line 441:
per-group activation quantization in the 4-bit setting).  CPU only.  Each check is against something other than the
functions themselves: a hand-worked vector, the already pinned per-token path in the case where the two coincide, a
dequantize-then-multiply brute force in exact rational arithmetic, and scaling invariants."""
from fractions import Fraction
import os

import numpy as np

import oracle
import synth

HERE = os.path.dirname(os.path.abspath(__file__))


def _layer(seed, N, K, bs, budget):
    W = synth.gen_weight(seed, N, K)
    return oracle.algorithm1(W, None, bs, budget)


def test_o2g_hand_vector():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "o2g_hand_vector_group.txt"))
            if l.strip() and not l.startswith("#")]
    x = np.array([float(r[1]) for r in rows], np.float16)[None, :]
    assert np.array_equal(x.astype(np.float64), np.array([[float(r[1]) for r in rows]]))   # exact in fp16
    qa, sa = oracle.quantize_act_group(x, 4)
    assert qa.shape == (1, 12) and sa.shape == (1, 3)
    assert qa[0].tolist() == [int(r[2]) for r in rows]
    assert sa[0].tolist() == [float(rows[4 * g][3]) for g in range(3)]


def test_o2g_one_group_is_per_token_and_groups_are_independent():
    A = synth.gen_act(5, 6, 256)
    q1, s1 = oracle.quantize_act(A)
    qg, sg = oracle.quantize_act_group(A, 256)
    assert np.array_equal(q1, qg) and np.array_equal(s1, sg[:, 0])
    # a group's codes and scale depend only on that group's values: quantizing the slice alone gives the same
    qg, sg = oracle.quantize_act_group(A, 64)
    for g in range(4):
        for m in range(6):
            q, s = oracle.quantize_row(A[m, 64 * g:64 * g + 64].astype(np.float32))
            assert np.array_equal(q, qg[m, 64 * g:64 * g + 64]) and s == sg[m, g]
    # every group reaches +-7 at its absmax and |a - s q| <= s / 2 inside the group
    a = A.astype(np.float64).reshape(6, 4, 64)
    assert (np.abs(qg.reshape(6, 4, 64)).max(axis=2) == 7).all()
    assert (np.abs(a - sg[:, :, None].astype(np.float64) * qg.reshape(6, 4, 64)) <= sg[:, :, None] / 2 * (1 + 2 ** -20)).all()
    # scaling ONE group by a power of two moves only that group's scale
    B = A.copy()
    B[:, 64:128] = np.ldexp(A[:, 64:128].astype(np.float32), -3).astype(np.float16)
    qb, sb = oracle.quantize_act_group(B, 64)
    assert np.array_equal(qb, qg)
    assert np.array_equal(sb[:, [0, 2, 3]], sg[:, [0, 2, 3]]) and np.array_equal(sb[:, 1] * 8, sg[:, 1])


def test_forward_group_with_one_group_equals_per_token_forward():
    L = _layer(11, 128, 256, 64, 3)
    A = synth.gen_act(11, 5, 256)
    want = oracle.forward(A, L)          # pinned in test_oracle_pins.py
    got = oracle.forward_group(A, L, 256)
    assert np.array_equal(got["acc0"], want["acc0"]) and np.array_equal(got["acc1"], want["acc1"])
    assert np.allclose(got["Y"], want["Y"], rtol=1e-14, atol=0)
    assert np.array_equal(got["acc0_g"][0], want["acc0"])


def test_forward_group_is_the_two_level_dequantized_product_brute_force():
    # Y[m,n] = sum_k (s_a[m, k // g] q_a[m,k]) * (s_w[n] q_w[n,k] + s_r[n] (M.q_r)[n,k]) -- dequantize first, multiply
    # after, in exact rationals, element by element (Eq.2 P:82 and Eq.4 P:106 with a K-varying activation scale).
    N, K, bs, g = 128, 128, 64, 32
    L = _layer(12, N, K, bs, 2)
    assert L.nnz == 2
    A = synth.gen_act(12, 3, K)
    out = oracle.forward_group(A, L, g)
    qa, sa = out["qa"], out["sa"]
    sel = {(int(bn), int(bk)) for bn, bk in zip(L.blk_n, L.blk_k)}
    rng = np.random.default_rng(0)
    for m in range(3):
        for n in rng.choice(N, 12, replace=False):
            y = Fraction(0)
            for k in range(K):
                a = Fraction(float(sa[m, k // g])) * int(qa[m, k])
                w = Fraction(float(L.d.sw[n])) * int(L.d.qw[n, k])
                if (n // bs, k // bs) in sel:
                    w += Fraction(float(L.d.sr[n])) * int(L.d.qr[n, k])
                y += a * w
            assert abs(float(y) - out["Y"][m, n]) <= 1e-12 * out["mag"][m, n] + 1e-300
    # integer accumulators: per-group sums add up to the whole-K integer GEMM of the same codes (O8, pinned)
    acc0, acc1 = oracle.gemm(qa, L.d.qw, L.d.qr, bs, L.blk_n, L.blk_k)
    assert np.array_equal(out["acc0"], acc0) and np.array_equal(out["acc1"], acc1)


def test_forward_group_budget_zero_and_group_scale_linearity():
    N, K, g = 128, 256, 128
    L0 = _layer(13, N, K, 64, 0)
    A = synth.gen_act(13, 4, K)
    out = oracle.forward_group(A, L0, g)
    assert not out["acc1_g"].any()
    # doubling the inputs of group 1 doubles exactly that group's contribution to Y
    B = A.copy()
    B[:, g:] = (A[:, g:].astype(np.float32) * 2).astype(np.float16)
    out2 = oracle.forward_group(B, L0, g)
    sw = L0.d.sw.astype(np.float64)[None, :]
    c1 = out["sa"][:, 1].astype(np.float64)[:, None] * (sw * out["acc0_g"][1])
    assert np.allclose(out2["Y"] - out["Y"], c1, rtol=1e-12, atol=1e-12 * np.abs(out["mag"]).max())
    # cols / rows restriction is a plain slice of the full result
    cols, rows = np.array([3, 77, 120]), np.array([2, 0])
    sub = oracle.forward_group(A, L0, g, cols=cols, rows=rows)
    assert np.array_equal(sub["Y"], out["Y"][np.ix_(rows, cols)])
