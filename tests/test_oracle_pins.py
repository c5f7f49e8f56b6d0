"""Pins for the CPU oracle (oracle/mq_oracle.cpp): each O-step is checked against something
other than itself -- closed forms, exact rational arithmetic, brute force, library routines,
and the invariants PAPER.md states (citations "P:<line>").  CPU only.

A plausible mistake (dropped term, wrong sign/index, transposed operand, wrong tie rule)
fails at least one test here.
"""
from fractions import Fraction
from itertools import combinations

import numpy as np
import pytest

import oracle
import synth


# ----------------------------------------------------------------------------- O1 quantizer
def test_o1_hand_vector_rne():
    # golden: tests/golden/o1_hand_vector.txt (Eq.1 P:77 with q_max=7, RNE; readings A1, A3)
    rows = [l.split() for l in open(__file__.replace("test_oracle_pins.py", "golden/o1_hand_vector.txt"))
            if l.strip() and not l.startswith("#")]
    x = np.array([float(r[0]) for r in rows], np.float32)
    want = np.array([int(r[1]) for r in rows], np.int8)
    q, s = oracle.quantize_row(x)
    assert s == np.float32(1.0)
    assert q.tolist() == want.tolist()


def test_o1_scale_is_correctly_rounded_quotient_and_q_is_nearest():
    rng = np.random.default_rng(1)
    for trial in range(20):
        x = (rng.standard_normal(257) * 10 ** rng.uniform(-3, 3)).astype(np.float32)
        q, s = oracle.quantize_row(x)
        amax = Fraction(float(np.abs(x).max()))
        exact = amax / 7
        # s is the binary32 nearest to amax/7 (Eq.1: s = max|X|/q_max): neither neighbour is closer
        sf = Fraction(float(s))
        lo = Fraction(float(np.nextafter(s, np.float32(0))))
        hi = Fraction(float(np.nextafter(s, np.float32(np.inf))))
        assert abs(sf - exact) <= abs(lo - exact) and abs(sf - exact) <= abs(hi - exact)
        # q = round(x/s): within half a step (+1 ulp of the binary32 quotient, reading A3)
        for xi, qi in zip(x, q):
            t = Fraction(float(xi)) / sf
            assert abs(t - int(qi)) <= Fraction(1, 2) + abs(t) * Fraction(1, 2 ** 23)
        i = int(np.abs(x).argmax())
        assert abs(int(q[i])) == 7 and np.sign(q[i]) == np.sign(x[i])
        assert np.abs(q).max() <= 7
        # |x - s q| <= s/2 (no clipping under absmax scaling)
        assert np.all(np.abs(x.astype(np.float64) - float(s) * q) <= float(s) / 2 * (1 + 2 ** -20))


def test_o1_symmetry_pow2_zero_requant():
    rng = np.random.default_rng(2)
    x = rng.standard_normal(300).astype(np.float32)
    q, s = oracle.quantize_row(x)
    qn, sn = oracle.quantize_row(-x)
    assert sn == s and np.array_equal(qn, -q)
    for e in (-9, 3, 20):
        q2, s2 = oracle.quantize_row(np.ldexp(x, e).astype(np.float32))
        assert np.array_equal(q2, q) and s2 == np.float32(np.ldexp(np.float64(s), e))
    qz, sz = oracle.quantize_row(np.zeros(17, np.float32))
    assert sz == np.float32(1.0) and not qz.any()
    # re-quantizing the dequantized row returns the same integers (max|q| = 7)
    q3, _ = oracle.quantize_row((np.float64(s) * q).astype(np.float32))
    assert np.array_equal(q3, q)


def test_o1_ties_on_fp16_grid_round_half_even():
    # amax = 7 * 2^-3 -> s = 2^-3 exactly; x = (n + 1/2) * 2^-3 are exact fp16 ties
    n = np.arange(-6, 7)
    x = np.concatenate([[7 / 8], (n + 0.5) / 8]).astype(np.float16).astype(np.float32)
    q, s = oracle.quantize_row(x)
    assert s == np.float32(0.125)
    want = [7] + [int(2 * round((k + 0.5) / 2)) for k in n]  # python round = half-even on exact halves
    assert q.tolist() == want


# ---- O1's per-element quotient, pinned in exact rational arithmetic (Eq.1, reading A3) --------------
def _rne_int(t: Fraction) -> int:
    """Round a rational to the nearest integer, halves to even."""
    f = t.numerator // t.denominator
    r = t - f
    if r > Fraction(1, 2) or (r == Fraction(1, 2) and f % 2 == 1):
        f += 1
    return f


def _round_to_binary32(t: Fraction) -> Fraction:
    """The IEEE-754 binary32 value nearest to the rational t (ties to even), as an exact rational.
    Written out by hand: scale to a 24-bit integer significand, round half to even, scale back."""
    if t == 0:
        return Fraction(0)
    sign, a = (-1 if t < 0 else 1), abs(t)
    e = a.numerator.bit_length() - a.denominator.bit_length()      # 2^(e-1) < a < 2^(e+1)
    if Fraction(2) ** e > a:
        e -= 1                                                      # now 2^e <= a < 2^(e+1)
    e = max(e, -126)                                                # subnormals share the exponent -126
    ulp = Fraction(2) ** (e - 23)
    m = _rne_int(a / ulp)                                           # 2^23 <= m <= 2^24 (or < 2^23: subnormal)
    assert e + 1 <= 127
    return sign * m * ulp


def _expected_code(x: float, s: float, qmax: int) -> int:
    """Eq.1 as reading A3 fixes it: q = clamp(RNE(fl32(x / s)))."""
    t32 = _round_to_binary32(Fraction(x) / Fraction(s))
    return max(-qmax, min(qmax, _rne_int(t32)))


def _code_with_reciprocal(x: float, s: float, qmax: int) -> int:
    """What `x * (1.0f / s)` would give (the mutation this pin must catch): two roundings."""
    r32 = _round_to_binary32(Fraction(1) / Fraction(s))
    t32 = _round_to_binary32(Fraction(x) * r32)
    return max(-qmax, min(qmax, _rne_int(t32)))


@pytest.mark.parametrize("bits", [4, 8])
def test_o1_quotient_is_one_correctly_rounded_binary32_division(bits):
    """Reading A3 of Eq.1: x / s is ONE IEEE binary32 division, then round half to even.  Rows are
    built next to the ties (k + 1/2) * s for scales that are not powers of two, where a product with the
    reciprocal of s lands on the other side of the tie; the expected codes come from exact rationals with
    the binary32 rounding written out by hand (no floating-point division anywhere on the expected side).
    The test also counts the elements on which `x * (1.0f / s)` would differ: the pin is only a pin if
    that count is positive."""
    qmax = 7 if bits == 4 else 127
    rng = np.random.default_rng(40 + bits)
    flips = 0
    for amax in [5.0, 0.3, 1234.0, 2.2, 6.0e-5, 3.3, 0.0417, 97.0]:
        amax32 = np.float32(amax)
        s = float(_round_to_binary32(Fraction(float(amax32)) / qmax))          # the scale, by hand as well
        ks = rng.integers(-qmax, qmax, size=96)
        xs = [float(amax32)]
        for k in ks:
            centre = np.float32(float(_round_to_binary32((Fraction(int(k)) + Fraction(1, 2)) * Fraction(s))))
            v = centre
            for _ in range(3):                                                  # fp32 neighbours on both sides
                v = np.nextafter(v, np.float32(-np.inf))
            for _ in range(7):
                if abs(float(v)) <= float(amax32):
                    xs.append(float(v))
                v = np.nextafter(v, np.float32(np.inf))
        x = np.array(xs, np.float32)
        q, s_got = oracle.quantize_row(x, bits=bits)
        assert float(s_got) == s
        want = [_expected_code(float(v), s, qmax) for v in x]
        assert q.tolist() == want, f"amax {amax}: codes differ from the exactly rounded quotient"
        flips += sum(1 for v, w in zip(x, want) if _code_with_reciprocal(float(v), s, qmax) != w)
    assert flips > 0, "the rows no longer discriminate a division from a reciprocal product"


@pytest.mark.parametrize("dt", ["f16", "bf16"])
def test_o2_near_ties_on_16bit_grids_match_exact_rationals(dt):
    """The same pin through O2 (per-token activations) on 16-bit inputs: the fp16 / bf16 neighbours
    of (k + 1/2) * s for non-power-of-two scales, expected codes from exact rationals."""
    rng = np.random.default_rng(44)
    K, rows = 256, []
    for amax in [5.0, 0.3, 1234.0, 2.2, 3.3, 97.0]:
        if dt == "f16":
            a16 = float(np.float16(amax))
        else:
            a16 = float((np.array([amax], np.float32).view(np.uint32) & 0xFFFF0000).view(np.float32)[0])
        s = float(_round_to_binary32(Fraction(a16) / 7))
        x = (rng.integers(-7, 7, size=K).astype(np.float64) + 0.5) * s
        if dt == "f16":
            nb = x.astype(np.float16).view(np.int16) + rng.integers(-2, 3, size=K).astype(np.int16)
            row = nb.view(np.float16).copy()
            row[0] = np.float16(a16)
            row = np.where(np.abs(row.astype(np.float32)) <= a16, row, np.float16(0)).view(np.uint16)
            vals = row.view(np.float16).astype(np.float64)
        else:
            b = (x.astype(np.float32).view(np.uint32) >> 16).astype(np.uint16) + rng.integers(0, 3, size=K).astype(np.uint16)
            b[0] = np.uint16(np.array([a16], np.float32).view(np.uint32)[0] >> 16)
            f = (b.astype(np.uint32) << 16).view(np.float32)
            row = np.where(np.abs(f) <= a16, b, np.uint16(0)).astype(np.uint16)
            vals = (row.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
        rows.append((row, vals, s))
    bits16 = np.stack([r[0] for r in rows])
    qa, sa = oracle.quantize_act(bits16.view(np.float16) if dt == "f16" else (bits16, "bf16"))
    for i, (_, vals, s) in enumerate(rows):
        assert float(sa[i]) == s
        assert qa[i].tolist() == [_expected_code(float(v), s, 7) for v in vals]


def test_o1_8bit_activations_w4a8():
    """The W4A8 variant (Table 1 W4A8 rows): the same quantizer with q_max = 127.  Hand vector
    (tests/golden/o1_hand_vector_8bit.txt), correctly rounded scale, nearest code, no clipping, symmetry,
    power-of-two scaling, exact ties, and the per-token activation path on 16-bit inputs."""
    rows = [l.split() for l in open(__file__.replace("test_oracle_pins.py", "golden/o1_hand_vector_8bit.txt"))
            if l.strip() and not l.startswith("#")]
    x = np.array([float(r[0]) for r in rows], np.float32)
    q, s = oracle.quantize_row(x, bits=8)
    assert s == np.float32(1.0) and q.tolist() == [int(r[1]) for r in rows]
    rng = np.random.default_rng(8)
    for trial in range(10):
        x = (rng.standard_normal(300) * 10 ** rng.uniform(-3, 3)).astype(np.float32)
        q, s = oracle.quantize_row(x, bits=8)
        exact = Fraction(float(np.abs(x).max())) / 127
        sf = Fraction(float(s))
        lo = Fraction(float(np.nextafter(s, np.float32(0))))
        hi = Fraction(float(np.nextafter(s, np.float32(np.inf))))
        assert abs(sf - exact) <= abs(lo - exact) and abs(sf - exact) <= abs(hi - exact)
        for xi, qi in zip(x, q):
            t = Fraction(float(xi)) / sf
            assert abs(t - int(qi)) <= Fraction(1, 2) + abs(t) * Fraction(1, 2 ** 23)
        i = int(np.abs(x).argmax())
        assert abs(int(q[i])) == 127 and np.sign(q[i]) == np.sign(x[i]) and np.abs(q.astype(np.int32)).max() <= 127
        assert np.all(np.abs(x.astype(np.float64) - float(s) * q) <= float(s) / 2 * (1 + 2 ** -20))
        qn, sn = oracle.quantize_row(-x, bits=8)
        assert sn == s and np.array_equal(qn, -q)
        q2, s2 = oracle.quantize_row(np.ldexp(x, 5).astype(np.float32), bits=8)
        assert np.array_equal(q2, q) and s2 == np.float32(np.ldexp(np.float64(s), 5))
    # exact ties on the fp16 grid: amax = 127 * 2^-4 -> s = 2^-4; x = (n + 1/2) * 2^-4
    n = np.arange(-126, 127, 7)
    x = np.concatenate([[127 / 16], (n + 0.5) / 16]).astype(np.float16).astype(np.float32)
    q, s = oracle.quantize_row(x, bits=8)
    assert s == np.float32(1 / 16) and q.tolist() == [127] + [int(2 * round((k + 0.5) / 2)) for k in n]
    # O2 at 8 bits: per token, row by row equal to O1 on the exactly converted fp16 row
    A = (rng.standard_normal((5, 64)) * 3).astype(np.float16)
    qa, sa = oracle.quantize_act(A, bits=8)
    for m in range(5):
        qr, sr = oracle.quantize_row(A[m].astype(np.float32), bits=8)
        assert np.array_equal(qa[m], qr) and sa[m] == sr
    qz, sz = oracle.quantize_row(np.zeros(9, np.float32), bits=8)
    assert sz == np.float32(1.0) and not qz.any()


def test_o2_fp16_bf16_conversion_exact_and_per_token():
    rng = np.random.default_rng(3)
    A = (rng.standard_normal((9, 128)) * 3).astype(np.float16)
    A[4] = 0
    A[5, 7] = np.float16(6e-8)  # subnormal fp16
    qa, sa = oracle.quantize_act(A)
    for m in range(A.shape[0]):
        q, s = oracle.quantize_row(A[m].astype(np.float32))  # numpy's fp16->fp32 is the library conversion
        assert np.array_equal(q, qa[m]) and s == sa[m]
    # bf16: bits << 16 is the definition of the format
    f = (rng.standard_normal((5, 64)) * 2).astype(np.float32)
    bits = (f.view(np.uint32) >> 16).astype(np.uint16)
    fb = (bits.astype(np.uint32) << 16).view(np.float32)
    qb, sb = oracle.quantize_act((bits, "bf16"))
    for m in range(5):
        q, s = oracle.quantize_row(fb[m])
        assert np.array_equal(q, qb[m]) and s == sb[m]


# ----------------------------------------------------------------------- O3/O4 decomposition
def test_o3_o4_bounds_and_exact_residual(tiny_case):
    W, L = tiny_case["W"], tiny_case["L"]
    d = L.d
    sw, sr = d.sw.astype(np.float64), d.sr.astype(np.float64)
    assert np.all(np.abs(d.R) <= (sw / 2 * (1 + 2 ** -22))[:, None])
    assert np.all(sr <= sw / 14 * (1 + 1e-6))
    rec = sw[:, None] * d.qw + sr[:, None] * d.qr
    assert np.all(np.abs(W.astype(np.float64) - rec) <= (sr / 2 * (1 + 1e-5))[:, None] + 1e-12)
    # R = fl32(W - s_w q_w) with the difference exact in rationals (Alg.1 line 1)
    rng = np.random.default_rng(0)
    for n, k in zip(rng.integers(0, 256, 64), rng.integers(0, 256, 64)):
        exact = Fraction(float(W[n, k])) - Fraction(float(d.sw[n])) * int(d.qw[n, k])
        assert Fraction(float(d.R[n, k])) == Fraction(float(np.float32(float(exact))))
    # per-channel: row n of qw only depends on row n of W
    d2 = oracle.decompose(W[10:20])
    assert np.array_equal(d2.qw, d.qw[10:20]) and np.array_equal(d2.sr, d.sr[10:20])


# ------------------------------------------------------------------------------ O5 h_j
def test_o5_closed_forms():
    X = np.full((8, 5), 3.0, np.float32)
    assert np.allclose(oracle.hessian_diag(X), 2 * 9.0, rtol=0, atol=0)  # h = (2/N) * N * c^2
    X = np.zeros((4, 4), np.float32)
    X[2, 1] = 5.0
    assert oracle.hessian_diag(X).tolist() == [0.0, 2 / 4 * 25.0, 0.0, 0.0]
    rng = np.random.default_rng(5)
    X = rng.standard_normal((33, 17)).astype(np.float32)
    want = 2.0 / 33 * (X.astype(np.float64) ** 2).sum(0)   # column index j = input channel (A9)
    assert np.allclose(oracle.hessian_diag(X), want, rtol=1e-13)


# --------------------------------------------------------------------------- O6 scores
def test_o6_closed_form_block():
    # handmade inputs: R = 1 on block (0,1), Q(R) = (1/8)*7 there -> A = sum h, B = sum h / 64
    N, K, bs = 8, 12, 4
    R = np.zeros((N, K), np.float32)
    qr = np.zeros((N, K), np.int8)
    R[0:4, 4:8] = 1.0
    qr[0:4, 4:8] = 7
    sr = np.full(N, 0.125, np.float32)
    h = np.arange(1, K + 1, dtype=np.float32)
    d = oracle.Decomp(None, None, R, qr, sr)
    sc = oracle.scores(d, h, bs)
    hs = float(h[4:8].sum()) * 4
    want_A = np.zeros(6)
    want_A[1] = hs
    assert np.array_equal(sc.A_B, want_A)
    assert sc.B_B[1] == hs / 64 and sc.delta[1] == hs - hs / 64 and sc.S[1] == sc.delta[1]
    assert not sc.S[[0, 2, 3, 4, 5]].any()
    # the [.]_+ guard: a candidate that makes things worse gets S = 0, delta < 0
    qr[4:8, 0:4] = 7  # R = 0 there, Q(R) = 7/8
    sc = oracle.scores(oracle.Decomp(None, None, R, qr, sr), h, bs)
    assert sc.delta[3] < 0 and sc.S[3] == 0.0


def _surrogate(R, QR, h, mask_blocks, bs):
    """L~(S) = sum_ij h_j (R_ij - (M_S o Q(R))_ij)^2, evaluated directly."""
    M = np.zeros_like(R)
    nbk = R.shape[1] // bs
    for b in mask_blocks:
        bn, bk = divmod(int(b), nbk)
        M[bn * bs:(bn + 1) * bs, bk * bs:(bk + 1) * bs] = 1.0
    E = R - M * QR
    return float((h[None, :] * E * E).sum())


def test_o6_delta_nonnegative_and_identity(tiny_case):
    L, h = tiny_case["L"], tiny_case["h"].astype(np.float64)
    d, sc = L.d, L.sc
    assert np.all(sc.delta >= 0)             # implied by round-to-nearest with unclipped scale
    assert np.array_equal(sc.S, sc.delta)    # so [.]_+ is a no-op
    R = d.R.astype(np.float64)
    QR = d.sr.astype(np.float64)[:, None] * d.qr
    L0 = _surrogate(R, QR, h, [], 64)
    assert np.isclose(L0, sc.A_B.sum(), rtol=1e-12)
    rng = np.random.default_rng(7)
    for _ in range(10):
        S = rng.choice(16, size=rng.integers(1, 16), replace=False)
        assert np.isclose(_surrogate(R, QR, h, S, 64), L0 - sc.delta[S].sum(), rtol=1e-12)


# ------------------------------------------------------------------------ O7 selection
def test_o7_theorem_4_1_brute_force(tiny_case):
    L, h = tiny_case["L"], tiny_case["h"].astype(np.float64)
    R = L.d.R.astype(np.float64)
    QR = L.d.sr.astype(np.float64)[:, None] * L.d.qr
    best, best_S = None, None
    for r in (0, 1, 2):
        for S in combinations(range(16), r):
            v = _surrogate(R, QR, h, S, 64)
            if best is None or v < best:
                best, best_S = v, S
    got = sorted((L.blk_n.astype(int) * 4 + L.blk_k).tolist())
    assert sorted(best_S) == got and len(got) == 2      # Theorem 4.1


def test_o7_ties_zero_scores_budget():
    S = np.array([0.0, 3.0, 5.0, 3.0, 0.0, 5.0, 1.0])
    assert oracle.select(S, 3).tolist() == [2, 5, 1]         # ties -> lower index (A7)
    assert oracle.select(S, 4).tolist() == [2, 5, 1, 3]
    assert oracle.select(S, 100).tolist() == [2, 5, 1, 3, 6]  # zero-score blocks omitted
    assert oracle.select(S, 0).tolist() == []
    assert oracle.select(np.zeros(4), 2).tolist() == []


def test_o7_zero_sensitivity_columns_never_selected(tiny_case):
    W = tiny_case["W"]
    h = np.ones(256, np.float32)
    h[64:256] = 0.0                              # only block-column 0 matters
    L = oracle.algorithm1(W, h, 64, 8)
    assert L.nnz == 4 and set(L.blk_k.tolist()) == {0}     # nnz < budget


def test_o7_offdiag_zero_matches_exact_output_distortion(tiny_case):
    # O = 0: orthogonal calibration columns -> L(S) = (2/N)||X E_S^T||_F^2 equals L~(S)
    L = tiny_case["L"]
    K = 256
    c = np.linspace(0.5, 2.0, K)
    X = np.diag(c).astype(np.float32)            # N_cal = K tokens, mutually orthogonal columns
    h = oracle.hessian_diag(X)
    R = L.d.R.astype(np.float64)
    QR = L.d.sr.astype(np.float64)[:, None] * L.d.qr
    for S in ([], [3], [0, 9], [5, 6, 15]):
        Mk = np.zeros_like(R)
        for b in S:
            bn, bk = divmod(b, 4)
            Mk[bn * 64:(bn + 1) * 64, bk * 64:(bk + 1) * 64] = 1
        E = R - Mk * QR
        exact = 2.0 / K * np.linalg.norm(X.astype(np.float64) @ E.T, "fro") ** 2
        assert np.isclose(exact, _surrogate(R, QR, h, S, 64), rtol=1e-10)


# ------------------------------------------------------------------------------ O8 GEMM
def test_o8_brute_force_python_ints():
    rng = np.random.default_rng(11)
    M, K, N, bs = 3, 16, 8, 4
    qa = rng.integers(-7, 8, (M, K)).astype(np.int8)
    qw = rng.integers(-7, 8, (N, K)).astype(np.int8)
    qr = rng.integers(-7, 8, (N, K)).astype(np.int8)
    blk_n = np.array([0, 1, 1], np.int32)
    blk_k = np.array([2, 0, 3], np.int32)
    a0, a1 = oracle.gemm(qa, qw, qr, bs, blk_n, blk_k)
    for m in range(M):
        for n in range(N):
            w0 = sum(int(qa[m, k]) * int(qw[n, k]) for k in range(K))
            w1 = 0
            for bn, bk in zip(blk_n, blk_k):
                if bn * bs <= n < (bn + 1) * bs:
                    w1 += sum(int(qa[m, k]) * int(qr[n, k]) for k in range(bk * bs, (bk + 1) * bs))
            assert a0[m, n] == w0 and a1[m, n] == w1


def test_o8_library_matmul_budget0_linearity_extremes(tiny_case):
    L, A = tiny_case["L"], tiny_case["A"]
    qa, sa = oracle.quantize_act(A)
    d = L.d
    a0, a1 = oracle.gemm(qa, d.qw, d.qr, 64, L.blk_n, L.blk_k)
    assert np.array_equal(a0, qa.astype(np.int64) @ d.qw.astype(np.int64).T)
    Mk = np.zeros((256, 256), np.int64)
    for bn, bk in zip(L.blk_n, L.blk_k):
        Mk[bn * 64:(bn + 1) * 64, bk * 64:(bk + 1) * 64] = 1
    assert np.array_equal(a1, qa.astype(np.int64) @ (Mk * d.qr).T)
    e = np.zeros(0, np.int32)
    b0, b1 = oracle.gemm(qa, d.qw, d.qr, 64, e, e)
    assert np.array_equal(b0, a0) and not b1.any()          # budget 0 == dense-only W4A4
    # linearity over disjoint block sets
    s1 = oracle.gemm(qa, d.qw, d.qr, 64, L.blk_n[:1], L.blk_k[:1])[1]
    s2 = oracle.gemm(qa, d.qw, d.qr, 64, L.blk_n[1:], L.blk_k[1:])[1]
    assert np.array_equal(s1 + s2, a1)
    # extremes: all +-7 -> |acc0| = 49 K exactly
    K = 512
    p = np.full((2, K), 7, np.int8)
    p[1] = -7
    w = np.full((3, K), 7, np.int8)
    x0, _ = oracle.gemm(p, w, w, 64, e, e)
    assert x0.tolist() == [[49 * K] * 3, [-49 * K] * 3]


def test_o8_o9_all_blocks_equals_two_level_dequantized_weight(tiny_case):
    W, A, h = tiny_case["W"], tiny_case["A"], tiny_case["h"]
    L = oracle.algorithm1(W, None, 64, 16)
    assert L.nnz == 16
    r = oracle.forward(A, L)
    d = L.d
    Wmq = d.sw.astype(np.float64)[:, None] * d.qw + d.sr.astype(np.float64)[:, None] * d.qr   # W_MQ, Alg.1 last line
    Aq = r["sa"].astype(np.float64)[:, None] * r["qa"]
    want = Aq @ Wmq.T
    assert np.allclose(r["Y"], want, rtol=1e-12, atol=1e-14)


def test_o9_closed_form_and_monotone_in_budget(tiny_case):
    Y, mag = oracle.output(np.array([[3, -2]], np.int64), np.array([[5, 0]], np.int64), np.array([0.5], np.float32),
                           np.array([2.0, 4.0], np.float32), np.array([0.25, 1.0], np.float32), want_mag=True)
    assert Y.tolist() == [[0.5 * (6 + 1.25), 0.5 * (-8.0)]] and mag.tolist() == [[0.5 * 7.25, 4.0]]
    # Eq.5/Eq.6 sanity: with the same Q(X), more residual blocks -> smaller output error
    W, A, h = tiny_case["W"], tiny_case["A"], tiny_case["h"]
    qa, sa = oracle.quantize_act(A)
    Aq = sa.astype(np.float64)[:, None] * qa
    ref = Aq @ W.astype(np.float64).T
    errs = []
    for budget in (0, 2, 8, 16):
        L = oracle.algorithm1(W, h, 64, budget)
        errs.append(np.linalg.norm(oracle.forward(A, L)["Y"] - ref))
    assert errs[0] > errs[1] > errs[2] > errs[3] > 0


def test_round_to_bf16_matches_torch():
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(13)
    y = np.concatenate([rng.standard_normal(4000) * 10 ** rng.uniform(-6, 6, 4000), [0.0, 1.0, 1.00390625, -3.0]])
    y32 = y.astype(np.float32).astype(np.float64)   # values exactly representable in fp32: one rounding either way
    want = torch.from_numpy(y32).to(torch.float32).to(torch.bfloat16).to(torch.float64).numpy()
    assert np.array_equal(oracle.round_to_bf16(y32), want)


def test_golden_config1_digest(tiny_case):
    """Drift guard: digests written by tests/golden/make_golden.py (which calls only oracle/ and synth/)."""
    import hashlib
    import json
    import os
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "config1_digest.json")))
    L, A = tiny_case["L"], tiny_case["A"]
    r = oracle.forward(A, L)
    def dig(a): return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()[:16]
    got = dict(qa=dig(r["qa"]), sa=dig(r["sa"]), acc0=dig(r["acc0"].astype(np.int32)),
               acc1=dig(r["acc1"].astype(np.int32)), qw=dig(L.d.qw), qr=dig(L.d.qr),
               blocks=sorted((L.blk_n.astype(int) * 4 + L.blk_k).tolist()))
    assert got == {k: g[k] for k in got}


def test_forward_timed_is_the_three_steps_in_sequence(tiny_case):
    """bench.py times oracle.forward_timed (O2 + O8 + O9 through one C call); it must return exactly what
    the three separately pinned steps return."""
    Y = oracle.forward_timed(tiny_case["A"], tiny_case["L"])
    assert np.array_equal(Y, oracle.forward(tiny_case["A"], tiny_case["L"])["Y"])
