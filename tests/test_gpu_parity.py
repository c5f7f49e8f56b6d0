"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Bars (north_star): activation ints/scales and both int32
accumulators bit-exact; Y within 2e-3 relative (helpers.assert_parity).

Run with:  python -m pytest tests -m gpu
"""
import numpy as np
import pytest

import oracle
import synth
from helpers import (Case, assert_parity, f32_to_bf16_bits, make_case, oracle_act, oracle_forward, pack_from_oracle,
                     run_cuda, to_device_act)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mq():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    assert torch.cuda.get_device_capability() == (10, 0), "libmq targets sm_100a (B200) only"
    import paper_2606_15652_b200 as m
    m.lib()  # raises if the extension is missing: no fallback
    yield m
    m.mq_set_option("split_k", 0)
    m.mq_set_option("token_tile", 0)
    m.mq_set_option("max_ctas", 0)


# ------------------------------------------------------------------ kernel (i): activation quantize
@pytest.mark.parametrize("M,K,dt", [(1, 128, "f16"), (16, 256, "f16"), (37, 4096, "f16"), (5, 14336, "f16"),
                                    (3, 28672, "bf16"), (130, 1024, "bf16"), (1, 4096, "bf16")])
def test_quantize_act_bit_exact(mq, M, K, dt):
    import torch
    case = make_case(7 + M, M, K, 128, rho=0.0, a_dtype=dt, calib_tokens=4)
    want_q, want_s = oracle_act(case)
    A = to_device_act(case)
    qA, sA = mq.mq_quantize_act(A)
    got_q = mq.mq_unpack_act(qA, M, K).cpu().numpy()
    torch.cuda.synchronize()
    assert np.array_equal(sA.cpu().numpy().view(np.uint32), want_s.view(np.uint32))
    assert np.array_equal(got_q, want_q)
    # canonical nibble packing (include/mq.h): byte i = element 2i | element 2i+1 << 4
    raw = qA.cpu().numpy()
    lo = (want_q[:, 0::2].astype(np.int16) & 0xF).astype(np.uint8)
    hi = (want_q[:, 1::2].astype(np.int16) & 0xF).astype(np.uint8)
    assert np.array_equal(raw, lo | (hi << 4))


def test_quantize_act_edge_rows(mq):
    """all-zero row (A2), exact ties on the fp16 grid (A3: half to even), +-amax, strided input."""
    import torch
    K = 256
    A = np.zeros((4, K), np.float16)
    A[1, :9] = [7, -7, 3.5, 2.5, 1.5, 0.5, -0.5, -2.5, 0]       # tests/golden/o1_hand_vector.txt
    A[2, :] = np.float16(-3.0)
    A[3, ::2] = np.float16(6.5e4)
    A[3, 1::2] = np.float16(6e-8)                                 # fp16 subnormal
    want_q, want_s = oracle.quantize_act(A)
    big = torch.zeros((4, K + 64), dtype=torch.float16, device="cuda")
    big[:, :K] = torch.from_numpy(A).cuda()
    qA, sA = mq.mq_quantize_act(big[:, :K])                       # lda = K + 64
    got = mq.mq_unpack_act(qA, 4, K).cpu().numpy()
    assert np.array_equal(got, want_q)
    assert np.array_equal(sA.cpu().numpy().view(np.uint32), want_s.view(np.uint32))
    assert want_s[0] == 1.0 and not want_q[0].any()
    assert want_q[1, :9].tolist() == [7, -7, 4, 2, 2, 0, 0, -2, 0]


@pytest.mark.parametrize("dt", ["f16", "bf16"])
def test_quantize_act_near_ties_bit_exact(mq, dt):
    """The kernels multiply by 1/s and divide only near half-integers (A3): rows made of the
    16-bit neighbours of (k + 1/2) * s, for power-of-two scales (exact ties) and for scales that are not
    representable nicely, plus tiny-scale rows (reciprocal unusable), must quantize exactly like the
    oracle's IEEE division (the fused mq_linear path shares quant1() and is checked against the two-call path)."""
    import torch
    rng = np.random.default_rng(5)
    K, rows = 512, []
    amaxes = [7.0, 3.5, 56.0, 1.0, 5.0, 0.3, 1234.0, 6.0e-5, 2.2]
    if dt == "bf16":
        amaxes += [3.0e-38, 1.0e-30, 1.7e38]
    for amax in amaxes:
        amax16 = np.float32(np.float16(amax)) if dt == "f16" else None
        if dt == "bf16":
            amax16 = (np.array([amax], np.float32).view(np.uint32) & 0xFFFF0000).view(np.float32)[0]
        s = np.float32(amax16) / np.float32(7.0)
        x = np.zeros(K, np.float32)
        ks = rng.integers(-7, 7, size=K).astype(np.float32) + np.float32(0.5)
        x[:] = ks * s                                            # near a tie; snapped to the 16-bit grid below
        x[0] = amax16
        if dt == "f16":
            base = x.astype(np.float16)
            nb = base.view(np.int16) + rng.integers(-2, 3, size=K).astype(np.int16)   # neighbours on the grid
            row = nb.view(np.float16)
            row[0] = np.float16(amax16)
            row = np.where(np.isfinite(row) & (np.abs(row.astype(np.float32)) <= amax16), row, np.float16(0))
        else:
            bits = (x.view(np.uint32) >> 16).astype(np.uint16) + rng.integers(0, 3, size=K).astype(np.uint16)
            row = bits
            row[0] = np.uint16(np.array([amax16], np.float32).view(np.uint32)[0] >> 16)
            f = (row.astype(np.uint32) << 16).view(np.float32)
            row = np.where(np.isfinite(f) & (np.abs(f) <= amax16), row, np.uint16(0))
        rows.append(row)
    A16 = np.stack(rows)
    want_q, want_s = oracle.quantize_act(A16 if dt == "f16" else (A16, "bf16"))
    if dt == "f16":
        A = torch.from_numpy(A16).cuda()
    else:
        A = torch.from_numpy(A16.view(np.int16)).cuda().view(torch.bfloat16)
    qA, sA = mq.mq_quantize_act(A)
    got = mq.mq_unpack_act(qA, A.shape[0], K).cpu().numpy()
    assert np.array_equal(sA.cpu().numpy().view(np.uint32), want_s.view(np.uint32))
    assert np.array_equal(got, want_q), f"{int((got != want_q).sum())} codes differ"
    assert (np.abs(want_q) == 7).any(axis=1).all()


# ------------------------------------------------------------------ packing
@pytest.mark.parametrize("bs", [64, 128])
def test_pack_prequantized_roundtrip(mq, bs):
    case = make_case(11, 4, 512, 384, bs=bs, rho=0.25)
    w = pack_from_oracle(case)
    e = w.export()
    L = case.L
    assert np.array_equal(e["qW"], L.d.qw)
    assert np.array_equal(e["sW"].view(np.uint32), L.d.sw.view(np.uint32))
    assert np.array_equal(e["sR"].view(np.uint32), L.d.sr.view(np.uint32))
    order = np.lexsort((L.blk_k, L.blk_n))
    assert e["nnz"] == L.nnz
    assert np.array_equal(e["blk_n"], L.blk_n[order]) and np.array_equal(e["blk_k"], L.blk_k[order])
    assert np.array_equal(e["qR"], L.qr_blocks()[order])
    info = w.info()
    assert (info["N"], info["K"], info["block"], info["nnz"]) == (384, 512, bs, L.nnz)


@pytest.mark.parametrize("N,K,bs,rho", [(256, 256, 64, 2 / 16), (384, 1024, 64, 0.05), (256, 512, 128, 0.25),
                                        (1024, 2048, 64, 0.10)])
def test_pack_weights_matches_algorithm1(mq, N, K, bs, rho):
    """mq_pack_weights (the library's own Algorithm 1) against the oracle's: same base ints and
    scales, same residual scales, same selected set, same Q(R) on it."""
    seed = 0 if N == 256 and K == 256 else 21
    case = make_case(seed, 16, K, N, bs=bs, rho=rho, n_outlier_ch=2 if seed == 0 else None)
    budget = synth.budget_from_density(rho, N, K, bs)
    w = mq.mq_pack_weights(case.W, case.h, bs, budget)
    e = w.export()
    L = case.L
    assert np.array_equal(e["qW"], L.d.qw)
    assert np.array_equal(e["sW"].view(np.uint32), L.d.sw.view(np.uint32))
    assert np.array_equal(e["sR"].view(np.uint32), L.d.sr.view(np.uint32))
    order = np.lexsort((L.blk_k, L.blk_n))
    assert e["nnz"] == L.nnz and L.nnz > 0
    assert np.array_equal(e["blk_n"], L.blk_n[order]) and np.array_equal(e["blk_k"], L.blk_k[order])
    assert np.array_equal(e["qR"], L.qr_blocks()[order])


@pytest.mark.parametrize("N,K,bs,rho", [(256, 256, 64, 2 / 16), (384, 1024, 64, 0.05), (256, 512, 128, 0.25),
                                        (1024, 2048, 64, 0.10), (512, 14336, 64, 0.05)])
def test_pack_weights_device_matches_algorithm1(mq, N, K, bs, rho):
    """mq_pack_weights_device (Algorithm 1's O(N*K) part on the GPU) against the oracle's
    Algorithm 1 and against the host packer: same base ints and scale bits, same selected set (the fp64 score
    sums keep the host's order, so even near-ties fall the same way), same Q(R) on it."""
    import torch
    seed = 0 if N == 256 and K == 256 else 21
    case = make_case(seed, 16, K, N, bs=bs, rho=rho, n_outlier_ch=2 if seed == 0 else None)
    budget = synth.budget_from_density(rho, N, K, bs)
    Wd = torch.from_numpy(np.ascontiguousarray(case.W, np.float32)).cuda()
    hd = torch.from_numpy(np.ascontiguousarray(case.h, np.float32)).cuda()
    e = mq.mq_pack_weights_device(Wd, hd, bs, budget).export()
    L = case.L
    assert np.array_equal(e["qW"], L.d.qw)
    assert np.array_equal(e["sW"].view(np.uint32), L.d.sw.view(np.uint32))
    assert np.array_equal(e["sR"].view(np.uint32), L.d.sr.view(np.uint32))
    order = np.lexsort((L.blk_k, L.blk_n))
    assert e["nnz"] == L.nnz and L.nnz > 0
    assert np.array_equal(e["blk_n"], L.blk_n[order]) and np.array_equal(e["blk_k"], L.blk_k[order])
    assert np.array_equal(e["qR"], L.qr_blocks()[order])
    eh = mq.mq_pack_weights(case.W, case.h, bs, budget).export()
    for k in ("qW", "sW", "sR", "blk_n", "blk_k", "qR"):
        assert np.array_equal(e[k], eh[k]), k
    # h = NULL (all ones), budget 0, budget larger than the number of positive scores, an all-zero row
    W2 = case.W.copy()
    W2[3] = 0.0
    W2d = torch.from_numpy(W2).cuda()
    for (hh, bud) in ((None, 5), (case.h, 0), (case.h, 10 ** 6)):
        a = mq.mq_pack_weights_device(W2d, None if hh is None else hd, bs, bud).export()
        b = mq.mq_pack_weights(W2, hh, bs, bud).export()
        assert a["nnz"] == b["nnz"]
        for k in ("qW", "sW", "sR", "blk_n", "blk_k", "qR"):
            assert np.array_equal(a[k], b[k]), (k, bud)


def test_pack_weights_zero_h_columns_and_null_h(mq):
    """blocks whose score is zero are never selected (nnz < budget); h = NULL means all ones."""
    N, K, bs = 256, 512, 64
    W = synth.gen_weight(5, N, K)
    h = np.ones(K, np.float32)
    h[128:] = 0.0                       # only block-columns 0,1 can score
    w = mq.mq_pack_weights(W, h, bs, 1000)
    L = oracle.algorithm1(W, h, bs, 1000)
    e = w.export()
    assert e["nnz"] == L.nnz == 8 and set(e["blk_k"].tolist()) == {0, 1}
    w1 = mq.mq_pack_weights(W, None, bs, 5)
    L1 = oracle.algorithm1(W, None, bs, 5)
    e1 = w1.export()
    order = np.lexsort((L1.blk_k, L1.blk_n))
    assert np.array_equal(e1["blk_n"], L1.blk_n[order]) and np.array_equal(e1["blk_k"], L1.blk_k[order])


def test_pack_rejects_bad_input(mq):
    qW = np.zeros((128, 128), np.int8)
    s = np.ones(128, np.float32)
    qW[3, 3] = -8                                                  # A1: code -8 is rejected
    with pytest.raises(mq.MqError):
        mq.mq_pack_prequantized(qW, s, 64, np.zeros(0, np.int32), np.zeros(0, np.int32), np.zeros((0, 64, 64), np.int8), s)
    qW[3, 3] = 0
    bn = np.array([0, 0], np.int32)
    bk = np.array([1, 1], np.int32)                               # duplicate block
    with pytest.raises(mq.MqError):
        mq.mq_pack_prequantized(qW, s, 64, bn, bk, np.zeros((2, 64, 64), np.int8), s)
    with pytest.raises(mq.MqError):
        mq.mq_pack_prequantized(qW, s, 64, np.array([5], np.int32), np.array([0], np.int32),
                                np.zeros((1, 64, 64), np.int8), s)  # out of range


# ------------------------------------------------------------------ fused GEMM
def test_config1_tiny(mq):
    """BASELINE.json configs[0]: M=16, K=N=256, 64x64 blocks, top-2 of 16, seed 0."""
    W = synth.gen_weight(0, 256, 256)
    A = synth.gen_act(0, 16, 256, n_outlier_ch=2)
    h = oracle.hessian_diag(A.astype(np.float32)).astype(np.float32)
    L = oracle.algorithm1(W, h, 64, 2)
    case = Case(16, 256, 256, 64, W, h, A, "f16", L)
    want = oracle_forward(case)
    w = mq.mq_pack_weights(W, h, 64, 2)                           # the library's own Algorithm 1
    got = run_cuda(case, w=w)
    assert_parity(got, want, what="config1")
    assert np.abs(want["acc1"]).sum() > 0


SHAPES = [
    # M, K, N, bs, rho, dtype
    (1, 512, 256, 64, 0.10, "f16"),
    (8, 1024, 384, 64, 0.05, "f16"),
    (17, 640, 256, 64, 0.20, "bf16"),       # ragged M, K-steps = 5
    (33, 1024, 512, 128, 0.25, "f16"),
    (100, 512, 384, 64, 0.10, "bf16"),
    (128, 768, 256, 64, 0.10, "f16"),
    (130, 512, 256, 128, 0.50, "f16"),      # two token tiles, ragged tail of 2
    (300, 1024, 640, 64, 0.05, "bf16"),     # several tiles both ways
]


@pytest.mark.parametrize("out_dtype", ["bf16", "f16"])
@pytest.mark.parametrize("M,K,N,bs,rho,dt", SHAPES)
def test_gemm_parity_small(mq, M, K, N, bs, rho, dt, out_dtype):
    case = make_case(100 + M, M, K, N, bs=bs, rho=rho, a_dtype=dt)
    want = oracle_forward(case)
    got = run_cuda(case, out_dtype=out_dtype)      # f16: north_star's 2e-3; bf16: half an ulp
    assert_parity(got, want, what=f"M{M} K{K} N{N} bs{bs} {out_dtype}")


@pytest.mark.parametrize("bt", [16, 32, 64, 128])
def test_gemm_every_token_tile(mq, bt):
    """Each template instantiation (token tile) on a shape with a ragged token tail."""
    M = {16: 40, 32: 70, 64: 150, 128: 260}[bt]
    case = make_case(200 + bt, M, 768, 384, bs=64, rho=0.15)
    want = oracle_forward(case)
    mq.mq_set_option("token_tile", bt)
    try:
        got = run_cuda(case)
    finally:
        mq.mq_set_option("token_tile", 0)
    assert_parity(got, want, what=f"token_tile {bt}")


@pytest.mark.parametrize("mode,ctas", [(2, 3), (2, 7), (2, 50), (2, 0), (1, 5), (1, 0)])
def test_gemm_stream_k_exact_and_workspace_reusable(mq, mode, ctas):
    """Stream-K partial tiles are summed as int32, so the accumulators stay bit-exact however the
    K-steps are cut across CTAs; the workspace is reusable from call to call (include/mq.h)."""
    case = make_case(300 + ctas, 24, 2048, 384, bs=64, rho=0.10)
    want = oracle_forward(case)
    w = pack_from_oracle(case)
    mq.mq_set_option("split_k", mode)
    mq.mq_set_option("max_ctas", ctas)
    try:
        ws = mq.new_workspace(mq.mq_gemm_workspace_bytes(w, case.M))
        assert (ws is not None) == (mode == 2)
        for rep in range(3):
            got = run_cuda(case, w=w, workspace=ws)
            assert_parity(got, want, what=f"split_k {mode} ctas {ctas} rep {rep}")
    finally:
        mq.mq_set_option("split_k", 0)
        mq.mq_set_option("max_ctas", 0)


@pytest.mark.parametrize("M,bt", [(70, 32), (200, 64), (300, 128)])
def test_gemm_stream_k_many_token_tiles(mq, M, bt):
    """Stream-K with several token tiles per weight tile (tile order nt-major) and a ragged tail."""
    case = make_case(400 + M, M, 1024, 256, bs=64, rho=0.10)
    want = oracle_forward(case)
    mq.mq_set_option("split_k", 2)
    mq.mq_set_option("token_tile", bt)
    mq.mq_set_option("max_ctas", 11)
    try:
        got = run_cuda(case)
    finally:
        mq.mq_set_option("split_k", 0)
        mq.mq_set_option("token_tile", 0)
        mq.mq_set_option("max_ctas", 0)
    assert_parity(got, want, what=f"stream-K M{M} bt{bt}")


def test_gemm_budget_zero_equals_dense_w4a4(mq):
    """north_star invariant: K=0 blocks == the dense-only W4A4 GEMM (acc1 == 0)."""
    case = make_case(41, 20, 1024, 256, bs=64, budget=0)
    want = oracle_forward(case)
    got = run_cuda(case)
    assert_parity(got, want, what="budget 0")
    assert not got["acc1"].any()
    dense = want["sa"][:, None].astype(np.float64) * (want["acc0"] * case.L.d.sw[None, :].astype(np.float64))
    assert np.allclose(got["Y"], dense, rtol=4e-3, atol=1e-6)


@pytest.mark.parametrize("bs", [64, 128])
def test_gemm_all_blocks_equals_two_level_dequant(mq, bs):
    """north_star invariant: selecting every block == the two-level dequantized weight."""
    N, K, M = 256, 512, 12
    case = make_case(43, M, K, N, bs=bs, budget=(N // bs) * (K // bs))
    L = case.L
    assert L.nnz == (N // bs) * (K // bs)
    want = oracle_forward(case)
    got = run_cuda(case)
    assert_parity(got, want, what="all blocks")
    W2 = L.d.sw[:, None].astype(np.float64) * L.d.qw + L.d.sr[:, None].astype(np.float64) * L.d.qr
    Aq = want["sa"][:, None].astype(np.float64) * want["qa"]
    assert np.allclose(got["Y"], Aq @ W2.T, rtol=4e-3, atol=1e-5)


def test_gemm_extreme_values(mq):
    """all +-7 operands: |acc0| = 49 K exactly (int32 head-room of the x16 unpack)."""
    import torch
    M, K, N = 8, 4096, 128
    qw = np.full((N, K), 7, np.int8)
    qw[1::2] = -7
    s1 = np.ones(N, np.float32)
    bn = np.array([0, 1], np.int32)
    bk = np.array([0, K // 64 - 1], np.int32)
    qr = np.full((2, 64, 64), -7, np.int8)
    w = mq.mq_pack_prequantized(qw, s1, 64, bn, bk, qr, s1)
    A = torch.full((M, K), 7.0, dtype=torch.float16, device="cuda")
    qA, sA = mq.mq_quantize_act(A)
    Y, d0, d1 = mq.mq_gemm(w, qA, sA, M, dbg=True)
    d0, d1 = d0.cpu().numpy(), d1.cpu().numpy()
    assert (d0[:, 0::2] == 49 * K).all() and (d0[:, 1::2] == -49 * K).all()
    assert (d1 == -49 * 64).all()
    assert np.allclose(sA.cpu().numpy(), 1.0)


def test_gemm_fp16_output_and_strided_y(mq):
    import torch
    case = make_case(47, 9, 512, 256, bs=64, rho=0.10)
    want = oracle_forward(case)
    w = pack_from_oracle(case)
    A = to_device_act(case)
    qA, sA = mq.mq_quantize_act(A)
    big = torch.full((9, 256 + 32), 123.0, dtype=torch.float16, device="cuda")
    mq.mq_gemm(w, qA, sA, 9, Y=big[:, :256])
    got = big.float().cpu().numpy().astype(np.float64)
    assert (got[:, 256:] == 123.0).all()
    err = np.abs(got[:, :256] - want["Y"])
    assert (err <= 1e-3 * np.abs(want["Y"]) + 1e-6 * want["mag"]).all()


def test_linear_matches_two_calls(mq):
    import torch
    case = make_case(49, 40, 1024, 384, bs=64, rho=0.05)
    w = pack_from_oracle(case)
    A = to_device_act(case)
    qA, sA = mq.mq_quantize_act(A)
    Y2 = mq.mq_gemm(w, qA, sA, case.M)
    Y1 = mq.mq_linear(w, A)
    torch.cuda.synchronize()
    assert torch.equal(Y1, Y2)
    assert mq.mq_last_launch_count() == 2


@pytest.mark.parametrize("dt", ["f16", "bf16"])
@pytest.mark.parametrize("M,K,N,rho", [(1, 256, 128, 0.5), (3, 1024, 384, 0.1), (8, 2048, 512, 0.3), (8, 4096, 4096, 0.05),
                                       (5, 14336, 1024, 0.05)])
def test_linear_fused_quantization_small_m(mq, M, K, N, rho, dt):
    """mq_linear with M <= 8 and option fused_quant = 1 runs the activation quantizer INSIDE the GEMM kernel
    (one launch): Y must be bit-identical to mq_quantize_act + mq_gemm, which is checked against the oracle;
    repeated calls on one workspace (grid-wide absmax control block returns to zero) stay identical."""
    import torch
    case = make_case(600 + M + K, M, K, N, bs=64, rho=rho, a_dtype=dt)
    want = oracle_forward(case)
    w = pack_from_oracle(case)
    got = run_cuda(case, w=w)
    assert_parity(got, want, what=f"two-call path M{M} K{K}")
    A = to_device_act(case)
    ws = mq.new_workspace(mq.mq_linear_workspace_bytes(w, M))
    try:
        mq.mq_set_option("fused_quant", 1)
        for rep in range(3):
            Y1 = mq.mq_linear(w, A, workspace=ws)
            torch.cuda.synchronize()
            assert mq.mq_last_launch_count() == 1
            assert np.array_equal(Y1.float().cpu().numpy().astype(np.float64), got["Y"]), f"fused path differs (rep {rep})"
        mq.mq_set_option("fused_quant", 0)
        Y2 = mq.mq_linear(w, A, workspace=ws)
        torch.cuda.synchronize()
        assert mq.mq_last_launch_count() == 2 and torch.equal(Y1, Y2)
    finally:
        mq.mq_set_option("fused_quant", 0)


def test_linear_host_buffers_end_to_end(mq):
    """mq_linear_host: host pointers in and out (the e2e entry bench.py times) equals the device path."""
    import torch
    for M in (3, 40):
        case = make_case(71 + M, M, 1024, 384, bs=64, rho=0.1)
        w = pack_from_oracle(case)
        got = run_cuda(case, w=w)
        A_host = torch.from_numpy(case.A16).pin_memory()
        Y_host = torch.empty((M, 384), dtype=torch.bfloat16).pin_memory()
        stg = torch.empty(mq.mq_linear_host_staging_bytes(w, M), dtype=torch.uint8, device="cuda")
        ws = mq.new_workspace(mq.mq_linear_workspace_bytes(w, M))
        for _ in range(2):
            mq.mq_linear_host(w, A_host, Y_host, stg, ws)
            torch.cuda.synchronize()
            assert np.array_equal(Y_host.float().numpy().astype(np.float64), got["Y"])


def test_linear_host_calls_on_their_own_streams(mq):
    """Independent mq_linear_host calls, each on its own stream with its own staging and workspace (how bench.py's
    end-to-end leg overlaps one call's copies with another's kernels): every result equals the device path."""
    import torch
    streams = [torch.cuda.Stream() for _ in range(3)]
    jobs = []
    for j, (M, K, N) in enumerate([(40, 1024, 384), (3, 512, 256), (70, 768, 640), (8, 1024, 384), (1, 2048, 128)]):
        case = make_case(171 + j, M, K, N, bs=64, rho=0.1)
        w = pack_from_oracle(case)
        got = run_cuda(case, w=w)
        jobs.append((w, torch.from_numpy(case.A16).pin_memory(), torch.empty((M, N), dtype=torch.bfloat16).pin_memory(),
                     torch.empty(mq.mq_linear_host_staging_bytes(w, M), dtype=torch.uint8, device="cuda"),
                     mq.new_workspace(mq.mq_linear_workspace_bytes(w, M)), got["Y"]))
    torch.cuda.synchronize()
    for rep in range(3):
        for j, (w, A_host, Y_host, stg, ws, _) in enumerate(jobs):
            Y_host.zero_()
            mq.mq_linear_host(w, A_host, Y_host, stg, ws, streams[j % 3])
        for s in streams:
            s.synchronize()
        for j, (_, _, Y_host, _, _, want) in enumerate(jobs):
            assert np.array_equal(Y_host.float().numpy().astype(np.float64), want), f"job {j}, round {rep}"


def test_m_zero_is_noop(mq):
    import torch
    case = make_case(51, 1, 256, 128, rho=0.0)
    w = pack_from_oracle(case)
    L = mq.lib()
    assert L.mq_gemm(w.handle, None, None, 0, None, 1, 128, None, None, None, 0, None) == 0
    assert L.mq_quantize_act(None, 0, 0, 256, 256, None, None, None) == 0
    torch.cuda.synchronize()


def _random_block_case(seed, M, K, N, bs, rho):
    """A case whose selected set is a seeded uniform-random block set (control pattern (u) of
    DESIGN.md section 4) instead of the Delta-score top-K: it produces residual cells with every
    quarter mask, including three and four 64x64 blocks inside one 128x128 cell."""
    import dataclasses
    case = make_case(seed, M, K, N, bs=bs, budget=0)
    nb = (N // bs) * (K // bs)
    rng = np.random.default_rng(seed)
    sel = np.sort(rng.choice(nb, size=int(rho * nb + 0.5), replace=False))
    L = dataclasses.replace(case.L, blk_n=(sel // (K // bs)).astype(np.int32), blk_k=(sel % (K // bs)).astype(np.int32))
    return dataclasses.replace(case, L=L)


@pytest.mark.gpu
@pytest.mark.parametrize("M,K,N,rho,mode", [
    (8, 2048, 512, 0.35, 0), (32, 2048, 512, 0.6, 0), (200, 2048, 512, 0.35, 1), (200, 2048, 512, 0.6, 2),
    (300, 1024, 1024, 1.0, 1),
])
def test_gemm_irregular_dense_residual_cells(mq, M, K, N, rho, mode):
    """Residual cells of every shape (1-4 quarters), many per tile, through every ring of the kernel:
    decode tiles, prefill tiles with whole tiles (mode 1) and with stream-K partial tiles (mode 2).
    Repeated calls on one workspace must stay bit-identical (ring/phase bookkeeping, counters)."""
    case = _random_block_case(77 + M, M, K, N, 64, rho)
    want = oracle_forward(case)
    try:
        mq.mq_set_option("split_k", mode)
        w = pack_from_oracle(case)
        ws = mq.new_workspace(mq.mq_gemm_workspace_bytes(w, M))
        for rep in range(3):
            got = run_cuda(case, w=w, workspace=ws)
            assert_parity(got, want, what=f"irregular residual M{M} rho{rho} mode{mode} rep{rep}")
    finally:
        mq.mq_set_option("split_k", 0)


@pytest.mark.gpu
def test_gemm_no_hooks_path_matches_hooked_path(mq):
    """The epilogue's hot path (no parity hooks) and the hooked path must give the same Y bits;
    back-to-back launches exercise programmatic dependent launch on one workspace."""
    import torch
    for (M, K, N) in [(4, 1024, 384), (160, 1024, 384), (260, 2048, 256)]:
        case = _random_block_case(5 + M, M, K, N, 64, 0.2)
        w = pack_from_oracle(case)
        A = to_device_act(case)
        qA, sA = mq.mq_quantize_act(A)
        ws = mq.new_workspace(mq.mq_gemm_workspace_bytes(w, M))
        Yh, _, _ = mq.mq_gemm(w, qA, sA, M, out_dtype=torch.bfloat16, dbg=True, workspace=ws)
        Y = torch.empty_like(Yh)
        for _ in range(4):
            mq.mq_gemm(w, qA, sA, M, Y=Y, workspace=ws)
        torch.cuda.synchronize()
        assert torch.equal(Y.view(torch.int16), Yh.view(torch.int16)), (M, K, N)


@pytest.mark.parametrize("bt", [64, 128])
@pytest.mark.parametrize("rho", [0.0, 0.2])
@pytest.mark.parametrize("odt", ["bf16", "f16"])
def test_gemm_prefill_fast_drain_matches_hooked_path(mq, bt, rho, odt):
    """Whole token tiles without parity hooks take the prefill epilogue's pipelined drain (token scales staged
    in shared memory, 8-token TMEM batches); its Y must be bit-identical to the hooked path's, with and without
    a residual accumulator, for both output types, including a ragged last token tile."""
    import torch
    dt = torch.bfloat16 if odt == "bf16" else torch.float16
    try:
        mq.mq_set_option("token_tile", bt)
        for M in (bt, 3 * bt, 3 * bt + 5):
            case = _random_block_case(900 + M + bt, M, 1024, 384, 64, rho)
            w = pack_from_oracle(case)
            A = to_device_act(case)
            qA, sA = mq.mq_quantize_act(A)
            ws = mq.new_workspace(mq.mq_gemm_workspace_bytes(w, M))
            Yh, _, _ = mq.mq_gemm(w, qA, sA, M, out_dtype=dt, dbg=True, workspace=ws)
            Y = torch.full_like(Yh, 7.0)
            for _ in range(3):
                mq.mq_gemm(w, qA, sA, M, Y=Y, workspace=ws)
            torch.cuda.synchronize()
            assert torch.equal(Y.view(torch.int16), Yh.view(torch.int16)), (M, bt, rho, odt)
    finally:
        mq.mq_set_option("token_tile", 0)


def test_gemm_seeded_fuzz_against_oracle(mq):
    """40 seeded random combinations of shape, block size, density (uniform-random block pattern) and
    launch options (token tile, split-K mode, CTA cap, PDL on/off): accumulators bit-exact and Y in
    tolerance against the oracle; the hot epilogue path must reproduce the hooked path's Y bits."""
    import torch
    rng = np.random.default_rng(2026)
    try:
        for ci in range(40):
            bs = int(rng.choice([64, 128]))
            K = int(rng.choice([128, 256, 640, 1024, 2048]))
            N = int(rng.choice([128, 256, 384, 512]))
            M = int(rng.choice([1, 2, 7, 16, 17, 32, 33, 64, 65, 100, 128, 129, 200, 300]))
            rho = float(rng.choice([0.0, 0.05, 0.1, 0.3, 0.6, 1.0]))
            opts = dict(split_k=int(rng.choice([0, 0, 1, 2])), max_ctas=int(rng.choice([0, 0, 7, 33])),
                        pdl=int(rng.choice([1, 1, 0])), token_tile=int(rng.choice([0, 0, 16, 32, 64, 128])))
            for k, v in opts.items():
                mq.mq_set_option(k, v)
            case = _random_block_case(3000 + ci, M, K, N, bs, rho)
            want = oracle_forward(case)
            w = pack_from_oracle(case)
            ws = mq.new_workspace(mq.mq_gemm_workspace_bytes(w, M))
            got = run_cuda(case, w=w, workspace=ws)
            assert_parity(got, want, what=f"fuzz {ci}: M{M} K{K} N{N} bs{bs} rho{rho} {opts}")
            A = to_device_act(case)
            qA, sA = mq.mq_quantize_act(A)
            Y = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
            for _ in range(2):
                mq.mq_gemm(w, qA, sA, M, Y=Y, workspace=ws)
            torch.cuda.synchronize()
            assert np.array_equal(Y.float().cpu().numpy().astype(np.float64), got["Y"]), f"fuzz {ci}: hot path differs"
    finally:
        for k in ("split_k", "max_ctas", "token_tile"):
            mq.mq_set_option(k, 0)
        mq.mq_set_option("pdl", 1)
