"""Parity of the lean decode kernel (csrc/mq_decode.cu: M <= 32, row slabs, TMA ring + mma.sync) with the oracle:
bit-exact activations, scales and int32 accumulators, Y within tolerance (tests/helpers.py).
The cases aim at what is specific to this kernel: every (rows per CTA, token tile) instantiation with ragged token
counts, K that is not a multiple of a stage (zero-filled last stage), more stages than ring slots, the FIFO ring of
residual pieces under pressure (dense cells: more pieces than slots), both block sizes, slabs in either row half of
an n-tile, grids of more than one wave, and ONE workspace shared by different layers and kernels.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import synth
from helpers import Case, assert_parity, make_case, oracle_forward, pack_from_oracle, run_cuda, y_tolerance

pytestmark = pytest.mark.gpu

OPTS = ("split_k", "token_tile", "max_ctas", "decode_path", "decode_rows", "decode_big")


@pytest.fixture(scope="module")
def mq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_2606_15652_b200 as m
    m.lib()
    for k in OPTS:
        m.mq_set_option(k, 0)
    return m


def with_options(mq, fn, **opts):
    try:
        for k, v in opts.items():
            mq.mq_set_option(k, v)
        return fn()
    finally:
        for k in opts:
            mq.mq_set_option(k, 0)


@pytest.mark.parametrize("out_dtype", ["bf16", "f16"])
@pytest.mark.parametrize("M", [1, 2, 7, 8, 9, 16, 17, 31, 32])
def test_decode_every_token_count(mq, M, out_dtype):
    case = make_case(700 + M, M, 1536, 640, bs=64, rho=0.10, a_dtype="f16" if M % 2 else "bf16")
    want = oracle_forward(case)
    got = run_cuda(case, out_dtype=out_dtype)
    assert mq.mq_last_launch_count() == 1
    assert_parity(got, want, what=f"decode M{M} {out_dtype}")
    assert np.abs(want["acc1"]).sum() > 0


@pytest.mark.parametrize("big", [2, 1])
@pytest.mark.parametrize("rows", [16, 32, 64, 128])
@pytest.mark.parametrize("M,K", [(1, 1536), (8, 640), (5, 4480), (16, 1536), (24, 2176), (32, 1536)])
def test_decode_every_slab_height(mq, M, K, rows, big):
    """Every (rows, token tile) instantiation; K-steps 12 / 5 / 35 / 17: last stages with 4, 5, 3 and 1 K-steps for
    stages of 8, 4 and 2 K-steps, and more stages than ring slots; three calls in a row."""
    case = make_case(720 + rows + M, M, K, 640, bs=64, rho=0.15)
    want = oracle_forward(case)
    w = pack_from_oracle(case)

    def run():
        for rep in range(3):
            got = run_cuda(case, w=w)
            assert_parity(got, want, what=f"decode M{M} K{K} rows {rows} rep {rep}")
    with_options(mq, run, decode_rows=rows, decode_big=big)


def test_decode_more_ctas_than_one_wave(mq):
    case = make_case(741, 3, 1024, 128 * 42, bs=64, rho=0.05)   # 336 slabs of 16 channels
    want = oracle_forward(case)
    got = with_options(mq, lambda: run_cuda(case), decode_rows=16)
    assert_parity(got, want, what="decode 336 CTAs")


@pytest.mark.parametrize("rows", [0, 16, 32, 64, 128])
@pytest.mark.parametrize("bs,budget_frac", [(64, 1.0), (128, 1.0), (64, 0.5), (128, 0.3)])
@pytest.mark.parametrize("M", [5, 32])
def test_decode_dense_residual_cells(mq, M, bs, budget_frac, rows):
    """Every K-step owns a full cell: a stage needs up to 16 residual pieces and the piece ring has 16 slots, so
    the producer must wait for consumed stages to issue more; also the paper's all-blocks invariant."""
    N, K = 384, 2048 + 128
    nb = (N // bs) * (K // bs)
    case = make_case(750 + bs, M, K, N, bs=bs, budget=int(nb * budget_frac))
    want = oracle_forward(case)
    for big in (2, 1):
        got = with_options(mq, lambda: run_cuda(case), decode_rows=rows, decode_big=big)
        assert_parity(got, want, what=f"decode dense residual bs{bs} frac{budget_frac} rows{rows} big{big}")


def test_decode_irregular_block_pattern(mq):
    """Seeded random block sets (not the Delta-score's): isolated quarters in every position of a cell."""
    rng = np.random.default_rng(77)
    N, K, bs, M = 512, 2560, 64, 8
    W = synth.gen_weight(77, N, K)
    d = oracle.decompose(W)
    for trial in range(6):
        nb = (N // bs) * (K // bs)
        sel = np.sort(rng.choice(nb, size=int(nb * rng.choice([0.03, 0.2, 0.6])), replace=False))
        L = oracle.PackedLayer(N, K, bs, d, None, (sel // (K // bs)).astype(np.int32), (sel % (K // bs)).astype(np.int32))
        case = Case(M, K, N, bs, W, None, synth.gen_act(77 + trial, M, K), "f16", L)
        want = oracle_forward(case)
        got = with_options(mq, lambda: run_cuda(case), decode_rows=int(rng.choice([0, 16, 32, 64, 128])))
        assert_parity(got, want, what=f"decode irregular blocks trial {trial}")


def test_decode_budget_zero_and_extremes(mq):
    case = make_case(760, 6, 1024, 256, bs=64, budget=0)
    got = run_cuda(case)
    assert_parity(got, oracle_forward(case), what="decode budget 0")
    assert not got["acc1"].any()
    # all codes +-7: |acc0| = 49 K exactly (O8 pin), through the x256 accumulators
    N, K, M = 128, 4096, 3
    qw = np.full((N, K), 7, np.int8)
    qw[1::2] = -7
    import paper_2606_15652_b200 as m
    import torch
    w = m.mq_pack_prequantized(qw, np.ones(N, np.float32), 64, np.zeros(0, np.int32), np.zeros(0, np.int32),
                               np.zeros((0, 64, 64), np.int8), np.ones(N, np.float32))
    A = torch.full((M, K), 7.0, dtype=torch.float16, device="cuda")
    qA, sA = m.mq_quantize_act(A)
    Y, d0, d1 = m.mq_gemm(w, qA, sA, M, dbg=True)
    torch.cuda.synchronize()
    a0 = d0.cpu().numpy()
    assert (a0[:, 0::2] == 49 * K).all() and (a0[:, 1::2] == -49 * K).all() and not d1.cpu().numpy().any()


def test_one_workspace_shared_by_layers_tokens_and_kernels(mq):
    """include/mq.h workspace contract: the zero-state words sit in a plan-independent 16 KB prefix and
    every call returns them to zero, so ONE zeroed workspace of the largest size serves alternating layer shapes,
    token counts and kernels (decode kernel, tcgen05 stream-K, mq_linear)."""
    import torch
    cases = [make_case(770, 8, 2048, 384, rho=0.10), make_case(771, 32, 1024, 640, rho=0.10),
             make_case(772, 40, 2048, 256, rho=0.10), make_case(773, 1, 1536, 512, rho=0.10)]
    ws_ = [pack_from_oracle(c) for c in cases]
    wants = [oracle_forward(c) for c in cases]
    need = 0
    for c, w in zip(cases, ws_):
        need = max(need, mq.mq_gemm_workspace_bytes(w, c.M), mq.mq_linear_workspace_bytes(w, c.M))
        mq.mq_set_option("split_k", 2)
        need = max(need, mq.mq_gemm_workspace_bytes(w, c.M))
        mq.mq_set_option("split_k", 0)
    ws = mq.new_workspace(need)
    for rnd in range(3):
        for i, (c, w, want) in enumerate(zip(cases, ws_, wants)):
            opts = [dict(), dict(split_k=2), dict(decode_path=1)][(rnd + i) % 3]
            got = with_options(mq, lambda: run_cuda(c, w=w, workspace=ws), **opts)
            assert_parity(got, want, what=f"shared workspace round {rnd} case {i} opts {opts}")
            A = torch.from_numpy(c.A16).cuda()
            Y = mq.mq_linear(w, A, workspace=ws)
            torch.cuda.synchronize()
            err = np.abs(Y.float().cpu().numpy().astype(np.float64) - want["Y"])
            assert (err <= y_tolerance(want["Y"], want["mag"], "bf16")).all(), "mq_linear on the shared workspace: Y out of tolerance"
    assert not ws[:16384].any(), "the zero-state prefix did not return to zero"


def test_decode_matches_tcgen05_kernel(mq):
    """The two kernels agree on the integer accumulators bit for bit and on Y up to fp32 contraction."""
    case = make_case(780, 16, 2048, 512, rho=0.10)
    w = pack_from_oracle(case)
    a = run_cuda(case, w=w)
    b = with_options(mq, lambda: run_cuda(case, w=w), decode_path=1)
    assert np.array_equal(a["acc0"], b["acc0"]) and np.array_equal(a["acc1"], b["acc1"])
    assert np.allclose(a["Y"], b["Y"], rtol=2.0 ** -7, atol=1e-6)
