"""Block-local residual scales (second half; north_star "per-block scales"; reading A4b) on the
GPU against the oracle (oracle.algorithm1_blocklocal / forward_blocklocal): the packer's Algorithm 1 selects the same
blocks and produces the same codes and scale bits; acc0 and the integer sum of the block accumulators are bit-exact; Y
is within the output rounding plus the fp32 accumulation of the block terms (tolerance T3 in DESIGN.md section 4).
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import synth
from helpers import f32_to_bf16_bits, y_tolerance

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_2606_15652_b200 as m
    m.lib()
    for k in ("split_k", "token_tile", "max_ctas", "decode_path", "decode_rows", "decode_big"):
        m.mq_set_option(k, 0)
    return m


def make(seed, M, K, N, bs, budget):
    W = synth.gen_weight(seed, N, K)
    A = synth.gen_act(seed, M, K)
    X = synth.gen_calib(seed, K, 64)
    h = oracle.hessian_diag(X).astype(np.float32)
    return W, A, h, oracle.algorithm1_blocklocal(W, h, bs, budget)


def run(mq, w, A, M, out_dtype="bf16"):
    import torch
    At = torch.from_numpy(A).cuda()
    qA, sA = mq.mq_quantize_act(At)
    Y, d0, d1 = mq.mq_gemm(w, qA, sA, M, out_dtype=torch.bfloat16 if out_dtype == "bf16" else torch.float16, dbg=True)
    torch.cuda.synchronize()
    return Y.float().cpu().numpy().astype(np.float64), d0.cpu().numpy(), d1.cpu().numpy()


def check(got, want, K, out_dtype, what):
    Y, d0, d1 = got
    assert np.array_equal(d0.astype(np.int64), want["acc0"]), f"{what}: base accumulator not bit-exact"
    assert np.array_equal(d1.astype(np.int64), want["acc1sum"]), f"{what}: sum of the block accumulators not bit-exact"
    # T3: output rounding + one fp32 rounding per block term and per partial sum (at most 2 K / 64 + 8 of them)
    tol = y_tolerance(want["Y"], 0.0 * want["mag"], out_dtype) + (2 * K // 64 + 8) * 2.0 ** -24 * want["mag"]
    err = np.abs(Y - want["Y"])
    assert (err <= tol).all(), f"{what}: Y out of tolerance at {int((err > tol).sum())} of {err.size}"


@pytest.mark.parametrize("bs", [64, 128])
def test_pack_weights_blockscale_matches_algorithm1(mq, bs):
    N, K = 384, 1024
    W, A, h, L = make(810 + bs, 4, K, N, bs, 7)
    w = mq.mq_pack_weights_blockscale(W, h, bs, 7)
    assert w.is_blockscale()
    ex = w.export()
    order = np.lexsort((L.blk_k, L.blk_n))
    assert np.array_equal(ex["blk_n"], L.blk_n[order]) and np.array_equal(ex["blk_k"], L.blk_k[order])
    assert np.array_equal(ex["qW"], L.d.qw) and np.array_equal(ex["sW"].view(np.uint32), L.d.sw.view(np.uint32))
    assert np.array_equal(ex["qR"], L.qr_blocks()[order])
    assert np.array_equal(w.export_blockscale().view(np.uint32), L.sr_blocks()[order].view(np.uint32))
    check(run(mq, w, A, 4), oracle.forward_blocklocal(A, L), K, "bf16", f"blockscale alg1 bs{bs}")
    # per-channel handles are told apart, and the other GEMM entries refuse block-local handles
    assert not mq.mq_pack_weights(W, h, bs, 7).is_blockscale()
    import torch
    qg, sg = mq.mq_quantize_act_group(torch.from_numpy(A).cuda(), 128)
    with pytest.raises(mq.MqError):
        mq.mq_gemm_group(w, qg, sg, 128, 4)


@pytest.mark.parametrize("out_dtype", ["bf16", "f16"])
@pytest.mark.parametrize("M,rows", [(1, 0), (8, 16), (17, 32), (32, 64), (5, 128), (40, 0), (100, 32)])
def test_gemm_blockscale_parity(mq, M, rows, out_dtype):
    N, K, bs = 512, 1536 + 128, 64
    W, A, h, L = make(820 + M, M, K, N, bs, 40)
    w = mq.mq_pack_prequantized_blockscale(L.d.qw, L.d.sw, bs, L.blk_n, L.blk_k, L.qr_blocks(), L.sr_blocks())
    want = oracle.forward_blocklocal(A, L)
    mq.mq_set_option("decode_rows", rows)
    try:
        got = run(mq, w, A, M, out_dtype)
        assert mq.mq_last_launch_count() == (M + 31) // 32
    finally:
        mq.mq_set_option("decode_rows", 0)
    check(got, want, K, out_dtype, f"blockscale M{M} rows{rows} {out_dtype}")
    assert np.abs(want["acc1sum"]).sum() > 0


@pytest.mark.parametrize("bs,frac", [(64, 1.0), (128, 1.0), (128, 0.4)])
def test_gemm_blockscale_dense_cells_and_budget_zero(mq, bs, frac):
    N, K, M = 256, 1024, 9
    nb = (N // bs) * (K // bs)
    W, A, h, L = make(830 + bs, M, K, N, bs, int(nb * frac))
    w = mq.mq_pack_prequantized_blockscale(L.d.qw, L.d.sw, bs, L.blk_n, L.blk_k, L.qr_blocks(), L.sr_blocks())
    check(run(mq, w, A, M), oracle.forward_blocklocal(A, L), K, "bf16", f"blockscale dense bs{bs} {frac}")
    L0 = oracle.PackedLayerBlockLocal(N, K, bs, L.d, None, L.blk_n[:0], L.blk_k[:0])
    w0 = mq.mq_pack_prequantized_blockscale(L.d.qw, L.d.sw, bs, L0.blk_n, L0.blk_k, L0.qr_blocks(), L0.sr_blocks())
    got0 = run(mq, w0, A, M)
    check(got0, oracle.forward_blocklocal(A, L0), K, "bf16", "blockscale budget 0")
    assert not got0[2].any()


def test_gemm_blockscale_full_size_decode_layer(mq):
    """LLaMA3-8B o projection, M = 8, 5 % density: the library's own Algorithm 1 against the oracle's."""
    N, K, M, bs = 4096, 4096, 8, 64
    budget = synth.budget_from_density(0.05, N, K, bs)
    W, A, h, L = make(840, M, K, N, bs, budget)
    w = mq.mq_pack_weights_blockscale(W, h, bs, budget)
    ex = w.export()
    assert sorted(zip(ex["blk_n"].tolist(), ex["blk_k"].tolist())) == sorted(zip(L.blk_n.tolist(), L.blk_k.tolist()))
    check(run(mq, w, A, M), oracle.forward_blocklocal(A, L), K, "bf16", "blockscale o M=8")
