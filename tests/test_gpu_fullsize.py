"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default options,
mq_pack_weights = the library's own Algorithm 1 at 5 % density, cold first call and repeated calls on
one workspace): every output column of a seeded sample of token rows is compared with the oracle
(bit-exact int32 accumulators, Y within tolerance), and the selected block set must equal the
oracle's Delta-score top-K.  The oracle computes the sampled rows one by one (O2 + O8 + O9).
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import synth
from helpers import assert_parity, make_case, oracle_forward, run_cuda

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_2606_15652_b200 as m
    m.lib()
    for k in ("split_k", "token_tile", "max_ctas"):
        m.mq_set_option(k, 0)
    return m


FULL = [
    # name, M, K, N   -- every (M, projection) bench.py times for BASELINE.json configs[1] / configs[2] (LLaMA3-8B)
    ("decode qkv M=1", 1, 4096, 6144),
    ("decode o M=8", 8, 4096, 4096),
    ("decode gate_up M=1", 1, 4096, 28672),
    ("decode gate_up M=32", 32, 4096, 28672),
    ("decode down M=8", 8, 14336, 4096),
    ("decode down M=32", 32, 14336, 4096),
    ("prefill qkv M=512", 512, 4096, 6144),
    ("prefill o M=512 (split-K off for large tiles)", 512, 4096, 4096),
    ("prefill gate_up M=512", 512, 4096, 28672),
    ("prefill down M=512", 512, 14336, 4096),
    ("prefill qkv M=2048", 2048, 4096, 6144),
    ("prefill o M=2048", 2048, 4096, 4096),
    ("prefill gate_up M=2048", 2048, 4096, 28672),
    ("prefill down M=2048", 2048, 14336, 4096),
    ("prefill qkv M=8192", 8192, 4096, 6144),
    ("prefill o M=8192", 8192, 4096, 4096),
    ("prefill gate_up M=8192 (14336 tiles, 97 per CTA)", 8192, 4096, 28672),
    ("prefill down M=8192", 8192, 14336, 4096),
    # configs[3] Qwen3-8B
    ("qwen3 gate_up M=128", 128, 4096, 24576),
    # configs[4] LLaMA3-70B: all four projections at M = 1 / 16 / 4096
    ("llama3-70B qkv M=1", 1, 8192, 10240),
    ("llama3-70B qkv M=16", 16, 8192, 10240),
    ("llama3-70B o M=16", 16, 8192, 8192),
    ("llama3-70B gate_up M=1", 1, 8192, 57344),
    ("llama3-70B gate_up M=16", 16, 8192, 57344),
    ("llama3-70B down M=16 (224 K-steps)", 16, 28672, 8192),
    ("llama3-70B qkv M=4096", 4096, 8192, 10240),
    ("llama3-70B o M=4096", 4096, 8192, 8192),
    ("llama3-70B gate_up M=4096", 4096, 8192, 57344),
    ("llama3-70B down M=4096", 4096, 28672, 8192),
]


_LAYER_CACHE = {}


def layer_case(K, N, bs, rho, M):
    """Weights, calibration and the oracle's Algorithm 1 depend on (K, N, bs, rho) only: built once per layer."""
    key = (K, N, bs, rho)
    if key not in _LAYER_CACHE:
        _LAYER_CACHE.clear()                      # one layer at a time (a 70B projection is 1.9 GB of fp32)
        _LAYER_CACHE[key] = make_case(9000 + K // 128 + N, 1, K, N, bs=bs, rho=rho, calib_tokens=64)
    base = _LAYER_CACHE[key]
    A16 = synth.gen_act(9000 + M + N, M, K)
    from helpers import Case
    return Case(M, K, N, bs, base.W, base.h, A16, "f16", base.L)


_PACKED = {}


def packed_layer(mq, case, bs, rho):
    key = (case.K, case.N, bs, rho)
    if key not in _PACKED:
        _PACKED.clear()
        w = mq.mq_pack_weights(case.W, case.h, bs, synth.budget_from_density(rho, case.N, case.K, bs))
        ex = w.export()
        sel_gpu = sorted(zip(ex["blk_n"].tolist(), ex["blk_k"].tolist()))
        sel_orc = sorted(zip(case.L.blk_n.tolist(), case.L.blk_k.tolist()))
        assert sel_gpu == sel_orc, "selected block set differs from the oracle's top-K"
        _PACKED[key] = w
    return _PACKED[key]


@pytest.mark.parametrize("name,M,K,N", sorted(FULL, key=lambda c: (c[2], c[3], c[1])))
def test_full_size_sampled_rows(mq, name, M, K, N):
    case = layer_case(K, N, 64, 0.05, M)
    w = packed_layer(mq, case, 64, 0.05)
    rng = np.random.default_rng(M * 7 + N)
    n_rows = 64 if M * N <= 2 ** 27 else 16       # 16 sampled token rows on the largest outputs (oracle time)
    rows = np.arange(M) if M <= 64 else np.sort(rng.choice(M, size=n_rows, replace=False))
    want = oracle_forward(case, rows=rows)
    ws = mq.new_workspace(mq.mq_gemm_workspace_bytes(w, M))
    for rep in range(2):
        got = run_cuda(case, w=w, workspace=ws, rows=rows)
        assert_parity(got, want, rows=rows, what=f"{name} rep {rep}")


# BASELINE.json configs[3]: the Qwen3-8B density / block-size sweep (0 %, 1 %, 5 %, 10 %; 64 and 128)
SWEEP = [(1, 4096, 6144, 64, 0.0), (1, 4096, 6144, 64, 0.01), (128, 4096, 4096, 64, 0.10), (1, 12288, 4096, 128, 0.05),
         (128, 4096, 6144, 128, 0.10), (4096, 4096, 4096, 128, 0.01),
         (4096, 4096, 24576, 64, 0.10), (4096, 4096, 24576, 128, 0.10), (4096, 12288, 4096, 64, 0.10), (4096, 12288, 4096, 128, 0.10),
         (1, 4096, 24576, 64, 0.10), (128, 12288, 4096, 64, 0.05)]


@pytest.mark.parametrize("M,K,N,bs,rho", SWEEP)
def test_qwen3_density_and_block_sweep(mq, M, K, N, bs, rho):
    case = make_case(9500 + M + N + bs, M, K, N, bs=bs, rho=rho, calib_tokens=64)
    budget = synth.budget_from_density(rho, N, K, bs)
    w = mq.mq_pack_weights(case.W, case.h, bs, budget)
    ex = w.export()
    assert sorted(zip(ex["blk_n"].tolist(), ex["blk_k"].tolist())) == sorted(zip(case.L.blk_n.tolist(), case.L.blk_k.tolist()))
    rng = np.random.default_rng(M + N + bs)
    rows = np.arange(M) if M <= 64 else np.sort(rng.choice(M, size=64 if M * N <= 2 ** 25 else 16, replace=False))
    want = oracle_forward(case, rows=rows)
    got = run_cuda(case, w=w, rows=rows)
    assert_parity(got, want, rows=rows, what=f"qwen3 sweep M{M} K{K} N{N} bs{bs} rho{rho}")
    if rho == 0.0:
        assert not got["acc1"].any()


def test_w4a8_and_group_paths_at_the_largest_prefill_shape(mq):
    """One M = 8192 case each for the W4A8 variant and the per-group path (sampled rows x columns)."""
    import torch
    from helpers import to_device_act, y_tolerance
    M, K, N = 8192, 4096, 4096
    case = layer_case(K, N, 64, 0.05, M)
    w = packed_layer(mq, case, 64, 0.05)
    rng = np.random.default_rng(5)
    rows = np.sort(rng.choice(M, size=16, replace=False))
    want8 = oracle_forward(case, rows=rows, bits=8)
    got8 = run_cuda(case, w=w, bits=8, rows=rows)
    assert_parity(got8, want8, rows=rows, what="W4A8 M=8192 o")
    cols = np.sort(rng.choice(N, size=256, replace=False))
    wg = oracle.forward_group(case.A16, case.L, 128, cols=cols, rows=rows)
    qg, sg = mq.mq_quantize_act_group(to_device_act(case), 128)
    Yg = mq.mq_gemm_group(w, qg, sg, 128, M)
    torch.cuda.synchronize()
    assert np.array_equal(sg.cpu().numpy()[rows].view(np.uint32), wg["sa"].view(np.uint32))
    Y = Yg.float().cpu().numpy().astype(np.float64)[np.ix_(rows, cols)]
    tol = y_tolerance(wg["Y"], 0.0 * wg["mag"], "bf16") + (2 * (K // 128) + 4) * 2.0 ** -24 * wg["mag"]
    assert (np.abs(Y - wg["Y"]) <= tol).all(), "per-group path M=8192: Y out of tolerance"
