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
    # name, M, K, N        (LLaMA3-8B projections of configs[1] / configs[2]; Qwen3-8B gate_up of configs[3])
    ("decode qkv M=1", 1, 4096, 6144),
    ("decode o M=8", 8, 4096, 4096),
    ("decode gate_up M=32", 32, 4096, 28672),
    ("decode down M=32", 32, 14336, 4096),
    ("prefill qkv M=2048", 2048, 4096, 6144),
    ("prefill o M=512 (split-K off for large tiles)", 512, 4096, 4096),
    ("qwen3 gate_up M=128", 128, 4096, 24576),
    ("llama3-70B o M=16", 16, 8192, 8192),
    ("llama3-70B down M=16 (224 K-steps)", 16, 28672, 8192),
]


@pytest.mark.parametrize("name,M,K,N", FULL)
def test_full_size_sampled_rows(mq, name, M, K, N):
    case = make_case(9000 + M + N, M, K, N, bs=64, rho=0.05, calib_tokens=64)
    w = mq.mq_pack_weights(case.W, case.h, 64, synth.budget_from_density(0.05, N, K, 64))
    ex = w.export()
    sel_gpu = sorted(zip(ex["blk_n"].tolist(), ex["blk_k"].tolist()))
    sel_orc = sorted(zip(case.L.blk_n.tolist(), case.L.blk_k.tolist()))
    assert sel_gpu == sel_orc, f"{name}: selected block set differs from the oracle's top-K"
    rng = np.random.default_rng(M * 7 + N)
    rows = np.arange(M) if M <= 64 else np.sort(rng.choice(M, size=64, replace=False))
    want = oracle_forward(case, rows=rows)
    ws = mq.new_workspace(mq.mq_gemm_workspace_bytes(w, M))
    for rep in range(2):
        got = run_cuda(case, w=w, workspace=ws)
        assert_parity(got, want, rows=rows, what=f"{name} rep {rep}")


# BASELINE.json configs[3]: the Qwen3-8B density / block-size sweep (0 %, 1 %, 5 %, 10 %; 64 and 128)
SWEEP = [(1, 4096, 6144, 64, 0.0), (1, 4096, 6144, 64, 0.01), (128, 4096, 4096, 64, 0.10), (1, 12288, 4096, 128, 0.05),
         (128, 4096, 6144, 128, 0.10), (4096, 4096, 4096, 128, 0.01)]


@pytest.mark.parametrize("M,K,N,bs,rho", SWEEP)
def test_qwen3_density_and_block_sweep(mq, M, K, N, bs, rho):
    case = make_case(9500 + M + N + bs, M, K, N, bs=bs, rho=rho, calib_tokens=64)
    budget = synth.budget_from_density(rho, N, K, bs)
    w = mq.mq_pack_weights(case.W, case.h, bs, budget)
    ex = w.export()
    assert sorted(zip(ex["blk_n"].tolist(), ex["blk_k"].tolist())) == sorted(zip(case.L.blk_n.tolist(), case.L.blk_k.tolist()))
    rng = np.random.default_rng(M + N + bs)
    rows = np.arange(M) if M <= 64 else np.sort(rng.choice(M, size=64, replace=False))
    want = oracle_forward(case, rows=rows)
    got = run_cuda(case, w=w)
    assert_parity(got, want, rows=rows, what=f"qwen3 sweep M{M} K{K} N{N} bs{bs} rho{rho}")
    if rho == 0.0:
        assert not got["acc1"].any()
