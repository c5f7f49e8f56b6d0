"""mq_pack_weights_device (Algorithm 1 entirely on the GPU): radix-select TopK, residual layout and
Q(R) as kernels.  Beyond test_gpu_parity.py::test_pack_weights_device_matches_algorithm1: exact score ties (the tie
rule A7: lower linear block index first), rows too long for the shared-memory residual row, a full-size layer, and the
handle running through mq_gemm against the oracle."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import synth
from helpers import Case, assert_parity, oracle_forward, run_cuda

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_2606_15652_b200 as m
    m.lib()
    return m


def same_as_oracle(mq, W, h, bs, budget):
    import torch
    Wd = torch.from_numpy(np.ascontiguousarray(W, np.float32)).cuda()
    hd = None if h is None else torch.from_numpy(np.ascontiguousarray(h, np.float32)).cuda()
    w = mq.mq_pack_weights_device(Wd, hd, bs, budget)
    e = w.export()
    L = oracle.algorithm1(W, h, bs, budget)
    order = np.lexsort((L.blk_k, L.blk_n))
    assert e["nnz"] == L.nnz
    assert np.array_equal(e["blk_n"], L.blk_n[order]) and np.array_equal(e["blk_k"], L.blk_k[order]), "selected set differs"
    assert np.array_equal(e["qW"], L.d.qw) and np.array_equal(e["sW"].view(np.uint32), L.d.sw.view(np.uint32))
    assert np.array_equal(e["sR"].view(np.uint32), L.d.sr.view(np.uint32))
    assert np.array_equal(e["qR"], L.qr_blocks()[order])
    return w, L


@pytest.mark.parametrize("bs", [64, 128])
def test_exact_ties_go_to_the_lower_block_index(mq, bs):
    """Block-rows that are copies of each other have bit-identical scores: with a budget that cuts through a group of
    ties, the lower linear indices must be taken (A7), on the device exactly as in the oracle's stable sort."""
    N, K = 512, 1024
    W = synth.gen_weight(31, N, K)
    W[bs:2 * bs] = W[0:bs]               # block-row 1 == block-row 0
    W[3 * bs:4 * bs] = W[0:bs]           # block-row 3 == block-row 0
    sc = oracle.algorithm1(W, None, bs, 0).sc.S
    nbk = K // bs
    assert np.array_equal(sc[:nbk], sc[nbk:2 * nbk]) and np.array_equal(sc[:nbk], sc[3 * nbk:4 * nbk])
    for budget in (1, 2, 3, 4, 5, 7, 11, nbk, 3 * nbk + 1, (N // bs) * nbk):
        same_as_oracle(mq, W, None, bs, budget)
    # all scores equal (every block-row identical, h = 1 on one column block only): pure index order
    W2 = np.tile(W[0:bs], (N // bs, 1))
    h2 = np.zeros(K, np.float32)
    h2[:bs] = 1.0
    for budget in (1, 3, N // bs):
        w, L = same_as_oracle(mq, W2, h2, bs, budget)
        assert L.blk_n.tolist() == list(range(budget)) and set(L.blk_k.tolist()) == {0}


def test_rows_longer_than_shared_memory(mq):
    """K = 53248: the residual row (208 KB of fp32) does not fit shared memory: it is recomputed from W (round 1's K <= 51200 cap)."""
    N, K, bs = 128, 53248, 64
    W = synth.gen_weight(33, N, K)
    X = synth.gen_calib(33, K, 16)
    h = oracle.hessian_diag(X).astype(np.float32)
    same_as_oracle(mq, W, h, bs, synth.budget_from_density(0.05, N, K, bs))


def test_full_size_layer_runs_through_the_gemm(mq):
    """LLaMA3-8B qkv (4096 -> 6144), 5 %: device packing equals the oracle's Algorithm 1, and the handle serves mq_gemm."""
    N, K, bs, M = 6144, 4096, 64, 8
    W = synth.gen_weight(35, N, K)
    X = synth.gen_calib(35, K, 64)
    h = oracle.hessian_diag(X).astype(np.float32)
    w, L = same_as_oracle(mq, W, h, bs, synth.budget_from_density(0.05, N, K, bs))
    case = Case(M, K, N, bs, W, h, synth.gen_act(35, M, K), "f16", L)
    assert_parity(run_cuda(case, w=w), oracle_forward(case), what="device-packed qkv M=8")
    case2 = Case(100, K, N, bs, W, h, synth.gen_act(36, 100, K), "f16", L)
    assert_parity(run_cuda(case2, w=w), oracle_forward(case2), what="device-packed qkv M=100")
