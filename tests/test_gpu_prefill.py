"""Parity of the whole-tile prefill kernels (csrc/mq_prefill.cu: M >= 64, 128 x 128 output tiles dealt to persistent
CTAs; one CTA per tile, or CTA pairs issuing tcgen05.mma.cta_group::2) with the oracle: bit-exact activations, scales
and int32 accumulators, Y within tolerance (tests/helpers.py).

mq_gemm picks these kernels by itself only when the last round of tiles is mostly full (the full-size cases of
test_gpu_fullsize.py); here option "prefill_path" forces them (2 = one CTA per tile, 3 = pairs where the layer has an
even number of n-tiles) on shapes the oracle finishes in seconds.  The cases aim at what is specific to these kernels:
ragged last token tiles (rows past M are read as zero and never stored), K-steps that are not a multiple of the ring
depths or of the 32-K-step metadata chunk, more tiles than CTAs (several tiles per CTA: both accumulator buffers, the
single residual accumulator handed back and forth), residual cells in every K-step (an operand-ring item after every
base item) and in none, n-tile pairs where only one CTA owns a cell, both block sizes, both output types, and calls
repeated on one workspace shared with the other kernels.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import synth
from helpers import Case, assert_parity, make_case, oracle_forward, pack_from_oracle, run_cuda

pytestmark = pytest.mark.gpu

OPTS = ("split_k", "token_tile", "max_ctas", "decode_path", "prefill_path")
PATHS = [2, 3]


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


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("out_dtype", ["bf16", "f16"])
@pytest.mark.parametrize("M", [64, 65, 127, 128, 129, 200, 256, 333])
def test_prefill_token_counts(mq, M, out_dtype, path):
    """Whole and ragged token tiles; N = 512: two n-tile pairs."""
    case = make_case(900 + M, M, 640, 512, bs=64, rho=0.10, a_dtype="f16" if M % 2 else "bf16")
    want = oracle_forward(case)
    got = with_options(mq, lambda: run_cuda(case, out_dtype=out_dtype), prefill_path=path)
    assert mq.mq_last_launch_count() == 1
    assert_parity(got, want, what=f"prefill path {path} M{M} {out_dtype}")
    assert np.abs(want["acc1"]).sum() > 0


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("K", [128, 256, 384, 1152, 2176, 4224, 4480])
def test_prefill_k_steps(mq, K, path):
    """1, 2, 3, 9, 17, 33 and 35 K-steps: fewer than the ring depths, not a multiple of them, one more than the
    32-K-step metadata chunk; three calls in a row on one handle."""
    case = make_case(930 + K // 128, 192, K, 256, bs=64, rho=0.12)
    want = oracle_forward(case)
    w = pack_from_oracle(case)

    def run():
        for rep in range(3):
            got = run_cuda(case, w=w)
            assert_parity(got, want, what=f"prefill path {path} K{K} rep {rep}")
    with_options(mq, run, prefill_path=path)


@pytest.mark.parametrize("path", PATHS)
def test_prefill_more_tiles_than_ctas(mq, path):
    """N = 3072, M = 1100: 24 x 9 = 216 tiles (108 tile pairs) for 148 CTAs (74 pairs): CTAs with one and with two
    tiles, ragged last token tile, both accumulator buffers in use."""
    case = make_case(951, 1100, 512, 3072, bs=64, rho=0.06)
    rows = np.unique(np.concatenate([np.arange(0, 1100, 37), np.arange(1020, 1100)]))
    want = oracle_forward(case, rows=rows)
    got = with_options(mq, lambda: run_cuda(case, rows=rows), prefill_path=path)
    assert_parity(got, want, rows=rows, what=f"prefill path {path} 216 tiles")


@pytest.mark.parametrize("path", PATHS)
def test_prefill_many_tiles_per_cta(mq, path):
    """N = 2048, M = 4100: 16 x 33 = 528 tiles: three to four tiles per CTA (seven to eight per pair)."""
    case = make_case(952, 4100, 384, 2048, bs=64, rho=0.08)
    rows = np.unique(np.concatenate([np.arange(0, 4100, 131), np.arange(4090, 4100)]))
    want = oracle_forward(case, rows=rows)
    got = with_options(mq, lambda: run_cuda(case, rows=rows), prefill_path=path)
    assert_parity(got, want, rows=rows, what=f"prefill path {path} 528 tiles")


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("bs,budget_frac", [(64, 1.0), (128, 1.0), (64, 0.5), (128, 0.25), (64, 0.0)])
def test_prefill_residual_density(mq, bs, budget_frac, path):
    """Every block selected (a residual item after every base item, all four quarters), half of them, none."""
    case = make_case(960 + bs, 160, 1024, 512, bs=bs, rho=budget_frac)
    want = oracle_forward(case)
    got = with_options(mq, lambda: run_cuda(case), prefill_path=path)
    assert_parity(got, want, what=f"prefill path {path} bs {bs} budget {budget_frac}")
    if budget_frac == 0.0:
        assert np.abs(want["acc1"]).sum() == 0


@pytest.mark.parametrize("path", PATHS)
def test_prefill_cells_in_one_n_tile_of_a_pair(mq, path):
    """A chosen block set (not the Delta-score's): blocks only in the channels of ONE n-tile of each pair (n-tile 1 =
    the odd CTA of pair 0, n-tile 2 = the even CTA of pair 1) and only in some K-steps, single quarters in every
    position of a cell.  The CTA without a cell supplies zero residual operands for the pair's MMAs, and its half of
    the second accumulator stays zero."""
    N, K, M, bs = 512, 1536, 130, 64
    W = synth.gen_weight(970, N, K)
    d = oracle.decompose(W)
    blocks = [(2, 0), (3, 1), (2, 10), (4, 10), (5, 23), (4, 22), (3, 22), (2, 11), (3, 11), (5, 4)]   # (n-block, k-block)
    blk_n = np.array([b[0] for b in blocks], np.int32)
    blk_k = np.array([b[1] for b in blocks], np.int32)
    order = np.argsort(blk_n * (K // bs) + blk_k)
    L = oracle.PackedLayer(N, K, bs, d, None, blk_n[order], blk_k[order])
    case = Case(M, K, N, bs, W, None, synth.gen_act(970, M, K), "f16", L)
    want = oracle_forward(case)
    assert np.abs(want["acc1"][:, :128]).sum() == 0 and np.abs(want["acc1"][:, 384:]).sum() == 0
    assert np.abs(want["acc1"][:, 128:256]).sum() > 0 and np.abs(want["acc1"][:, 256:384]).sum() > 0
    got = with_options(mq, lambda: run_cuda(case), prefill_path=path)
    assert_parity(got, want, what=f"prefill path {path} one-sided cells")


@pytest.mark.parametrize("path", PATHS)
def test_prefill_irregular_block_pattern(mq, path):
    """Seeded random block sets at three densities: every mix of quarters per cell, runs of K-steps with and without
    cells (the item numbering of the operand ring shifts with every cell)."""
    rng = np.random.default_rng(975)
    N, K, bs, M = 512, 2560, 64, 150
    W = synth.gen_weight(975, N, K)
    d = oracle.decompose(W)
    for trial, dens in enumerate([0.03, 0.2, 0.6]):
        nb = (N // bs) * (K // bs)
        sel = np.sort(rng.choice(nb, size=int(nb * dens), replace=False))
        L = oracle.PackedLayer(N, K, bs, d, None, (sel // (K // bs)).astype(np.int32), (sel % (K // bs)).astype(np.int32))
        case = Case(M, K, N, bs, W, None, synth.gen_act(975 + trial, M, K), "f16", L)
        want = oracle_forward(case)
        got = with_options(mq, lambda: run_cuda(case), prefill_path=path)
        assert_parity(got, want, what=f"prefill path {path} irregular blocks, density {dens}")


def test_prefill_pairs_need_even_n_tiles(mq):
    """N = 384: three n-tiles; path 3 falls back to one CTA per tile."""
    case = make_case(980, 140, 512, 384, bs=64, rho=0.10)
    want = oracle_forward(case)
    got = with_options(mq, lambda: run_cuda(case), prefill_path=3)
    assert mq.mq_last_launch_count() == 1
    assert_parity(got, want, what="prefill path 3, odd n-tiles")


def test_prefill_shares_workspace_with_other_kernels(mq):
    """One workspace for a decode call, a stream-K call and both prefill kernels in turn, twice: nobody leaves
    state behind (the prefill kernels do not touch the workspace at all)."""
    import torch
    case_p = make_case(985, 192, 768, 512, bs=64, rho=0.10)
    case_d = make_case(986, 8, 768, 512, bs=64, rho=0.10)
    want_p, want_d = oracle_forward(case_p), oracle_forward(case_d)
    wp, wd = pack_from_oracle(case_p), pack_from_oracle(case_d)
    nbytes = max(mq.mq_gemm_workspace_bytes(wp, 192), mq.mq_gemm_workspace_bytes(wd, 8), 1 << 20)
    ws = mq.new_workspace(nbytes)
    for rep in range(2):
        assert_parity(run_cuda(case_d, w=wd, workspace=ws), want_d, what=f"decode rep {rep}")
        assert_parity(with_options(mq, lambda: run_cuda(case_p, w=wp, workspace=ws), prefill_path=1), want_p, what=f"stream-K rep {rep}")
        for path in PATHS:
            assert_parity(with_options(mq, lambda: run_cuda(case_p, w=wp, workspace=ws), prefill_path=path), want_p,
                          what=f"prefill path {path} rep {rep}")
    assert int(ws[:16384].to(torch.int32).sum().item()) == 0


def test_prefill_extreme_values(mq):
    """All codes at +-7 with aligned signs: |acc0| = 49 K and |acc1| = 49 * 64 exactly, the largest accumulators the
    x16 operands produce at K = 4096 (int32 head-room of the unpack)."""
    import torch
    M, K, N = 130, 4096, 256
    qw = np.full((N, K), 7, np.int8)
    qw[1::2] = -7
    s1 = np.ones(N, np.float32)
    bn = np.array([0, 1, 2], np.int32)
    bk = np.array([0, K // 64 - 1, 5], np.int32)
    qr = np.full((3, 64, 64), -7, np.int8)
    w = mq.mq_pack_prequantized(qw, s1, 64, bn, bk, qr, s1)
    A = torch.full((M, K), 7.0, dtype=torch.float16, device="cuda")
    qA, sA = mq.mq_quantize_act(A)
    for path in PATHS:
        Y, d0, d1 = with_options(mq, lambda: mq.mq_gemm(w, qA, sA, M, dbg=True), prefill_path=path)
        torch.cuda.synchronize()
        d0, d1 = d0.cpu().numpy(), d1.cpu().numpy()
        assert (d0[:, 0::2] == 49 * K).all() and (d0[:, 1::2] == -49 * K).all(), f"path {path}"
        assert (d1[:, :192] == -49 * 64).all() and not d1[:, 192:].any(), f"path {path}"
