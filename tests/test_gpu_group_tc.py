"""Per-group activation scales on the tcgen05 path (csrc/mq_group_tc.cu: group = 128, M >= 64, PAPER.md
line 441) against the oracle (oracle.quantize_act_group, oracle.forward_group): codes and scale bits equal, the per-group
int32 accumulators [K/128, M, N] bit-exact (parity hooks = the kernel's second instantiation), Y within tolerance T2
(tests/test_gpu_group.py), for the hooked AND the hook-free instantiation.

The cases aim at what is specific to this kernel: an accumulator that is drained after EVERY K-step (two buffers, handed
back and forth between the MMA warp and eight epilogue warps), a residual accumulator handed over per cell, group scales
requested two K-steps ahead across tile boundaries, channel scales applied once per tile (and the tiles where that is
not possible), ragged last token tiles, K-step counts around the ring depths and the
32-K-step metadata chunk, tiles with a cell in every K-step and in none, more tiles than CTAs, both output types, the
transposed (vector) and the unaligned (scalar) output store, and repeated calls on a long-K layer that must give the
same bits every time (the packed-stage hand-off hazard this kernel exposed).
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import synth
from helpers import Case, make_case, pack_from_oracle, to_device_act
from test_gpu_group import check, run_group

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_2606_15652_b200 as m
    m.lib()
    for k in ("group_simt", "split_k", "token_tile", "max_ctas"):
        m.mq_set_option(k, 0)
    m.mq_set_option("group_tc", 1)
    return m


def want_of(case, rows=None, cols=None):
    A = case.A16 if case.a_dtype == "f16" else (case.A16, "bf16")
    return oracle.forward_group(A, case.L, 128, cols=cols, rows=rows)


@pytest.mark.parametrize("out_dtype", ["bf16", "f16"])
@pytest.mark.parametrize("M", [64, 65, 127, 128, 129, 200, 333])
def test_group_tc_token_counts(mq, M, out_dtype):
    case = make_case(1400 + M, M, 640, 256, bs=64, rho=0.10, a_dtype="f16" if M % 2 else "bf16")
    w = pack_from_oracle(case)
    want = want_of(case)
    for dbg in (True, False):
        got = run_group(mq, case, 128, w, out_dtype=out_dtype, dbg=dbg)
        assert mq.mq_last_launch_count() == 1
        check(got, want, 128, case.K, out_dtype, f"group tc M{M} {out_dtype} dbg {dbg}")
    assert np.abs(want["acc1_g"]).sum() > 0


@pytest.mark.parametrize("K", [128, 256, 384, 1152, 2176, 4224, 4480])
def test_group_tc_k_steps(mq, K):
    """1, 2, 3, 9, 17, 33 and 35 K-steps (groups); three calls in a row on one handle."""
    case = make_case(1430 + K // 128, 192, K, 256, bs=64, rho=0.12)
    w = pack_from_oracle(case)
    want = want_of(case)
    for rep in range(3):
        got = run_group(mq, case, 128, w, dbg=(rep == 0))
        check(got, want, 128, K, "bf16", f"group tc K{K} rep {rep}")


@pytest.mark.parametrize("bs,budget_frac", [(64, 1.0), (128, 1.0), (64, 0.5), (128, 0.25), (64, 0.0)])
def test_group_tc_residual_density(mq, bs, budget_frac):
    """A cell (a residual item and a residual epilogue pass) in every K-step, in some, in none."""
    case = make_case(1460 + bs, 160, 1024, 512, bs=bs, rho=budget_frac)
    w = pack_from_oracle(case)
    want = want_of(case)
    for dbg in (True, False):
        got = run_group(mq, case, 128, w, dbg=dbg)
        check(got, want, 128, case.K, "bf16", f"group tc bs {bs} budget {budget_frac} dbg {dbg}")


def test_group_tc_irregular_block_pattern(mq):
    rng = np.random.default_rng(1475)
    N, K, bs, M = 512, 2560, 64, 150
    W = synth.gen_weight(1475, N, K)
    d = oracle.decompose(W)
    for trial, dens in enumerate([0.03, 0.2, 0.6]):
        nb = (N // bs) * (K // bs)
        sel = np.sort(rng.choice(nb, size=int(nb * dens), replace=False))
        L = oracle.PackedLayer(N, K, bs, d, None, (sel // (K // bs)).astype(np.int32), (sel % (K // bs)).astype(np.int32))
        case = Case(M, K, N, bs, W, None, synth.gen_act(1475 + trial, M, K), "f16", L)
        w = pack_from_oracle(case)
        got = run_group(mq, case, 128, w, dbg=(trial != 1))
        check(got, want_of(case), 128, K, "bf16", f"group tc irregular blocks, density {dens}")


def test_group_tc_channels_with_a_zero_scale(mq):
    """The kernel keeps its running sums in units of s_w (channel scale applied once per tile) and falls back to units
    of 1 for a tile that holds a channel with s_w = 0.  (a) all-zero weight rows (the oracle gives them scale 1 and
    codes 0: output exactly 0), (b) a channel whose base scale is forced to 0 while its residual blocks and s_r stay
    (only the residual term is left) and one with both scales forced to 0 (output 0), next to regular tiles in the same
    launch."""
    rng = np.random.default_rng(1477)
    N, K, bs, M = 384, 1024, 64, 150
    W = synth.gen_weight(1477, N, K)
    W[5, :] = 0.0
    W[130:134, :] = 0.0
    d = oracle.decompose(W)
    assert not d.qw[5].any() and not d.qr[5].any()
    nb = (N // bs) * (K // bs)
    sel = np.sort(rng.choice(nb, size=nb // 4, replace=False))
    L = oracle.PackedLayer(N, K, bs, d, None, (sel // (K // bs)).astype(np.int32), (sel % (K // bs)).astype(np.int32))
    case = Case(M, K, N, bs, W, None, synth.gen_act(1477, M, K), "f16", L)
    for variant in ("zero rows", "base scale forced to 0"):
        if variant != "zero rows":
            d.sw[200] = 0.0          # tile 1 of 3; its blocks and s_r stay
            d.sw[201] = 0.0
            d.sr[201] = 0.0
            assert d.sr[200] != 0.0
        w = pack_from_oracle(case)
        want = want_of(case)
        for dbg in (True, False):
            got = run_group(mq, case, 128, w, dbg=dbg)
            check(got, want, 128, K, "bf16", f"group tc, {variant}, dbg {dbg}")
        assert not got["Y"][:, 5].any() and not got["Y"][:, 130:134].any()
    assert np.abs(want["Y"][:, 200]).sum() > 0 and not got["Y"][:, 201].any()


def test_group_tc_more_tiles_than_ctas(mq):
    """N = 2048, M = 2100: 16 x 17 = 272 tiles for 148 CTAs: one and two tiles per CTA, ragged last token tile."""
    case = make_case(1480, 2100, 512, 2048, bs=64, rho=0.06)
    w = pack_from_oracle(case)
    rows = np.unique(np.concatenate([np.arange(0, 2100, 53), np.arange(2040, 2100)]))
    want = want_of(case, rows=rows)
    got = run_group(mq, case, 128, w, dbg=False)
    check(got, want, 128, case.K, "bf16", "group tc 272 tiles", rows=rows)


def test_group_tc_unaligned_output_rows(mq):
    """Y with a row stride that is not a multiple of 8 elements: the scalar store path of the transposed tile."""
    import torch
    case = make_case(1485, 140, 512, 256, bs=64, rho=0.10)
    w = pack_from_oracle(case)
    want = want_of(case)
    A = to_device_act(case)
    qA, sA = mq.mq_quantize_act_group(A, 128)
    big = torch.zeros((140, 256 + 3), dtype=torch.bfloat16, device="cuda")
    Y = big[:, :256]
    mq.mq_gemm_group(w, qA, sA, 128, 140, Y=Y)
    torch.cuda.synchronize()
    assert not big[:, 256:].any(), "wrote past the row"
    q = mq.mq_unpack_act(qA, 140, 512)
    got = dict(qa=q.cpu().numpy(), sa=sA.cpu().numpy(), Y=Y.float().cpu().numpy().astype(np.float64), acc0_g=None, acc1_g=None)
    check(got, want, 128, 512, "bf16", "group tc, unaligned Y rows")


def test_group_tc_matches_the_mma_sync_kernel_and_repeats_bit_for_bit(mq):
    """A long-K layer (112 K-steps, 2048 tiles): five calls give the same bits, and, where no K-step owns a cell, the
    bits of the mma.sync kernel (same arithmetic in the same order).  Before the packed-stage hand-off was made to
    depend on the loaded data, a few tiles per call came out with another K-step's tokens."""
    import torch
    K, N, M = 14336, 4096, 8192
    rng = np.random.default_rng(1490)
    qw = rng.integers(-7, 8, size=(N, K)).astype(np.int8)
    w = mq.mq_pack_prequantized(qw, np.ones(N, np.float32), 64, np.zeros(0, np.int32), np.zeros(0, np.int32),
                                np.zeros((0, 64, 64), np.int8), np.ones(N, np.float32))
    A = torch.randn((M, K), device="cuda", dtype=torch.float16, generator=torch.Generator(device="cuda").manual_seed(1490))
    qg, sg = mq.mq_quantize_act_group(A, 128)
    try:
        mq.mq_set_option("group_tc", 0)
        ref = mq.mq_gemm_group(w, qg, sg, 128, M, out_dtype=torch.float16).clone()
    finally:
        mq.mq_set_option("group_tc", 1)
    for rep in range(5):
        y = mq.mq_gemm_group(w, qg, sg, 128, M, out_dtype=torch.float16)
        torch.cuda.synchronize()
        assert torch.equal(y.view(torch.int16), ref.view(torch.int16)), f"call {rep} differs"
