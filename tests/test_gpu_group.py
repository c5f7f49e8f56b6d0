"""per-group activation quantization through the C ABI
(mq_quantize_act_group, mq_gemm_group) against the oracle (oracle.quantize_act_group, oracle.forward_group):
codes and scale bits equal, the per-group int32 accumulators [K/group, M, N] bit-exact, Y within

    |Y - Y_exact| <= (output rounding: half a bf16 ulp / 2e-3 relative + 2^-25 absolute for fp16) + (2 G + 4) 2^-24 mag

mag = sum_g s_a (|s_w acc0_g| + |s_r acc1_g|): the base and the residual product of every group are each rounded once
and added to the fp32 running sum, together (mma.sync kernel: G additions) or one after the other (tcgen05 kernel: up to
2 G additions), tolerance T2.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import synth
from helpers import make_case, pack_from_oracle, to_device_act, y_tolerance

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_2606_15652_b200 as m
    m.lib()
    return m


def run_group(mq, case, group, w, out_dtype="bf16", dbg=True):
    import torch
    A = to_device_act(case)
    odt = torch.bfloat16 if out_dtype == "bf16" else torch.float16
    qA, sA = mq.mq_quantize_act_group(A, group)
    assert mq.mq_last_launch_count() == (1 if case.M else 0)
    if dbg:
        Y, d0, d1 = mq.mq_gemm_group(w, qA, sA, group, case.M, out_dtype=odt, dbg=True)
    else:
        Y, d0, d1 = mq.mq_gemm_group(w, qA, sA, group, case.M, out_dtype=odt), None, None
    torch.cuda.synchronize()
    q = mq.mq_unpack_act(qA, case.M, case.K)
    return dict(qa=q.cpu().numpy(), sa=sA.cpu().numpy(), Y=Y.float().cpu().numpy().astype(np.float64),
                acc0_g=None if d0 is None else d0.cpu().numpy(), acc1_g=None if d1 is None else d1.cpu().numpy())


def check(got, want, group, K, out_dtype, what, rows=None, cols=None):
    sel = (lambda x: x) if rows is None else (lambda x: x[rows])
    assert np.array_equal(sel(got["sa"]).view(np.uint32), want["sa"].view(np.uint32)), f"{what}: group scales differ"
    assert np.array_equal(sel(got["qa"]), want["qa"]), f"{what}: activation codes differ"
    def sub(x):
        if rows is not None:
            x = x[:, rows] if x.ndim == 3 else x[rows]
        if cols is not None:
            x = x[..., cols]
        return x
    if got["acc0_g"] is not None:
        assert np.array_equal(sub(got["acc0_g"]).astype(np.int64), want["acc0_g"]), f"{what}: base group accumulators not bit-exact"
        assert np.array_equal(sub(got["acc1_g"]).astype(np.int64), want["acc1_g"]), f"{what}: residual group accumulators not bit-exact"
    G = K // group
    tol = y_tolerance(want["Y"], 0.0 * want["mag"], out_dtype) + (2 * G + 4) * 2.0 ** -24 * want["mag"]
    if out_dtype == "f16":
        tol = tol + 2.0 ** -25    # fp16 values are never closer than 2^-24 (subnormal spacing): half of it
    err = np.abs(sub(got["Y"]) - want["Y"])
    bad = err > tol
    assert not bad.any(), f"{what}: Y out of tolerance at {int(bad.sum())} of {bad.size} (max excess {float((err - tol).max()):.3e})"


def A_of(case):
    return case.A16 if case.a_dtype == "f16" else (case.A16, "bf16")


# several n-tiles and token tiles, ragged token tails, K-split on and off, both block sizes, dense rows of cells
SHAPES = [
    (16, 256, 256, 64, None, "f16"),      # BASELINE configs[0] (budget 2 of 16)
    (1, 512, 256, 64, 0.10, "f16"), (8, 1024, 384, 64, 0.05, "bf16"), (17, 640, 256, 64, 0.20, "f16"),
    (33, 1024, 512, 128, 0.25, "f16"), (64, 2048, 256, 64, 0.3, "f16"), (100, 512, 384, 64, 0.10, "bf16"),
    (130, 512, 256, 128, 0.50, "f16"), (300, 1024, 640, 64, 0.05, "bf16"), (5, 4096, 128, 64, 1.0, "f16"),
    (700, 256, 5120, 64, 0.05, "f16"),    # >= 296 CTAs: no K-split
]


@pytest.mark.parametrize("group", [32, 64, 128])
@pytest.mark.parametrize("M,K,N,bs,rho,dt", SHAPES)
def test_group_parity_small(mq, M, K, N, bs, rho, dt, group):
    case = make_case(1200 + M, M, K, N, bs=bs, rho=rho, budget=2 if rho is None else None, a_dtype=dt)
    want = oracle.forward_group(A_of(case), case.L, group)
    w = pack_from_oracle(case)
    out = "bf16" if (M + group) % 3 else "f16"
    got = run_group(mq, case, group, w, out_dtype=out)
    check(got, want, group, K, out, f"group {group} M{M} K{K} N{N} bs{bs} {out}")


@pytest.mark.parametrize("M,K,N,bs,rho,dt", [SHAPES[0], SHAPES[1], SHAPES[3], SHAPES[4], SHAPES[8]])
def test_group_parity_simt_kernel_every_m(mq, M, K, N, bs, rho, dt):
    """Option group_simt = 1: the dp4a kernel (not used by default) on single- and multi-token shapes."""
    case = make_case(1200 + M, M, K, N, bs=bs, rho=rho, budget=2 if rho is None else None, a_dtype=dt)
    w = pack_from_oracle(case)
    try:
        mq.mq_set_option("group_simt", 1)
        for group in (32, 128):
            want = oracle.forward_group(A_of(case), case.L, group)
            got = run_group(mq, case, group, w)
            check(got, want, group, K, "bf16", f"simt group {group} M{M} K{K} N{N}")
    finally:
        mq.mq_set_option("group_simt", 0)


@pytest.mark.parametrize("rows", [16, 32, 64, 128])
@pytest.mark.parametrize("M", [1, 7, 8, 9, 16, 17, 31, 32])
def test_group128_decode_kernel_variants(mq, rows, M):
    """Group 128 at M <= 32 runs in the row-slab decode kernel (csrc/mq_decode.cu, GRP form: the sums of a K-step are
    converted and added right after its MMAs).  Every slab height (option decode_rows) x every token-count class (8 / 16
    / 32 token columns, ragged), K-step counts that do not fill the last stage (5, 9, 19 K-steps), a cell in most
    K-steps, hooks on and off, both output types; one launch."""
    K = {16: 640, 32: 1152, 64: 2432, 128: 640}[rows]
    case = make_case(1500 + 40 * rows + M, M, K, 256, bs=64, rho=0.35, a_dtype="bf16" if M % 2 else "f16")
    w = pack_from_oracle(case)
    want = oracle.forward_group(A_of(case), case.L, 128)
    assert np.abs(want["acc1_g"]).sum() > 0
    try:
        mq.mq_set_option("decode_rows", rows)
        for dbg in (True, False):
            out = "bf16" if (M + rows // 16 + dbg) % 2 else "f16"
            got = run_group(mq, case, 128, w, out_dtype=out, dbg=dbg)
            assert mq.mq_last_launch_count() == 1
            check(got, want, 128, K, out, f"group 128 decode kernel rows {rows} M{M} dbg {dbg}")
    finally:
        mq.mq_set_option("decode_rows", 0)


def test_group128_decode_kernel_and_mma_sync_kernel_agree(mq):
    """The same launch through both kernels (option group_tc = 0 selects the mma.sync kernel for every M): the same
    integer sums, both outputs within T2 of the oracle (their fp32 additions are ordered differently), K = 4096."""
    case = make_case(1590, 32, 4096, 512, bs=64, rho=0.10)
    w = pack_from_oracle(case)
    want = oracle.forward_group(A_of(case), case.L, 128)
    got1 = run_group(mq, case, 128, w, out_dtype="f16")
    try:
        mq.mq_set_option("group_tc", 0)
        got2 = run_group(mq, case, 128, w, out_dtype="f16")
    finally:
        mq.mq_set_option("group_tc", 1)
    assert np.array_equal(got1["acc0_g"], got2["acc0_g"]) and np.array_equal(got1["acc1_g"], got2["acc1_g"])
    check(got1, want, 128, 4096, "f16", "group 128, M 32, decode kernel")
    check(got2, want, 128, 4096, "f16", "group 128, M 32, mma.sync kernel")


def test_group_budget_zero_and_whole_row_group(mq):
    """Budget 0: acc1_g == 0 and Y is the dense-only product.  Activations constant along K in magnitude per group:
    every group scale equal, so the per-group result must agree with the per-token path (mq_gemm) to rounding."""
    import torch
    case = make_case(1300, 24, 1024, 256, bs=64, budget=0)
    w = pack_from_oracle(case)
    for group in (32, 128):
        want = oracle.forward_group(A_of(case), case.L, group)
        got = run_group(mq, case, group, w)
        assert not got["acc1_g"].any()
        check(got, want, group, case.K, "bf16", f"budget 0 group {group}")
    # +-c per token: one scale for every group of a row, identical codes on both paths
    rng = np.random.default_rng(5)
    sign = rng.choice([-1.0, 1.0], size=(24, 1024))
    amp = rng.uniform(0.5, 2.0, size=(24, 1)).astype(np.float16)
    case2 = make_case(1301, 24, 1024, 256, bs=64, rho=0.2)
    case2.A16 = (sign * amp).astype(np.float16)
    w2 = pack_from_oracle(case2)
    got = run_group(mq, case2, 64, w2)
    A = to_device_act(case2)
    qA, sA = mq.mq_quantize_act(A)
    Yt, d0, d1 = mq.mq_gemm(w2, qA, sA, 24, dbg=True)
    torch.cuda.synchronize()
    assert np.array_equal(got["acc0_g"].sum(0), d0.cpu().numpy()) and np.array_equal(got["acc1_g"].sum(0), d1.cpu().numpy())
    assert np.array_equal(got["sa"], np.repeat(sA.cpu().numpy()[:, None], 16, axis=1))
    want = oracle.forward_group(A_of(case2), case2.L, 64)
    check(got, want, 64, 1024, "bf16", "constant-magnitude rows")


def test_group_empty_and_errors(mq):
    import torch
    case = make_case(1400, 4, 2048, 256, bs=64, rho=0.1)    # 16 K-steps, 2 CTAs: the K-split is on
    w = pack_from_oracle(case)
    A = to_device_act(case)
    for bad in (0, 16, 48, 256):
        with pytest.raises(mq.MqError) as e:
            mq.mq_quantize_act_group(A, bad)
        assert e.value.status == -2
    qA, sA = mq.mq_quantize_act_group(A, 64)
    with pytest.raises(mq.MqError):
        mq.mq_gemm_group(w, qA, sA, 48, 4)
    Y = torch.full((0, 256), 0, dtype=torch.bfloat16, device="cuda")
    mq.mq_gemm_group(w, qA, sA, 64, 0, Y=Y)
    assert mq.mq_last_launch_count() == 0
    need = mq.mq_gemm_group_workspace_bytes(w, 4)
    assert need > 0
    small = torch.empty(16, dtype=torch.uint8, device="cuda")
    with pytest.raises(mq.MqError) as e:
        mq.mq_gemm_group(w, qA, sA, 64, 4, workspace=small)
    assert e.value.status == -7
    # strided Y (ldy > N) and repeated calls give the same bits
    Yw = torch.zeros((4, 384), dtype=torch.bfloat16, device="cuda")
    mq.mq_gemm_group(w, qA, sA, 64, 4, Y=Yw[:, :256])
    Y2 = mq.mq_gemm_group(w, qA, sA, 64, 4)
    torch.cuda.synchronize()
    assert torch.equal(Yw[:, :256], Y2) and not Yw[:, 256:].any()


FULL = [("decode qkv M=1", 1, 4096, 6144, 128), ("decode gate_up M=32", 32, 4096, 28672, 64),
        ("decode down M=8", 8, 14336, 4096, 32), ("prefill o M=512", 512, 4096, 4096, 128)]


@pytest.mark.parametrize("name,M,K,N,group", FULL)
def test_group_full_size_sampled(mq, name, M, K, N, group):
    """BASELINE.json configs[1] / configs[2] sizes, the library's own Algorithm 1 packing, no parity hooks (the launch a
    user makes): sampled token rows x sampled output channels against the oracle."""
    case = make_case(9000 + M + N, M, K, N, bs=64, rho=0.05, calib_tokens=64)
    w = mq.mq_pack_weights(case.W, case.h, 64, synth.budget_from_density(0.05, N, K, 64))
    rng = np.random.default_rng(M + N + group)
    rows = np.arange(M) if M <= 32 else np.sort(rng.choice(M, size=32, replace=False))
    cols = np.sort(rng.choice(N, size=512, replace=False))
    want = oracle.forward_group(A_of(case), case.L, group, cols=cols, rows=rows)
    got = run_group(mq, case, group, w, dbg=False)
    check(got, want, group, K, "bf16", name, rows=rows, cols=cols)
