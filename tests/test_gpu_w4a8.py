"""W4A8 variant (Table 1 W4A8 rows): per-token int8 activations against the
same packed int4 base + residual weights.  Same parity bar as W4A4: quantized activations and scales
bit-exact against the oracle (q_max = 127), acc0 / acc1 bit-exact, Y within tolerance."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from helpers import assert_parity, make_case, oracle_forward, pack_from_oracle, run_cuda

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


SHAPES = [
    (1, 512, 256, 64, 0.10, "f16"), (8, 1024, 384, 64, 0.05, "bf16"), (17, 640, 256, 64, 0.20, "f16"),
    (33, 1024, 512, 128, 0.25, "f16"), (64, 2048, 256, 64, 0.3, "f16"), (100, 512, 384, 64, 0.10, "bf16"),
    (130, 512, 256, 128, 0.50, "f16"), (300, 1024, 640, 64, 0.05, "bf16"),
]


@pytest.mark.parametrize("out_dtype", ["bf16", "f16"])
@pytest.mark.parametrize("M,K,N,bs,rho,dt", SHAPES)
def test_w4a8_parity_small(mq, M, K, N, bs, rho, dt, out_dtype):
    case = make_case(700 + M, M, K, N, bs=bs, rho=rho, a_dtype=dt)
    want = oracle_forward(case, bits=8)
    assert np.abs(want["qa"].astype(np.int32)).max() == 127
    got = run_cuda(case, out_dtype=out_dtype, bits=8)
    assert_parity(got, want, what=f"W4A8 M{M} K{K} N{N} bs{bs} {out_dtype}")


@pytest.mark.parametrize("rows", [16, 32, 64, 128])
@pytest.mark.parametrize("M", [1, 7, 8, 9, 16, 17, 32])
def test_w4a8_decode_kernel_variants(mq, rows, M):
    """W4A8 at M <= 32 runs in the row-slab decode kernel's A8 form (csrc/mq_decode.cu: int8 tokens as they are, weight
    nibbles expanded in canonical order): every slab height (option decode_rows) x every token-count class, K-step counts
    that do not fill the last stage, a residual piece in most K-steps; one launch where the form is eligible (32 token
    columns need slabs of 64 channels or more; the stream-K kernel takes the rest), two calls on one handle."""
    K = {16: 640, 32: 1152, 64: 2432, 128: 640}[rows]
    case = make_case(1700 + 40 * rows + M, M, K, 256, bs=64, rho=0.35, a_dtype="bf16" if M % 2 else "f16")
    want = oracle_forward(case, bits=8)
    assert np.abs(want["acc1"]).sum() > 0
    w = pack_from_oracle(case)
    ws = mq.new_workspace(mq.mq_gemm_workspace_bytes(w, M))
    try:
        mq.mq_set_option("decode_rows", rows)
        for rep in range(2):
            got = run_cuda(case, w=w, workspace=ws, out_dtype="bf16" if rep else "f16", bits=8)
            if M <= 16 or rows >= 64:
                assert mq.mq_last_launch_count() == 1
            assert_parity(got, want, what=f"W4A8 decode kernel rows {rows} M{M} rep {rep}")
    finally:
        mq.mq_set_option("decode_rows", 0)


@pytest.mark.parametrize("mode,ctas,bt", [(2, 0, 0), (2, 7, 0), (2, 33, 32), (1, 0, 64), (2, 5, 128), (1, 0, 16)])
def test_w4a8_stream_k_and_token_tiles(mq, mode, ctas, bt):
    M = 40 if bt in (0, 64) else (12 if bt == 16 else (30 if bt == 32 else 150))
    case = make_case(800 + bt + ctas, M, 2048, 384, bs=64, rho=0.2)
    want = oracle_forward(case, bits=8)
    try:
        mq.mq_set_option("split_k", mode)
        mq.mq_set_option("max_ctas", ctas)
        mq.mq_set_option("token_tile", bt)
        w = pack_from_oracle(case)
        ws = mq.new_workspace(mq.mq_gemm_workspace_bytes(w, M))
        for rep in range(2):
            got = run_cuda(case, w=w, workspace=ws, bits=8)
            assert_parity(got, want, what=f"W4A8 split_k {mode} ctas {ctas} bt {bt} rep {rep}")
    finally:
        for k in ("split_k", "max_ctas", "token_tile"):
            mq.mq_set_option(k, 0)


def test_w4a8_extreme_values_and_full_size(mq):
    """all +-127 x +-7: |acc0| = 889 K exactly (int32 head-room of the x16 weight expansion); then a
    LLaMA3-8B-sized decode and prefill projection on sampled rows."""
    import torch
    M, K, N = 8, 4096, 128
    qw = np.full((N, K), 7, np.int8)
    qw[1::2] = -7
    s1 = np.ones(N, np.float32)
    w = mq.mq_pack_prequantized(qw, s1, 64, np.zeros(0, np.int32), np.zeros(0, np.int32), np.zeros((0, 64, 64), np.int8), s1)
    A = torch.full((M, K), 3.0, dtype=torch.float16, device="cuda")
    q8, sA = mq.mq_quantize_act8(A)
    assert int(q8.min()) == 127
    Y, d0, d1 = mq.mq_gemm_a8(w, q8, sA, M, dbg=True)
    torch.cuda.synchronize()
    assert np.array_equal(np.abs(d0.cpu().numpy()), np.full((M, N), 889 * K)) and not d1.cpu().numpy().any()
    for (Mf, Kf, Nf) in [(8, 4096, 6144), (512, 4096, 4096)]:
        case = make_case(880 + Mf, Mf, Kf, Nf, bs=64, rho=0.05, calib_tokens=64)
        rows = np.arange(Mf) if Mf <= 64 else np.sort(np.random.default_rng(1).choice(Mf, size=64, replace=False))
        want = oracle_forward(case, rows=rows, bits=8)
        got = run_cuda(case, bits=8)
        assert_parity(got, want, rows=rows, what=f"W4A8 full size M{Mf}")


def test_w4a8_seeded_fuzz_against_oracle(mq):
    """30 seeded random combinations of shape, block size, density (uniform-random block pattern: cells with
    every quarter mask) and launch options: int8 codes, scales and accumulators bit-exact, Y in tolerance; the
    epilogue's hot path (no parity hooks) must reproduce the hooked path's Y bits."""
    import dataclasses
    import torch
    from helpers import to_device_act
    rng = np.random.default_rng(4242)
    try:
        for ci in range(30):
            bs = int(rng.choice([64, 128]))
            K = int(rng.choice([128, 256, 640, 1024, 2048]))
            N = int(rng.choice([128, 256, 384, 512]))
            M = int(rng.choice([1, 3, 16, 17, 32, 33, 64, 65, 100, 128, 129, 256, 300]))
            rho = float(rng.choice([0.0, 0.05, 0.1, 0.3, 0.6, 1.0]))
            opts = dict(split_k=int(rng.choice([0, 0, 1, 2])), max_ctas=int(rng.choice([0, 0, 7, 33])),
                        pdl=int(rng.choice([1, 1, 0])), token_tile=int(rng.choice([0, 0, 16, 32, 64, 128])))
            for k, v in opts.items():
                mq.mq_set_option(k, v)
            case = make_case(5000 + ci, M, K, N, bs=bs, budget=0)
            nb = (N // bs) * (K // bs)
            sel = np.sort(np.random.default_rng(5000 + ci).choice(nb, size=int(rho * nb + 0.5), replace=False))
            case = dataclasses.replace(case, L=dataclasses.replace(
                case.L, blk_n=(sel // (K // bs)).astype(np.int32), blk_k=(sel % (K // bs)).astype(np.int32)))
            want = oracle_forward(case, bits=8)
            w = pack_from_oracle(case)
            ws = mq.new_workspace(mq.mq_gemm_workspace_bytes(w, M))
            got = run_cuda(case, w=w, workspace=ws, bits=8)
            assert_parity(got, want, what=f"W4A8 fuzz {ci}: M{M} K{K} N{N} bs{bs} rho{rho} {opts}")
            q8, s8 = mq.mq_quantize_act8(to_device_act(case))
            Y = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
            for _ in range(2):
                mq.mq_gemm_a8(w, q8, s8, M, Y=Y, workspace=ws)
            torch.cuda.synchronize()
            assert np.array_equal(Y.float().cpu().numpy().astype(np.float64), got["Y"]), f"W4A8 fuzz {ci}: hot path differs"
    finally:
        for k in ("split_k", "max_ctas", "token_tile"):
            mq.mq_set_option(k, 0)
        mq.mq_set_option("pdl", 1)


# ---------------------------------------------------------------------------------------------------------------------
# W4A8 on the whole-tile kernel (csrc/mq_prefill.cu, template A8: the int8 token tile of a K-step goes by TMA straight
# into the MMA's operand stage, the weights are expanded in canonical element order).  mq_gemm_a8 picks it by itself for
# large M (the full-size cases of test_gpu_fullsize.py); option "prefill_path" = 2 forces it on small shapes.
def with_prefill(mq, fn, path=2):
    try:
        mq.mq_set_option("prefill_path", path)
        return fn()
    finally:
        mq.mq_set_option("prefill_path", 0)


@pytest.mark.parametrize("out_dtype", ["bf16", "f16"])
@pytest.mark.parametrize("M", [64, 65, 128, 129, 200, 333])
def test_w4a8_whole_tile_token_counts(mq, M, out_dtype):
    case = make_case(1500 + M, M, 640, 512, bs=64, rho=0.10, a_dtype="f16" if M % 2 else "bf16")
    want = oracle_forward(case, bits=8)
    got = with_prefill(mq, lambda: run_cuda(case, out_dtype=out_dtype, bits=8))
    assert mq.mq_last_launch_count() == 1
    assert_parity(got, want, what=f"W4A8 whole-tile M{M} {out_dtype}")
    assert np.abs(want["acc1"]).sum() > 0


@pytest.mark.parametrize("K", [128, 384, 1152, 4224, 4480])
def test_w4a8_whole_tile_k_steps(mq, K):
    case = make_case(1530 + K // 128, 192, K, 256, bs=64, rho=0.12)
    want = oracle_forward(case, bits=8)
    w = pack_from_oracle(case)

    def run():
        for rep in range(3):
            assert_parity(run_cuda(case, w=w, bits=8), want, what=f"W4A8 whole-tile K{K} rep {rep}")
    with_prefill(mq, run)


@pytest.mark.parametrize("bs,budget_frac", [(64, 1.0), (128, 1.0), (64, 0.5), (64, 0.0)])
def test_w4a8_whole_tile_residual_density(mq, bs, budget_frac):
    case = make_case(1560 + bs, 160, 1024, 512, bs=bs, rho=budget_frac)
    want = oracle_forward(case, bits=8)
    got = with_prefill(mq, lambda: run_cuda(case, bits=8))
    assert_parity(got, want, what=f"W4A8 whole-tile bs {bs} budget {budget_frac}")


def test_w4a8_whole_tile_many_tiles_and_path_3(mq):
    """N = 2048, M = 1100: 16 x 9 = 144 tiles; option 3 (CTA pairs) falls back to the single-CTA form for W4A8."""
    case = make_case(1570, 1100, 512, 2048, bs=64, rho=0.06)
    rows = np.unique(np.concatenate([np.arange(0, 1100, 37), np.arange(1020, 1100)]))
    want = oracle_forward(case, rows=rows, bits=8)
    for path in (2, 3):
        got = with_prefill(mq, lambda: run_cuda(case, rows=rows, bits=8), path)
        assert_parity(got, want, rows=rows, what=f"W4A8 whole-tile 144 tiles, path {path}")


def test_w4a8_whole_tile_extremes(mq):
    """+-127 tokens against +-7 weights: |acc0| = 127 * 7 * K exactly through the x16 accumulators."""
    import torch
    M, K, N = 130, 4096, 256
    qw = np.full((N, K), 7, np.int8)
    qw[1::2] = -7
    s1 = np.ones(N, np.float32)
    w = mq.mq_pack_prequantized(qw, s1, 64, np.array([0, 1], np.int32), np.array([0, K // 64 - 1], np.int32),
                                np.full((2, 64, 64), -7, np.int8), s1)
    A = torch.full((M, K), 127.0, dtype=torch.float16, device="cuda")
    q8, sA = mq.mq_quantize_act8(A)
    Y, d0, d1 = with_prefill(mq, lambda: mq.mq_gemm_a8(w, q8, sA, M, dbg=True))
    torch.cuda.synchronize()
    d0, d1 = d0.cpu().numpy(), d1.cpu().numpy()
    assert (d0[:, 0::2] == 127 * 7 * K).all() and (d0[:, 1::2] == -127 * 7 * K).all()
    assert (d1[:, :128] == -127 * 7 * 64).all() and not d1[:, 128:].any()
