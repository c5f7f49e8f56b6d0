"""mq_linear_static (include/mq.h): mq_linear on the library's built-in `static __device__` scratch array, for callers
that cannot allocate device memory.  Checked against the existing path (mq_linear with a caller workspace) on the same
inputs: same kernels, same arithmetic, so Y must be bit-identical (and, like the existing path's, inside tolerance T1 of
tests/helpers.py against the oracle), on two calls in a row (the array keeps the previous call's
contents), for the three GEMM kernels (decode kernel, stream-K kernel: the one that keeps counters and partial tiles in
the scratch, whole-tile kernel), and for sizes beyond the array (refused, nothing allocated).

The file name sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide other tests.
It passes alone in a fresh process and after the other GPU tests (it resets the options it depends on).
"""
from __future__ import annotations

import numpy as np
import pytest

from helpers import make_case, oracle_forward, pack_from_oracle, to_device_act, y_tolerance

pytestmark = pytest.mark.gpu

OPTS = ("split_k", "token_tile", "max_ctas", "fused_quant", "decode_path", "decode_rows", "decode_big", "prefill_path")


@pytest.fixture(scope="module")
def mq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_2606_15652_b200 as m
    m.lib()
    for k in OPTS:
        m.mq_set_option(k, 0)
    m.mq_set_option("pdl", 1)
    return m


# (M, K, N, options): decode kernel; stream-K kernel with split tiles (counters, flags and partial tiles live in the
# scratch array); stream-K kernel, M between the two specialised kernels; whole-tile kernel (CTA pairs), ragged tile
CASES = [
    (8, 2048, 512, {}),
    (16, 2048, 256, {"decode_path": 1}),
    (40, 1024, 512, {}),
    (200, 1024, 512, {}),
]


@pytest.mark.parametrize("M,K,N,opts", CASES)
def test_static_scratch_matches_workspace_path_twice(mq, M, K, N, opts):
    import torch
    case = make_case(1200 + M, M, K, N, bs=64, rho=0.10)
    w = pack_from_oracle(case)
    A = to_device_act(case)
    assert mq.mq_linear_workspace_bytes(w, M) <= mq.mq_linear_static_max_bytes()
    try:
        for k, v in opts.items():
            mq.mq_set_option(k, v)
        Y_ref = mq.mq_linear(w, A)                     # existing path: caller workspace (zeroed by the binding)
        torch.cuda.synchronize()
        n_launch = mq.mq_last_launch_count()
        outs = []
        for rep in range(2):                           # two calls in a row on the shared array
            Y = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device="cuda")
            before = torch.cuda.memory_allocated()
            mq.mq_linear_static(w, A, Y)
            assert torch.cuda.memory_allocated() == before
            assert mq.mq_last_launch_count() == n_launch
            torch.cuda.synchronize()
            outs.append(Y)
    finally:
        for k in opts:
            mq.mq_set_option(k, 0)
    want = oracle_forward(case)
    tol = y_tolerance(want["Y"], want["mag"], "bf16")
    ref = Y_ref.float().cpu().numpy().astype(np.float64)
    assert (np.abs(ref - want["Y"]) <= tol).all(), "existing path out of tolerance"
    for rep, Y in enumerate(outs):
        got = Y.float().cpu().numpy().astype(np.float64)
        assert (np.abs(got - want["Y"]) <= tol).all(), f"call {rep}: out of tolerance T1 against the oracle"
        assert torch.equal(Y.view(torch.int16), Y_ref.view(torch.int16)), f"call {rep}: differs from mq_linear"


def test_static_scratch_alternating_layers(mq):
    """Calls for different layers, block sizes and token counts (all three kernels) alternate on the one array: a call
    finds the previous call's partial tiles, flags and packed activations there and must not depend on them."""
    import torch
    cases = [make_case(1300, 12, 1536, 384, bs=64, rho=0.10), make_case(1301, 48, 768, 256, bs=128, rho=0.2),
             make_case(1302, 150, 512, 512, bs=64, rho=0.05)]
    ws = [pack_from_oracle(c) for c in cases]
    As = [to_device_act(c) for c in cases]
    refs = [mq.mq_linear(w, A) for w, A in zip(ws, As)]
    torch.cuda.synchronize()
    for rnd in range(3):
        for i in (2, 0, 1, 0, 2):
            Y = torch.empty_like(refs[i])
            mq.mq_linear_static(ws[i], As[i], Y)
            torch.cuda.synchronize()
            assert torch.equal(Y.view(torch.int16), refs[i].view(torch.int16)), f"round {rnd} layer {i}"


def test_static_scratch_rejects_sizes_beyond_the_array(mq):
    import torch
    case = make_case(1310, 4, 4096, 128, bs=64, rho=0.05)
    w = pack_from_oracle(case)
    M = 16384                                          # packed activations alone: 16384 x 2048 B = 32 MiB > 16 MiB
    assert mq.mq_linear_workspace_bytes(w, M) > mq.mq_linear_static_max_bytes() == 16 << 20
    A = torch.zeros((M, 4096), dtype=torch.float16, device="cuda")
    Y = torch.full((M, 128), 3.0, dtype=torch.bfloat16, device="cuda")
    before = torch.cuda.memory_allocated()
    with pytest.raises(mq.MqError) as e:
        mq.mq_linear_static(w, A, Y)
    assert e.value.status == -8 and "16 MiB" in str(e.value)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    assert bool((Y == 3.0).all()), "a refused call must not touch Y"
    # M = 0 is a no-op, as for mq_linear
    mq.mq_linear_static(w, A[:0], Y[:0])
