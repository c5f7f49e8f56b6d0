"""The paper's naive 3-kernel pipeline (Fig.3), built for the
fused-vs-naive ablation: dense GEMM with the residual switched off, a separate sparse-block GEMM that writes the
int32 partial output acc1, a reduce-add.  acc1 must be bit-exact against the oracle; Y is rounded twice (the dense
GEMM's 16-bit output, then the sum), so its tolerance is one 16-bit unit of the larger of |Y0| and |Y|."""
from __future__ import annotations

import numpy as np
import pytest

from helpers import Y_MAG_TOL, make_case, oracle_forward, pack_from_oracle, to_device_act

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_2606_15652_b200 as m
    m.lib()
    return m


@pytest.mark.parametrize("out_dtype", ["bf16", "f16"])
@pytest.mark.parametrize("M,K,N,bs,rho", [(1, 512, 256, 64, 0.10), (8, 1024, 384, 64, 0.05), (17, 640, 256, 64, 0.3),
                                          (33, 1024, 512, 128, 0.25), (130, 512, 256, 64, 0.5), (300, 2048, 640, 64, 0.05),
                                          (16, 1024, 256, 64, 0.0)])
def test_naive_pipeline_parity(mq, M, K, N, bs, rho, out_dtype):
    import torch
    case = make_case(1200 + M, M, K, N, bs=bs, rho=rho)
    want = oracle_forward(case)
    w = pack_from_oracle(case)
    qA, sA = mq.mq_quantize_act(to_device_act(case))
    dt = torch.bfloat16 if out_dtype == "bf16" else torch.float16
    Y, acc1 = mq.mq_gemm_naive(w, qA, sA, M, out_dtype=dt)
    Yf = mq.mq_gemm(w, qA, sA, M, out_dtype=dt)
    torch.cuda.synchronize()
    assert np.array_equal(acc1.cpu().numpy().astype(np.int64), want["acc1"]), "sparse-block GEMM: acc1 not bit-exact"
    y = Y.float().cpu().numpy().astype(np.float64)
    sa = want["sa"].astype(np.float64)[:, None]
    y0 = sa * (case.L.d.sw.astype(np.float64)[None, :] * want["acc0"])          # the dense kernel's exact output
    ulp = 2.0 ** -8 if out_dtype == "bf16" else 2.0 ** -11
    tol = ulp * (np.abs(y0) + np.abs(want["Y"])) + Y_MAG_TOL * want["mag"]
    err = np.abs(y - want["Y"])
    assert (err <= tol).all(), f"naive Y out of tolerance at {int((err > tol).sum())} (max excess {float((err - tol).max()):.3e})"
    # and it stays within two 16-bit units of the fused kernel's Y
    yf = Yf.float().cpu().numpy().astype(np.float64)
    assert (np.abs(y - yf) <= 2 * ulp * (np.abs(y0) + np.abs(want["Y"])) + Y_MAG_TOL * want["mag"]).all()


def test_naive_pipeline_rejects_small_scratch(mq):
    import torch
    case = make_case(1300, 8, 512, 256, bs=64, rho=0.1)
    w = pack_from_oracle(case)
    qA, sA = mq.mq_quantize_act(to_device_act(case))
    assert mq.mq_gemm_naive_scratch_bytes(w, 8) == 8 * 256 * 4
    small = torch.empty(16, dtype=torch.int32, device="cuda")
    with pytest.raises(RuntimeError):
        mq.mq_gemm_naive(w, qA, sA, 8, scratch=small)
