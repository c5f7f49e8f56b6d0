"""Writes tests/golden/config1_digest.json: digests of the ORACLE's outputs on BASELINE.json
configs[0] (M=16, K=256, N=256, 64x64 blocks, top-2 of 16, seed 0).  Calls only oracle/ and
synth/ -- never the CUDA path.  A drift guard, not a correctness pin: re-run (and say why in the
commit message) only when a PAPER.md passage or a DESIGN.md reading changes the oracle's arithmetic.

    python tests/golden/make_golden.py
"""
import hashlib
import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import oracle  # noqa: E402
import synth   # noqa: E402


def dig(a):
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()[:16]


W = synth.gen_weight(0, 256, 256)
A = synth.gen_act(0, 16, 256, n_outlier_ch=2)
h = oracle.hessian_diag(A.astype(np.float32)).astype(np.float32)
L = oracle.algorithm1(W, h, 64, 2)
r = oracle.forward(A, L)
out = dict(qa=dig(r["qa"]), sa=dig(r["sa"]), acc0=dig(r["acc0"].astype(np.int32)), acc1=dig(r["acc1"].astype(np.int32)),
           qw=dig(L.d.qw), qr=dig(L.d.qr), blocks=sorted((L.blk_n.astype(int) * 4 + L.blk_k).tolist()))
path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_digest.json")
json.dump(out, open(path, "w"), indent=1)
print(out)
