"""Build libmq.so (the C-ABI library, include/mq.h) in-tree for sm_100a.

    python -m paper_2606_15652_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so lands next to this file and is git-ignored
(it still travels to the GPU box with the repo snapshot).  Translation units are compiled
in parallel and only when they (or a shared header) changed.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libmq.so")
SOURCES = ["mq_quant.cu", "mq_pack.cu", "mq_gemm.cu", "mq_group.cu", "mq_group_tc.cu", "mq_decode.cu", "mq_prefill.cu", "mq_pack_device.cu", "mq_probe.cu"]
HEADERS = ["mq_internal.h", "mq_ptx.cuh", os.path.join("..", "..", "include", "mq.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC,-O2,-Wall,-ffp-contract=off",
    "-Xptxas", "-v",
]


def _mtime(path: str) -> float:
    return os.path.getmtime(path) if os.path.exists(path) else 0.0


def _compile(src: str, verbose: bool) -> str:
    o = os.path.join(CSRC, src.replace(".cu", ".o"))
    cmd = [NVCC, *FLAGS, "-c", os.path.join(CSRC, src), "-o", o]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}")
    return o


def build(force: bool = False, verbose: bool = False) -> str:
    sources = [s for s in SOURCES if os.path.exists(os.path.join(CSRC, s))]
    common = max([_mtime(os.path.join(CSRC, h)) for h in HEADERS] + [_mtime(os.path.abspath(__file__))])
    objs = [os.path.join(CSRC, s.replace(".cu", ".o")) for s in sources]
    stale = [s for s, o in zip(sources, objs)
             if force or _mtime(o) < max(common, _mtime(os.path.join(CSRC, s)))]
    if stale:
        with ThreadPoolExecutor(max_workers=min(len(stale), os.cpu_count() or 4)) as ex:
            list(ex.map(lambda s: _compile(s, verbose), stale))
    if stale or _mtime(OUT) < max(_mtime(o) for o in objs):
        r = subprocess.run([NVCC, "-shared", "-o", OUT, *objs, "-lpthread"], capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("link failed")
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
