"""CPU-only checks of the boundary: libmq.so builds, loads, exports every symbol include/mq.h
declares, validates arguments on the host, and FAILS LOUDLY (no fallback) without a B200."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def mqlib():
    from paper_2606_15652_b200 import build
    build.build()
    import paper_2606_15652_b200 as mq
    return mq


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "mq.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mq_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_all_exported(mqlib):
    names = _declared_symbols()
    assert "mq_gemm" in names and "mq_quantize_act" in names and "mq_pack_weights" in names
    L = mqlib.lib()
    for n in names:
        assert hasattr(L, n), f"libmq.so does not export {n}"
    assert sorted(mqlib.EXPORTS) == names, "binding EXPORTS and include/mq.h disagree"


def test_binding_has_same_names(mqlib):
    for n in _declared_symbols():
        if n in ("mq_status_string", "mq_weights_export", "mq_weights_info", "mq_weights_free", "mq_weights_clone",
                 "mq_weights_export_blockscale", "mq_weights_is_blockscale"):
            continue  # exposed as status_string / Weights methods
        assert hasattr(mqlib, n), n


def test_status_strings(mqlib):
    assert mqlib.status_string(0) == "ok"
    seen = {mqlib.status_string(-i) for i in range(0, 9)}
    assert len(seen) == 9
    assert "unknown" in mqlib.status_string(-99)


def test_qact_bytes_and_options(mqlib):
    assert mqlib.mq_qact_bytes(16, 256) == 16 * 128
    assert mqlib.mq_qact_bytes(0, 256) == 0
    mqlib.mq_set_option("split_k", 3)
    mqlib.mq_set_option("split_k", 0)
    mqlib.mq_set_option("token_tile", 64)
    mqlib.mq_set_option("token_tile", 0)
    with pytest.raises(mqlib.MqError):
        mqlib.mq_set_option("token_tile", 48)
    with pytest.raises(mqlib.MqError):
        mqlib.mq_set_option("no_such_option", 1)


def test_host_side_argument_checks(mqlib):
    L = mqlib.lib()
    # shape errors are detected before any device work
    assert L.mq_quantize_act(None, 0, 4, 100, 100, None, None, None) == -2      # K % 128
    assert L.mq_quantize_act(None, 7, 4, 128, 128, None, None, None) == -1      # bad dtype
    assert L.mq_quantize_act(None, 0, 0, 128, 128, None, None, None) == 0       # M == 0 no-op
    assert L.mq_quantize_act(None, 0, 4, 128, 128, None, None, None) == -1      # NULL pointers
    out = C.c_void_p()
    W = np.zeros((128, 128), np.float32)
    assert L.mq_pack_weights(W.ctypes.data_as(C.c_void_p), 128, 100, None, 64, 1, C.byref(out), None) == -2
    assert L.mq_pack_weights(W.ctypes.data_as(C.c_void_p), 128, 128, None, 32, 1, C.byref(out), None) == -2
    assert L.mq_pack_weights(None, 128, 128, None, 64, 1, C.byref(out), None) == -1
    assert L.mq_gemm(None, None, None, 1, None, 0, 0, None, None, None, 0, None) == -1
    assert L.mq_gemm_workspace_bytes(None, 4) == 0


def test_no_fallback_without_b200(mqlib):
    """On a machine without a compute-capability-10.0 GPU the compute calls must return an
    error, never a CPU result."""
    import torch
    if torch.cuda.is_available() and torch.cuda.get_device_capability() == (10, 0):
        pytest.skip("a B200 is present")
    L = mqlib.lib()
    out = C.c_void_p()
    W = np.ones((128, 128), np.float32)
    rc = L.mq_pack_weights(W.ctypes.data_as(C.c_void_p), 128, 128, None, 64, 1, C.byref(out), None)
    assert rc in (-3, -4) and not out.value
    a = np.zeros((1, 128), np.float16)
    q = np.zeros((1, 64), np.uint8)
    s = np.zeros(1, np.float32)
    # (host pointers: the call must be refused at the device check, before any launch)
    rc = L.mq_quantize_act(a.ctypes.data_as(C.c_void_p), 0, 1, 128, 128, q.ctypes.data_as(C.c_void_p),
                           s.ctypes.data_as(C.c_void_p), None)
    assert rc in (-3, -4)


def test_product_does_not_import_oracle():
    """The product path must not reference oracle/ (independence)."""
    pkg = os.path.join(ROOT, "paper_2606_15652_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "mq_oracle" not in txt, f
    orc = os.path.join(ROOT, "oracle")
    for f in os.listdir(orc):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(orc, f)).read()
            assert "libmq.so" not in txt and "paper_2606_15652_b200 import" not in txt and "import paper_2606_15652_b200" not in txt, f
