"""CPU-only checks of the C-ABI library: it builds for sm_100a, loads, exports every symbol include/aceapex.h
declares, and validates headers on the host (no compute calls: there is no GPU here and no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2606_04268_b200 as ax
from streams import build_stream

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    return ctypes.CDLL(ax.build())


def test_exports_match_header(lib):
    hdr = open(os.path.join(ROOT, "include", "aceapex.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(aceapex_[a-z_]+)\s*\(", hdr))
    assert declared == set(ax.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_no_torch_types_in_header():
    hdr = open(os.path.join(ROOT, "include", "aceapex.h")).read()
    assert "torch" not in hdr.lower().replace("pytorch types", "") and "at::" not in hdr and "std::" not in hdr


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2606_04268_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "aceapex_oracle" not in src, f


def _plan_rc(buf):
    L = ax._lib()
    h = ctypes.c_void_p()
    rc = L.aceapex_plan(buf.ctypes.data, buf.size, 0, ctypes.byref(h))
    if rc == 0:
        L.aceapex_free(h)
    return rc


def test_plan_rejects_malformed_headers_on_host():
    s = build_stream([[(b"abcdefgh", 8, 0), (b"WX", 8, 0), (b"z", 5, 26)]], 32, flags=5)
    assert _plan_rc(s) in (ax.OK, ax.E_CUDA)          # valid: OK on a GPU box, E_CUDA here (no device, no fallback)

    def mut(off, vals):
        t = s.copy()
        t[off:off + len(vals)] = np.frombuffer(bytes(vals), np.uint8)
        return t
    assert _plan_rc(mut(0, b"X")) == ax.E_MAGIC
    assert _plan_rc(mut(8, [2])) == ax.E_VERSION
    assert _plan_rc(mut(28, [2])) == ax.E_HEADER       # n_blocks != ceil(raw / B)
    assert _plan_rc(mut(64, [64])) == ax.E_HEADER      # payload offset misaligned / inside the metadata
    assert _plan_rc(mut(72, [0])) == ax.E_HEADER       # n_seq == 0
    assert _plan_rc(mut(48, [4])) == ax.E_HEADER       # total_seq mismatch
    assert _plan_rc(mut(12, [1])) == ax.E_HEADER       # HAS_DEP flag missing
    assert _plan_rc(s[:100].copy()) == ax.E_TRUNCATED
    assert _plan_rc(s[:200].copy()) == ax.E_TRUNCATED
    assert _plan_rc(s[:32].copy()) == ax.E_TRUNCATED
    L = ax._lib()
    assert L.aceapex_plan(None, 0, 0, ctypes.byref(ctypes.c_void_p())) == ax.E_ARG
    L.aceapex_free(None)
    assert L.aceapex_strerror(ax.E_STREAM).decode().startswith("token stream")
