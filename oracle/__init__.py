"""ctypes front end of the CPU oracle (``aceapex_oracle.c``).  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It never imports ``paper_2606_04268_b200`` and shares no code with it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libaceapex_oracle.so")

ERRORS = {0: "OK", -1: "E_MAGIC", -2: "E_VERSION", -3: "E_TRUNCATED", -4: "E_HEADER", -5: "E_CAPACITY",
          -6: "E_NOMEM", -7: "E_ARG", -11: "E_I1", -12: "E_I2", -13: "E_I3", -14: "E_I4", -15: "E_I5"}


class OracleError(RuntimeError):
    def __init__(self, code, where=""):
        self.code = code
        self.name = ERRORS.get(code, str(code))
        super().__init__(f"oracle: {self.name} {where}")


class EncParams(ctypes.Structure):
    _fields_ = [("block_size", ctypes.c_uint32), ("min_match", ctypes.c_uint32), ("max_chain", ctypes.c_uint32),
                ("window", ctypes.c_uint64), ("flatten", ctypes.c_uint32), ("depth_limit", ctypes.c_uint32),
                ("prefer_shallow", ctypes.c_uint32), ("hash_bits", ctypes.c_uint32)]


class Report(ctypes.Structure):
    _fields_ = [(n, ctypes.c_uint64) for n in ("raw_bytes", "comp_bytes", "lit_bytes", "match_bytes",
                                               "match_src_bytes", "n_seq", "n_match")] + \
               [(n, ctypes.c_uint32) for n in ("n_blocks", "block_size", "max_depth", "depth_limit", "flags",
                                               "fail_block")] + [("fail_seq", ctypes.c_uint64)]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "aceapex_oracle.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-Wall", "-shared", "-fPIC", "-pthread", "-o", _SO, src])
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp, u64 = ctypes.c_void_p, ctypes.c_uint64
        L.orc_raw_size.argtypes = [vp, u64]; L.orc_raw_size.restype = u64
        L.orc_decode_seq.argtypes = [vp, u64, vp, u64]; L.orc_decode_seq.restype = ctypes.c_int
        L.orc_decode_mt.argtypes = [vp, u64, vp, u64, ctypes.c_int]; L.orc_decode_mt.restype = ctypes.c_int
        L.orc_encode.argtypes = [vp, u64, ctypes.POINTER(EncParams), ctypes.POINTER(vp), ctypes.POINTER(u64)]
        L.orc_encode.restype = ctypes.c_int
        L.orc_free.argtypes = [vp]; L.orc_free.restype = None
        L.orc_validate.argtypes = [vp, u64, ctypes.POINTER(Report)]; L.orc_validate.restype = ctypes.c_int
        L.orc_asap.argtypes = [vp, u64, vp, u64]; L.orc_asap.restype = ctypes.c_int64
        _lib = L
    return _lib


def _u8(a) -> np.ndarray:
    a = np.frombuffer(a, dtype=np.uint8) if isinstance(a, (bytes, bytearray, memoryview)) else np.asarray(a)
    assert a.dtype == np.uint8
    return np.ascontiguousarray(a)


def encode(raw, block_size=1 << 20, min_match=4, max_chain=32, window=0, flatten=True, depth_limit=0,
           prefer_shallow=False, hash_bits=0) -> np.ndarray:
    """Greedy hash-chain encoder; returns the serialized stream (uint8)."""
    raw = _u8(raw)
    P = EncParams(block_size, min_match, max_chain, window, int(flatten), depth_limit, int(prefer_shallow), hash_bits)
    out, n = ctypes.c_void_p(), ctypes.c_uint64()
    rc = _load().orc_encode(raw.ctypes.data, raw.size, ctypes.byref(P), ctypes.byref(out), ctypes.byref(n))
    if rc:
        raise OracleError(rc, "encode")
    try:
        buf = np.ctypeslib.as_array(ctypes.cast(out, ctypes.POINTER(ctypes.c_uint8)), shape=(n.value,)).copy()
    finally:
        _load().orc_free(out)
    return buf


def raw_size(comp) -> int:
    comp = _u8(comp)
    n = _load().orc_raw_size(comp.ctypes.data, comp.size)
    if n == 2**64 - 1:
        raise OracleError(-4, "raw_size")
    return n


def _open_code(comp) -> int:
    r = Report()
    return _load().orc_validate(comp.ctypes.data, comp.size, ctypes.byref(r))


def decode(comp, threads: int = 0, out: np.ndarray | None = None) -> np.ndarray:
    """Sequential decode (threads == 0: the definition) or block-parallel."""
    comp = _u8(comp)
    L = _load()
    n = L.orc_raw_size(comp.ctypes.data, comp.size)
    if n == 2**64 - 1:
        probe = np.empty(0, np.uint8)
        raise OracleError(L.orc_decode_seq(comp.ctypes.data, comp.size, probe.ctypes.data, 0), "decode")
    if out is None:
        out = np.zeros(n, dtype=np.uint8)
    if threads <= 0:
        rc = L.orc_decode_seq(comp.ctypes.data, comp.size, out.ctypes.data, out.size)
    else:
        rc = L.orc_decode_mt(comp.ctypes.data, comp.size, out.ctypes.data, out.size, threads)
    if rc:
        raise OracleError(rc, "decode")
    return out[:n]


def validate(comp) -> dict:
    """Invariants I0-I4; raises OracleError naming the violated invariant, else returns the recount."""
    comp = _u8(comp)
    r = Report()
    rc = _load().orc_validate(comp.ctypes.data, comp.size, ctypes.byref(r))
    if rc:
        raise OracleError(rc, f"validate block {r.fail_block} seq {r.fail_seq}")
    return r.as_dict()


def asap(comp):
    """Invariant I5: wave-by-wave simulation; returns (rounds, bytes built wave by wave)."""
    comp = _u8(comp)
    n = raw_size(comp)
    out = np.zeros(n, dtype=np.uint8)
    r = _load().orc_asap(comp.ctypes.data, comp.size, out.ctypes.data, out.size)
    if r < 0:
        raise OracleError(int(r), "asap")
    return int(r), out
