"""paper_2606_04268_b200 — thin ctypes binding of libaceapex (include/aceapex.h).

Argument marshalling only: every step of the decode runs in the CUDA kernels under ``csrc/``.  PyTorch is
used by callers for device memory and streams; nothing here computes.  There is no CPU fallback: if the
shared library is missing or does not load, importing the binding's functions raises.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_SO = os.path.join(_HERE, "libaceapex.so")
_SOURCES = ["k_index.cu", "k_tilesum.cu", "k_pre.cu", "k_match.cu", "k_pass.cu", "k_chain.cu", "api.cu"]
_HEADERS = [os.path.join(_CSRC, "common.cuh"), os.path.join(_CSRC, "copy.cuh"), os.path.join(os.path.dirname(_HERE), "include", "aceapex.h")]

OK = 0
E_MAGIC, E_VERSION, E_TRUNCATED, E_HEADER, E_CAPACITY, E_ALIGN, E_CUDA, E_ARG, E_STREAM, E_NOMEM, E_NOALLOC_LIMIT = range(-1, -12, -1)
PHASE_PRE, PHASE_MATCH, PHASE_ALL = 1, 2, 3
WAVES_AUTO, WAVES_LAUNCH, WAVES_GRAPH, WAVES_PERSISTENT, WAVES_PASSES, WAVES_CHAIN = 0, 1, 2, 3, 4, 5
STRATEGY_NAMES = {0: "auto", 1: "launch", 2: "graph", 3: "persistent", 4: "passes", 5: "chain"}
F_BLOCK_SUM, F_SOURCE, F_DEPTH, F_PLACEHOLDER, F_INDEX = 1, 2, 4, 8, 16

EXPORTS = ["aceapex_plan", "aceapex_raw_bytes", "aceapex_out_bytes", "aceapex_scratch_bytes", "aceapex_set_strategy",
           "aceapex_decode", "aceapex_decode_host", "aceapex_get_stats", "aceapex_depth_hist", "aceapex_strerror",
           "aceapex_last_cuda_error", "aceapex_free", "aceapex_decode_noalloc", "aceapex_get_stats_noalloc",
           "aceapex_noalloc_max_scratch_bytes"]


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu for sm_100a into libaceapex.so next to this file (nvcc cross-compiles without a GPU)."""
    srcs = [os.path.join(_CSRC, s) for s in _SOURCES]
    newest = max(os.path.getmtime(f) for f in srcs + _HEADERS)
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < newest:
        cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--cudart", "shared",
               "-shared", "-Xcompiler", "-fPIC", "-o", _SO, *srcs, "-Xlinker", "-rpath=/usr/local/cuda/lib64"]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.check_call(cmd)
    return _SO


class Stats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_uint64) for n in ("raw_bytes", "comp_bytes", "lit_bytes", "match_bytes", "match_src_bytes",
                                               "n_seq", "n_match")] + \
               [(n, ctypes.c_uint32) for n in ("n_blocks", "block_size", "min_match", "max_depth", "depth_limit", "flags",
                                               "strategy", "n_launches", "fault_flags", "fault_block")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class AceapexError(RuntimeError):
    def __init__(self, code, what=""):
        self.code = code
        msg = _lib().aceapex_strerror(code).decode() if _LIB is not None else str(code)
        super().__init__(f"aceapex: {what}: {msg} ({code})")


_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(_SO)
        vp, sz, u32 = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_uint32
        L.aceapex_plan.argtypes = [vp, sz, ctypes.c_int, ctypes.POINTER(vp)]; L.aceapex_plan.restype = ctypes.c_int
        for n in ("aceapex_raw_bytes", "aceapex_out_bytes", "aceapex_scratch_bytes"):
            getattr(L, n).argtypes = [vp]; getattr(L, n).restype = sz
        L.aceapex_set_strategy.argtypes = [vp, ctypes.c_int]; L.aceapex_set_strategy.restype = ctypes.c_int
        L.aceapex_decode.argtypes = [vp, vp, vp, sz, vp, sz, ctypes.c_uint, vp]; L.aceapex_decode.restype = ctypes.c_int
        L.aceapex_decode_host.argtypes = [vp, vp, sz, vp, sz, vp, vp, sz, vp, sz, vp]
        L.aceapex_decode_host.restype = ctypes.c_int
        L.aceapex_get_stats.argtypes = [vp, vp, ctypes.POINTER(Stats)]; L.aceapex_get_stats.restype = ctypes.c_int
        L.aceapex_depth_hist.argtypes = [vp, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64), u32]
        L.aceapex_depth_hist.restype = ctypes.c_int64
        L.aceapex_strerror.argtypes = [ctypes.c_int]; L.aceapex_strerror.restype = ctypes.c_char_p
        L.aceapex_last_cuda_error.argtypes = [vp]; L.aceapex_last_cuda_error.restype = ctypes.c_int
        L.aceapex_free.argtypes = [vp]; L.aceapex_free.restype = None
        L.aceapex_decode_noalloc.argtypes = [vp, vp, vp, sz, vp]; L.aceapex_decode_noalloc.restype = ctypes.c_int
        L.aceapex_get_stats_noalloc.argtypes = [vp, ctypes.POINTER(Stats)]; L.aceapex_get_stats_noalloc.restype = ctypes.c_int
        L.aceapex_noalloc_max_scratch_bytes.argtypes = []; L.aceapex_noalloc_max_scratch_bytes.restype = sz
        _LIB = L
    return _LIB


def _check(rc, what):
    if rc != 0:
        raise AceapexError(rc, what)


class Plan:
    """aceapex_plan / aceapex_decode / aceapex_free with the same argument meaning as include/aceapex.h."""

    def __init__(self, comp_host_ptr: int, comp_bytes: int, device: int = 0):
        self._h = ctypes.c_void_p()
        self._L = _lib()
        _check(self._L.aceapex_plan(comp_host_ptr, comp_bytes, device, ctypes.byref(self._h)), "plan")
        self.comp_bytes = comp_bytes

    @property
    def raw_bytes(self) -> int:
        return self._L.aceapex_raw_bytes(self._h)

    @property
    def out_bytes(self) -> int:
        return self._L.aceapex_out_bytes(self._h)

    @property
    def scratch_bytes(self) -> int:
        return self._L.aceapex_scratch_bytes(self._h)

    def set_strategy(self, s: int):
        _check(self._L.aceapex_set_strategy(self._h, s), "set_strategy")

    def decode(self, comp_dev: int, out_dev: int, out_capacity: int, scratch_dev: int, scratch_bytes: int,
               phases: int = PHASE_ALL, stream: int = 0):
        rc = self._L.aceapex_decode(self._h, comp_dev, out_dev, out_capacity, scratch_dev, scratch_bytes, phases, stream)
        _check(rc, "decode" if rc != E_CUDA else f"decode (cudaError {self._L.aceapex_last_cuda_error(self._h)})")

    def decode_host(self, comp_host: int, comp_bytes: int, out_host: int, out_host_capacity: int, comp_dev: int,
                    out_dev: int, out_capacity: int, scratch_dev: int, scratch_bytes: int, stream: int = 0):
        _check(self._L.aceapex_decode_host(self._h, comp_host, comp_bytes, out_host, out_host_capacity, comp_dev, out_dev,
                                           out_capacity, scratch_dev, scratch_bytes, stream), "decode_host")

    def decode_noalloc(self, comp_dev: int, out_dev: int, out_capacity: int, stream: int = 0):
        """aceapex_decode_noalloc: full decode with the library's static device scratch (no allocation; one call at a time)."""
        rc = self._L.aceapex_decode_noalloc(self._h, comp_dev, out_dev, out_capacity, stream)
        _check(rc, "decode_noalloc" if rc != E_CUDA else f"decode_noalloc (cudaError {self._L.aceapex_last_cuda_error(self._h)})")

    def stats_noalloc(self, check: bool = True) -> dict:
        s = Stats()
        rc = self._L.aceapex_get_stats_noalloc(self._h, ctypes.byref(s))
        if rc != 0 and (check or rc != E_STREAM):
            raise AceapexError(rc, "get_stats_noalloc")
        d = s.as_dict()
        d["rc"] = rc
        return d

    def stats(self, scratch_dev: int = 0, check: bool = True) -> dict:
        s = Stats()
        rc = self._L.aceapex_get_stats(self._h, scratch_dev, ctypes.byref(s))
        if rc != 0 and (check or rc != E_STREAM):
            raise AceapexError(rc, "get_stats")
        d = s.as_dict()
        d["rc"] = rc
        return d

    def depth_hist(self):
        n = self._L.aceapex_depth_hist(self._h, None, None, 0)
        _check(min(n, 0), "depth_hist")
        a = (ctypes.c_uint64 * n)()
        b = (ctypes.c_uint64 * n)()
        self._L.aceapex_depth_hist(self._h, a, b, n)
        return list(a), list(b)

    def close(self):
        if self._h:
            self._L.aceapex_free(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
