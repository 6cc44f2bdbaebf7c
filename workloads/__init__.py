"""Seeded synthetic input generators (raw bytes only) shared by the oracle tests and the CUDA tests.

Holds none of the method's arithmetic (no tokens, offsets or depths): see ``gen.c``.  The five named
workloads mirror BASELINE.json ``configs[0..4]``; DESIGN.md "Input recipe" states every parameter.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libaceapex_workloads.so")
BASE_SEED = 260604268
MiB = 1 << 20

# name -> (generator symbol, raw bytes, seed)
CONFIGS = {
    "synth4m":   ("wl_markov", 4 * MiB,    BASE_SEED + 0),
    "text256m":  ("wl_text",   256 * MiB,  BASE_SEED + 1),
    "fastq1g":   ("wl_fastq",  1024 * MiB, BASE_SEED + 2),
    "text1g_d4": ("wl_text",   1024 * MiB, BASE_SEED + 1),   # config 1's generator scaled up, same seed
    "stress2g":  ("wl_stress", 2048 * MiB, BASE_SEED + 4),
}


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "gen.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-o", _SO, src, "-lm"])
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        for name in ("wl_markov", "wl_text", "wl_fastq", "wl_stress"):
            fn = getattr(_lib, name)
            fn.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint64]
            fn.restype = ctypes.c_int
    return _lib


def generate(kind: str, n: int, seed: int) -> np.ndarray:
    """kind in {markov, text, fastq, stress}; returns a uint8 array of exactly n bytes."""
    out = np.empty(n, dtype=np.uint8)
    if n:
        rc = getattr(_load(), "wl_" + kind)(out.ctypes.data, n, seed)
        if rc != 0:
            raise MemoryError(f"wl_{kind} failed ({rc})")
    return out


def config_bytes(name: str, n: int | None = None) -> np.ndarray:
    """Raw bytes of a named BASELINE config (optionally truncated/extended to n bytes, same seed)."""
    sym, size, seed = CONFIGS[name]
    return generate(sym[3:], size if n is None else n, seed)
