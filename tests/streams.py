"""Hand-built ACEAPEX streams for the tests, written from docs/FORMAT.md alone.

Pure Python + numpy; imports neither ``oracle`` nor the CUDA package, so a stream built here is an input
that neither side produced.  ``py_decode`` is a byte-at-a-time loop used to pin the oracle decoder.
"""
from __future__ import annotations

import struct

import numpy as np


def _pad(b: bytes, m: int) -> bytes:
    return b + b"\0" * ((-len(b)) % m)


def py_depths(blocks, block_size):
    """dep per sequence by the recursive rule of PAPER.md:155 (dep = level + 1); returns (deps, byte depths)."""
    n = sum(len(l) + ml for blk in blocks for (l, ml, _off) in blk)
    bd = [0] * n
    deps = []
    p = 0
    for blk in blocks:
        d = []
        for lit, mlen, off in blk:
            p += len(lit)
            if mlen:
                se = min(off + mlen, p)
                dep = 1 + max(bd[off:se])
                for i in range(mlen):
                    bd[p + i] = dep
                p += mlen
            else:
                dep = 0
            d.append(dep)
        deps.append(d)
    return deps, bd


def build_stream(blocks, block_size, *, flags=None, deps=None, min_match=4, depth_limit=0, raw_size=None,
                 max_depth=None) -> np.ndarray:
    """blocks: list (per block) of sequences (lit: bytes, mlen: int, off: int).  Returns the serialized stream."""
    if deps is None:
        deps, _ = py_depths(blocks, block_size)
    n = sum(len(l) + ml for blk in blocks for (l, ml, _o) in blk)
    if raw_size is None:
        raw_size = n
    md = max([0] + [d for blk in deps for d in blk]) if max_depth is None else max_depth
    hc = [0] * (md + 1)
    hb = [0] * (md + 1)
    for blk, dd in zip(blocks, deps):
        for (lit, mlen, _o), d in zip(blk, dd):
            if len(lit):
                hc[0] += 1
                hb[0] += len(lit)
            if mlen and d <= md:
                hc[d] += 1
                hb[d] += mlen
    if flags is None:
        flags = 4 | (2 if depth_limit else 0)
    nb = len(blocks)
    meta = 64 + 16 * nb + 16 * (md + 1)
    meta_p = (meta + 127) // 128 * 128
    payloads, dirs, po = [], [], meta_p
    tot_seq = tot_lit = 0
    for blk, dd in zip(blocks, deps):
        ns = len(blk)
        cmd = np.array([len(l) for l, _, _ in blk], dtype="<u2").tobytes()
        ln = np.array([m for _, m, _ in blk], dtype="<u2").tobytes()
        dp = np.array(dd, dtype="<u2").tobytes()
        off = np.array([o for _, _, o in blk], dtype="<u4").tobytes()
        lit = b"".join(l for l, _, _ in blk)
        pay = _pad(cmd, 16) + _pad(ln, 16) + _pad(dp, 16) + _pad(off, 16) + _pad(lit, 16)
        pay = _pad(pay, 128)
        dirs.append(struct.pack("<QII", po, ns, len(lit)))
        payloads.append(pay)
        po += len(pay)
        tot_seq += ns
        tot_lit += len(lit)
    hdr = b"ACEAPEX1" + struct.pack("<IIQIIIIIIQQ", 1, flags, raw_size, block_size, nb, min_match, depth_limit,
                                    md, 0, tot_seq, tot_lit)
    assert len(hdr) == 64
    hist = b"".join(struct.pack("<IIQ", hc[d], 0, hb[d]) for d in range(md + 1))
    buf = _pad(hdr + b"".join(dirs) + hist, 128) + b"".join(payloads)
    return np.frombuffer(buf, dtype=np.uint8).copy()


def py_decode(blocks) -> bytes:
    """Byte-at-a-time LZ77 decode of the hand-built description (textbook rule, ascending copy)."""
    out = bytearray()
    for blk in blocks:
        for lit, mlen, off in blk:
            out += lit
            assert mlen == 0 or off < len(out)
            for i in range(mlen):
                out.append(out[off + i])
    return bytes(out)


def parse_stream(comp: np.ndarray):
    """Inverse of build_stream (used to inspect what the oracle encoder emitted)."""
    c = comp.tobytes()
    assert c[:8] == b"ACEAPEX1"
    ver, flags, raw, B, nb, mm, dl, md, _r, ts, tl = struct.unpack_from("<IIQIIIIIIQQ", c, 8)
    hdr = dict(version=ver, flags=flags, raw_size=raw, block_size=B, n_blocks=nb, min_match=mm, depth_limit=dl,
               max_depth=md, total_seq=ts, total_lit=tl)
    blocks, deps = [], []
    for b in range(nb):
        po, ns, nl = struct.unpack_from("<QII", c, 64 + 16 * b)
        p16 = lambda x: (x + 15) // 16 * 16
        cmd = np.frombuffer(c, "<u2", ns, po)
        ln = np.frombuffer(c, "<u2", ns, po + p16(2 * ns))
        dp = np.frombuffer(c, "<u2", ns, po + 2 * p16(2 * ns))
        off = np.frombuffer(c, "<u4", ns, po + 3 * p16(2 * ns))
        lo = po + 3 * p16(2 * ns) + p16(4 * ns)
        lit = c[lo:lo + nl]
        blk, li = [], 0
        for j in range(ns):
            blk.append((lit[li:li + int(cmd[j])], int(ln[j]), int(off[j])))
            li += int(cmd[j])
        blocks.append(blk)
        deps.append([int(x) for x in dp])
    hist = [struct.unpack_from("<IIQ", c, 64 + 16 * nb + 16 * d) for d in range(md + 1)]
    hdr["hist"] = [(h[0], h[2]) for h in hist]
    return hdr, blocks, deps


def random_blocks(rng: np.random.Generator, block_size: int, n_blocks: int, *, last_short=True, p_match=0.6,
                  max_lit=12, max_len=40, overlap_bias=0.3):
    """Encoder-free fuzz: random literal runs and random matches with off < mdst."""
    blocks, p = [], 0
    for b in range(n_blocks):
        end = p + block_size
        if last_short and b == n_blocks - 1 and block_size > 1:
            end = p + int(rng.integers(1, block_size + 1))
        blk = []
        while p < end:
            nl = int(rng.integers(0, max_lit + 1))
            if p == 0:
                nl = max(nl, 1)
            nl = min(nl, end - p)
            lit = rng.integers(0, 256, nl, dtype=np.uint8).tobytes()
            p += nl
            mlen = off = 0
            if p < end and p > 0 and rng.random() < p_match:
                mlen = min(int(rng.integers(4, max_len + 1)), end - p)
                if rng.random() < overlap_bias:
                    off = p - int(rng.integers(1, min(p, 20) + 1))      # short period: self-overlap
                else:
                    off = int(rng.integers(0, p))
            if nl == 0 and mlen == 0:
                continue
            blk.append((lit, mlen, off))
            p += mlen
        blocks.append(blk)
    return blocks


def flatten_blocks(blocks, block_size):
    """Make a hand-built description satisfy invariant I3 (after chain flattening no match reads a byte
    another match of its own block produced) without changing the decoded bytes: a match whose effective source range
    touches a match-written byte of its own block is replaced by literals of the same bytes."""
    exp = py_decode(blocks)
    out, p = [], 0
    for blk in blocks:
        lo = p
        is_match = bytearray(block_size + 1)                      # per byte of this block: written by a match
        nb = []
        for lit, mlen, off in blk:
            p += len(lit)
            if mlen:
                se = min(off + mlen, p)
                if any(is_match[i - lo] for i in range(max(off, lo), se)):
                    nb.append((lit + exp[p:p + mlen], 0, 0))
                else:
                    nb.append((lit, mlen, off))
                    for i in range(p, p + mlen):
                        is_match[i - lo] = 1
                p += mlen
            else:
                nb.append((lit, 0, 0))
        out.append(nb)
    assert py_decode(out) == exp
    return out
