"""Pins for the CPU oracle (decoder, validator, ASAP simulation, encoder) against what the paper and the
mathematics fix.  CPU only.  Nothing here comes from the CUDA path."""
import os

import numpy as np
import pytest

import oracle
import workloads
from streams import build_stream, parse_stream, py_decode, py_depths, random_blocks

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [tuple(int(x) for x in ln.split()) for ln in f if ln.strip() and not ln.startswith("#")]


E1_IN = b"abcdefghabcdefghWXabcdefghzzzzzz"
E2_IN = b"abcdefgh" * 4


# ---------------------------------------------------------------- decoder: the paper's printed example
def test_t1_absolute_offsets():
    """the bytes at 5 000 are off=5000 from 5 100 and from 5 300."""
    rows = _rows("t1_absolute_offsets.txt")
    assert [(r[0], r[1]) for r in rows] == [(5100, 5000), (5300, 5000)]
    assert all(m - o == dist for m, o, dist in rows)          # what relative LZ77 would have stored
    rng = np.random.default_rng(1)
    lit0 = rng.integers(0, 256, 5100, dtype=np.uint8).tobytes()
    lit1 = rng.integers(0, 256, 150, dtype=np.uint8).tobytes()
    blocks = [[(lit0, 50, 5000), (lit1, 50, 5000), (b"tail", 0, 0)]]
    assert len(lit0) == rows[0][0] and len(lit0) + 50 + len(lit1) == rows[1][0]
    s = build_stream(blocks, 1 << 20)
    out = oracle.decode(s).tobytes()
    assert out[5100:5150] == lit0[5000:5050] == out[5300:5350]
    assert out == py_decode(blocks)
    oracle.validate(s)


# ---------------------------------------------------------------- decoder: special cases = library routines
def test_all_literal_is_memcpy():
    rng = np.random.default_rng(2)
    raw = rng.integers(0, 256, 3 * 64 + 17, dtype=np.uint8).tobytes()
    blocks = [[(raw[i:i + 64], 0, 0)] for i in range(0, len(raw), 64)]
    s = build_stream(blocks, 64)
    assert oracle.decode(s).tobytes() == raw


def test_period_one_is_memset():
    blocks = [[(b"Q", 65535, 0), (b"", 65535, 0), (b"", 1000, 7)]]
    s = build_stream(blocks, 1 << 20)
    assert oracle.decode(s).tobytes() == b"Q" * (1 + 65535 * 2 + 1000)
    # match 0 reads the literal (dep 1); matches 1 and 2 read bytes match 0 wrote (dep 2)
    assert oracle.validate(s)["max_depth"] == 2


@pytest.mark.parametrize("k", [2, 3, 4, 5, 7, 8, 9, 15, 16, 17, 31, 32, 33])
def test_period_k_is_tile(k):
    """Overlapping source = periodic extension of out[off..mdst) (Q3) = np.tile."""
    pat = bytes(range(65, 65 + k))
    blocks = [[(b"xy" + pat, 1000, 2)]]
    s = build_stream(blocks, 4096)
    exp = b"xy" + (pat * (1000 // k + 2))[:k + 1000]
    assert oracle.decode(s).tobytes() == exp
    r = oracle.validate(s)
    assert r["match_src_bytes"] == k and r["max_depth"] == 1


def test_non_overlap_edges():
    """off+len == mdst (plain copy) and off+len == mdst+1 (one byte of overlap)."""
    lit = bytes(range(40))
    for off, ln in [(30, 10), (31, 10)]:
        blocks = [[(lit, ln, off)]]
        s = build_stream(blocks, 64)
        assert oracle.decode(s).tobytes() == py_decode(blocks)
    blocks = [[(bytes(range(16)), 0, 0)], [(b"", 16, 8)]]          # source straddles the block boundary
    s = build_stream(blocks, 16)
    assert oracle.decode(s).tobytes() == py_decode(blocks)
    assert oracle.validate(s)["max_depth"] == 1


# ---------------------------------------------------------------- decoder + ASAP: brute force on fuzzed streams
@pytest.mark.parametrize("bs,nb,seed", [(16, 9, 0), (64, 7, 1), (4096, 3, 2), (16, 40, 3), (64, 30, 4)])
def test_fuzz_decode_vs_python_loop(bs, nb, seed):
    rng = np.random.default_rng(100 + seed)
    for it in range(40 if bs < 4096 else 6):
        blocks = random_blocks(rng, bs, nb)
        deps, _ = py_depths(blocks, bs)
        s = build_stream(blocks, bs, deps=deps, min_match=1)
        exp = py_decode(blocks)
        assert oracle.decode(s).tobytes() == exp
        assert oracle.decode(s, threads=3).tobytes() == exp
        r = oracle.validate(s)                                   # recursive depth rule agrees with py_depths
        assert r["max_depth"] == max([0] + [d for dd in deps for d in dd])
        rounds, wave_out = oracle.asap(s)                        # I5: ASAP simulation agrees too
        assert rounds == r["max_depth"] and wave_out.tobytes() == exp


def test_edge_sizes():
    for n in (0, 1, 15, 16, 17):
        raw = np.arange(n, dtype=np.uint8)
        s = oracle.encode(raw, block_size=16)
        assert oracle.raw_size(s) == n
        assert oracle.decode(s).tobytes() == raw.tobytes()
        assert oracle.validate(s)["n_blocks"] == (n + 15) // 16


# ---------------------------------------------------------------- encoder: the paper's flattening examples
def _enc_rows(raw, **kw):
    s = oracle.encode(np.frombuffer(raw, np.uint8), **kw)
    hdr, blocks, deps = parse_stream(s)
    rows = [(b, j, len(l), m, o, deps[b][j]) for b, blk in enumerate(blocks) for j, (l, m, o) in enumerate(blk)]
    return s, hdr, rows


@pytest.mark.parametrize("flatten", [1, 0])
def test_e1_chain_flattening(flatten):
    """A -> B -> C(literal) becomes A -> C."""
    exp = [r[1:] for r in _rows("e1_flatten.txt") if r[0] == flatten]
    s, hdr, rows = _enc_rows(E1_IN, block_size=32, flatten=bool(flatten))
    assert [r[1:] for r in rows] == exp
    assert hdr["hist"] == ([(3, 11), (3, 21)] if flatten else [(3, 11), (2, 13), (1, 8)])
    assert oracle.decode(s).tobytes() == E1_IN
    oracle.validate(s)
    assert oracle.asap(s)[0] == (1 if flatten else 2)


def test_e1_golden_bytes():
    """docs/FORMAT.md layout: the oracle encoder's serialization equals the hand-built golden stream."""
    with open(os.path.join(GOLD, "e1_stream.hex")) as f:
        gold = bytes.fromhex("".join(ln.strip() for ln in f if not ln.startswith("#")))
    s = oracle.encode(np.frombuffer(E1_IN, np.uint8), block_size=32, flatten=True)
    assert s.tobytes() == gold


@pytest.mark.parametrize("D", [0, 1])
def test_e2_cross_block(D):
    """a chain that leaves the block is not flattened; depth limit."""
    exp = [r[1:] for r in _rows("e2_crossblock.txt") if r[0] == D]
    s, hdr, rows = _enc_rows(E2_IN, block_size=16, flatten=True, depth_limit=D)
    assert rows == exp
    assert hdr["max_depth"] == (2 if D == 0 else 1)
    assert oracle.decode(s).tobytes() == E2_IN
    oracle.validate(s)


# ---------------------------------------------------------------- encoder: round trip + invariants I0-I6
CASES = [("markov", dict()), ("markov", dict(flatten=False)), ("markov", dict(depth_limit=2)),
         ("text", dict()), ("text", dict(depth_limit=4)), ("fastq", dict()), ("stress", dict()),
         ("stress", dict(flatten=False)), ("stress", dict(depth_limit=1)), ("markov", dict(prefer_shallow=True))]


@pytest.mark.parametrize("kind,kw", CASES)
def test_round_trip_and_invariants(kind, kw):
    n = 3 * 4096 + 1234 if kind != "stress" else 300_000
    bs = 4096 if kind != "stress" else 65536
    raw = workloads.generate(kind, n, 7)
    s = oracle.encode(raw, block_size=bs, **kw)
    r = oracle.validate(s)                                        # I0-I4
    assert r["raw_bytes"] == n and r["lit_bytes"] + r["match_bytes"] == n
    assert np.array_equal(oracle.decode(s), raw)                  # I6
    assert np.array_equal(oracle.decode(s, threads=4), raw)
    if kw.get("depth_limit"):
        assert r["max_depth"] <= kw["depth_limit"]                # I4 / PAPER.md:228
    if n <= 20000:
        rounds, out = oracle.asap(s)                              # I5
        assert rounds == r["max_depth"] and np.array_equal(out, raw)
    hdr, blocks, deps = parse_stream(s)
    mydeps, bd = py_depths(blocks, bs)                            # independent recount of PAPER.md:155
    assert mydeps == deps
    if kw.get("flatten", True):                                   # I3 recount: in-block sources are literals
        p = 0
        for b, blk in enumerate(blocks):
            for lit, mlen, off in blk:
                p += len(lit)
                if mlen:
                    lo = max(off, b * bs)
                    assert all(bd[q] == 0 for q in range(lo, min(off + mlen, p)))
                p += mlen


def test_flatten_off_deep_chains():
    raw = workloads.generate("markov", 64 * 4096, 3)
    s = oracle.encode(raw, block_size=4096, flatten=False)
    r = oracle.validate(s)
    assert r["max_depth"] > 8 and np.array_equal(oracle.decode(s), raw)
    s2 = oracle.encode(raw, block_size=4096, flatten=True)
    assert oracle.validate(s2)["max_depth"] <= r["max_depth"]


def test_long_literal_and_long_run():
    rng = np.random.default_rng(5)
    raw = rng.integers(0, 256, 200_000, dtype=np.uint8)           # incompressible: runs > 65535 split
    s = oracle.encode(raw)
    hdr, blocks, _ = parse_stream(s)
    assert len(blocks[0]) >= 4 and max(len(l) for l, _, _ in blocks[0]) <= 65535
    assert oracle.validate(s)["lit_bytes"] > 199_000            # chance 4-byte matches only
    assert np.array_equal(oracle.decode(s), raw)
    raw = np.full(200_000, 0x41, np.uint8)                        # period-1 run: matches split at 65535; flattening (I3)
    # forbids reading same-block match bytes, so each piece restarts from one fresh literal: all dep 1
    s = oracle.encode(raw)
    r = oracle.validate(s)
    assert r["max_depth"] == 1 and r["lit_bytes"] == 4 and np.array_equal(oracle.decode(s), raw)


# ---------------------------------------------------------------- validator rejects each violation
def test_malformed_streams_rejected():
    good = [[(b"abcdefgh", 8, 0), (b"WX", 8, 0), (b"z", 5, 26)]]
    s = build_stream(good, 32, flags=5)
    oracle.validate(s)

    def bad(mut, name):
        t = s.copy()
        mut(t)
        with pytest.raises(oracle.OracleError) as e:
            oracle.validate(t)
        assert e.value.name == name, (e.value.name, name)

    def setb(off, vals):
        def f(t):
            t[off:off + len(vals)] = np.frombuffer(bytes(vals), np.uint8)
        return f
    po = 128
    bad(setb(0, b"X"), "E_MAGIC")
    bad(setb(8, [2]), "E_VERSION")
    bad(setb(28, [2]), "E_HEADER")                    # n_blocks != ceil(raw/B)
    bad(setb(64, [64]), "E_HEADER")                   # payload offset not a multiple of 128 / inside metadata
    bad(setb(po, [9]), "E_I1")                        # cmd[0] 8 -> 9: lengths no longer sum
    bad(setb(po + 16 + 2, [3]), "E_I2")               # len[1] 8 -> 3 < min_match
    bad(setb(po + 48 + 4, [200]), "E_I2")             # off[1] >= mdst
    bad(setb(po + 32 + 2, [2]), "E_I4")               # dep[1] wrong
    u = build_stream([[(b"abcdefgh", 8, 0), (b"WX", 8, 8), (b"z", 5, 26)]], 32, flags=5)
    with pytest.raises(oracle.OracleError) as e:
        oracle.validate(u)                            # FLATTENED flag but a same-block match-written source
    assert e.value.name == "E_I3"
    with pytest.raises(oracle.OracleError):
        oracle.validate(s[:100])                      # truncated
    with pytest.raises(oracle.OracleError):
        oracle.decode(s[:150])


# ---------------------------------------------------------------- generators are pinned by checksum
GEN_SHA256_1MIB = {   # docs/WORKLOADS.md: SHA-256 (first 32 hex digits) of the first MiB of each BASELINE config's generator
    "synth4m": "e7fa8a03e69a46a24ae67c373dc440aa",
    "text256m": "e9dc67a497379fe02db0cc26cfa8438f",
    "fastq1g": "27f782f45a4cb36c2a25834aad865f9c",
    "text1g_d4": "e9dc67a497379fe02db0cc26cfa8438f",
    "stress2g": "5fc6eaa5080fbd29d8bc5771414ceb5a",
}


def test_generators_pinned_by_checksum():
    """generator parameters are frozen in docs/WORKLOADS.md and pinned by a checksum of each output.  The
    generators are prefix-stable, so the first MiB pins the recipe of the full-size configs too."""
    import hashlib
    for name, want in GEN_SHA256_1MIB.items():
        a = workloads.config_bytes(name, 1 << 20)
        assert hashlib.sha256(a.tobytes()).hexdigest()[:32] == want, name
        b = workloads.config_bytes(name, (1 << 20) + 4321)
        assert np.array_equal(a, b[:1 << 20]), f"{name}: not prefix-stable"


def test_generators_deterministic():
    a = workloads.generate("text", 100_000, 11)
    b = workloads.generate("text", 100_000, 11)
    assert np.array_equal(a, b)
    assert not np.array_equal(a, workloads.generate("text", 100_000, 12))
    for kind in ("markov", "text", "fastq", "stress"):
        x = workloads.generate(kind, 50_000, 1)
        assert x.size == 50_000 and len(set(x.tolist())) > 3
    fq = workloads.generate("fastq", 2000, 1).tobytes().split(b"\n")
    assert fq[0].startswith(b"@SIM:") and fq[2] == b"+" and len(fq[1]) == 150 == len(fq[3])
    assert set(fq[1]) <= set(b"ACGTN")


# ---------------------------------------------------------------- the oracle under ASan + UBSan
def test_oracle_under_sanitizers(tmp_path):
    """Every oracle entry point on BASELINE config 0 (synth4m: 4 blocks of 1 MB) in a build with
    -fsanitize=address,undefined: tests/asan_driver.c includes oracle/aceapex_oracle.c as is."""
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    exe = str(tmp_path / "asan_driver")
    subprocess.check_call(["gcc", "-O1", "-g", "-std=gnu11", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-pthread",
                           os.path.join(root, "tests", "asan_driver.c"), "-o", exe])
    raw = workloads.config_bytes("synth4m")
    f = tmp_path / "synth4m.raw"
    raw.tofile(f)
    r = subprocess.run([exe, str(f), str(1 << 20)], capture_output=True, text=True, timeout=600,
                       env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0"))
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.count("ok") == 3
