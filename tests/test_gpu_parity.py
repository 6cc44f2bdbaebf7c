"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit-exact, on the same seeded inputs.
Every test here needs a B200 (``-m gpu``)."""
import os

import numpy as np
import pytest

import oracle
import workloads
import paper_2606_04268_b200 as ax
from streams import build_stream, flatten_blocks, py_decode, py_depths, random_blocks

pytestmark = pytest.mark.gpu

STRATS = [ax.WAVES_LAUNCH, ax.WAVES_GRAPH, ax.WAVES_PERSISTENT]       # wave lists for every depth, three ways of sequencing
ALL_STRATS = STRATS + [ax.WAVES_PASSES]                               # + one streaming pass per depth (shallow streams only)


def chain_ok(comp):
    """Strategy CHAIN needs the header's FLATTENED flag (offset 12, bit 0): invariant I3."""
    return bool(int(np.frombuffer(comp[12:16].tobytes(), "<u4")[0]) & 1)


def passes_ok(comp):
    """Strategy PASSES runs one streaming pass per depth and accepts at most 16 of them."""
    return int(np.frombuffer(comp[40:44].tobytes(), "<u4")[0]) <= 16


def strats_for(comp):
    return STRATS + ([ax.WAVES_CHAIN] if chain_ok(comp) else []) + ([ax.WAVES_PASSES] if passes_ok(comp) else [])


def gpu_decode(comp, strategy=0, check=True):
    from paper_2606_04268_b200.torch_io import Decoder
    d = Decoder(comp, 0, strategy)
    try:
        d.run()
        out = d.output()
        st = d.stats(check=check)
        return out, st
    finally:
        d.close()


def assert_parity(comp, raw=None, strategies=STRATS):
    want = oracle.decode(comp)
    rep = oracle.validate(comp)
    if strategies is STRATS:
        strategies = strats_for(comp)
    for s in strategies:
        got, st = gpu_decode(comp, s)
        assert got.size == want.size
        if not np.array_equal(got, want):
            bad = np.flatnonzero(got != want)
            raise AssertionError(f"strategy {s}: {bad.size} bytes differ, first at {bad[0]}")
        assert st["match_src_bytes"] == rep["match_src_bytes"] and st["n_match"] == rep["n_match"]
    if raw is not None:
        assert np.array_equal(want, raw)


# ---------------------------------------------------------------- hand-built streams (tests/streams.py)
def test_paper_examples():
    E1 = [[(b"abcdefgh", 8, 0), (b"WX", 8, 0), (b"z", 5, 26)]]
    assert_parity(build_stream(E1, 32, flags=5))
    E1b = [[(b"abcdefgh", 8, 0), (b"WX", 8, 8), (b"z", 5, 26)]]                 # flatten off: depth 2
    assert_parity(build_stream(E1b, 32))
    E2 = [[(b"abcdefgh", 8, 0)], [(b"", 16, 8)]]                                # PAPER.md:63 cross-block, overlap period 8
    assert_parity(build_stream(E2, 16))
    rng = np.random.default_rng(1)
    lit0 = rng.integers(0, 256, 5100, dtype=np.uint8).tobytes()
    lit1 = rng.integers(0, 256, 150, dtype=np.uint8).tobytes()
    T1 = [[(lit0, 50, 5000), (lit1, 50, 5000), (b"tail", 0, 0)]]
    s = build_stream(T1, 1 << 20)
    got, _ = gpu_decode(s)
    assert got.tobytes() == py_decode(T1)


def test_empty_and_tiny():
    for n in (0, 1, 15, 16, 17):
        raw = np.arange(n, dtype=np.uint8)
        comp = oracle.encode(raw, block_size=16)
        got, _ = gpu_decode(comp)
        assert got.tobytes() == raw.tobytes()


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5, 7, 8, 9, 15, 16, 17, 31, 32, 33, 100])
@pytest.mark.parametrize("n", [5, 31, 32, 33, 1000, 65535])
def test_periodic_overlap(k, n):
    """Self-overlapping copies = periodic replication (Q3), short (one thread) and long (one warp)."""
    pat = bytes((65 + i) % 251 for i in range(k))
    for lead in (b"", b"xy", b"0123456789abcde"):                               # vary destination alignment
        blocks = [[(lead + pat, n, len(lead))]]
        s = build_stream(blocks, 1 << 17, flags=5)
        exp = lead + (pat * (n // k + 2))[:k + n]
        for strat in (ax.WAVES_CHAIN, ax.WAVES_PASSES, ax.WAVES_LAUNCH, ax.WAVES_PERSISTENT):
            got, _ = gpu_decode(s, strat)
            assert got.tobytes() == exp, strat


def test_long_copies_all_alignments():
    """Non-overlapping long matches and long literal runs at every (src, dst) alignment mod 16."""
    rng = np.random.default_rng(3)
    base = rng.integers(0, 256, 4096, dtype=np.uint8).tobytes()
    seqs = [(base, 0, 0)]
    for sa in range(16):
        for da in range(0, 16, 3):
            lit = rng.integers(0, 256, 17 + da, dtype=np.uint8).tobytes()
            seqs.append((lit, 33 + 7 * sa + da, 100 + sa))
    blocks = [seqs]
    s = build_stream(blocks, 1 << 20, flags=5)                                  # every source is literal: I3 holds
    for strat in (ax.WAVES_CHAIN, ax.WAVES_PASSES, ax.WAVES_LAUNCH, ax.WAVES_PERSISTENT):
        got, _ = gpu_decode(s, strat)
        assert got.tobytes() == py_decode(blocks), strat


@pytest.mark.parametrize("bs,nb,seed", [(16, 9, 0), (64, 37, 1), (4096, 5, 2), (1 << 16, 3, 3)])
def test_fuzz_streams(bs, nb, seed):
    """Encoder-free fuzz: random valid streams, arbitrary depths (deep chains), random overlaps."""
    rng = np.random.default_rng(200 + seed)
    for it in range(6):
        blocks = random_blocks(rng, bs, nb, max_len=40 if bs < 4096 else 300, max_lit=12 if bs < 4096 else 40)
        s = build_stream(blocks, bs, min_match=1)
        exp = py_decode(blocks)
        for strat in strats_for(s):
            got, _ = gpu_decode(s, strat)
            assert got.tobytes() == exp, (bs, nb, seed, it, strat)


# ---------------------------------------------------------------- oracle-encoded workloads
CASES = [("markov", 1 << 20, dict(block_size=1 << 18)),
         ("markov", (1 << 20) + 4321, dict(block_size=1 << 16, flatten=False)),           # deep chains: hundreds of waves
         ("markov", 1 << 20, dict(block_size=1 << 18, depth_limit=2)),
         ("text", 3 << 20, dict()),
         ("text", 3 << 20, dict(depth_limit=4)),
         ("fastq", (3 << 20) + 77, dict()),
         ("stress", 6 << 20, dict()),
         ("stress", 4 << 20, dict(flatten=False)),
         ("stress", 4 << 20, dict(depth_limit=1)),
         ("text", 3 << 20, dict(min_match=11)),                                          # token-cost-aware regime (Q4):
         ("fastq", (3 << 20) + 5, dict(min_match=11, depth_limit=4)),                    # long literal runs, fewer and longer matches
         ("fastq", 2 << 20, dict(min_match=11, max_chain=4, flatten=False)),
         ("text", 16 << 20, dict(block_size=8 << 20, max_chain=4)),      # ~1900 tiles per block: more than k_chain keeps resident
         ("markov", 1 << 20, dict(block_size=4096))]                     # 256 blocks of one tile each: one chain hop per tile


@pytest.mark.parametrize("kind,n,kw", CASES)
def test_workload_parity(kind, n, kw):
    raw = workloads.generate(kind, n, 260604268)
    comp = oracle.encode(raw, **kw)
    assert_parity(comp, raw)


def test_config0_synth4m():
    """BASELINE config 0 at full size: 4 blocks of 1 MB, flatten on, no depth limit."""
    raw = workloads.config_bytes("synth4m")
    comp = oracle.encode(raw)
    assert_parity(comp, raw)


def test_deeper_than_smem_bins():
    """max_depth + 1 > 4096 takes the global-atomic bucketing path."""
    n = 6000
    blocks = [[(b"abcd", 0, 0)] + [(b"", 4, 4 * i) for i in range(n)]]
    s = build_stream(blocks, 1 << 20)
    got, st = gpu_decode(s, ax.WAVES_PERSISTENT)
    assert st["max_depth"] == n and got.tobytes() == b"abcd" * (n + 1)


def test_incompressible_and_runs():
    rng = np.random.default_rng(5)
    raw = rng.integers(0, 256, (2 << 20) + 5, dtype=np.uint8)
    assert_parity(oracle.encode(raw), raw, [0])
    raw = np.full(3 << 20, 0x41, np.uint8)
    assert_parity(oracle.encode(raw), raw, [0])


# ---------------------------------------------------------------- phases, reuse, faults
def test_phases_and_replay():
    from paper_2606_04268_b200.torch_io import Decoder
    raw = workloads.generate("text", 2 << 20, 9)
    comp = oracle.encode(raw, depth_limit=4)
    for strat in ALL_STRATS + [ax.WAVES_CHAIN]:
        d = Decoder(comp, 0, strat)
        d.run(ax.PHASE_PRE)
        d.run(ax.PHASE_MATCH)
        assert np.array_equal(d.output(), raw)
        for _ in range(3):                                 # plan + scratch reuse; MATCH alone replays on PRE's lists
            d.out_dev.zero_()
            d.run(ax.PHASE_ALL)
            assert np.array_equal(d.output(), raw)
        d.run(ax.PHASE_MATCH)
        assert np.array_equal(d.output(), raw)
        d.close()


def test_decode_host_entry():
    import torch
    raw = workloads.generate("fastq", 2 << 20, 4)
    comp = oracle.encode(raw)
    p = ax.Plan(comp.ctypes.data, comp.size, 0)
    ch = torch.from_numpy(comp).pin_memory()
    oh = torch.zeros(p.raw_bytes, dtype=torch.uint8).pin_memory()
    cd = torch.empty(comp.size, dtype=torch.uint8, device="cuda")
    od = torch.empty(p.out_bytes, dtype=torch.uint8, device="cuda")
    sc = torch.empty(p.scratch_bytes, dtype=torch.uint8, device="cuda")
    p.decode_host(ch.data_ptr(), comp.size, oh.data_ptr(), oh.numel(), cd.data_ptr(), od.data_ptr(), od.numel(),
                  sc.data_ptr(), sc.numel(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert p.stats(sc.data_ptr())["rc"] == 0
    assert np.array_equal(oh.numpy(), raw)
    p.close()


def test_argument_errors():
    import torch
    raw = workloads.generate("markov", 100000, 1)
    comp = oracle.encode(raw, block_size=1 << 16)
    p = ax.Plan(comp.ctypes.data, comp.size, 0)
    cd = torch.from_numpy(comp).cuda()
    od = torch.empty(p.out_bytes + 16, dtype=torch.uint8, device="cuda")
    sc = torch.empty(p.scratch_bytes + 16, dtype=torch.uint8, device="cuda")
    L = ax._lib()
    rc = lambda *a: L.aceapex_decode(p._h, *a)
    assert rc(cd.data_ptr(), od.data_ptr(), p.out_bytes - 16, sc.data_ptr(), sc.numel(), 3, 0) == ax.E_CAPACITY
    assert rc(cd.data_ptr(), od.data_ptr(), od.numel(), sc.data_ptr(), p.scratch_bytes - 1, 3, 0) == ax.E_CAPACITY
    assert rc(cd.data_ptr(), od.data_ptr() + 1, od.numel() - 1, sc.data_ptr(), sc.numel(), 3, 0) == ax.E_ALIGN
    assert rc(cd.data_ptr(), od.data_ptr(), od.numel(), sc.data_ptr(), sc.numel(), 0, 0) == ax.E_ARG
    assert rc(None, od.data_ptr(), od.numel(), sc.data_ptr(), sc.numel(), 3, 0) == ax.E_ARG
    p.close()


def test_device_faults_are_flagged_not_fatal():
    """Token-level faults: flagged through get_stats (E_STREAM), never an out-of-bounds access; the guard bytes
    behind the output stay untouched."""
    import torch
    from paper_2606_04268_b200.torch_io import Decoder
    good = [[(b"abcdefgh", 8, 0), (b"WX", 8, 0), (b"z", 5, 26)]]
    s = build_stream(good, 32, flags=5)
    po = 128

    def run(t, strat=0):
        d = Decoder(t, 0, strat)
        guard = torch.full((4096,), 0xEE, dtype=torch.uint8, device="cuda")
        big = torch.cat([torch.zeros(d.plan.out_bytes, dtype=torch.uint8, device="cuda"), guard])
        d.out_dev = big
        st = None
        d.plan.decode(d.comp_dev.data_ptr(), big.data_ptr(), d.plan.out_bytes, d.scratch.data_ptr(), d.scratch.numel(), 3,
                      torch.cuda.current_stream().cuda_stream)
        st = d.stats(check=False)
        assert bool((big[d.plan.out_bytes:] == 0xEE).all())
        d.close()
        return st

    def mut(off, vals):
        t = s.copy()
        t[off:off + len(vals)] = np.frombuffer(bytes(vals), np.uint8)
        return t
    assert run(s)["rc"] == 0
    for strat in ALL_STRATS + [ax.WAVES_CHAIN]:
        st = run(mut(po, [9]), strat)                         # cmd[0] 8 -> 9: block no longer sums
        assert st["rc"] == ax.E_STREAM and st["fault_flags"] & ax.F_BLOCK_SUM and st["fault_block"] == 0
        st = run(mut(po + 48 + 4, [200]), strat)              # off[1] >= mdst
        assert st["rc"] == ax.E_STREAM and st["fault_flags"] & ax.F_SOURCE
        st = run(mut(po + 32 + 2, [0]), strat)                # dep[1] = 0 on a match
        assert st["rc"] == ax.E_STREAM and st["fault_flags"] & ax.F_DEPTH
        st = run(mut(po + 32 + 2, [9]), strat)                # dep[1] > max_depth
        assert st["rc"] == ax.E_STREAM and st["fault_flags"] & ax.F_DEPTH
        st = run(mut(po + 16 + 2, [200, 200]), strat)         # len[1] huge: would run past the block
        assert st["rc"] == ax.E_STREAM and st["fault_flags"] & ax.F_BLOCK_SUM
    two = build_stream([[(b"abcdefgh", 8, 0), (b"WX", 8, 8), (b"z", 5, 26)]], 32)   # depths 1,2,1
    t = two.copy()
    t[po + 32 + 2] = 1                                        # dep[1] 2 -> 1: counts disagree with the histogram
    for strat in [0] + ALL_STRATS:
        st = run(t, strat)
        assert st["rc"] == ax.E_STREAM and st["fault_flags"] & ax.F_DEPTH


# ---------------------------------------------------------------- BASELINE configs at full size (bench.py's launch configuration)
# Every config of BASELINE.json, full size, AUTO strategy, the buffers bench.py uses: the WHOLE output is compared with
# the oracle's sequential decode (the definition) and with the generator's bytes, and the device-side recount of M_src /
# n_match with the oracle validator's.  The streams are encoded by the CPU oracle encoder (5-8 MB/s per core): all of
# them are prepared concurrently, one process each, when the first of these tests runs (about 6 minutes of wall time on
# the GPU box, then a few seconds per test); bench.py finds them in the same cache afterwards.
FULL = {   # id -> (workload, encoder overrides)
    "text256m": ("text256m", {}),
    "fastq1g": ("fastq1g", {}),
    "text1g_d4": ("text1g_d4", {}),
    "stress2g": ("stress2g", {}),                                 # flatten on, D unlimited
    "stress2g_d4": ("stress2g", {"depth_limit": 4}),              # flatten on, D = 4
    "stress2g_noflat": ("stress2g", {"flatten": False}),          # flatten OFF: tens of thousands of waves
}


@pytest.fixture(scope="session")
def full_streams():
    import subprocess
    import sys
    import time
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    t0 = time.time()
    procs = []
    for wl, enc in FULL.values():
        cmd = [sys.executable, os.path.join(root, "bench.py"), "--workload", wl, "--prepare-only"]
        if "depth_limit" in enc:
            cmd += ["--depth-limit", str(enc["depth_limit"])]
        if "flatten" in enc:
            cmd += ["--flatten", str(int(enc["flatten"]))]
        procs.append(subprocess.Popen(cmd, cwd=root))
    for pr in procs:
        assert pr.wait() == 0
    print(f"\n[full_streams] {len(procs)} streams generated + encoded concurrently in {time.time() - t0:.0f} s")
    return True


@pytest.mark.parametrize("case", list(FULL))
def test_full_size(case, full_streams):
    from bench import load_workload
    wl, enc = FULL[case]
    raw, comp = load_workload(wl, None, enc)
    got, st = gpu_decode(comp)
    assert got.size == raw.size
    want = oracle.decode(comp)                                    # sequential: the definition
    assert np.array_equal(want, raw)
    if not np.array_equal(got, want):
        bad = np.flatnonzero(got != want)
        raise AssertionError(f"{case}: {bad.size} bytes differ, first at {bad[0]}")
    rep = oracle.validate(comp)
    assert st["match_src_bytes"] == rep["match_src_bytes"] and st["n_match"] == rep["n_match"]


@pytest.mark.parametrize("seed", range(4))
def test_fuzz_shallow_streams_passes(seed):
    """Encoder-free fuzz restricted to shallow depths (sources drawn from literal bytes or shallow matches): the
    per-depth passes see random overlaps, tile-straddling sources and multi-tile blocks."""
    rng = np.random.default_rng(900 + seed)
    for bs, nb in ((64, 40), (4096, 6), (1 << 16, 3), (1 << 18, 2)):
        blocks = random_blocks(rng, bs, nb, max_len=60 if bs < 4096 else 400, max_lit=12 if bs < 4096 else 60, p_match=0.7)
        deps, bd = py_depths(blocks, bs)
        # cut chains: a match deeper than 12 is replaced by literals of the same bytes
        exp = py_decode(blocks)
        pos, nblocks = 0, []
        for blk, dd in zip(blocks, deps):
            nb_ = []
            for (lit, mlen, off), d in zip(blk, dd):
                pos += len(lit)
                if mlen and d > 12:
                    nb_.append((lit + exp[pos:pos + mlen], 0, 0))
                else:
                    nb_.append((lit, mlen, off))
                pos += mlen
            nblocks.append(nb_)
        assert py_decode(nblocks) == exp
        s = build_stream(nblocks, bs, min_match=1)
        for strat in (ax.WAVES_PASSES, ax.WAVES_LAUNCH, ax.WAVES_PERSISTENT):
            got, _ = gpu_decode(s, strat)
            assert got.tobytes() == exp, (bs, nb, seed, strat)


@pytest.mark.parametrize("seed", range(4))
def test_fuzz_flattened_streams_chain(seed):
    """Encoder-free fuzz of strategy CHAIN: random streams made to satisfy I3 (tests/streams.py flatten_blocks), so
    chains run ACROSS blocks only — arbitrary depths, random overlaps, sources straddling tiles and blocks, blocks of
    one or many tiles, a short last block."""
    rng = np.random.default_rng(1300 + seed)
    for bs, nb in ((64, 40), (4096, 9), (1 << 16, 4), (1 << 18, 3)):
        blocks = flatten_blocks(random_blocks(rng, bs, nb, max_len=60 if bs < 4096 else 400, max_lit=12 if bs < 4096 else 60,
                                              p_match=0.7), bs)
        exp = py_decode(blocks)
        s = build_stream(blocks, bs, flags=5, min_match=1)
        for strat in (ax.WAVES_CHAIN, ax.WAVES_LAUNCH):
            got, st = gpu_decode(s, strat)
            assert got.tobytes() == exp, (bs, nb, seed, strat)
    # I3 broken under a FLATTENED header (an in-block source that a match produced): flagged, not decoded
    bad = [[(b"abcdefgh", 8, 0), (b"WX", 8, 8), (b"z", 5, 26)]]
    got, st = gpu_decode(build_stream(bad, 32, flags=5), ax.WAVES_CHAIN, check=False)
    assert st["rc"] == ax.E_STREAM and st["fault_flags"] & ax.F_DEPTH


def test_chain_needs_flattened_flag():
    s = build_stream([[(b"abcdefgh", 8, 0)]], 32)               # flags = HAS_DEP only
    p = ax.Plan(s.ctypes.data, s.size, 0)
    with pytest.raises(ax.AceapexError):
        p.set_strategy(ax.WAVES_CHAIN)
    p.close()


def test_understated_depth_is_undefined_but_in_bounds():
    """dep[] is trusted for scheduling (include/aceapex.h, docs/FORMAT.md "Trust").  A stream whose dep[]
    understates a depth, with a histogram to match, is rejected by the oracle validator (I4); the GPU library raises no
    fault, stays inside its buffers, and its bytes are undefined — the documented limitation, pinned here."""
    import torch
    seqs = [[(b"abcdefgh", 8, 0), (b"WX", 8, 8), (b"z", 5, 26)]]            # true depths 1, 2, 1
    s = build_stream(seqs, 32, deps=[[1, 1, 1]])
    with pytest.raises(oracle.OracleError) as e:
        oracle.validate(s)
    assert e.value.name == "E_I4"
    G = 4096
    for strat in ALL_STRATS:
        p = ax.Plan(s.ctypes.data, s.size, 0)
        p.set_strategy(strat)
        cd = torch.from_numpy(s).cuda()
        ob, sb = p.out_bytes, (p.scratch_bytes + 255) & ~255
        big_o = torch.full((G + ob + G,), 0xEE, dtype=torch.uint8, device="cuda")
        big_s = torch.full((G + sb + G,), 0xEE, dtype=torch.uint8, device="cuda")
        p.decode(cd.data_ptr(), big_o.data_ptr() + G, ob, big_s.data_ptr() + G, sb, ax.PHASE_ALL, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert p.stats(big_s.data_ptr() + G, check=False)["rc"] == 0
        assert bool((big_o[:G] == 0xEE).all()) and bool((big_o[G + ob:] == 0xEE).all())
        assert bool((big_s[:G] == 0xEE).all()) and bool((big_s[G + sb:] == 0xEE).all())
        p.close()


def test_adjacent_merges_and_plain_stores_in_one_wave():
    """within one wave, short non-overlapping matches are OR-merged as whole 8-byte words (red.or.b64) while
    overlapping short matches and long matches use plain 1..16-byte stores; neighbours of both kinds share 8-byte words.
    Many such neighbours, every alignment, one wave: the bytes must come out right (the L2 applies reductions and byte-
    enabled stores to disjoint bytes of a word independently — DESIGN.md 6.1)."""
    rng = np.random.default_rng(77)
    base = rng.integers(0, 256, 600, dtype=np.uint8).tobytes()
    seqs = [(base, 0, 0)]
    for i in range(3000):
        kind = i % 3
        if kind == 0:
            seqs.append((b"", int(rng.integers(4, 17)), int(rng.integers(0, 500))))          # simple: merged
        elif kind == 1:
            seqs.append((bytes([65 + i % 20]), int(rng.integers(5, 30)), 0))                 # placeholder, fixed below
        else:
            seqs.append((b"", int(rng.integers(33, 90)), int(rng.integers(0, 400))))         # long: warp copy
    # kind 1 becomes a self-overlapping short match: source = the literal byte just before it (period 1)
    pos, fixed = 0, []
    for lit, ml, off in seqs:
        pos += len(lit)
        fixed.append((lit, ml, pos - 1) if (len(lit) == 1 and ml) else (lit, ml, off))
        pos += ml
    blocks = [fixed]
    s = build_stream(blocks, 1 << 20, flags=5)                                               # every source is a literal: one wave
    exp = py_decode(blocks)
    for strat in (ax.WAVES_LAUNCH, ax.WAVES_PERSISTENT, ax.WAVES_PASSES, ax.WAVES_CHAIN):
        for _ in range(3):
            got, st = gpu_decode(s, strat)
            assert st["max_depth"] == 1 and got.tobytes() == exp, strat


def test_guard_bands_all_strategies():
    """compute-sanitizer is closed on this GPU pool, so out-of-bounds writes are hunted with guard bands: the output
    and the scratch sit inside larger tensors filled with 0xEE; after a decode with every strategy the guards are
    intact and the bytes are right.  Sizes chosen so the last block is short and the output is not a multiple of 16."""
    import torch
    G = 8192
    cases = [("stress", (3 << 20) + 13, dict(block_size=1 << 18)), ("text", (2 << 20) + 5, dict(depth_limit=4)),
             ("markov", (1 << 20) + 777, dict(block_size=1 << 16, flatten=False)), ("fastq", (2 << 20) + 1, dict(depth_limit=2))]
    for kind, n, kw in cases:
        raw = workloads.generate(kind, n, 77)
        comp = oracle.encode(raw, **kw)
        for strat in strats_for(comp):
            p = ax.Plan(comp.ctypes.data, comp.size, 0)
            p.set_strategy(strat)
            cd = torch.from_numpy(comp).cuda()
            ob, sb = p.out_bytes, (p.scratch_bytes + 255) & ~255
            big_o = torch.full((G + ob + G,), 0xEE, dtype=torch.uint8, device="cuda")
            big_s = torch.full((G + sb + G,), 0xEE, dtype=torch.uint8, device="cuda")
            for _ in range(2):                                   # twice: scratch reuse must not leak either
                p.decode(cd.data_ptr(), big_o.data_ptr() + G, ob, big_s.data_ptr() + G, sb, ax.PHASE_ALL,
                         torch.cuda.current_stream().cuda_stream)
            torch.cuda.synchronize()
            assert p.stats(big_s.data_ptr() + G)["rc"] == 0
            assert bool((big_o[:G] == 0xEE).all()) and bool((big_o[G + ob:] == 0xEE).all()), (kind, strat, "output guard")
            assert bool((big_s[:G] == 0xEE).all()) and bool((big_s[G + sb:] == 0xEE).all()), (kind, strat, "scratch guard")
            assert np.array_equal(big_o[G:G + n].cpu().numpy(), raw), (kind, strat)
            p.close()


def test_sparse_depths_empty_waves():
    """Stored depths may be larger than necessary (any order-preserving labelling decodes correctly): here every
    depth is doubled, so every odd wave is empty — empty waves, empty passes and histogram entries of 0."""
    rng = np.random.default_rng(31)
    for bs, nb in ((4096, 5), (1 << 16, 3)):
        blocks = random_blocks(rng, bs, nb, max_len=200, max_lit=30, p_match=0.7)
        deps, _ = py_depths(blocks, bs)
        exp = py_decode(blocks)
        # keep the test in the shallow range as well: cut chains deeper than 6 (stored depth 12)
        pos, nblocks = 0, []
        for blk, dd in zip(blocks, deps):
            nb_ = []
            for (lit, mlen, off), d in zip(blk, dd):
                pos += len(lit)
                nb_.append((lit + exp[pos:pos + mlen], 0, 0) if (mlen and d > 6) else (lit, mlen, off))
                pos += mlen
            nblocks.append(nb_)
        deps2, _ = py_depths(nblocks, bs)
        doubled = [[2 * d for d in dd] for dd in deps2]
        s = build_stream(nblocks, bs, deps=doubled, min_match=1)
        for strat in [0] + ALL_STRATS:
            got, st = gpu_decode(s, strat)
            assert got.tobytes() == exp, (bs, strat)
            assert st["max_depth"] % 2 == 0
