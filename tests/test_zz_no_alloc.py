"""aceapex_decode_noalloc: the decode for callers that cannot allocate device scratch (include/aceapex.h).

Collected last on purpose (the suite runs with ``pytest -x``).  The new entry point must give exactly the bytes of the
existing path (caller-provided scratch) and of the oracle — this is byte work: the tolerance is zero, as everywhere in
tests/test_gpu_parity.py — on calls in a row that share the library's static scratch array, whatever the previous call
left in it."""
import numpy as np
import pytest

import oracle
import workloads
import paper_2606_04268_b200 as ax

pytestmark = pytest.mark.gpu


def _existing_path(comp, strategy):
    from paper_2606_04268_b200.torch_io import Decoder
    d = Decoder(comp, 0, strategy)
    try:
        d.run()
        return d.output(), d.stats()
    finally:
        d.close()


def _noalloc(comp, strategy, out_dev=None):
    import torch
    p = ax.Plan(comp.ctypes.data, comp.size, 0)
    try:
        if strategy:
            p.set_strategy(strategy)
        cd = torch.from_numpy(comp).cuda()
        od = out_dev if out_dev is not None else torch.full((max(p.out_bytes, 16),), 0xA5, dtype=torch.uint8, device="cuda")
        p.decode_noalloc(cd.data_ptr(), od.data_ptr(), od.numel(), torch.cuda.current_stream().cuda_stream)
        st = p.stats_noalloc()                       # synchronises the stream; must precede the next call (shared scratch)
        return od[:p.raw_bytes].cpu().numpy(), st
    finally:
        p.close()


def test_noalloc_matches_existing_path_on_calls_in_a_row():
    streams = []
    raw_a = workloads.generate("markov", (1 << 20) + 12345, 260604268)
    raw_b = workloads.generate("text", (2 << 20) + 77, 260604269)
    streams.append((raw_a, oracle.encode(raw_a, block_size=1 << 16), [ax.WAVES_AUTO, ax.WAVES_CHAIN, ax.WAVES_PERSISTENT]))
    streams.append((raw_b, oracle.encode(raw_b, block_size=1 << 18, depth_limit=4), [ax.WAVES_AUTO, ax.WAVES_PASSES, ax.WAVES_GRAPH]))
    streams.append((raw_a, oracle.encode(raw_a, block_size=1 << 16, flatten=False), [ax.WAVES_AUTO, ax.WAVES_LAUNCH]))
    want = {}
    for i, (raw, comp, strats) in enumerate(streams):
        assert np.array_equal(oracle.decode(comp), raw)
        for s in strats:
            if s != ax.WAVES_GRAPH:
                got, st = _existing_path(comp, s)
                assert np.array_equal(got, raw)
                want[(i, s)] = st
    # two rounds over every (stream, strategy), back to back: each call finds the previous call's scratch contents
    for rnd in range(2):
        for i, (raw, comp, strats) in enumerate(streams):
            for s in strats:
                got, st = _noalloc(comp, s)
                assert got.size == raw.size
                if not np.array_equal(got, raw):
                    bad = np.flatnonzero(got != raw)
                    raise AssertionError(f"round {rnd} stream {i} strategy {s}: {bad.size} bytes differ, first at {bad[0]}")
                ref = want.get((i, s)) or want[(i, ax.WAVES_AUTO)]
                assert st["match_src_bytes"] == ref["match_src_bytes"] and st["n_match"] == ref["n_match"] and st["rc"] == 0
                if s == ax.WAVES_GRAPH:
                    assert st["strategy"] == ax.WAVES_LAUNCH          # instantiating a graph would allocate


def test_noalloc_allocates_nothing_and_rejects_oversize():
    import torch
    L = ax._lib()
    cap = L.aceapex_noalloc_max_scratch_bytes()
    assert cap == 16 << 20
    raw = workloads.config_bytes("synth4m")                          # BASELINE config 0 fits the static buffer
    comp = oracle.encode(raw)
    p = ax.Plan(comp.ctypes.data, comp.size, 0)
    assert p.scratch_bytes <= cap
    cd = torch.from_numpy(comp).cuda()
    od = torch.zeros(p.out_bytes, dtype=torch.uint8, device="cuda")
    sp = torch.cuda.current_stream().cuda_stream
    p.decode_noalloc(cd.data_ptr(), od.data_ptr(), od.numel(), sp)    # warm-up: module load, symbol address
    assert p.stats_noalloc()["rc"] == 0
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        od.fill_(0xA5)
        p.decode_noalloc(cd.data_ptr(), od.data_ptr(), od.numel(), sp)
        assert p.stats_noalloc()["rc"] == 0
        assert np.array_equal(od[:raw.size].cpu().numpy(), raw)
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < (1 << 20), "device memory was allocated by the no-allocation entry point"
    # argument errors behave like aceapex_decode's
    assert L.aceapex_decode_noalloc(p._h, cd.data_ptr(), od.data_ptr(), p.out_bytes - 16, sp) == ax.E_CAPACITY
    assert L.aceapex_decode_noalloc(p._h, cd.data_ptr(), od.data_ptr() + 1, od.numel(), sp) == ax.E_ALIGN
    assert L.aceapex_decode_noalloc(p._h, None, od.data_ptr(), od.numel(), sp) == ax.E_ARG
    p.close()
    # a stream whose scratch exceeds the stated maximum is rejected with a clear error, nothing is launched
    big = workloads.generate("text", 24 << 20, 5)
    cbig = oracle.encode(big, max_chain=4)
    pb = ax.Plan(cbig.ctypes.data, cbig.size, 0)
    assert pb.scratch_bytes > cap
    cdb = torch.from_numpy(cbig).cuda()
    odb = torch.full((pb.out_bytes,), 0x5A, dtype=torch.uint8, device="cuda")
    rc = L.aceapex_decode_noalloc(pb._h, cdb.data_ptr(), odb.data_ptr(), odb.numel(), sp)
    assert rc == ax.E_NOALLOC_LIMIT
    assert b"static no-allocation buffer" in L.aceapex_strerror(rc)
    torch.cuda.synchronize()
    assert bool((odb == 0x5A).all())
    pb.close()
