"""-m gpu: "all work is enqueued on psl_config.stream" (include/psl.h).  The library on caller-created, non-blocking
streams: nothing may land on the default stream, and two contexts fed alternately on two streams must not disturb one
another.  Results against the oracle, bit for bit, as everywhere."""
import numpy as np
import pytest

import workloads as W
from helpers import assert_matches_oracle, dirty, library_result
from oracle import psl_oracle as O

pytestmark = pytest.mark.gpu


def test_a_side_stream_never_touches_the_default_stream():
    """the default stream is blocked by a long spin kernel; a context on a non-blocking stream must load, build and
    report while that kernel is still running -- anything the library put on stream 0 would sit behind it"""
    import torch

    import paper_1302_1861_b200 as P

    side = torch.cuda.Stream()
    cases = [(W.config(2, 150_000), None), (W.config(3, 150_000), W.config(3).beams[0]), (W.config(4, 150_000), W.config(4).beams[0])]
    prepared = []
    for w, beam in cases:
        r = dirty(w.records(), 5)
        ctx = P.PslContext(w.grid, w.geometry, w.mode, max_records=len(r), stream=side, max_launch_records=1 << 18)
        lib_beam = None if beam is None else ctx.beam(beam)  # uploads the map on the side stream
        prepared.append((w, beam, lib_beam, r, ctx))
    pinned = [torch.from_numpy(np.ascontiguousarray(r).view(np.uint8).reshape(-1).copy()).pin_memory() for _, _, _, r, _ in prepared]
    w2 = prepared[0][0]

    def everything():
        for (w, beam, lib_beam, r, ctx), host in zip(prepared, pinned):
            ctx.reset()
            half = (len(r) // 2) // 4 * 4
            ctx.load_chunk(host[:half * 28])
            ctx.load_chunk(host[half * 28:])
            ctx.build_batches(lib_beam)
            st = ctx.get_stats()  # synchronises the context's stream only
            assert st["n_in"] == len(r)
            if w.mode == P.MODE_INDEX:  # the sampling layer too (it synchronises its own stream)
                total, lens = ctx.plan_set([lib_beam], 50_000, seed=3)
                t, ie = divmod(max(range(len(lens)), key=lambda i: lens[i]), w.grid["n_ebins"])
                assert 0 < ctx.sample_batch(t, ie)["n_list"] <= 50_000
                ctx.build_batches(None)
                ctx.get_stats()
                ctx.build_batches(lib_beam)
                ctx.get_stats()
            else:
                assert ctx.flush_schedule(4096)["n_events"] > 0
        with torch.cuda.stream(side):
            P.count_static(w2.grid, w2.geometry, dev, counts, stream=side)

    with torch.cuda.stream(side):
        dev = pinned[0].to("cuda", non_blocking=True)
        counts = torch.zeros(w2.n_keys, dtype=torch.int32, device="cuda")
    everything()  # once without the blocker: the first launch of a kernel loads its module, which may wait for the device
    torch.cuda.synchronize()
    blocker = torch.cuda.Event()
    torch.cuda._sleep(int(6e9))  # about three seconds on the default stream
    blocker.record()             # ... and an event behind it
    everything()
    side.synchronize()
    assert not blocker.query(), "the default stream finished first: the timing of this test proves nothing"
    torch.cuda.synchronize()
    for w, beam, lib_beam, r, ctx in prepared:
        with torch.cuda.stream(side):
            lib = library_result(ctx)
        side.synchronize()
        assert_matches_oracle(lib, O.Oracle(w.grid, w.geometry).build(r, beam))
        ctx.destroy()
    want = O.Oracle(w2.grid, w2.geometry).build(prepared[0][3], None)["counts"]
    assert np.array_equal(counts.cpu().numpy().view(np.uint32), want)


def test_two_contexts_fed_alternately_on_two_streams():
    import torch

    import paper_1302_1861_b200 as P

    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    w1, w2 = W.config(3, 400_000), W.config(5, 400_000)
    r1, r2 = dirty(w1.records(), 1), dirty(w2.records(), 2)
    c1 = P.PslContext(w1.grid, w1.geometry, w1.mode, max_records=len(r1), stream=s1)
    c2 = P.PslContext(w2.grid, w2.geometry, w2.mode, max_records=len(r2), stream=s2)
    h1 = torch.from_numpy(np.ascontiguousarray(r1).view(np.uint8).reshape(-1).copy()).pin_memory()
    h2 = torch.from_numpy(np.ascontiguousarray(r2).view(np.uint8).reshape(-1).copy()).pin_memory()
    step = 50_000
    for first in range(0, 400_000, step):  # chunks of the two phase-spaces in turn, nothing waited for
        c1.load_chunk(h1[first * 28:(first + step) * 28])
        c2.load_chunk(h2[first * 28:(first + step) * 28])
    b1 = c1.beam(w1.beams[0])
    beams2 = [c2.beam(b) for b in w2.beams[:3]]
    o1, o2 = O.Oracle(w1.grid, w1.geometry), O.Oracle(w2.grid, w2.geometry)
    for k in range(3):
        c1.build_batches(b1 if k != 1 else None)
        c2.build_batches(beams2[k])
        with torch.cuda.stream(s1):
            l1 = library_result(c1)
        with torch.cuda.stream(s2):
            l2 = library_result(c2)
        torch.cuda.synchronize()
        assert_matches_oracle(l1, o1.build(r1, w1.beams[0] if k != 1 else None))
        assert_matches_oracle(l2, o2.build(r2, w2.beams[k]))
    c1.destroy()
    c2.destroy()
