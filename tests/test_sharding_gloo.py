"""-m "not gpu": the N > 1 path on CPU -- two gloo ranks shard the record stream the way bench.py does and
exchange counts[K]; the per-rank global slots must tile the oracle's single-run result exactly."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as W
from oracle import psl_oracle as O
from paper_1302_1861_b200 import sharding as S


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_total, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.config(3, n_total)
        first, n = S.shard_range(rank, world, n_total)
        rec = W.generate(w.gen, first, n)
        res = O.Oracle(w.grid, w.geometry).build(rec, w.beams[0])
        counts = torch.from_numpy(res["counts"].astype(np.int64))
        slot0, total = S.global_offsets(counts)
        ms = S.max_over_ranks(float(rank + 1))
        q.put((rank, first, n, res["src_index"] + first, res["offsets"].astype(np.int64), slot0.numpy(), total.numpy(), ms))
    finally:
        dist.destroy_process_group()


def test_two_rank_shards_tile_the_single_run_result():
    world, n_total = 2, 30_001
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_total, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # shards: contiguous, disjoint, complete, multiples of 4 except the last
    assert got[0][1] == 0 and got[0][1] + got[0][2] == got[1][1] and got[1][1] + got[1][2] == n_total
    assert got[0][2] % 4 == 0
    w = W.config(3, n_total)
    whole = O.Oracle(w.grid, w.geometry).build(W.generate(w.gen, 0, n_total), w.beams[0])
    K = len(whole["counts"])
    assert np.array_equal(got[0][6], whole["counts"]) and np.array_equal(got[1][6], whole["counts"])
    out = np.full(whole["n_survivors"], -1, dtype=np.int64)
    for rank, first, n, src, off, slot0, total, ms in got:
        assert ms == float(world)  # max over ranks
        for k in range(K):
            c = off[k + 1] - off[k]
            out[slot0[k]:slot0[k] + c] = src[off[k]:off[k + 1]]
    assert np.array_equal(out, whole["src_index"].astype(np.int64))  # the global stable order, particle by particle


def test_shard_range_edges():
    assert S.shard_range(0, 1, 10) == (0, 10)
    assert S.shard_range(3, 4, 10) == (10, 0)          # 4-record granularity leaves the last shard empty
    assert [S.shard_range(r, 3, 100) for r in range(3)] == [(0, 36), (36, 36), (72, 28)]
