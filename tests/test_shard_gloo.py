"""N > 1 path on CPU: event sharding and the gather of per-event results over torch.distributed (gloo, world size 2).
The kernels are not involved (no GPU here); each rank runs the oracle on its shard, which also shows that sharded
processing equals whole-batch processing event by event."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import hough_c as C
from paper_2511_02742_b200 import shard, synth
from util import params_of


def test_shard_events_covers_and_balances():
    rng = np.random.default_rng(5)
    for world in (1, 2, 3, 8):
        for _ in range(20):
            n = int(rng.integers(0, 40))
            offsets = np.concatenate([[0], np.cumsum(rng.integers(0, 50, size=n))]).astype(np.int64)
            r = shard.shard_events(offsets, world)
            assert len(r) == world and r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1)) and all(a <= b for a, b in r)
            total = int(offsets[-1])
            if total and n:
                biggest = int(np.diff(offsets).max())
                for k in range(1, world):      # every cut is within one event of its ideal position
                    assert abs(int(offsets[r[k][0]]) - total * k / world) <= biggest
    assert shard.shard_events(np.zeros(5, np.int64), 2) == [(0, 2), (2, 4)]      # no hits: split the events


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = synth.workload(1)
        b = synth.generate(wl, 0, 24)
        p = params_of(wl)
        ranges = shard.shard_events(b.offsets, world)
        u, v, off = shard.local_batch(b.u, b.v, b.offsets, ranges[rank])
        o = C.run_batch(u, v, off, p)
        n_found = shard.gather_per_event(torch.from_numpy(o["n_found"].astype(np.int32)), ranges)
        votes0 = shard.gather_per_event(torch.from_numpy(np.ascontiguousarray(o["cands"]["votes"][:, :4]).astype(np.int32)), ranges)
        hits = torch.tensor([float(len(u))], dtype=torch.float64)
        dist.all_reduce(hits, op=dist.ReduceOp.SUM)
        if rank == 0:
            q.put((n_found.numpy(), votes0.numpy(), float(hits.item()), ranges))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_ranks_gloo_equal_whole_batch():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    n_found, votes0, hits, ranges = q.get()
    for pr in procs:
        pr.join(120)
        assert pr.exitcode == 0
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 24)
    whole = C.run_batch(b.u, b.v, b.offsets, params_of(wl))
    np.testing.assert_array_equal(n_found, whole["n_found"])
    np.testing.assert_array_equal(votes0, whole["cands"]["votes"][:, :4])
    assert hits == b.n_hits and ranges[0][1] == ranges[1][0] and 0 < ranges[0][1] < 24
