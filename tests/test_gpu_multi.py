"""N > 1 on GPUs: every rank runs the LIBRARY on its shard of one batch (shard.shard_events), the per-event results are
all-gathered over NCCL and compared with the oracle on the whole batch.  Skipped unless two CUDA devices are visible (the
gloo / oracle variant in test_shard_gloo.py covers the host logic on CPU)."""
import os
import socket

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_2511_02742_b200 import hough as H
    from paper_2511_02742_b200 import shard, synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    try:
        wl = synth.workload(1)
        b = synth.generate(wl, 0, 600)
        ranges = shard.shard_events(b.offsets, world)
        u, v, off = shard.local_batch(b.u, b.v, b.offsets, ranges[rank])
        plan = H.plan_for_workload(wl, len(off) - 1, len(u), int(np.diff(off).max()), device=rank)
        du, dv, do = (torch.from_numpy(np.ascontiguousarray(a)).cuda(rank) for a in (u, v, off))
        cands, n_found = H.hough_find_clusters(plan, du, dv, do)
        labels = H.hough_assign_hits(plan, du, dv, do, cands, n_found)
        torch.cuda.synchronize(rank)
        nf = shard.gather_per_event(n_found, ranges)
        votes = shard.gather_per_event(cands[:, :4, 2].contiguous(), ranges)        # votes of the first four records
        n_lab = torch.tensor([float((labels >= 0).sum().item())], dtype=torch.float64, device=f"cuda:{rank}")
        dist.all_reduce(n_lab, op=dist.ReduceOp.SUM)
        if rank == 0:
            q.put((nf.cpu().numpy(), votes.cpu().numpy(), float(n_lab.item())))
        H.hough_plan_destroy(plan)
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(600)
@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two CUDA devices")
def test_two_ranks_run_the_library_on_their_shards():
    import torch.multiprocessing as mp
    from oracle import hough_c as C
    from paper_2511_02742_b200 import synth
    from util import params_of
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    nf, votes, n_lab = q.get()
    for pr in procs:
        pr.join(300)
        assert pr.exitcode == 0
    wl = synth.workload(1)
    b = synth.generate(wl, 0, 600)
    o = C.run_batch(b.u, b.v, b.offsets, params_of(wl))
    np.testing.assert_array_equal(nf, o["n_found"])
    np.testing.assert_array_equal(votes, o["cands"]["votes"][:, :4])
    assert n_lab == float((o["labels"] >= 0).sum())
