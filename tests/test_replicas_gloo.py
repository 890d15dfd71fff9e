"""world_size-2 gloo test (CPU) of the multi-GPU plumbing: replicas draw independent samples of
the same config, the job time is the max over ranks, the rate is the whole-job aggregate."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1912_04232_b200 import replicas as R
    from paper_1912_04232_b200 import workloads as W
    assert R.world() == (rank, world)
    w = W.config(0, replica=R.replica_index(rank))
    # every rank holds the same box and a different sample of the positions
    digest = torch.tensor([float(np.float64(w.pos[:, :3]).sum()), float(w.box[0])], dtype=torch.float64)
    both = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(both, digest)
    assert both[0][1] == both[1][1] and both[0][0] != both[1][0]
    t = R.max_over_ranks(1.0 + rank)            # rank 1 is the slow one
    assert t == float(world)
    rate = R.whole_job_rate(units_per_rank=w.n * 100, seconds_max=t)
    assert rate == world * w.n * 100 / t
    dist.barrier()
    if rank == 0:
        out.put((t, rate))
    dist.destroy_process_group()


def test_two_replicas_over_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    t, rate = out.get()
    assert t == 2.0 and rate == 2 * 864 * 100 / 2.0


def test_single_process_defaults():
    from paper_1912_04232_b200 import replicas as R
    assert R.world() == (0, 1)
    assert R.max_over_ranks(3.5) == 3.5
    assert R.whole_job_rate(10.0, 2.0) == 5.0
