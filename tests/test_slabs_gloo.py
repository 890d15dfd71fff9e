"""The message layer of the slab decomposition (paper_1912_04232_b200/slabs.py DistComm) over
torch.distributed with the gloo backend on CPU: variable-length (rows, ids) messages to the previous and
the next rank, world sizes 2 (the other rank is both neighbours) and 3, and the flag all-reduce."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1912_04232_b200 import slabs as SL


def _msg(src, direction, k):
    """A recognisable message: k rows whose content names the sender and the direction."""
    rows = torch.full((k, 8), float(10 * src + direction)) + torch.arange(k, dtype=torch.float32)[:, None]
    ids = torch.arange(k, dtype=torch.int32) + 1000 * src + 100 * direction
    return rows, ids


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        comm = SL.DistComm()
        ok = True
        for rnd in range(3):
            kp, kn = (rank + rnd) % 3, (2 * rank + rnd + 1) % 4          # 0 rows happens too
            (fp, fn), = comm.shift([_msg(rank, 0, kp)], [_msg(rank, 1, kn)])
            prev, nxt = (rank - 1) % world, (rank + 1) % world
            want_p = _msg(prev, 1, (2 * prev + rnd + 1) % 4)              # what prev sent to ITS next
            want_n = _msg(nxt, 0, (nxt + rnd) % 3)                        # what next sent to ITS previous
            ok &= torch.equal(fp[0], want_p[0]) and torch.equal(fp[1], want_p[1])
            ok &= torch.equal(fn[0], want_n[0]) and torch.equal(fn[1], want_n[1])
            # plain tensors (the per-step position rows)
            (tp, tn), = comm.shift([torch.full((rank + 1, 4), float(rank))], [torch.full((rank + 2, 4), -float(rank))])
            ok &= torch.equal(tp, torch.full((prev + 2, 4), -float(prev))) and torch.equal(tn, torch.full((nxt + 1, 4), float(nxt)))
            # the step exchange: row counts known to both ends, the receive buffers reused from step to step
            for _ in range(2):
                (tp, tn), = comm.shift_rows([torch.full((rank + 1, 4), float(rank + rnd))], [torch.full((rank + 2, 4), -float(rank + rnd))],
                                            [(prev + 2, nxt + 1)])
                ok &= torch.equal(tp, torch.full((prev + 2, 4), -float(prev + rnd))) and torch.equal(tn, torch.full((nxt + 1, 4), float(nxt + rnd)))
        flags = []
        for r in list(range(world)) + [-1]:
            words = torch.tensor([1 if rank == r else 0, 0, 5, 0], dtype=torch.int32)
            comm.share_flag(words)                                   # only the flag word travels
            ok &= words.tolist()[1:] == [0, 5, 0]
            flags.append(bool(words[0]))
        none = flags.pop()
        q.put((rank, bool(ok), flags, none))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_neighbour_messages_gloo(world):
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = {}
    for _ in procs:
        r, ok, flags, none = q.get(timeout=120)
        got[r] = (ok, flags, none)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        assert got[r] == (True, [True] * world, False)


def test_local_comm_is_the_same_shift():
    world = 4
    comm = SL.LocalComm(world)
    got = comm.shift([("p", r) for r in range(world)], [("n", r) for r in range(world)])
    for r in range(world):
        assert got[r] == (("n", (r - 1) % world), ("p", (r + 1) % world))
