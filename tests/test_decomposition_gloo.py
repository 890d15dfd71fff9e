"""Host logic of the split-list multi-GPU loop (paper_1912_04232_b200/decomposition.py)
on CPU: the ranges, and the slot exchange over torch.distributed with the gloo backend, world_size 2."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1912_04232_b200 import decomposition as D


def test_ranges_cover_and_align():
    for n in (1, 31, 32, 33, 864, 16384, 256000, 1048576):
        for world in (1, 2, 3, 4, 8):
            rs = D.ranges(n, world)
            assert rs[0][0] == 0 and rs[-1][1] == n
            for (b0, e0), (b1, e1) in zip(rs, rs[1:]):
                assert e0 == b1
            for b, e in rs:
                assert (b % 32 == 0 or b == e == n) and (e % 32 == 0 or e == n) and b <= e      # empty: (n, n)
            sizes = [e - b for b, e in rs if e > b]
            assert max(sizes) - min(sizes) <= 32 or n % 32
            assert D.slot_rows(n, world) == max(e - b for b, e in rs) + 1


def test_pack_unpack_roundtrip():
    n, world = 200, 3
    x = torch.arange(n * 4, dtype=torch.float32).reshape(n, 4)
    rows = D.slot_rows(n, world)
    for flags in ([0, 0, 0], [0, 1, 0]):
        slots = torch.stack([D.pack(x, rg, rows, torch.tensor([f], dtype=torch.int32))
                             for rg, f in zip(D.ranges(n, world), flags)])
        out = torch.zeros_like(x)
        assert bool(D.unpack(slots, n, world, out)) == bool(sum(flags))
        assert torch.equal(out, x)


def _worker(rank, world, port, n, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ex = D.DistExchange()
        g = torch.Generator().manual_seed(7)
        full = torch.rand(n, 4, generator=g)                    # the state every rank should end with
        mine = torch.zeros(n, 4)
        b, e = D.ranges(n, world)[rank]
        mine[b:e] = full[b:e]                                   # a rank only has its own range right
        rows = D.slot_rows(n, world)
        results = []
        for step_flag in (0, 1):                                # rank 1 raises its flag in the second round
            flag = torch.tensor([step_flag if rank == 1 else 0], dtype=torch.int32)
            slots = ex.all_gather(D.pack(mine, (b, e), rows, flag))
            out = mine.clone()
            any_flag = bool(D.unpack(slots, n, world, out))
            results.append((any_flag, bool(torch.equal(out, full))))
        q.put((rank, results))
    finally:
        dist.destroy_process_group()


def test_exchange_gloo_world2():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    world, n = 2, 1000
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        assert got[r] == [(False, True), (True, True)]          # every rank sees the flag and the full state
