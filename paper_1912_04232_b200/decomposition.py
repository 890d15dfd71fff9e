"""Multi-GPU velocity-Verlet loop by replicated positions and a split neighbor list (
DESIGN.md §8).

One process per GPU.  Every rank holds all positions and runs the same (deterministic) cell list and
re-sort; rank r builds list rows, computes forces and integrates only for its own range of the
cell-sorted particles (md_set_range).  Per step the ranks exchange their position ranges together with
their half-skin flags in ONE all-gather; at a rebuild they also exchange their velocity ranges, because
the re-sort moves particles -- and with them ownership -- between ranges.  What is split is the list
(4 * capacity bytes per particle) and the work on it; a position is 16 bytes.

This module is plumbing only: ranges, the packing of what travels, and the order of the C-ABI calls.
All arithmetic runs in the library's kernels, and a run on P ranks is bit-identical to md_nve_step on
one (same kernels, same per-particle operation order).  `exchange` is torch.distributed's all-gather
(NCCL over NVLink on GPUs, gloo in the CPU test); for tests on one GPU `run_local` steps P contexts
of one process in lockstep.
"""
from __future__ import annotations

import torch

TILE = 32


def ranges(n: int, world: int) -> list[tuple[int, int]]:
    """Contiguous particle ranges, whole list tiles each, sizes differing by at most one tile.
    Ranks beyond the number of tiles get an empty range (begin == end)."""
    ntiles = (n + TILE - 1) // TILE
    base, extra = divmod(ntiles, world)
    out, t = [], 0
    for r in range(world):
        k = base + (1 if r < extra else 0)
        out.append((min(t * TILE, n), min((t + k) * TILE, n)))
        t += k
    return out


def slot_rows(n: int, world: int) -> int:
    """Rows of one rank's slot in the exchange buffer: the largest range plus one row for the flag."""
    return max(e - b for b, e in ranges(n, world)) + 1


def pack(x: torch.Tensor, rng: tuple[int, int], rows: int, flag: torch.Tensor | None = None,
         out: torch.Tensor | None = None) -> torch.Tensor:
    """This rank's slot: x[begin:end], zero padding, and in the last row the flag (as a float).
    `out`: a slot buffer to reuse (its padding rows stay as they are: zero from its creation)."""
    b, e = rng
    slot = out if out is not None else torch.zeros(rows, x.shape[1], dtype=x.dtype, device=x.device)
    slot[: e - b] = x[b:e]
    slot[rows - 1, 0] = flag.to(x.dtype)[0] if flag is not None else 0.0
    return slot


def unpack(slots: torch.Tensor, n: int, world: int, out: torch.Tensor, skip: int = -1) -> torch.Tensor:
    """slots [world, rows, 4] -> out[begin_r:end_r] for every r but `skip` (the caller's own range, which
    it already holds); returns the OR of the flags (0-d bool)."""
    rows = slots.shape[1]
    for r, (b, e) in enumerate(ranges(n, world)):
        if r != skip:
            out[b:e] = slots[r, : e - b]
    return (slots[:, rows - 1, 0] != 0).any()


class DistExchange:
    """All-gather over torch.distributed (one process per GPU)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.world, self.rank = dist.get_world_size(group), dist.get_rank(group)

    def all_gather(self, slot: torch.Tensor) -> torch.Tensor:
        parts = [torch.empty_like(slot) for _ in range(self.world)]
        self.dist.all_gather(parts, slot, group=self.group)
        return torch.stack(parts)


class RankLoop:
    """The step loop of one rank around a binding.System (which owns the tensors)."""

    def __init__(self, system, rank: int, world: int):
        from . import binding as B
        self.B, self.S, self.rank, self.world = B, system, rank, world
        self.n = system.n
        self.range = ranges(self.n, world)[rank]
        if self.range[0] == self.range[1]:
            raise ValueError(f"rank {rank} of {world} owns no list tile of {self.n} particles")
        self.rows = slot_rows(self.n, world)
        if not system.cfg.resort:
            raise ValueError("a split list needs resort = 1: ranges are ranges of the cell-sorted order")
        B.md_set_range(system.sys, *self.range)
        self.rebuilds = 0
        self.slot = torch.zeros(self.rows, 4, dtype=torch.float32, device=system.pos.device)    # reused every step

    # -- the phases of one step; `exchange` sits between them
    def start(self):
        """List rows and forces of the own range for the initial (replicated) state."""
        self.S.build()
        self.force()

    def move(self) -> torch.Tensor:
        w = self.S.w
        self.B.md_kick_drift(self.S.sys, self.S.pos, self.S.vel, self.S.force, w.dt, w.mass, self.S.flag)
        return pack(self.S.pos, self.range, self.rows, self.S.flag, out=self.slot)

    def absorb_positions(self, slots: torch.Tensor) -> bool:
        return bool(unpack(slots, self.n, self.world, self.S.pos, skip=self.rank))

    def velocity_slot(self) -> torch.Tensor:
        return pack(self.S.vel, self.range, self.rows, out=self.slot)

    def rebuild(self, vel_slots: torch.Tensor):
        unpack(vel_slots, self.n, self.world, self.S.vel, skip=self.rank)
        self.S.build()                     # global cell list + re-sort, list rows of the own range
        self.rebuilds += 1

    def force(self):
        self.S.compute_force(want_energy=False)

    def force_and_kick(self):
        """The second half of the step in one launch (md_nve_step's own closing kernel)."""
        S, w = self.S, self.S.w
        self.B.md_force_half_kick(S.sys, S.pot, S.pos, S.nbr_idx, S.nbr_count, S.force, S.vel, w.dt, w.mass)


def run(loop: RankLoop, exchange, nsteps: int) -> None:
    """nsteps on this rank; every rank of the group must make the same call."""
    for _ in range(nsteps):
        slots = exchange.all_gather(loop.move())
        if loop.absorb_positions(slots):
            loop.rebuild(exchange.all_gather(loop.velocity_slot()))
        loop.force_and_kick()


def gather_state(loop: RankLoop, exchange) -> None:
    """After a run: make velocities and forces complete on every rank (positions already are)."""
    for x in (loop.S.vel, loop.S.force):
        unpack(exchange.all_gather(pack(x, loop.range, loop.rows)), loop.n, loop.world, x)


def run_local(loops: list[RankLoop], nsteps: int) -> None:
    """The same protocol for P contexts of ONE process (tests on one GPU): the phases of all ranks run
    one after the other, the all-gather is a stack of their slots."""
    for _ in range(nsteps):
        slots = torch.stack([lp.move() for lp in loops])
        flags = [lp.absorb_positions(slots) for lp in loops]
        assert all(f == flags[0] for f in flags)
        if flags[0]:
            vel = torch.stack([lp.velocity_slot() for lp in loops])
            for lp in loops:
                lp.rebuild(vel)
        for lp in loops:
            lp.force_and_kick()


def gather_state_local(loops: list[RankLoop]) -> None:
    for name in ("vel", "force"):
        slots = torch.stack([pack(getattr(lp.S, name), lp.range, lp.rows) for lp in loops])
        for lp in loops:
            unpack(slots, lp.n, lp.world, getattr(lp.S, name))
