"""One system over several GPUs by SPATIAL decomposition: slabs along x with halos (SURVEY.md §8e / §8f-f1,
second version).

Rank r owns the particles whose x lies in its slab [lo_r, hi_r) and, beside them, copies of the particles
of other ranks (or periodic images of its own, never needed for world >= 2) within the list radius
R = r_cut + skin of the slab: its HALO.  Owned + halo particles form an ordinary periodic system of the
library on a LOCAL box (x side: slab + two halos + an empty gap >= R, so that nothing an owned particle
sees comes through the local box's own periodic wrap; y, z: the full box), and every step of the path --
cell list, neighbor list, force, velocity Verlet -- runs in the library's kernels on that local system:

    every step      md_slab_step_open: kick and drift of the owned particles, x put back on the global fp32
                    grid, half-skin test (a device flag word), the new positions of the BORDER particles
                    (the owned ones that are somebody's halo; index lists fixed since the last rebuild) packed
                    for the two neighbors; the exchange; md_slab_step_close: the received rows over the halo
                    copies, force and second half-kick.  The host enqueues batches of steps and reads one
                    device word per batch: once a flag is up every later call of the batch is a no-op.
    at a rebuild    owned particles that left the slab MIGRATE to the neighbor (position, velocity, id);
                    halos are re-selected; the local system is re-created for the new particle count;
                    md_cell_list_build + md_neighbor_list_build; the list counts of halo copies are set to
                    0, so the force kernels give them zero force and zero energy.  Five device phases
                    (md_slab_split / append / border / load / plan); the host reads two count arrays.

Exactness.  A local x coordinate is the global one minus a non-negative multiple of 2^-8 (or, for the one
image each of rank 0 and the last rank takes through the box boundary, the Sterbenz-exact x - L plus the
local box length, resp. the raw x): every such translation is exact in fp32 (the result is never larger
than the coordinate it comes from, so it lies on that coordinate's grid), pair displacements in a local
frame are bit-identical to the global ones, and after every drift the local x is rounded the way the
global coordinate would be.  A decomposed run therefore differs from md_nve_step only in the order forces
are summed (list order), not in any pair term.

This module is plumbing: geometry, index lists, the order of the C-ABI calls, and the exchange.  `SlabRun`
steps all ranks inside ONE process on one GPU (the exchange is a gather / scatter between the ranks'
tensors) -- what the tests run; across processes the same index lists feed send / recv of the packed rows
to the previous and next rank (`exchange_plan` returns exactly what travels).
No multi-GPU timing exists: this run has one GPU.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np
import torch

Q = 2.0 ** -8          # slab boundaries and translations are multiples of this (exact fp32 shifts)


@dataclasses.dataclass
class Frame:
    """The local frame of one rank (all numbers exactly representable in fp32)."""
    rank: int
    world: int
    lo: float              # slab [lo, hi) in global x
    hi: float
    T: float               # local x = global x - T for everything that is not a periodic image
    Lx: float              # local box length in x
    H: float               # halo width
    G: float               # gap
    L: float               # global box length in x

    @property
    def first(self) -> bool:
        return self.rank == 0

    @property
    def last(self) -> bool:
        return self.rank == self.world - 1

    @property
    def g2l_thr(self) -> float:
        """Global x that separates plain copies from periodic images (global_to_local)."""
        return 0.5 * (self.hi + self.L) if self.first else (0.5 * self.lo if self.last else 0.0)

    @property
    def l2g_thr(self) -> float:
        """Local x that separates the zone of the images from the rest (local_to_global)."""
        return self.hi + self.H + 0.5 * self.G if self.first else (self.H + 0.5 * self.G if self.last else 0.0)

    def abi(self, B):
        """The frame as the library's md_slab_frame (md.h)."""
        return B.md_slab_frame(0 if self.first else (2 if self.last else 1), self.T, self.Lx, self.L,
                               self.g2l_thr, self.l2g_thr)


def frames(box_x: float, R: float, world: int) -> list[Frame]:
    """Slab frames for `world` >= 2 ranks.  Layouts in local x (H = halo width = R rounded up to Q, G = gap):
    rank 0:        [slab | high halo | gap | low halo = images of x in [L - H, L) at (x - L) + Lx]     T = 0
    middle ranks:  [low halo | slab | high halo | gap]                                                  T = lo - H
    last rank:     [high halo = images of x in [0, H) at their raw x | gap | low halo | slab]           T = lo - 2H - G,
                                                                                                        Lx = L - T
    In the first and the last frame the local box's own periodic wrap IS the global one: a particle of rank 0
    that drifts below 0 reappears at the top of the local box, where the images of x near L live."""
    if world < 2:
        raise ValueError("a slab decomposition needs at least 2 ranks (one rank is md_nve_step itself)")
    L = float(np.float32(box_x))
    H = math.ceil(R / Q) * Q
    W = L / world
    los = [round(r * W / Q) * Q for r in range(world)] + [L]

    def gap_for(base):
        # at least R, and such that Lx / R sits mid-way between integers (the library refuses a box whose
        # cell side is within 1e-5 of R)
        k = math.floor((base + R) / R)
        g = (k + 0.5) * R - base
        while g < R:
            g += R
        return math.ceil(g / Q) * Q

    out = []
    for r in range(world):
        lo, hi = los[r], los[r + 1]
        width = hi - lo
        G = gap_for(width + 2 * H)
        if width < H:                    # a halo must come from the two adjacent slabs only
            raise ValueError(f"box side {L} too small for {world} slabs of list radius {R}")
        if r == 0:
            fr = Frame(r, world, lo, hi, 0.0, width + 2 * H + G, H, G, L)
        elif r == world - 1:
            T = lo - 2 * H - G
            if T < 0 or float(np.float32(L - T)) != L - T:
                raise ValueError(f"box side {L} too small for {world} slabs of list radius {R}")
            fr = Frame(r, world, lo, hi, T, L - T, H, G, L)
        else:
            fr = Frame(r, world, lo, hi, lo - H, width + 2 * H + G, H, G, L)
        out.append(fr)
    # images and plain copies must be told apart by x alone (global_to_local): rank 0's slab ends well
    # below L - H, the last rank's begins well above H
    if L - out[0].hi < 2 * (H + 1.0) or out[-1].lo < 2 * (H + 1.0):
        raise ValueError(f"box side {L} too small for {world} slabs of list radius {R}")
    return out


def owner_of(xg: torch.Tensor, frs: list[Frame]) -> torch.Tensor:
    """Rank whose slab holds global x (fp32 tensor)."""
    bounds = torch.tensor([f.lo for f in frs[1:]], dtype=torch.float32, device=xg.device)
    return torch.bucketize(xg.contiguous(), bounds, right=True)


def global_to_local(xg: torch.Tensor, fr: Frame) -> torch.Tensor:
    """Local x in frame fr of a particle at global x in [0, L) that lives in fr's slab or halo (fp32,
    every operation exact: see the module text)."""
    f32 = np.float32
    if fr.first:
        # x near L is the image through x = 0: (x - L) is Sterbenz-exact, + Lx lands on x's own grid
        img = xg >= f32(fr.g2l_thr)
        return torch.where(img, (xg - f32(fr.L)) + f32(fr.Lx), xg)
    if fr.last:
        # x near 0 is the image through x = L: x + L - T = x (mod Lx = L - T): the raw coordinate
        img = xg < f32(fr.g2l_thr)
        return torch.where(img, xg, xg - f32(fr.T))
    return xg - f32(fr.T)


def local_to_global(xl: torch.Tensor, fr: Frame) -> torch.Tensor:
    """Global x in [0, L) of local x (the inverse of global_to_local; for a coordinate a drift has just
    produced this is also where the global fp32 rounding happens)."""
    f32 = np.float32
    if fr.first:
        img = xl >= f32(fr.l2g_thr)                            # the zone of the images at the top of the box
        xg = torch.where(img, (xl - f32(fr.Lx)) + f32(fr.L), xl)
    elif fr.last:
        img = xl < f32(fr.l2g_thr)                             # the zone of the raw images at the bottom
        xg = torch.where(img, xl, xl + f32(fr.T))
    else:
        xg = xl + f32(fr.T)
    return torch.where(xg >= f32(fr.L), torch.zeros_like(xg), xg)    # x - tiny + L rounding to L


def halo_select(xg: torch.Tensor, fr: Frame) -> torch.Tensor:
    """Which particles (global x in [0, L)) are in fr's halo: within H below lo or above hi, periodically."""
    f32 = np.float32
    lo, hi, H, L = f32(fr.lo), f32(fr.hi), f32(fr.H), f32(fr.L)
    high = (xg < H) if fr.last else ((xg >= hi) & (xg < hi + H))
    low = (xg >= L - H) if fr.first else ((xg >= lo - H) & (xg < lo))
    return high | low


class LocalSystem:
    """Device buffers of one rank with room for `cap` particles; the md_system is re-created at every
    rebuild for the current count (allocation only; no arithmetic)."""

    def __init__(self, B, w, fr: Frame, cap: int, device):
        self.B, self.w, self.fr, self.cap, self.device = B, w, fr, cap, torch.device(device)
        box = [fr.Lx, float(w.box[1]), float(w.box[2])]
        self.cfg = B.make_config(w.dim, box, w.r_cut, w.skin, w.capacity, 1)
        self.pot = B.make_potential(w.kind, w.epsilon, w.sigma, w.r_cut, w.shift, getattr(w, "alpha", 0.0))
        dev = self.device
        self.workspace = torch.empty(B.md_workspace_bytes(self.cfg, cap), dtype=torch.uint8, device=dev)
        self.pos = torch.zeros(cap, 4, dtype=torch.float32, device=dev)
        self.vel = torch.zeros(cap, 4, dtype=torch.float32, device=dev)
        self.force = torch.zeros(cap, 4, dtype=torch.float32, device=dev)
        self.id = torch.zeros(cap, dtype=torch.int32, device=dev)          # global id; -1 - id for a halo copy
        self.sys = None
        self.n = 0
        self.perm = torch.zeros(cap, dtype=torch.int32, device=dev)
        self.nbr_count = torch.zeros(cap, dtype=torch.int32, device=dev)
        self.status = torch.zeros(2, dtype=torch.int32, device=dev)
        self.flag = torch.zeros(1, dtype=torch.int32, device=dev)
        self.energy = torch.zeros(1, dtype=torch.float64, device=dev)
        self.nbr_idx = torch.empty(((cap + 31) // 32) * 32 * self.cfg.capacity, dtype=torch.int32, device=dev)
        self.cell_start = None

    def resize(self, n: int):
        """A system of n particles over the same buffers (pos / vel / id are filled by the caller)."""
        B = self.B
        if n > self.cap:
            raise RuntimeError(f"rank {self.fr.rank}: {n} local particles exceed the reserved {self.cap}")
        if self.sys is not None:
            B.md_destroy(self.sys)          # its kernels have finished: the caller has just read this rebuild's counts
        self.n = n
        self.sys = B.md_create(self.cfg, n, self.workspace)
        ncell = B.md_num_cells(self.sys)
        cells = ncell[0] * ncell[1] * ncell[2]
        if self.cell_start is None or self.cell_start.numel() != cells + 1:
            self.cell_start = torch.zeros(cells + 1, dtype=torch.int32, device=self.device)

    def build(self):
        B = self.B
        B.md_cell_list_build(self.sys, self.pos, self.vel, self.id, self.cell_start, self.perm)
        B.md_neighbor_list_build(self.sys, self.pos, self.cell_start, self.perm, self.nbr_idx, self.nbr_count, self.status)

    def close(self):
        if self.sys is not None:
            torch.cuda.synchronize(self.device)
            self.B.md_destroy(self.sys)
            self.sys = None


class SlabRank:
    """One rank of the decomposition: its frame, its local system, and the phases of a step and of a rebuild.
    Every phase is a call into the library (md_slab_*): the host sizes messages from small count arrays and
    moves no particle data.  What leaves a phase for another rank is a pair (float32 rows, int32 ids); what
    arrives comes from the PREVIOUS and the NEXT rank only (periodically: rank 0's previous rank is the last)."""

    def __init__(self, B, w, fr: Frame, device, reserve: float = 1.35):
        self.B, self.w, self.fr = B, w, fr
        share = (fr.hi - fr.lo + 2 * fr.H) / fr.L
        cap = int(reserve * w.n * share) + 2048
        self.S = LocalSystem(B, w, fr, cap, device)
        self.frames = frames(fr.L, float(np.float32(w.r_cut) + np.float32(w.skin)), fr.world)
        self.prev, self.next = (fr.rank - 1) % fr.world, (fr.rank + 1) % fr.world
        self.frame = fr.abi(B)      # the coordinate arithmetic of every phase runs in the library (md_slab_*)
        self.rebuilds = 0
        dev = self.S.device
        f32 = dict(dtype=torch.float32, device=dev)
        i32 = dict(dtype=torch.int32, device=dev)
        # owned particles between the phases of a rebuild (x global)
        self.own_pos, self.own_vel = torch.zeros(cap, 4, **f32), torch.zeros(cap, 4, **f32)
        self.own_id = torch.zeros(cap, **i32)
        self.n_own = 0
        # messages: migrants (position | velocity) and border rows (position), for (prev, next)
        self.cap_rows = int(reserve * w.n * fr.H / fr.L) + 2048
        self.mig_rows = tuple(torch.zeros(self.cap_rows, 8, **f32) for _ in range(2))
        self.mig_ids = tuple(torch.zeros(self.cap_rows, **i32) for _ in range(2))
        self.bor_rows = tuple(torch.zeros(self.cap_rows, 4, **f32) for _ in range(2))
        self.bor_ids = tuple(torch.zeros(self.cap_rows, **i32) for _ in range(2))
        self.step_rows_buf = tuple(torch.zeros(self.cap_rows, 4, **f32) for _ in range(2))
        self.counts = torch.zeros(8, **i32)      # [0:4] split, [4:7] border, [7] errors of append
        # global id -> position in a message, -1 between rebuilds
        self.map_prev, self.map_next, self.map_halo = (torch.full((w.n,), -1, **i32) for _ in range(3))
        self.border_slots = tuple(torch.zeros(self.cap_rows, **i32) for _ in range(2))
        self.halo_slots = torch.zeros(2 * self.cap_rows, **i32)
        self.border = (None, None)  # local slots of my border particles for (prev, next)
        self.halo = (None, None)    # local slots of the copies that came from (prev, next), in arrival order
        # {flag: a list is stale, stop: every step call is a no-op, done: steps completed}; the ranks of one
        # process share the words (attach), ranks in different processes all-reduce the flag every step
        self.words = torch.zeros(4, **i32)

    def attach(self, words: torch.Tensor):
        self.words = words

    def _read_counts(self):
        c = self.counts.tolist()                                # the host read of this phase
        if c[3] or c[6]:
            raise RuntimeError(f"rank {self.fr.rank}: message buffers of {self.cap_rows} rows are too small")
        if c[7]:
            raise RuntimeError("a particle moved past a neighbouring slab between two rebuilds")
        return c

    # ---- start and rebuild ------------------------------------------------------------------
    def take_initial(self, pos_g, vel, gid):
        """From the (replicated) initial state: my owned particles."""
        mine = owner_of(pos_g[:, 0].contiguous(), self.frames) == self.fr.rank
        k = int(mine.sum())
        self.own_pos[:k] = pos_g[mine]; self.own_vel[:k] = vel[mine]; self.own_id[:k] = gid[mine]
        self.n_own = k

    def leavers(self):
        """Owned particles whose x has left the slab since the last rebuild: ((rows, ids) for prev, for next);
        the stayers are kept for adopt()."""
        S, fr, B = self.S, self.fr, self.B
        B.md_slab_split(self.frame, np.float32(fr.lo), np.float32(fr.hi), S.pos, S.vel, S.id, S.n,
                        self.own_pos, self.own_vel, self.own_id, self.mig_rows[0], self.mig_ids[0],
                        self.mig_rows[1], self.mig_ids[1], self.cap_rows, self.counts)
        c = self._read_counts()
        self.n_own = c[0]
        return (self.mig_rows[0][: c[1]], self.mig_ids[0][: c[1]]), (self.mig_rows[1][: c[2]], self.mig_ids[1][: c[2]])

    def adopt(self, from_prev, from_next):
        """Migrants from the neighbours join my owned particles."""
        fr = self.fr
        for rows, ids in (from_prev, from_next):
            m = 0 if rows is None else int(rows.shape[0])
            if m:
                if self.n_own + m > self.S.cap:
                    raise RuntimeError(f"rank {fr.rank}: more than the reserved {self.S.cap} particles")
                self.B.md_slab_append(rows, ids, m, np.float32(fr.lo), np.float32(fr.hi), self.own_pos, self.own_vel,
                                      self.own_id, self.n_own, self.counts[7:])
                self.n_own += m

    def border_rows(self):
        """My owned particles within H of my slab's faces: ((positions, ids) for prev, for next).  They
        become the neighbours' halo copies; their ids, in this order, define what travels every step."""
        fr, f32 = self.fr, np.float32
        self.B.md_slab_border(f32(fr.lo + fr.H), f32(fr.hi - fr.H), self.own_pos, self.own_id, self.n_own,
                              self.bor_rows[0], self.bor_ids[0], self.bor_rows[1], self.bor_ids[1], self.cap_rows,
                              self.map_prev, self.map_next, self.counts[4:])
        c = self._read_counts()
        self.n_border = (c[4], c[5])
        return (self.bor_rows[0][: c[4]], self.bor_ids[0][: c[4]]), (self.bor_rows[1][: c[5]], self.bor_ids[1][: c[5]])

    def rebuild(self, halo_prev, halo_next):
        """Local system = owned + the copies the neighbours sent; lists; index lists of the step exchange."""
        S, B = self.S, self.B
        hp, hn = int(halo_prev[0].shape[0]), int(halo_next[0].shape[0])
        if hp + hn > self.halo_slots.numel():
            raise RuntimeError(f"rank {self.fr.rank}: more halo copies than the reserved {self.halo_slots.numel()}")
        n = self.n_own + hp + hn
        S.resize(n)
        B.md_slab_load(self.frame, self.own_pos, self.own_vel, self.own_id, self.n_own, halo_prev[0].contiguous(),
                       halo_prev[1].contiguous(), hp, halo_next[0].contiguous(), halo_next[1].contiguous(), hn,
                       S.pos, S.vel, S.id, self.map_halo)
        S.build()
        B.md_slab_plan(S.id, n, S.nbr_count, self.map_prev, self.map_next, self.map_halo, self.border_slots[0],
                       self.border_slots[1], self.halo_slots)
        self.border = tuple(self.border_slots[k][: self.n_border[k]] for k in range(2))
        self.halo = (self.halo_slots[:hp], self.halo_slots[hp: hp + hn])
        self.rows_out = tuple(self.step_rows_buf[k][: self.n_border[k]] for k in range(2))
        self.rebuilds += 1

    # ---- the phases of an ordinary step ------------------------------------------------------
    def open_step(self):
        """v += dt/2m F, r = mu(r, dt v) on my owned particles, x back on the global fp32 grid; raises the flag
        word when one of them is more than skin / 2 from where the lists were built; a no-op once the stop word
        is up.  Returns the new positions (global x) of my border particles, for (prev, next)."""
        B, S, w = self.B, self.S, self.w
        B.md_slab_step_open(S.sys, self.frame, S.pos, S.vel, S.force, S.id, w.dt, w.mass, self.words[0:1],
                            self.words[1:2], self.border[0], self.rows_out[0], self.border[1], self.rows_out[1])
        return self.rows_out

    def close_step(self, from_prev, from_next, count: bool = False):
        """The neighbours' rows into my halo copies (the image follows from x), then F = F(r), v += dt/2m F:
        a no-op that raises the stop word while the flag word is up.  count: this rank's call is the one that
        counts the step in the done word."""
        B, S, w = self.B, self.S, self.w
        B.md_slab_step_close(S.sys, self.frame, S.pot, from_prev, self.halo[0], from_next, self.halo[1], S.pos,
                             S.nbr_idx, S.nbr_count, S.force, S.vel, w.dt, w.mass, self.words[0:1], self.words[1:2],
                             self.words[2:3] if count else None)

    def force_kick(self):
        """F = F(r), v += dt/2m F on the lists just rebuilt (the second half of an interrupted step)."""
        S, w = self.S, self.w
        self.B.md_force_half_kick(S.sys, S.pot, S.pos, S.nbr_idx, S.nbr_count, S.force, S.vel, w.dt, w.mass)

    def first_force(self):
        S = self.S
        self.B.md_pair_energy_force(S.sys, S.pot, S.pos, S.nbr_idx, S.nbr_count, S.force, None)


def rebuild_all(ranks, comm, initial=None):
    """The rebuild protocol: migration to the neighbours, then the halo rows from the neighbours.
    comm.shift(to_prev, to_next) delivers, for every rank, (what its previous rank sent to ITS next,
    what its next rank sent to ITS previous)."""
    if initial is None:
        out = [r.leavers() for r in ranks]
        got = comm.shift([o[0] for o in out], [o[1] for o in out])
        for r, (fp, fn) in zip(ranks, got):
            r.adopt(fp, fn)
    else:
        for r in ranks:
            r.take_initial(*initial)
    out = [r.border_rows() for r in ranks]
    got = comm.shift([o[0] for o in out], [o[1] for o in out])
    for r, (fp, fn) in zip(ranks, got):
        r.rebuild(fp, fn)


def step_all(ranks, comm, nsteps: int, state=None):
    """nsteps velocity-Verlet steps of the ranks this process drives (one per process across GPUs).  The host
    runs ahead of the device: it enqueues a batch of steps (drift, flag, exchange, force) and reads the done
    word once per batch.  From the step whose drift finds a stale list on any rank every later call of the
    batch is a no-op on the device; the host then rebuilds, finishes that step and goes on.  state: dict that
    carries the batch length from call to call (the last rebuild interval)."""
    state = {} if state is None else state
    words = ranks[0].words
    left = nsteps
    interval = state.get("interval", 8)                  # steps between the last two rebuilds
    since = state.get("since", 0)                        # steps since the last rebuild
    while left > 0:
        # up to where the next rebuild is expected in one batch, short batches beyond it
        k = min(left, max(1, interval - since) if since < interval else max(1, interval // 4))
        words.zero_()
        for _ in range(k):
            out = [r.open_step() for r in ranks]
            comm.share_flag(words)
            got = comm.shift_rows([o[0] for o in out], [o[1] for o in out], [tuple(h.numel() for h in r.halo) for r in ranks])
            for i, (r, (fp, fn)) in enumerate(zip(ranks, got)):
                r.close_step(fp, fn, count=(i == 0))
        done = int(words[2])                               # the one host read of the batch
        left -= done
        since += done
        if done < k:                                       # step done + 1 has drifted and waits for its lists
            rebuild_all(ranks, comm)
            words.zero_()
            for r in ranks:
                r.force_kick()
            left -= 1
            interval, since = max(1, since), 0
    state["interval"], state["since"] = interval, since


class LocalComm:
    """All ranks live in this process (tests on one GPU): a shift is a re-indexing of the lists."""

    def __init__(self, world: int):
        self.world = world

    def shift(self, to_prev: list, to_next: list):
        P = self.world
        return [(to_next[(r - 1) % P], to_prev[(r + 1) % P]) for r in range(P)]

    def shift_rows(self, to_prev: list, to_next: list, sizes):
        return self.shift(to_prev, to_next)

    def share_flag(self, words):
        pass                                             # the ranks of one process share the words


class DistComm:
    """One rank per process over torch.distributed (NCCL across GPUs, gloo in the CPU test).  A message is a
    tensor or a (rows, ids) pair of variable length: its row count travels first."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.world, self.rank = dist.get_world_size(group), dist.get_rank(group)
        self.prev, self.next = (self.rank - 1) % self.world, (self.rank + 1) % self.world

    def _pairs(self, s_prev, s_next, r_prev, r_next):
        """Point-to-point ops in an order both ends agree on without tags (NCCL has none): between two
        ranks messages match in the order they are issued.  With world = 2 the other rank is both
        neighbours: its first send (to its previous = me) is what I receive as `from next`."""
        dist = self.dist
        sends = [(s_prev, self.prev), (s_next, self.next)]
        recvs = [(r_next, self.next), (r_prev, self.prev)] if self.world == 2 else [(r_prev, self.prev), (r_next, self.next)]
        ops = [dist.P2POp(dist.isend, t, p, self.group) for t, p in sends if t is not None]
        ops += [dist.P2POp(dist.irecv, t, p, self.group) for t, p in recvs if t is not None]
        if ops:
            for q in dist.batch_isend_irecv(ops):
                q.wait()

    def _sendrecv(self, t_prev: torch.Tensor, t_next: torch.Tensor, width, dtype):
        dev = t_prev.device
        n_out = torch.tensor([t_prev.shape[0], t_next.shape[0]], dtype=torch.int64, device=dev)
        n_in = torch.zeros(2, dtype=torch.int64, device=dev)
        self._pairs(n_out[0:1], n_out[1:2], n_in[0:1], n_in[1:2])
        k_prev, k_next = int(n_in[0]), int(n_in[1])
        r_prev = torch.empty((k_prev,) + tuple(width), dtype=dtype, device=dev)
        r_next = torch.empty((k_next,) + tuple(width), dtype=dtype, device=dev)
        # empty messages do not travel: both ends know the counts
        self._pairs(t_prev.contiguous() if t_prev.shape[0] else None, t_next.contiguous() if t_next.shape[0] else None,
                    r_prev if k_prev else None, r_next if k_next else None)
        return r_prev, r_next

    def shift(self, to_prev: list, to_next: list):
        """Lists of length 1 (this process drives one rank)."""
        a, b = to_prev[0], to_next[0]
        if isinstance(a, tuple):
            rp, rn = self._sendrecv(a[0], b[0], a[0].shape[1:], a[0].dtype)
            ip, inn = self._sendrecv(a[1], b[1], (), a[1].dtype)
            return [((rp, ip), (rn, inn))]
        rp, rn = self._sendrecv(a, b, a.shape[1:], a.dtype)
        return [(rp, rn)]

    def shift_rows(self, to_prev: list, to_next: list, sizes):
        """The step exchange: both ends know the row counts from the rebuild, nothing passes through the host."""
        a, b = to_prev[0], to_next[0]
        k_prev, k_next = sizes[0]
        key = (k_prev, k_next, a.device, a.dtype)
        if getattr(self, "_rows_key", None) != key:
            self._rows_key = key
            self._rows = (torch.empty((k_prev,) + tuple(a.shape[1:]), dtype=a.dtype, device=a.device),
                          torch.empty((k_next,) + tuple(a.shape[1:]), dtype=a.dtype, device=a.device))
        r_prev, r_next = self._rows
        self._pairs(a if a.shape[0] else None, b if b.shape[0] else None, r_prev if k_prev else None, r_next if k_next else None)
        return [(r_prev, r_next)]

    def share_flag(self, words):
        self.dist.all_reduce(words[0:1], op=self.dist.ReduceOp.MAX, group=self.group)


class SlabRun:
    """`world` ranks of one process on one device, stepped in lockstep through LocalComm (tests, and
    `bench.py --slabs`): the same SlabRank phases and the same neighbour-only messages a run with one
    process per GPU makes through DistComm."""

    def __init__(self, B, w, world: int, device="cuda:0", reserve: float = 1.35):
        if w.dim != 3:
            raise ValueError("slabs are implemented for 3-D systems")
        self.B, self.w, self.world = B, w, world
        R = float(np.float32(w.r_cut) + np.float32(w.skin))
        self.frames = frames(float(np.float32(w.box[0])), R, world)
        dev = torch.device(device)
        self.device = dev
        self.comm = LocalComm(world)
        self.slab_ranks = [SlabRank(B, w, fr, dev, reserve) for fr in self.frames]
        self.ranks = [r.S for r in self.slab_ranks]
        for r in self.slab_ranks[1:]:
            r.attach(self.slab_ranks[0].words)
        self._step_state = {}
        pos = torch.from_numpy(w.pos).to(dev)
        vel = torch.from_numpy(w.vel).to(dev)
        gid = torch.arange(w.n, dtype=torch.int32, device=dev)
        rebuild_all(self.slab_ranks, self.comm, initial=(pos, vel, gid))
        for r in self.slab_ranks:
            r.first_force()

    @property
    def rebuilds(self) -> int:
        return self.slab_ranks[0].rebuilds - 1          # the initial build is not a rebuild

    def exchange_plan(self):
        """[(source rank, destination rank, rows)]: what travels every step (16 bytes per row)."""
        out = []
        for r in self.slab_ranks:
            out.append((r.fr.rank, r.prev, int(r.border[0].numel())))
            out.append((r.fr.rank, r.next, int(r.border[1].numel())))
        return out

    def step(self, nsteps: int):
        step_all(self.slab_ranks, self.comm, nsteps, self._step_state)

    # ---- results ------------------------------------------------------------------------------
    def gather(self, with_force: bool = False):
        """Owned particles of all ranks in global coordinates: (pos, vel, global id[, force])."""
        ps, vs, gs, fs = [], [], [], []
        for S in self.ranks:
            n = S.n
            owned = S.id[:n] >= 0
            p = S.pos[:n][owned].contiguous()
            self.B.md_slab_convert(S.fr.abi(self.B), p, p.shape[0], 0)
            ps.append(p); vs.append(S.vel[:n][owned]); gs.append(S.id[:n][owned])
            if with_force:
                fs.append(S.force[:n][owned])
        out = (torch.cat(ps), torch.cat(vs), torch.cat(gs))
        return out + (torch.cat(fs),) if with_force else out

    def energy(self) -> float:
        E = 0.0
        for S in self.ranks:
            self.B.md_pair_energy_force(S.sys, S.pot, S.pos, S.nbr_idx, S.nbr_count, S.force, S.energy)
            E += float(S.energy[0])
        return E

    def close(self):
        for S in self.ranks:
            S.close()
