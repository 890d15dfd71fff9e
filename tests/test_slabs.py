"""Slab decomposition with halos (paper_1912_04232_b200/slabs.py).

CPU: the geometry -- frames, exact local <-> global coordinates, ownership, halo selection -- against
fp64 arithmetic written out here.  GPU: 2, 4 and 8 slabs of config 2 stepped in lockstep on one device
against the ORACLE (forces / energy of the gathered state at the north_star tolerances) and against
md_nve_step on one context (same trajectory to rounding)."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_1912_04232_b200 import slabs as SL

L2 = float(np.float32((32000 / 0.8442) ** (1.0 / 3.0)))


@pytest.mark.parametrize("L,world", [(L2, 2), (L2, 4), (L2, 8), (67.183848, 8), (107.494156, 5)])
def test_frames_are_exact_translations(L, world):
    R = float(np.float32(2.5) + np.float32(0.3))
    frs = SL.frames(L, R, world)
    Lf = float(np.float32(L))
    assert frs[0].lo == 0.0 and frs[-1].hi == Lf
    for a, b in zip(frs[:-1], frs[1:]):
        assert a.hi == b.lo
    rng = np.random.default_rng(1)
    x = rng.uniform(0, Lf, 300000).astype(np.float32)
    x = np.concatenate([x, np.float32([0.0, np.nextafter(np.float32(Lf), np.float32(0)), 1e-30, 2.0 ** -20])])
    x = x[x < np.float32(Lf)]
    xt = torch.from_numpy(x)
    own = SL.owner_of(xt, frs).numpy()
    x64 = x.astype(np.float64)
    for fr in frs:
        # every number of the frame is an fp32 number, the box holds >= 3 cells with a margin
        for v in (fr.lo, fr.hi, fr.T, fr.Lx, fr.H):
            assert float(np.float32(v)) == v
        assert fr.Lx / R >= 3.0 and abs(fr.Lx / R - round(fr.Lx / R)) > 0.2 and fr.G >= R and fr.H >= R
        mine = own == fr.rank
        assert np.array_equal(mine, (x64 >= fr.lo) & (x64 < fr.hi))
        # halo: within H of the slab, periodically (fp64)
        d_lo = np.mod(fr.lo - x64, Lf); d_hi = np.mod(x64 - fr.hi, Lf)
        want = ((d_lo > 0) & (d_lo <= fr.H) | (d_hi >= 0) & (d_hi < fr.H)) & ~mine
        got = SL.halo_select(xt, fr).numpy() & ~mine
        assert np.array_equal(got, want)
        m = mine | got
        xl = SL.global_to_local(xt[m], fr)
        # the local coordinate is the global one moved by an exact amount: T, or the periodic images
        xl64 = xl.numpy().astype(np.float64)
        shift = x64[m] - xl64
        ok = np.isclose(shift, fr.T, rtol=0, atol=0) | np.isclose(shift, Lf - fr.Lx if fr.first else -1e300, rtol=0, atol=0) \
            | (np.isclose(shift, 0.0, rtol=0, atol=0) if fr.last else False)
        assert ok.all()
        assert (xl64 >= 0).all() and (xl64 < fr.Lx).all()
        assert torch.equal(SL.local_to_global(xl, fr), xt[m])
        # owned particles and halo copies keep their distances: |x_i - x_j| identical in both frames (min image)
        k = min(2000, int(m.sum()))
        a, b = xl64[:k], xl64[-k:]
        dl = a - b; dl -= fr.Lx * np.round(dl / fr.Lx)
        ga, gb = x64[m][:k], x64[m][-k:]
        dg = ga - gb; dg -= Lf * np.round(dg / Lf)
        near = np.abs(dg) < fr.H
        assert np.array_equal(dl[near], dg[near])


def test_too_small_boxes_are_refused():
    with pytest.raises(ValueError):
        SL.frames(10.077577, 2.8, 2)           # config 0: 3 cells per side
    with pytest.raises(ValueError):
        SL.frames(L2, 2.8, 1)
    with pytest.raises(ValueError):
        SL.frames(L2, 2.8, 16)


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1912_04232_b200 import build
    build.build()
    from paper_1912_04232_b200 import binding
    binding.lib()
    return binding


def _oracle_force(orc, w, pos):
    idx, cnt, _ = orc.neighbor_list(pos, w.box, 3, w.r_cut, w.skin, w.capacity, predicate=1, method=1)
    return orc.energy_force(pos, None, w.box, 3, w.kind, w.epsilon, w.sigma, float(np.float32(w.r_cut)), w.shift, idx, cnt)


@pytest.mark.gpu
@pytest.mark.parametrize("world", [2, 5])
def test_library_translations_equal_the_written_out_ones(B, world):
    """md_slab_convert / md_slab_pack / md_slab_unpack (the kernels the runs use) against the torch
    expressions of this module, which the CPU test above pins to fp64: bit for bit."""
    frs = SL.frames(L2, 2.8, world)
    rng = np.random.default_rng(3)
    x = rng.uniform(0, float(np.float32(L2)), 100000).astype(np.float32)
    x = x[x < np.float32(L2)]
    xt = torch.from_numpy(x).cuda()
    own = SL.owner_of(xt, frs)
    for fr in frs:
        m = (own == fr.rank) | SL.halo_select(xt, fr)
        pos = torch.zeros(int(m.sum()), 4, device="cuda"); pos[:, 0] = xt[m]; pos[:, 1] = 7.0
        want = SL.global_to_local(xt[m], fr)
        B.md_slab_convert(fr.abi(B), pos, pos.shape[0], 1)
        assert torch.equal(pos[:, 0], want) and bool((pos[:, 1] == 7.0).all())
        slots = torch.randperm(pos.shape[0], device="cuda")[:1000].int()
        rows = torch.empty(1000, 4, device="cuda")
        B.md_slab_pack(fr.abi(B), pos, slots, rows)
        assert torch.equal(rows[:, 0], xt[m][slots.long()])
        pos2 = torch.zeros_like(pos)
        B.md_slab_unpack(fr.abi(B), rows, slots, pos2)
        assert torch.equal(pos2[slots.long(), 0], want[slots.long()])
        B.md_slab_convert(fr.abi(B), pos, pos.shape[0], 0)
        assert torch.equal(pos[:, 0], xt[m])


@pytest.mark.gpu
@pytest.mark.parametrize("world", [2, 4, 8])
def test_slabs_against_the_oracle_and_one_gpu(B, orc, W, world):
    w = W.config(2)
    steps = 100
    run = SL.SlabRun(B, w, world)
    n_local = [S.n for S in run.ranks]
    owned0 = [int((S.id[: S.n] >= 0).sum()) for S in run.ranks]
    assert sum(owned0) == w.n and all(a > b for a, b in zip(n_local, owned0))
    # only neighbours talk to each other
    for s, d, rows in run.exchange_plan():
        assert (s - d) % world in (1, world - 1) and rows > 0

    def state():
        pos, vel, gid, force = run.gather(with_force=True)
        g = gid.cpu().numpy().astype(np.int64)
        assert np.array_equal(np.sort(g), np.arange(w.n))
        out = []
        for t in (pos, vel, force):
            a = np.empty((w.n, 4), np.float32); a[g] = t.cpu().numpy(); out.append(a)
        return out

    def check(p, f, E):
        assert (p[:, 0] >= 0).all() and (p[:, 0] < w.box[0]).all()
        f_o, e_o, E_o = _oracle_force(orc, w, p)
        err = (np.linalg.norm(f[:, :3] - f_o, axis=1) / np.maximum(np.linalg.norm(f_o, axis=1), 1e-3)).max()
        assert err <= 1e-5, err
        assert abs(E - E_o) <= 1e-6 * abs(E_o), (E, E_o)

    p0, v0, f0 = state()
    assert np.array_equal(p0, w.pos) and np.array_equal(v0, w.vel)          # exact frames: nothing moved
    check(p0, f0, run.energy())
    mom0 = v0[:, :3].astype(np.float64).sum(0)
    run.step(steps)
    torch.cuda.synchronize()
    p1, v1, f1 = state()
    check(p1, f1, run.energy())
    assert np.abs(v1[:, :3].astype(np.float64).sum(0) - mom0).max() <= 2e-5 * np.sqrt(w.n) + 1e-3
    # the same trajectory as one GPU, up to the order forces are summed in
    one = B.System(w)
    one.build(); one.compute_force(); one.step(steps)
    torch.cuda.synchronize()
    ids = one.id.cpu().numpy().astype(np.int64)
    q = np.empty((w.n, 4), np.float32); q[ids] = one.pos.cpu().numpy()
    d = p1[:, :3].astype(np.float64) - q[:, :3]
    Lb = w.box.astype(np.float64)
    d -= Lb * np.round(d / Lb)
    assert np.abs(d).max() <= 2e-4, np.abs(d).max()
    r1 = int(one.stats[1])
    assert abs(run.rebuilds - r1) <= max(2, r1 // 3), (run.rebuilds, r1)
    one.close(); run.close()


@pytest.mark.gpu
def test_rebuild_phases_against_the_reference_selection(B, W):
    """md_slab_split / border / load / plan (the rebuild on the device) against the torch reference functions
    of slabs.py that the CPU tests above pin: who stays, who migrates where, who is border, and that the
    exchange plan pairs every border particle with its copy on the neighbour."""
    w = W.config(2)
    world = 4
    run = SL.SlabRun(B, w, world)
    run.step(37)
    torch.cuda.synchronize()
    f32 = np.float32
    ranks = run.slab_ranks
    migrants = 0
    for r in ranks:
        S, fr = r.S, r.fr
        n = S.n
        ids = S.id[:n]
        owned = ids >= 0
        gid = ids[owned]
        xg = SL.local_to_global(S.pos[:n, 0][owned], fr)
        own = SL.owner_of(xg, r.frames)
        (pr, pi), (nr, ni) = r.leavers()
        for rows, mids, rank in ((pr, pi, r.prev), (nr, ni, r.next)):
            want = gid[own == rank]
            assert sorted(mids.tolist()) == sorted(want.tolist())
            migrants += int(mids.numel())
            if mids.numel():
                # a row is (position with global x | velocity) of that particle
                slot = torch.full((w.n,), -1, dtype=torch.long, device=ids.device)
                slot[gid.long()] = torch.arange(n, device=ids.device)[owned]
                s = slot[mids.long()]
                assert torch.equal(rows[:, 1:4], S.pos[s, 1:4]) and torch.equal(rows[:, 4:], S.vel[s])
                assert torch.equal(rows[:, 0], SL.local_to_global(S.pos[s, 0], fr))
        stay = r.own_id[: r.n_own]
        assert sorted(stay.tolist()) == sorted(gid[own == fr.rank].tolist())
        (bp, bpi), (bn, bni) = r.border_rows()
        x_own, id_own = r.own_pos[: r.n_own, 0], r.own_id[: r.n_own]
        assert sorted(bpi.tolist()) == sorted(id_own[x_own < f32(fr.lo + fr.H)].tolist())
        assert sorted(bni.tolist()) == sorted(id_own[x_own >= f32(fr.hi - fr.H)].tolist())
        assert int((r.map_prev >= 0).sum()) == bpi.numel() and int((r.map_next >= 0).sum()) == bni.numel()
    assert migrants > 0
    # the whole protocol, then the plan
    SL.rebuild_all(ranks, run.comm)
    torch.cuda.synchronize()
    for r in ranks:
        S = r.S
        for m in (r.map_prev, r.map_next, r.map_halo):
            assert int((m >= 0).sum()) == 0
        ids = S.id[: S.n]
        assert int(S.nbr_count[: S.n][ids < 0].abs().sum()) == 0 and int(S.nbr_count[: S.n][ids >= 0].min()) > 0
        prev, nxt = ranks[r.prev], ranks[r.next]
        # what my previous rank sends to ITS next lands on my `from prev` copies, row by row
        sent_by_prev = S.id.new_tensor(prev.S.id[prev.border[1].long()].tolist())
        sent_by_next = S.id.new_tensor(nxt.S.id[nxt.border[0].long()].tolist())
        assert torch.equal(ids[r.halo[0].long()], -1 - sent_by_prev)
        assert torch.equal(ids[r.halo[1].long()], -1 - sent_by_next)
        assert torch.equal(S.id[r.border[0].long()], r.bor_ids[0][: r.n_border[0]])
        assert torch.equal(S.id[r.border[1].long()], r.bor_ids[1][: r.n_border[1]])
    run.close()
