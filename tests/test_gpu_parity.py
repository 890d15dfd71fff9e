"""GPU parity tests: the CUDA path (through the C ABI) against the fp64 CPU oracle,
element by element on the same seeded inputs (SURVEY.md §8c "Tolerances").

  neighbor rows   bit-exact after sorting each row (all `capacity` slots + counts)
  cells           identical membership, cell_start, canonical in-cell order
  forces          max_i ||F_gpu - F_or|| / max(||F_or||, 1e-3) <= 1e-5
  total energy    relative 1e-6
  config 0        positions after 100 NVE steps within 1e-4 (minimum image)
"""
import dataclasses

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

FORCE_TOL = 1e-5
ENERGY_TOL = 1e-6


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1912_04232_b200 import build
    build.build()
    from paper_1912_04232_b200 import binding
    binding.lib()
    return binding


def custom_workload(W, pos, box32, dim, kind, r_cut, skin, capacity, resort=1, vel=None, dt=0.005):
    n = pos.shape[0]
    return W.Workload(index=-1, name="custom", dim=dim, n=n, box=box32, kind=kind, epsilon=1.0,
                      sigma=1.0, r_cut=r_cut, skin=skin, capacity=capacity, shift=1 if kind == 0 else 0,
                      dt=dt, mass=1.0, temperature=0.0, steps=0, resort=resort, pos=pos,
                      vel=np.zeros((n, 4), np.float32) if vel is None else vel)


def gpu_rows_in_original_order(S):
    """Neighbor rows of the GPU list mapped back to original particle ids, sorted."""
    n, cap = S.n, S.capacity
    idx = S.nbr_rows().cpu().numpy().astype(np.int64)
    cnt = S.nbr_count.cpu().numpy()
    ids = S.id.cpu().numpy().astype(np.int64)
    lut = np.concatenate([ids, [n]])                 # pad value n maps to itself
    mapped = np.sort(lut[idx], axis=1)
    rows = np.empty_like(mapped)
    rows[ids] = mapped
    counts = np.empty_like(cnt)
    counts[ids] = cnt
    return rows.astype(np.int32), counts


def unpermute(S, t):
    ids = S.id.cpu().numpy().astype(np.int64)
    a = t.cpu().numpy()
    out = np.empty_like(a)
    out[ids] = a
    return out


def force_error(f_gpu, f_or):
    num = np.linalg.norm(f_gpu[:, :3].astype(np.float64) - f_or, axis=1)
    return (num / np.maximum(np.linalg.norm(f_or, axis=1), 1e-3)).max()


def check_cells(S, orc, w):
    """md_cell_list_build vs oracle O2 (run BEFORE anything re-orders S again)."""
    ncell, cell_of, cell_start_o, members_o = orc.cell_list(w.pos, w.box, w.dim, w.r_cut, w.skin)
    cs = S.cell_start.cpu().numpy()
    perm = S.perm.cpu().numpy()
    assert np.array_equal(cs, cell_start_o)
    assert cs[0] == 0 and cs[-1] == w.n and np.all(np.diff(cs) >= 0)
    assert np.array_equal(np.sort(perm), np.arange(w.n))
    # membership per cell is the oracle's (order inside a cell is free); the library's
    # canonical order is ascending x, ties by id (on the first build id == index)
    cell_of_slot = np.repeat(np.arange(len(cs) - 1), np.diff(cs))
    order = np.lexsort((perm, cell_of_slot))
    assert np.array_equal(perm[order], members_o)
    xs = w.pos[perm, 0]
    same = cell_of_slot[1:] == cell_of_slot[:-1]
    assert np.all((xs[1:] > xs[:-1]) | ((xs[1:] == xs[:-1]) & (perm[1:] > perm[:-1])) | ~same)
    if S.cfg.resort:
        assert np.array_equal(S.pos.cpu().numpy(), w.pos[perm])
        assert np.array_equal(S.vel.cpu().numpy(), w.vel[perm])
        assert np.array_equal(S.id.cpu().numpy(), perm)
    else:
        assert np.array_equal(S.pos.cpu().numpy(), w.pos)
        assert np.array_equal(S.id.cpu().numpy(), np.arange(w.n))


def check_list(S, orc, w, method):
    rows, counts = gpu_rows_in_original_order(S)
    idx_o, cnt_o, st_o = orc.neighbor_list(w.pos, w.box, w.dim, w.r_cut, w.skin, S.capacity,
                                           predicate=0, method=method)
    st = S.status.cpu().numpy()
    assert np.array_equal(counts, cnt_o)
    assert st[1] == st_o[1] and st[0] == st_o[0]
    if st_o[0] == 0:
        assert np.array_equal(rows, idx_o)
    return idx_o, cnt_o


def check_force(S, orc, w, idx_o=None, cnt_o=None):
    S.compute_force(want_energy=True)
    f = unpermute(S, S.force)
    E = float(S.energy.cpu()[0])
    diam = w.pos[:, 3].astype(np.float64)
    f_o, e_o, E_o = orc.energy_force(w.pos, diam, w.box, w.dim, w.kind, w.epsilon, w.sigma,
                                     float(np.float32(w.r_cut)), w.shift, idx_o, cnt_o)
    err = force_error(f, f_o)
    assert err <= FORCE_TOL, err
    assert abs(E - E_o) <= ENERGY_TOL * abs(E_o), (E, E_o)
    assert np.abs(f[:, 3] - e_o).max() <= 2e-6 * max(1.0, np.abs(e_o).max())
    if w.dim == 2:
        assert np.all(f[:, 2] == 0.0)
    zero = np.linalg.norm(f_o, axis=1) == 0.0
    if zero.any():
        assert np.linalg.norm(f[zero, :3], axis=1).max() <= 1e-8
    return err


# ----------------------------------------------------------------- configs 0, 1, 2 ------

@pytest.mark.parametrize("ci", [0, 1, 2])
@pytest.mark.parametrize("resort", [1, 0])
def test_config_build_and_force_parity(B, orc, W, ci, resort):
    w = W.config(ci)
    S = B.System(w, resort=resort)
    S.build()
    torch.cuda.synchronize()
    check_cells(S, orc, w)
    idx_o, cnt_o = check_list(S, orc, w, method=0)        # oracle brute force O(N^2)
    check_force(S, orc, w)                                # oracle all-pairs definition
    S.close()


def test_force_from_a_foreign_list(B, orc, W):
    """md_pair_energy_force consumes ANY list in the md_nbr_layout layout: feed it the oracle's
    brute-force rows (original particle order, resort = 0) and compare with the all-pairs
    definition.  Default path (fp32 pair terms + fp64 re-evaluation by error estimate): the
    north_star tolerances; fast32 = 0 (fp64 pair chain everywhere): only the fp32 store rounding
    is left."""
    w = W.config(2)
    S = B.System(w, resort=0)
    S.build()                                               # sets up cells; list replaced below
    idx_o, cnt_o, _ = orc.neighbor_list(w.pos, w.box, 3, w.r_cut, w.skin, w.capacity, 0, 1)
    S.set_nbr_rows(idx_o, cnt_o)
    f_o, _, E_o = orc.energy_force(w.pos, None, w.box, 3, 0, 1.0, 1.0, 2.5, 1)
    S.compute_force()
    assert force_error(S.force.cpu().numpy(), f_o) <= FORCE_TOL
    assert abs(float(S.energy.cpu()[0]) - E_o) <= ENERGY_TOL * abs(E_o)
    B.md_set_option(S.sys, "fast32", 0)
    S.compute_force()
    assert force_error(S.force.cpu().numpy(), f_o) <= 3e-7
    assert abs(float(S.energy.cpu()[0]) - E_o) <= 1e-9 * abs(E_o)
    S.close()


@pytest.mark.parametrize("tpp", [0, 1, 2, 4])
def test_threads_per_particle_variants(B, orc, W, tpp):
    """The fp64 force kernels (fast32 = 0), every lanes-per-particle variant."""
    w = W.config(0)
    S = B.System(w)
    S.build()
    B.md_set_option(S.sys, "fast32", 0)
    B.md_set_option(S.sys, "threads_per_particle", tpp)
    check_force(S, orc, w)
    S.close()


@pytest.mark.parametrize("parts", [1, 2, 4])
@pytest.mark.parametrize("ci,resort", [(0, 1), (1, 1), (2, 1), (2, 0)])
def test_builder_warps_per_tile(B, orc, W, ci, resort, parts):
    """1, 2 or 4 warps share a tile in the bit-mask builder: same rows, same counts, and the lists
    stay right through the rebuilds of a short run (incremental pads)."""
    w = W.config(ci)
    S = B.System(w, resort=resort)
    B.md_set_option(S.sys, "builder_parts", parts)
    S.build()
    torch.cuda.synchronize()
    check_list(S, orc, w, method=0 if ci < 2 else 1)
    S.compute_force()
    S.step(40)
    torch.cuda.synchronize()
    assert int(S.stats[1]) >= 2 and int(S.stats[2]) == -1
    pos = unpermute(S, S.pos)
    w2 = dataclasses.replace(w, pos=pos)
    S.build()                                   # a full build of the final state for comparison
    torch.cuda.synchronize()
    check_list(S, orc, w2, method=1)
    S.close()


@pytest.mark.parametrize("ci", [0, 1])
def test_first_design_builder(B, orc, W, ci):
    """builder = 1 (per-lane shared-memory columns) still builds the same rows."""
    w = W.config(ci)
    S = B.System(w)
    B.md_set_option(S.sys, "builder", 1)
    S.build()
    torch.cuda.synchronize()
    check_list(S, orc, w, method=0)
    S.close()


@pytest.mark.parametrize("dim", [3, 2])
def test_morse_force_energy_and_trajectory(B, orc, W, dim):
    """SURVEY §8f-f2, first potential beyond the two configs: Morse [75] on the
    fp64 pair chain.  Force / energy against the oracle's all-pairs definition, then 100 NVE
    steps against the oracle's fp64 trajectory (brute-force forces), on a jittered lattice."""
    D, r0 = float(np.float32(0.9)), float(np.float32(1.12))
    alpha, rc = float(np.float32(5.0)), 2.5
    if dim == 3:
        base = W.config(0)
        pos, vel, box = base.pos.copy(), base.vel.copy(), base.box
    else:
        rng = np.random.default_rng(9)
        g = np.arange(24.0)
        xy = np.stack(np.meshgrid(g, g, indexing="ij"), -1).reshape(-1, 2) * 1.15 + rng.normal(0, 0.04, (576, 2))
        box = np.array([24 * 1.15, 24 * 1.15, 1.0], np.float32)
        pos = np.zeros((576, 4), np.float32); pos[:, :2] = W.into_box_f32(xy, box); pos[:, 3] = 1.0
        vel = np.zeros((576, 4), np.float32); vel[:, :2] = rng.normal(0, 0.5, (576, 2)); vel[:, :2] -= vel[:, :2].mean(0)
    w = custom_workload(W, pos, box, dim, 2, rc, 0.3, 128, vel=vel, dt=0.005)
    w = dataclasses.replace(w, epsilon=D, sigma=r0, alpha=alpha, shift=1)
    S = B.System(w)
    S.build(); S.compute_force()
    f_o, e_o, E_o = orc.energy_force(w.pos, None, w.box, dim, 2, D, r0, rc, 1, alpha=alpha)
    f = unpermute(S, S.force)
    assert force_error(f, f_o) <= FORCE_TOL
    assert abs(float(S.energy.cpu()[0]) - E_o) <= ENERGY_TOL * abs(E_o)
    assert np.abs(f[:, 3] - e_o).max() <= 2e-6 * max(1.0, np.abs(e_o).max())
    p_o, v_o, _, _, _ = orc.nve_run(w.pos, w.vel, f_o, None, w.box, dim, 2, D, r0, rc, 1, w.dt, w.mass,
                                    100, want_energies=False, alpha=alpha)
    S.step(100)
    torch.cuda.synchronize()
    assert int(S.stats[0]) == 100 and int(S.stats[2]) == -1
    d = unpermute(S, S.pos)[:, :dim].astype(np.float64) - p_o[:, :dim]
    L = w.box[:dim].astype(np.float64)
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    S.close()


@pytest.mark.parametrize("which", ["soft2d", "lj3d"])
def test_fire_minimize_against_the_oracle(B, orc, W, which):
    """FIRE on the same drift / device-side rebuild / force sequence.  State after 20 /
    80 steps against the oracle's fp64 FIRE with all-pairs forces: positions to 1e-4, the device-side
    schedule (dt, alpha, n_pos) and the energy; then the run is continued from the returned state."""
    if which == "soft2d":
        w = W.soft_disks(1, 2048)                       # the paper's packing (L293-L305), smaller
        par = (0.01, 0.1, 5, 1.1, 0.5, 0.1, 0.99)
        diam = w.pos[:, 3].astype(np.float64)
    else:
        w = W.config(0)
        w = dataclasses.replace(w, vel=np.zeros_like(w.vel))
        par = (0.002, 0.02, 5, 1.1, 0.5, 0.1, 0.99)
        diam = None
    # fp32 state against an fp64 trajectory: in the packing's box (L = 51) one ulp of a position is
    # 3.8e-6, dt grows to 0.1 and contacts open and close: measured deviation 1.9e-6 after 1 step,
    # 3.5e-5 after 20, 4.6e-4 after 40.  The LJ lattice (L = 10) is benign.
    steps = 20 if which == "soft2d" else 80
    S = B.System(w)
    S.build(); S.compute_force()
    fp = B.md_fire_params(par[0], par[1], int(par[2]), par[3], par[4], par[5], par[6])
    state = torch.zeros(4, dtype=torch.float32, device="cuda")
    B.md_fire_minimize(S.sys, S.pot, fp, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, state, steps, S.stats)
    torch.cuda.synchronize()
    p_o, v_o, f_o, en, st_o = orc.fire_run(w.pos, w.vel, diam, w.box, w.dim, w.kind, w.epsilon, w.sigma,
                                           w.r_cut, w.shift, steps, par=par)
    st = state.cpu().numpy()
    assert int(S.stats[0]) == steps and int(S.stats[2]) == -1
    assert int(st[2]) == int(st_o[2])
    assert abs(st[0] - st_o[0]) <= 1e-5 * st_o[0] and abs(st[1] - st_o[1]) <= 1e-5 * st_o[1]
    d = unpermute(S, S.pos)[:, :w.dim].astype(np.float64) - p_o[:, :w.dim]
    L = w.box[:w.dim].astype(np.float64)
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    # the force md_fire_minimize leaves is F of ITS final positions (forces of two states 1e-5
    # apart differ by far more than the tolerance near a minimum): state-wise parity
    f_own, _, _ = orc.energy_force(unpermute(S, S.pos), diam, w.box, w.dim, w.kind, w.epsilon, w.sigma,
                                   w.r_cut, w.shift)
    assert force_error(unpermute(S, S.force), f_own) <= FORCE_TOL
    S.compute_force()
    E = float(S.energy.cpu()[0])
    assert abs(E - en[-1]) <= 1e-4 * abs(en[-1]) and en[-1] < en[0]
    # continuing from the returned state keeps the schedule going (no restart from dt_start)
    dt_before = float(state[0])
    B.md_fire_minimize(S.sys, S.pot, fp, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, state, 1, S.stats)
    torch.cuda.synchronize()
    assert float(state[0]) in (np.float32(dt_before), np.float32(min(dt_before * par[3], par[1])),
                               np.float32(dt_before * par[4]))
    S.close()


@pytest.mark.parametrize("which", ["lj3d_kT", "soft2d_descent"])
def test_brownian_and_gradient_descent_against_the_oracle(B, orc, W, which):
    """Brownian dynamics (and gradient descent, kT = 0) with the noise of the shared
    counter-based generator, keyed by the original particle id so the re-sort does not matter."""
    if which == "lj3d_kT":
        w, diam, dt, gamma, kT, steps = W.config(0), None, 2e-4, 1.0, 0.8, 60
    else:
        w = W.soft_disks(1, 2048)
        diam, dt, gamma, kT, steps = w.pos[:, 3].astype(np.float64), 0.02, 1.0, 0.0, 30
    seed = 77
    S = B.System(w)
    S.build(); S.compute_force()
    # one step: the increment is (dt/gamma) F + amp * xi(id)
    f0 = unpermute(S, S.force)[:, :w.dim].astype(np.float64)
    B.md_brownian_step(S.sys, S.pot, S.pos, S.force, S.id, S.nbr_idx, S.nbr_count, dt, gamma, kT, seed, 5, 1, S.stats)
    torch.cuda.synchronize()
    L = w.box[:w.dim].astype(np.float64)
    d = unpermute(S, S.pos)[:, :w.dim].astype(np.float64) - w.pos[:, :w.dim]
    d -= L * np.round(d / L)
    want = dt / gamma * f0 + np.sqrt(2 * kT * dt / gamma) * orc.normals(seed, 5, w.n, w.dim)[:, :w.dim]
    assert np.abs(d - want).max() <= 2e-6 * max(1.0, float(L.max()) / 10)     # fp32 positions
    S.close()
    # a run against the oracle
    S = B.System(w)
    S.build(); S.compute_force()
    B.md_brownian_step(S.sys, S.pot, S.pos, S.force, S.id, S.nbr_idx, S.nbr_count, dt, gamma, kT, seed, 0, steps, S.stats)
    torch.cuda.synchronize()
    p_o, f_o, en = orc.brownian_run(w.pos, diam, w.box, w.dim, w.kind, w.epsilon, w.sigma, w.r_cut, w.shift,
                                    dt, gamma, kT, seed, steps)
    assert int(S.stats[0]) == steps and int(S.stats[2]) == -1
    d = unpermute(S, S.pos)[:, :w.dim].astype(np.float64) - p_o[:, :w.dim]
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    f_own, _, _ = orc.energy_force(unpermute(S, S.pos), diam, w.box, w.dim, w.kind, w.epsilon, w.sigma,
                                   w.r_cut, w.shift)
    assert force_error(unpermute(S, S.force), f_own) <= FORCE_TOL
    if kT == 0.0:
        S.compute_force()
        assert abs(float(S.energy.cpu()[0]) - en[-1]) <= 1e-4 * abs(en[-1]) and en[-1] < en[0]
    S.close()


def test_langevin_against_the_oracle(B, orc, W):
    """BAOAB Langevin with the shared counter-based noise.  60 steps of the 3-D LJ
    system against the oracle; gamma = 0 must reproduce md_nve_step bit for bit."""
    w = W.config(0)
    dt, mass, gamma, kT, seed, steps = 0.004, 1.0, 2.0, 0.8, 9, 60
    S = B.System(w)
    S.build(); S.compute_force()
    f0 = unpermute(S, S.force)[:, :3].astype(np.float64)
    B.md_langevin_step(S.sys, S.pot, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, dt, mass, gamma, kT,
                       seed, 0, steps, S.stats)
    torch.cuda.synchronize()
    p_o, v_o, _ = orc.langevin_run(w.pos, w.vel, f0, None, w.box, 3, 0, 1.0, 1.0, 2.5, 1, dt, mass, gamma, kT, seed, steps)
    assert int(S.stats[0]) == steps and int(S.stats[1]) >= 3 and int(S.stats[2]) == -1
    L = w.box.astype(np.float64)
    d = unpermute(S, S.pos)[:, :3].astype(np.float64) - p_o
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    assert np.abs(unpermute(S, S.vel)[:, :3] - v_o).max() <= 2e-3
    S.close()
    A, N = B.System(w), B.System(w)
    for X in (A, N):
        X.build(); X.compute_force()
    B.md_langevin_step(A.sys, A.pot, A.pos, A.vel, A.force, A.id, A.nbr_idx, A.nbr_count, w.dt, w.mass, 0.0, 0.8,
                       seed, 0, 40, A.stats)
    B.md_set_option(N.sys, "fused", 0)
    N.step(40)
    torch.cuda.synchronize()
    # BAOAB with c1 = 1, c2 = 0 drifts in two half steps (one more rounding than r += dt v): close, not equal
    dd = (A.pos - N.pos)[:, :3].abs().max().item()
    assert dd <= 2e-5 and torch.equal(A.id, N.id)
    A.close(); N.close()


def test_nose_hoover_against_the_oracle(B, orc, W):
    """Nose-Hoover NVT (MTK splitting, thermostat state on the device).  80 steps of
    the 3-D LJ system quenched from T = 1 toward kT = 0.5 against the oracle: positions, velocities
    and the thermostat variables; the run split in two calls continues from the returned state."""
    w = W.config(0)
    dt, mass, kT, tau, steps = 0.004, 1.0, 0.5, 0.2, 80
    S = B.System(w)
    S.build(); S.compute_force()
    state = torch.zeros(2, dtype=torch.float64, device="cuda")
    B.md_nose_hoover_step(S.sys, S.pot, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, dt, mass, kT, tau,
                          state, steps, S.stats)
    torch.cuda.synchronize()
    p_o, v_o, f_o, cons, st_o = orc.nose_hoover_run(w.pos, w.vel, None, w.box, 3, 0, 1.0, 1.0, 2.5, 1, dt, mass, kT, tau, steps)
    assert int(S.stats[0]) == steps and int(S.stats[1]) >= 3 and int(S.stats[2]) == -1
    st = state.cpu().numpy()
    assert np.abs(st - st_o).max() <= 1e-4 * np.abs(st_o).max()
    L = w.box.astype(np.float64)
    d = unpermute(S, S.pos)[:, :3].astype(np.float64) - p_o
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    assert np.abs(unpermute(S, S.vel)[:, :3] - v_o).max() <= 2e-3
    assert (v_o ** 2).sum() < 0.8 * (w.vel[:, :3].astype(np.float64) ** 2).sum()      # it did cool
    S2 = B.System(w)
    S2.build(); S2.compute_force()
    state2 = torch.zeros(2, dtype=torch.float64, device="cuda")
    for k in (30, 50):
        B.md_nose_hoover_step(S2.sys, S2.pot, S2.pos, S2.vel, S2.force, S2.id, S2.nbr_idx, S2.nbr_count, dt, mass,
                              kT, tau, state2, k, S2.stats)
    torch.cuda.synchronize()
    assert torch.equal(S2.pos, S.pos) and torch.equal(S2.vel, S.vel) and torch.equal(state2, state)
    S.close(); S2.close()


def test_nose_hoover_chain_against_the_oracle(B, orc, W):
    """A chain of three thermostats ([67]; option "nh_chain"): 80 steps against the oracle -- positions,
    velocities and all six thermostat variables; graph and direct launches agree bit for bit; a chain
    of one is the default."""
    w = W.config(0)
    dt, mass, kT, tau, steps, M = 0.004, 1.0, 0.5, 0.2, 80, 3
    outs = []
    for graph in (1, 0):
        S = B.System(w)
        B.md_set_option(S.sys, "nh_chain", M)
        B.md_set_option(S.sys, "use_graph", graph)
        S.build(); S.compute_force()
        state = torch.zeros(2 * M, dtype=torch.float64, device="cuda")
        B.md_nose_hoover_step(S.sys, S.pot, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, dt, mass, kT, tau,
                              state, steps, S.stats)
        torch.cuda.synchronize()
        outs.append((S.pos.clone(), S.vel.clone(), state.clone(), unpermute(S, S.pos), unpermute(S, S.vel)))
        S.close()
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1]) and torch.equal(outs[0][2], outs[1][2])
    p_o, v_o, f_o, cons, st_o = orc.nose_hoover_run(w.pos, w.vel, None, w.box, 3, 0, 1.0, 1.0, 2.5, 1, dt, mass, kT, tau,
                                                    steps, chain=M)
    st = outs[0][2].cpu().numpy()
    assert np.abs(st_o[M:]).min() > 1e-3                                   # every link is in motion
    assert np.abs(st - st_o).max() <= 1e-4 * np.abs(st_o).max(), (st, st_o)
    L = w.box.astype(np.float64)
    d = outs[0][3][:, :3].astype(np.float64) - p_o
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    assert np.abs(outs[0][4][:, :3] - v_o).max() <= 2e-3
    S = B.System(w)
    with pytest.raises(B.MdError):
        B.md_set_option(S.sys, "nh_chain", 9)
    S.close()


def test_buckingham_force_energy_and_trajectory(B, orc, W):
    """Buckingham-type exp-6 (PAPER.md:L104 [71-73]) on the fp64 pair chain: force and
    energy against the all-pairs definition, then 100 NVE steps against the oracle."""
    # exp-6 with alpha = 14, eps = 1, r_m = 1.12: A = 6 eps e^alpha/(alpha-6), B = alpha/r_m, C = eps alpha r_m^6/(alpha-6)
    A, Bc, Cc, rc = float(np.float32(9.02e5)), float(np.float32(12.5)), float(np.float32(3.454)), 2.5
    base = W.config(0)
    w = custom_workload(W, base.pos.copy(), base.box, 3, 3, rc, 0.3, 128, vel=base.vel.copy(), dt=0.004)
    w = dataclasses.replace(w, epsilon=A, sigma=Cc, alpha=Bc, shift=1)
    S = B.System(w)
    S.build(); S.compute_force()
    f_o, e_o, E_o = orc.energy_force(w.pos, None, w.box, 3, 3, A, Cc, rc, 1, alpha=Bc)
    f = unpermute(S, S.force)
    assert force_error(f, f_o) <= FORCE_TOL
    assert abs(float(S.energy.cpu()[0]) - E_o) <= ENERGY_TOL * abs(E_o)
    p_o, v_o, _, _, _ = orc.nve_run(w.pos, w.vel, f_o, None, w.box, 3, 3, A, Cc, rc, 1, w.dt, w.mass, 100,
                                    want_energies=False, alpha=Bc)
    S.step(100)
    torch.cuda.synchronize()
    d = unpermute(S, S.pos)[:, :3].astype(np.float64) - p_o
    L = w.box.astype(np.float64)
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    S.close()


def test_species_lj_binary_mixture(B, orc, W):
    """species x species LJ.  The 80:20 Kob-Andersen
    mixture on the jittered lattice of config 0: force / energy against the all-pairs definition,
    100 NVE steps against the oracle, and equal tables reproducing plain LJ."""
    eps = np.array([[1.0, 1.5], [1.5, 0.5]], np.float32)
    sig = np.array([[1.0, 0.8], [0.8, 0.88]], np.float32)
    rc = (2.5 * sig).astype(np.float32)
    base = W.config(0)
    pos = base.pos.copy()
    pos[:, 3] = (np.arange(base.n) % 5 == 0).astype(np.float32)            # species in pos.w
    w = custom_workload(W, pos, base.box, 3, 4, 2.5, 0.3, 128, vel=base.vel.copy(), dt=0.004)
    w = dataclasses.replace(w, shift=1)
    S = B.System(w)
    B.md_set_species_lj(S.sys, eps, sig, rc)
    S.build(); S.compute_force()
    orc.set_species_lj(eps.astype(np.float64), sig.astype(np.float64), rc.astype(np.float64))
    sp = pos[:, 3].astype(np.float64)
    f_o, e_o, E_o = orc.energy_force(w.pos, sp, w.box, 3, 4, 0.0, 0.0, 0.0, 1)
    assert force_error(unpermute(S, S.force), f_o) <= FORCE_TOL
    assert abs(float(S.energy.cpu()[0]) - E_o) <= ENERGY_TOL * abs(E_o)
    p_o, v_o, _, _, _ = orc.nve_run(w.pos, w.vel, f_o, sp, w.box, 3, 4, 0.0, 0.0, 0.0, 1, w.dt, w.mass, 100,
                                    want_energies=False)
    S.step(100)
    torch.cuda.synchronize()
    d = unpermute(S, S.pos)[:, :3].astype(np.float64) - p_o
    L = w.box.astype(np.float64)
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    assert np.array_equal(unpermute(S, S.pos)[:, 3], pos[:, 3])            # species travel with the re-sort
    S.close()
    # equal tables: the fp64 LJ chain
    one = np.ones((2, 2), np.float32)
    S1, S0 = B.System(w), B.System(dataclasses.replace(w, kind=0))
    B.md_set_species_lj(S1.sys, one, one, 2.5 * one)
    B.md_set_option(S0.sys, "fast32", 0)
    for X in (S1, S0):
        X.build(); X.compute_force()
    torch.cuda.synchronize()
    assert (S1.force[:, :3] - S0.force[:, :3]).abs().max().item() <= 1e-5 * S0.force[:, :3].abs().max().item()
    S1.close(); S0.close()


def test_bks_type_binary_crystal(B, orc, W):
    """BKS-type potential (PAPER.md:L104 [71-73]; A27): exp-6 with distinct A, B, C
    per species pair plus damped shifted-force Coulomb between charges +-0.6 on the jittered lattice of
    config 0: force / energy against the all-pairs definition, 100 NVE steps against the oracle; zero
    charges and equal tables reproduce the Buckingham kind."""
    A0, B0, C0, rc = 9.02e5, 12.5, 3.454, 2.5
    f32 = lambda a: np.asarray(a, np.float32)
    Am = f32(A0 * np.array([[1.0, 0.7], [0.7, 0.5]])); Bm = f32(B0 * np.array([[1.0, 1.05], [1.05, 1.1]]))
    Cm = f32(C0 * np.array([[1.0, 0.6], [0.6, 0.3]])); q = f32([0.6, -0.6])
    alpha_c, ke = float(np.float32(0.3)), float(np.float32(1.0))
    base = W.config(0)
    pos = base.pos.copy()
    pos[:, 3] = (np.arange(base.n) % 2).astype(np.float32)
    w = custom_workload(W, pos, base.box, 3, 5, rc, 0.3, 128, vel=base.vel.copy(), dt=0.004)
    w = dataclasses.replace(w, shift=1)
    S = B.System(w)
    B.md_set_species_bks(S.sys, Am, Bm, Cm, q, alpha_c, ke)
    S.build(); S.compute_force()
    d64 = lambda a: np.asarray(a, np.float64)
    orc.set_species_bks(d64(Am), d64(Bm), d64(Cm), d64(q), alpha_c, ke)
    sp = pos[:, 3].astype(np.float64)
    f_o, e_o, E_o = orc.energy_force(w.pos, sp, w.box, 3, 5, 0.0, 0.0, rc, 1)
    assert force_error(unpermute(S, S.force), f_o) <= FORCE_TOL
    assert abs(float(S.energy.cpu()[0]) - E_o) <= ENERGY_TOL * abs(E_o)
    p_o, v_o, _, _, _ = orc.nve_run(w.pos, w.vel, f_o, sp, w.box, 3, 5, 0.0, 0.0, rc, 1, w.dt, w.mass, 100,
                                    want_energies=False)
    S.step(100)
    torch.cuda.synchronize()
    d = unpermute(S, S.pos)[:, :3].astype(np.float64) - p_o
    L = w.box.astype(np.float64)
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    S.close()
    # zero charges, equal tables: the Buckingham kind
    one = np.ones((2, 2), np.float32)
    S5 = B.System(w)
    B.md_set_species_bks(S5.sys, f32(A0) * one, f32(B0) * one, f32(C0) * one, f32([0.0, 0.0]), alpha_c, ke)
    w3 = dataclasses.replace(w, kind=3, epsilon=float(np.float32(A0)), sigma=float(np.float32(C0)), alpha=float(np.float32(B0)))
    S3 = B.System(w3)
    B.md_set_option(S3.sys, "fast32", 0)              # the fp64 Buckingham chain, term by term the same arithmetic
    for X in (S5, S3):
        X.build(); X.compute_force()
    torch.cuda.synchronize()
    assert (S5.force[:, :3] - S3.force[:, :3]).abs().max().item() <= 1e-5 * S3.force[:, :3].abs().max().item()
    assert abs(float(S5.energy[0]) - float(S3.energy[0])) <= 1e-9 * abs(float(S3.energy[0]))
    S5.close(); S3.close()
    Sx = B.System(w)
    with pytest.raises(B.MdError):
        Sx.build(); Sx.compute_force()                                   # tables not set
    Sx.close()


@pytest.mark.parametrize("rule", ["fire", "brownian", "langevin", "nose_hoover"])
def test_update_rules_graph_and_direct_launch_agree(B, W, rule):
    """Every update rule beyond NVE runs as CUDA graphs of 8 steps (rebuild in an IF node, step
    counter and rule state on the device) or, with use_graph = 0, as direct launches: same bits,
    also when the run is split into calls that mix both graph sizes."""
    w = W.config(0)
    out = []
    for graph, split in ((1, (37,)), (0, (37,)), (1, (5, 16, 16))):
        S = B.System(w)
        B.md_set_option(S.sys, "use_graph", graph)
        S.build(); S.compute_force()
        st32 = torch.zeros(4, dtype=torch.float32, device="cuda")
        st64 = torch.zeros(2, dtype=torch.float64, device="cuda")
        done = 0
        for k in split:
            if rule == "fire":
                fp = B.md_fire_params(0.002, 0.02, 5, 1.1, 0.5, 0.1, 0.99)
                B.md_fire_minimize(S.sys, S.pot, fp, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, st32, k, S.stats)
            elif rule == "brownian":
                B.md_brownian_step(S.sys, S.pot, S.pos, S.force, S.id, S.nbr_idx, S.nbr_count, 2e-4, 1.0, 0.8, 3, done, k, S.stats)
            elif rule == "langevin":
                B.md_langevin_step(S.sys, S.pot, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, 0.004, 1.0, 2.0, 0.8,
                                   3, done, k, S.stats)
            else:
                B.md_nose_hoover_step(S.sys, S.pot, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, 0.004, 1.0, 0.5,
                                      0.2, st64, k, S.stats)
            done += k
        torch.cuda.synchronize()
        out.append((S.pos.clone(), S.vel.clone(), S.force.clone(), S.id.clone(), st32.clone(), st64.clone()))
        S.close()
    for o in out[1:]:
        for x, y in zip(out[0], o):
            assert torch.equal(x, y)


def test_flocking_against_the_oracle(B, orc, W):
    """the boids energy model (App. B eqs. 3-10) by forward Euler on the same
    cell / neighbor list, headings in pos.w.
    (a) one step of 1024 boids against the oracle's all-pairs gradients (all three terms);
    (b) 60 steps with alignment + avoidance against the oracle, graph and direct launches bit-equal;
    (c) 20 steps with cohesion on isolated triplets.  Eq. 10 normalises D_i = sum (R_j - R_i), so the
        cohesion gradient is singular where the neighbors surround a boid evenly (|D| -> 0): in a
        uniform flock fp32 and fp64 trajectories part within two steps (measured 1.5e-2), which is the
        model's conditioning, not an error -- hence (a) there and trajectories only where |D| is
        bounded below."""
    rng = np.random.default_rng(17)
    n, L = 1024, 40.3
    box32 = np.array([L, L, 1.0], np.float32)
    pos = np.zeros((n, 4), np.float32)
    gq = (np.arange(32) + 0.5) * (L / 32)
    pos[:, :2] = W.into_box_f32(np.stack(np.meshgrid(gq, gq, indexing="ij"), -1).reshape(-1, 2)
                                + rng.normal(0, 0.15, (n, 2)), box32)
    pos[:, 3] = rng.uniform(-np.pi, np.pi, n).astype(np.float32)
    speed, dt = 0.5, 0.02
    w = custom_workload(W, pos, box32, 2, 1, 4.0, 0.5, 128)
    th0 = pos[:, 3].astype(np.float64)

    # (a) alpha = 3, 2 (compile-time integer powers) and 2.5 (pow)
    for alpha in (3.0, 2.0, 2.5):
        par = (1.0, 3.0, 10.0, 1.5, 0.5, 4.0, alpha)
        S = B.System(w)
        S.build()
        B.md_flock_step(S.sys, B.md_flock_params(*par, speed), S.pos, S.id, S.nbr_idx, S.nbr_count, dt, 1, S.stats)
        torch.cuda.synchronize()
        en, gR, gth = orc.flock_energy_grad(pos, th0, box32, par)
        one = unpermute(S, S.pos)
        d = one[:, :2].astype(np.float64) - pos[:, :2]
        d -= L * np.round(d / L)
        want = dt * (speed * np.stack([np.cos(th0), np.sin(th0)], 1) - gR)
        scale = max(1.0, np.abs(want).max())
        assert np.abs(d - want).max() <= 4e-6 * scale                  # fp32 positions at L = 40
        assert np.abs((one[:, 3].astype(np.float64) - th0) + dt * gth).max() <= 1e-6 * max(1.0, np.abs(gth).max())
        S.close()

    # (b)
    par = (1.0, 3.0, 10.0, 1.5, 0.0, 4.0, 3.0)
    steps = 60
    outs = []
    for graph in (1, 0):
        S = B.System(w)
        B.md_set_option(S.sys, "use_graph", graph)
        S.build()
        B.md_flock_step(S.sys, B.md_flock_params(*par, speed), S.pos, S.id, S.nbr_idx, S.nbr_count, dt, steps, S.stats)
        torch.cuda.synchronize()
        assert int(S.stats[0]) == steps and int(S.stats[2]) == -1
        outs.append((unpermute(S, S.pos), S.pos.clone(), S.id.clone()))
        S.close()
    assert torch.equal(outs[0][1], outs[1][1]) and torch.equal(outs[0][2], outs[1][2])
    p_o, th_o = orc.flock_run(pos, th0, box32, par, speed, dt, steps)
    d = outs[0][0][:, :2].astype(np.float64) - p_o[:, :2]
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    assert np.abs(outs[0][0][:, 3].astype(np.float64) - th_o).max() <= 1e-4

    # (c) 100 isolated triplets, 10 apart, each an irregular triangle of side ~2
    m = 10
    cen = (np.stack(np.meshgrid(np.arange(m), np.arange(m), indexing="ij"), -1).reshape(-1, 2) + 0.5) * 10.0
    tri = np.array([[0.0, 0.0], [2.0, 0.3], [0.7, 1.9]])
    p3 = np.zeros((300, 4), np.float32)
    p3[:, :2] = (cen[:, None, :] + tri[None, :, :] + rng.normal(0, 0.1, (100, 3, 2))).reshape(-1, 2)
    p3[:, 3] = rng.uniform(-np.pi, np.pi, 300).astype(np.float32)
    box3 = np.array([100.0 + 0.7, 100.0 + 0.7, 1.0], np.float32)
    par = (1.0, 3.0, 10.0, 1.5, 0.5, 4.0, 3.0)
    w3 = custom_workload(W, p3, box3, 2, 1, 4.0, 0.5, 32)
    S = B.System(w3)
    S.build()
    B.md_flock_step(S.sys, B.md_flock_params(*par, 0.2), S.pos, S.id, S.nbr_idx, S.nbr_count, 0.02, 20, S.stats)
    torch.cuda.synchronize()
    p_o, th_o = orc.flock_run(p3, p3[:, 3].astype(np.float64), box3, par, 0.2, 0.02, 20)
    got = unpermute(S, S.pos)
    d = got[:, :2].astype(np.float64) - p_o[:, :2]
    d -= box3[:2] * np.round(d / box3[:2])
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    assert np.abs(got[:, 3].astype(np.float64) - th_o).max() <= 1e-4
    S.close()

    # (d) disk obstacles (App. B.3.1, eq. 11): the obstacle term alone after one step, then 60 steps of
    #     alignment + avoidance + obstacles; one disk straddles the periodic boundary
    cen_o = np.array([[10.2, 11.7], [0.9, 30.1], [25.3, 20.4], [33.0, 5.5]], np.float32)
    rad_o = np.array([4.0, 3.0, 5.5, 2.5], np.float32)
    Jo = 4.0
    par0 = (0.0, 3.0, 0.0, 1.5, 0.0, 4.0, 3.0)
    S = B.System(w)
    B.md_flock_obstacles(S.sys, cen_o, rad_o, Jo)
    S.build()
    B.md_flock_step(S.sys, B.md_flock_params(*par0, speed), S.pos, S.id, S.nbr_idx, S.nbr_count, dt, 1, S.stats)
    torch.cuda.synchronize()
    e_ob, gR, gth = orc.flock_obstacle_energy_grad(pos, th0, box32, cen_o, rad_o, Jo, 3.0)
    assert e_ob > 0 and (np.abs(gR).sum(1) > 0).sum() > 50              # boids do sit inside the disks
    one = unpermute(S, S.pos)
    d = one[:, :2].astype(np.float64) - pos[:, :2]
    d -= L * np.round(d / L)
    want = dt * (speed * np.stack([np.cos(th0), np.sin(th0)], 1) - gR)
    assert np.abs(d - want).max() <= 4e-6 * max(1.0, np.abs(want).max())
    assert np.abs((one[:, 3].astype(np.float64) - th0) + dt * gth).max() <= 1e-6 * max(1.0, np.abs(gth).max())
    S.close()
    par = (1.0, 3.0, 10.0, 1.5, 0.0, 4.0, 3.0)
    S = B.System(w)
    B.md_flock_obstacles(S.sys, cen_o, rad_o, Jo)
    S.build()
    B.md_flock_step(S.sys, B.md_flock_params(*par, speed), S.pos, S.id, S.nbr_idx, S.nbr_count, dt, 60, S.stats)
    torch.cuda.synchronize()
    orc.flock_set_obstacles(cen_o, rad_o, Jo)
    try:
        p_o, th_o = orc.flock_run(pos, th0, box32, par, speed, dt, 60)
    finally:
        orc.flock_set_obstacles()
    got = unpermute(S, S.pos)
    d = got[:, :2].astype(np.float64) - p_o[:, :2]
    d -= L * np.round(d / L)
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    assert np.abs(got[:, 3].astype(np.float64) - th_o).max() <= 1e-4
    # removing the obstacles restores the plain model (and re-captures the graph)
    B.md_flock_obstacles(S.sys)
    S.reset(); S.build()
    B.md_flock_step(S.sys, B.md_flock_params(*par, speed), S.pos, S.id, S.nbr_idx, S.nbr_count, dt, 60, S.stats)
    torch.cuda.synchronize()
    assert torch.equal(S.pos, outs[0][1])
    with pytest.raises(B.MdError):
        B.md_flock_obstacles(S.sys, [[1.0, 1.0]], [30.0], 1.0)          # radius above half the box
    S.close()

    # (e) predators (App. B.3.2, eqs. 12-13) with obstacles.  One step of both populations on the uniform
    #     flock against the oracle's gradients; then 60 steps on four separated clumps of 64 boids with a
    #     predator beside each -- like eq. 10, the chase term is singular where the prey surrounds the
    #     predator evenly (|D_p| -> 0: in the uniform flock fp32 and fp64 runs part within 5 steps), so the
    #     trajectory is compared where |D_p| is bounded below.
    def run_both(wk, p0, t0, bx, Lb, pp0, pt0, ppar, cen, rad, steps, tol):
        S = B.System(wk)
        pred0 = np.zeros((len(pt0), 4), np.float32); pred0[:, :2] = pp0; pred0[:, 3] = pt0
        pred = torch.from_numpy(pred0).cuda()
        B.md_flock_obstacles(S.sys, cen, rad, Jo)
        B.md_flock_predators(S.sys, pred, B.md_predator_params(*ppar))
        S.build()
        B.md_flock_step(S.sys, B.md_flock_params(*par, speed), S.pos, S.id, S.nbr_idx, S.nbr_count, dt, steps, S.stats)
        torch.cuda.synchronize()
        orc.flock_set_obstacles(cen, rad, Jo)
        try:
            p_o, th_o, pp_o, pt_o = orc.flock_run_predators(p0, t0, bx, par, speed, dt, steps, pp0, pt0, ppar)
        finally:
            orc.flock_set_obstacles()
        got = unpermute(S, S.pos)
        d = got[:, :2].astype(np.float64) - p_o[:, :2]
        d -= Lb * np.round(d / Lb)
        assert np.abs(d).max() <= tol, (steps, np.abs(d).max())
        assert np.abs(got[:, 3].astype(np.float64) - th_o).max() <= tol
        gp = pred.cpu().numpy()
        dp = gp[:, :2].astype(np.float64) - pp_o
        dp -= Lb * np.round(dp / Lb)
        assert np.abs(dp).max() <= tol, (steps, np.abs(dp).max())
        assert np.abs(gp[:, 3].astype(np.float64) - pt_o).max() <= tol
        B.md_flock_predators(S.sys)                                      # removable
        S.close()
        return pp_o, pt_o

    par = (1.0, 3.0, 10.0, 1.5, 0.0, 4.0, 3.0)
    pp0 = np.array([[5.3, 6.1], [20.7, 21.9], [39.6, 12.2], [30.2, 33.3]], np.float32)
    pt0 = np.array([0.4, -2.1, 3.0, 1.2], np.float32)
    ppar = (5.0, 4.0, 3.0, 6.0, 0.8)
    run_both(w, pos, th0, box32, L, pp0, pt0, ppar, cen_o, rad_o, 1, 4e-6)
    _, gq, _ = orc.predator_energy_grad(pos, box32, pp0, pt0, ppar[2], ppar[3])
    e_f, _, _ = orc.flock_obstacle_energy_grad(pos, th0, box32, pp0, [ppar[1]] * 4, ppar[0], 3.0)
    assert np.abs(gq).max() > 0 and e_f > 0                # predators felt their prey, boids their predators
    Lc = 60.3
    boxc = np.array([Lc, Lc, 1.0], np.float32)
    cents = np.array([[15.0, 15.0], [45.0, 15.0], [15.0, 45.0], [45.0, 45.0]])
    g8 = (np.arange(8) - 3.5) * 1.0
    cl = np.stack(np.meshgrid(g8, g8, indexing="ij"), -1).reshape(-1, 2)
    pc = np.zeros((256, 4), np.float32)
    pc[:, :2] = (cents[:, None, :] + cl[None, :, :] + rng.normal(0, 0.12, (4, 64, 2))).reshape(-1, 2)
    pc[:, 3] = rng.uniform(-np.pi, np.pi, 256).astype(np.float32)
    ppc = (cents + np.array([[-6.0, 0.5], [0.4, 6.0], [6.0, -0.3], [-4.5, -4.5]])).astype(np.float32)
    ptc = np.array([2.0, 0.3, -1.0, 2.5], np.float32)
    wc = custom_workload(W, pc, boxc, 2, 1, 4.0, 0.5, 64)
    pp_o, pt_o = run_both(wc, pc, pc[:, 3].astype(np.float64), boxc, Lc, ppc, ptc, (5.0, 4.0, 3.0, 14.0, 0.8),
                          np.array([[18.5, 17.0], [45.0, 50.5]], np.float32), np.array([3.0, 4.0], np.float32), 60, 1e-4)
    assert np.abs(pp_o - ppc).max() > 0.5 and np.abs(pt_o - ptc).max() > 1.0     # they did turn and travel


def test_fast32_dimers_at_the_force_zero(B, orc, W):
    """Isolated pairs around r = 2^(1/6) sigma, where the LJ force changes sign: the coefficient and
    with it sum|coefficient| vanish while the fp32 rounding error does not, so the error estimate
    needs its floor there (md_force32.cuh).  64 dimers in a sparse 3-D box, sigma = 0.4."""
    rng = np.random.default_rng(5)
    sig = float(np.float32(0.4))
    box32 = np.array([30.3, 30.3, 30.3], np.float32)
    centers = (np.stack(np.meshgrid(*[np.arange(4)] * 3, indexing="ij"), -1).reshape(-1, 3) * 7.0 + 3.0)
    pos = np.zeros((128, 4), np.float32); pos[:, 3] = 1.0
    for k, c in enumerate(centers):
        u = rng.normal(size=3); u /= np.linalg.norm(u)
        r = 2.0 ** (1.0 / 6.0) * sig * (1.0 + (k - 32) * 1e-4)      # from 0.3 % inside to 0.3 % outside
        pos[2 * k, :3] = c + 0.5 * r * u
        pos[2 * k + 1, :3] = c - 0.5 * r * u
    w = custom_workload(W, pos, box32, 3, 0, 1.0, 0.25, 32)
    w = dataclasses.replace(w, sigma=0.4)
    S = B.System(w)
    S.build(); S.compute_force()
    f = unpermute(S, S.force)
    f_o, _, E_o = orc.energy_force(w.pos, None, w.box, 3, 0, 1.0, sig, 1.0, 1)
    assert np.linalg.norm(f_o, axis=1).max() < 1.0 and np.linalg.norm(f_o, axis=1).min() < 1e-2
    assert force_error(f, f_o) <= FORCE_TOL
    assert abs(float(S.energy.cpu()[0]) - E_o) <= ENERGY_TOL * abs(E_o)
    S.close()


@pytest.mark.parametrize("thr", [1e-3, 8.0, 1e9])
def test_fast32_re_evaluation(B, orc, W, thr):
    """The fp32 fast path: est_thr -> 0 sends every particle through the fp64 re-evaluation (must
    then match the fp64 kernels' accuracy), the default must hold the north_star tolerance, and
    est_thr -> inf (never re-evaluate, except at the cutoff) shows what the estimate is for."""
    w = W.config(2)
    S = B.System(w)
    S.build()
    B.md_set_option(S.sys, "est_thr", thr)
    cnt = torch.zeros(8, dtype=torch.int32, device="cuda")
    B.md_counters(S.sys, cnt, True)
    S.compute_force()
    B.md_counters(S.sys, cnt, True)
    f_o, _, E_o = orc.energy_force(w.pos, None, w.box, 3, 0, 1.0, 1.0, 2.5, 1)
    err = force_error(unpermute(S, S.force), f_o)
    fixed = int(cnt[0].item())
    if thr < 1.0:
        assert fixed == w.n and err <= 3e-7
    elif thr < 1e6:
        assert 0 < fixed < 0.25 * w.n and err <= FORCE_TOL
    else:
        assert fixed < 0.01 * w.n and err <= 1e-4
    assert abs(float(S.energy.cpu()[0]) - E_o) <= ENERGY_TOL * abs(E_o)
    S.close()


# --------------------------------------------------------------------- edge cases -------

def edge_positions(W, seed, n, dim, box, R):
    pos, box32 = W.random_box(seed, n, dim, box, diam=(1.0, 1.4))
    for k in range(dim):
        L = box32[k]
        nk = int(np.floor(float(L) / float(R)))
        specials = [np.float32(0.0), np.nextafter(L, np.float32(0.0), dtype=np.float32)]
        for c in range(1, nk):
            face = np.float32(c * float(L) / nk)
            specials += [face, np.nextafter(face, np.float32(0), dtype=np.float32),
                         np.nextafter(face, np.float32(1e9), dtype=np.float32)]
        for s, x in enumerate(specials):
            pos[(7 * s + 3 * k) % n, k] = x
    return pos, box32


@pytest.mark.parametrize("dim,box,n", [
    (3, [3.9, 5.2, 6.4], 700),       # 3 x 4 x 5 cells, ragged n
    (3, [3.76, 3.76, 3.76], 333),    # 3 cells per side: every cell is a periodic neighbor
    (2, [3.8, 6.3], 257),            # 2-D, 3 x 5 cells
    (2, [13.0, 4.0], 64),            # many empty cells
    (3, [5.01, 5.01, 5.01], 1),      # a single particle
    (3, [5.01, 5.01, 5.01], 2),
    (3, [40.5, 4.0, 4.0], 50),       # sparse: most cells empty
    (2, [200.7, 190.3], 5000),       # 160 x 152 = 24,320 cells: the two-launch cell scan
    (3, [40.3, 40.3, 41.1], 3000),   # 32 x 32 x 32 = 32,768 cells, almost all empty
])
@pytest.mark.parametrize("kind", [0, 1])
def test_edge_cases(B, orc, W, dim, box, n, kind):
    r_cut, skin = 1.0, 0.25
    R = np.float32(np.float32(r_cut) + np.float32(skin))
    pos, box32 = edge_positions(W, 100 + n, n, dim, box, R)
    if kind == 0:
        pos[:, 3] = 1.0
    else:
        pos[:, 3] = np.where(np.arange(n) < n // 2, 0.7, 1.0)   # d_ij <= 1.0 = list r_cut
    w = custom_workload(W, pos, box32, dim, kind, r_cut, skin, 192)
    if kind == 0:
        w = dataclasses.replace(w, sigma=0.4)    # keeps LJ forces representable at random overlaps
    for resort in (1, 0):
        S = B.System(w, resort=resort)
        S.build()
        torch.cuda.synchronize()
        check_cells(S, orc, w)
        check_list(S, orc, w, method=0)
        if kind == 1:
            check_force(S, orc, w)
        else:
            # random overlaps give |F| ~ 1e9: compare where the oracle force is sane
            S.compute_force()
            f = unpermute(S, S.force)
            # the ABI carries sigma as fp32: the oracle gets the same value (near the zero of the
            # pair force a 1.5e-8 difference in sigma is amplified a thousandfold)
            f_o, _, _ = orc.energy_force(w.pos, None, w.box, dim, 0, 1.0, float(np.float32(0.4)),
                                         float(np.float32(r_cut)), 1)
            sane = np.linalg.norm(f_o, axis=1) < 1e30        # beyond that fp32 cannot hold F
            num = np.linalg.norm(f[sane, :3].astype(np.float64) - f_o[sane], axis=1)
            if sane.any():
                assert (num / np.maximum(np.linalg.norm(f_o[sane], axis=1), 1e-3)).max() <= FORCE_TOL
            assert not np.isfinite(f[~sane, :3]).all(axis=1).any() or \
                np.linalg.norm(f[~sane, :3].astype(np.float64), axis=1).min() > 1e30
        S.close()


def test_overflow_flag(B, orc, W):
    """Static capacity: capacity 64 on config 0 overflows; counts stay true."""
    w = W.config(0)
    S = B.System(w, capacity=64)
    S.build()
    st = S.status.cpu().numpy()
    idx_o, cnt_o, st_o = orc.neighbor_list(w.pos, w.box, 3, w.r_cut, w.skin, 64)
    assert st[0] == 1 and st_o[0] == 1 and st[1] == st_o[1]
    _, counts = gpu_rows_in_original_order(S)
    assert np.array_equal(counts, cnt_o)
    # a later build with room clears the flag
    S2 = B.System(w, capacity=128)
    S2.build()
    assert S2.status.cpu().numpy()[0] == 0
    S.close(); S2.close()


def test_needs_rebuild_constructed(B, orc, W):
    """P9: half-skin criterion, strict, minimum image."""
    w = W.config(0)
    S = B.System(w, resort=0)
    S.build()
    ref = S.pos.clone()
    half = w.skin / 2
    u = np.array([1.0, 2.0, -2.0]) / 3.0

    def flag_for(p):
        B.md_needs_rebuild(S.sys, p, S.flag)
        return int(S.flag.cpu()[0])

    assert flag_for(ref) == 0
    for scale, want in [(1 - 1e-3, 0), (1 + 1e-3, 1)]:
        p = ref.clone()
        x = ref[100, :3].cpu().numpy().astype(np.float64) + u * half * scale
        p[100, :3] = torch.from_numpy(np.mod(x, w.box).astype(np.float32)).cuda()
        assert flag_for(p) == want
        o_flag, _ = orc.needs_rebuild(p.cpu().numpy(), ref.cpu().numpy(), w.box, 3, w.skin)
        assert o_flag == want
    # crossing the periodic boundary by 0.01 is a small displacement
    refc = ref.clone(); refc[5, 0] = 0.004
    S.pos.copy_(refc); S.build()
    p = S.pos.clone(); p[5, 0] = float(w.box[0]) - 0.006
    assert flag_for(p) == 0
    S.close()


# ------------------------------------------------------------------ NVE trajectory ------

def test_nve_config0_trajectory(B, orc, W):
    """north_star: positions after 100 NVE steps on config 0 within 1e-4 sigma."""
    w = W.config(0)
    S = B.System(w)
    S.build()
    S.compute_force()
    f0, _, E0 = orc.energy_force(w.pos, None, w.box, 3, 0, 1.0, 1.0, 2.5, 1)
    p_o, v_o, f_o, en, _ = orc.nve_run(w.pos, w.vel, f0, None, w.box, 3, 0, 1.0, 1.0, 2.5, 1,
                                       w.dt, w.mass, w.steps)          # brute force, no list
    S.step(w.steps)
    torch.cuda.synchronize()
    stats = S.stats.cpu().numpy()
    assert stats[0] == w.steps and 5 <= stats[1] <= 20 and stats[2] == -1 and 70 < stats[3] < 128
    p = unpermute(S, S.pos)[:, :3].astype(np.float64)
    d = p - p_o
    d -= w.box.astype(np.float64) * np.round(d / w.box.astype(np.float64))
    assert np.abs(d).max() <= 1e-4, np.abs(d).max()
    v = unpermute(S, S.vel)[:, :3].astype(np.float64)
    assert np.abs(v - v_o).max() <= 2e-3
    # positions stay inside the box; ids are a permutation
    pg = S.pos.cpu().numpy()
    assert pg[:, :3].min() >= 0 and np.all(pg[:, :3] < w.box)
    assert np.array_equal(np.sort(S.id.cpu().numpy()), np.arange(w.n))
    # the final force is F(final positions): snapshot parity
    w2 = dataclasses.replace(w, pos=unpermute(S, S.pos))
    f2, _, _ = orc.energy_force(w2.pos, None, w.box, 3, 0, 1.0, 1.0, 2.5, 1)
    assert force_error(unpermute(S, S.force), f2) <= FORCE_TOL
    # graph and direct launches give the same bits
    S2 = B.System(w)
    B.md_set_option(S2.sys, "use_graph", 0)
    S2.build(); S2.compute_force(); S2.step(w.steps)
    assert torch.equal(S2.pos, S.pos) and torch.equal(S2.vel, S.vel)
    # splitting the run does not change the result (stats restart per call)
    S3 = B.System(w)
    S3.build(); S3.compute_force(); S3.step(37); S3.step(w.steps - 37)
    assert torch.equal(S3.pos, S.pos) and torch.equal(S3.vel, S.vel)
    S.close(); S2.close(); S3.close()


def test_nve_run_host_matches_device_path(B, W):
    w = W.config(0)
    S = B.System(w)
    S.build(); S.compute_force(); S.step(50); S.compute_force()
    pos = w.pos.copy(); vel = w.vel.copy(); force = np.zeros_like(pos)
    stats = np.zeros(4, np.int32)
    E = B.md_nve_run_host(S.cfg, S.pot, pos, vel, force, w.dt, w.mass, 50, stats)
    assert np.array_equal(pos, unpermute(S, S.pos))
    assert np.array_equal(vel, unpermute(S, S.vel))
    assert np.array_equal(force, unpermute(S, S.force))
    assert abs(E - float(S.energy.cpu()[0])) <= 1e-9 * abs(E)
    assert np.array_equal(stats, S.stats.cpu().numpy())
    S.close()


@pytest.mark.parametrize("resort", [1, 0])
@pytest.mark.parametrize("ci,steps", [(0, 100), (2, 120)])
def test_fused_step_same_bits(B, W, ci, steps, resort):
    """The fused graph (force kernel opens the next step, positions ping-pong between two buffers)
    and the plain sequence k_kick_drift -> rebuild -> force give the same bits and the same
    rebuild history, for step counts that exercise both the 9-step and the 1-step graph."""
    w = W.config(ci)
    out = []
    for fused, graph in ((1, 1), (0, 1), (0, 0)):
        S = B.System(w, resort=resort)
        B.md_set_option(S.sys, "fused", fused)
        B.md_set_option(S.sys, "use_graph", graph)
        S.build(); S.compute_force(); S.step(steps)
        torch.cuda.synchronize()
        out.append((S.pos.clone(), S.vel.clone(), S.force.clone(), S.id.clone(), S.stats.clone()))
        S.close()
    for o in out[1:]:
        for x, y in zip(out[0], o):
            assert torch.equal(x, y)
    assert int(out[0][4][0]) == steps and int(out[0][4][1]) >= 5


@pytest.mark.parametrize("ci,steps,resort", [(0, 100, 1), (1, 60, 1), (2, 120, 1), (2, 61, 0)])
def test_rebuild_as_flagged_launches_or_if_node_same_bits(B, W, ci, steps, resort):
    """Inside the step graphs the rebuild is either two launches that return at once while the step's flag
    is 0 (cooperative cell list + builder; the default at these sizes) or the body of an IF node
    ("rebuild_flagged" = 0): same bits, same rebuild history, same lists -- for the fused 3-D LJ loop, the 2-D
    soft-sphere loop, and without the physical re-sort; and for one of the update rules."""
    w = W.config(ci)
    out = []
    for flagged in (1, 0):
        S = B.System(w, resort=resort)
        B.md_set_option(S.sys, "rebuild_flagged", flagged)
        assert B.md_get_option(S.sys, "rebuild_flagged") == flagged
        S.build(); S.compute_force(); S.step(steps)
        torch.cuda.synchronize()
        out.append((S.pos.clone(), S.vel.clone(), S.force.clone(), S.id.clone(), S.stats.clone(), S.nbr_rows().clone(),
                    S.nbr_count.clone()))
        S.close()
    for x, y in zip(out[0], out[1]):
        assert torch.equal(x, y)
    assert int(out[0][4][0]) == steps and int(out[0][4][1]) >= 3
    if w.dim == 3 and resort:
        # the fused loop with the flagged rebuild beside the force kernel ("step_fork", the default) or in front
        # of it, as graphs and as plain launches on two streams, over step counts that are and are not multiples
        # of the graph's nine steps and of the three flag words: same bits
        for nst in (steps, 9, 10, 13):
            res = []
            for fork, graph in ((1, 1), (0, 1), (1, 0)):
                S = B.System(w)
                B.md_set_option(S.sys, "step_fork", fork)
                B.md_set_option(S.sys, "use_graph", graph)
                S.build(); S.compute_force(); S.step(nst); S.step(nst)
                torch.cuda.synchronize()
                res.append((S.pos.clone(), S.vel.clone(), S.force.clone(), S.id.clone(), S.stats.clone(),
                            S.nbr_rows().clone(), S.nbr_count.clone()))
                S.close()
            for o in res[1:]:
                for x, y in zip(res[0], o):
                    assert torch.equal(x, y)
            if nst == steps:
                assert int(res[0][4][0]) == nst and int(res[0][4][1]) >= 2      # stats are per call
    if ci == 0:                                   # a rule other than NVE: Langevin through its own graphs
        res = []
        for flagged in (1, 0):
            S = B.System(w)
            B.md_set_option(S.sys, "rebuild_flagged", flagged)
            S.build(); S.compute_force()
            B.md_langevin_step(S.sys, S.pot, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, w.dt, w.mass, 1.0, 1.0,
                               7, 0, 50, S.stats)
            torch.cuda.synchronize()
            res.append((S.pos.clone(), S.vel.clone(), S.id.clone(), S.stats.clone()))
            S.close()
        for x, y in zip(res[0], res[1]):
            assert torch.equal(x, y)
        assert int(res[0][3][1]) >= 2


def test_nve_run_host_context_reuse(B, W):
    """md_nve_run_host keeps its device context between calls: a second call with the same
    (cfg, n) must give the same bits, a call with another system must replace the context, and
    going back must again give the first result."""
    w0, w2 = W.config(0), W.lj_fcc(0, 7, seed=7)

    def run(w):
        cfg = B.make_config(w.dim, w.box, w.r_cut, w.skin, w.capacity, w.resort)
        pot = B.make_potential(w.kind, w.epsilon, w.sigma, w.r_cut, w.shift)
        pos = w.pos.copy(); vel = w.vel.copy(); force = np.zeros_like(pos)
        stats = np.zeros(4, np.int32)
        E = B.md_nve_run_host(cfg, pot, pos, vel, force, w.dt, w.mass, 30, stats)
        return pos, vel, force, E, stats

    a = run(w0); b = run(w0); c = run(w2); d = run(w0)
    for x, y in ((a, b), (a, d)):
        assert all(np.array_equal(p, q) for p, q in zip(x[:3], y[:3])) and np.array_equal(x[4], y[4])
        assert abs(x[3] - y[3]) <= 1e-12 * abs(x[3])
    assert c[0].shape[0] == w2.n and np.isfinite(c[0]).all() and c[4][0] == 30
    B.md_nve_run_host_release()
    B.md_nve_run_host_release()          # idempotent
    e = run(w0)
    assert all(np.array_equal(p, q) for p, q in zip(a[:3], e[:3]))


def snapshot_checks(B, orc, W, w, steps, method=1):
    """State-wise parity along a trajectory (SURVEY §8c last row of P): run on the GPU, then
    hand the GPU snapshot to the oracle and compare list / force / energy at that state; plus
    momentum and energy invariants."""
    S = B.System(w)
    S.build(); S.compute_force()
    E_pot0 = float(S.energy.cpu()[0])
    ke0 = 0.5 * w.mass * float((S.vel[:, :3].double() ** 2).sum())
    mom0 = S.vel[:, :3].double().sum(0).cpu().numpy()
    S.step(steps)
    S.compute_force()
    torch.cuda.synchronize()
    stats = S.stats.cpu().numpy()
    assert stats[0] == steps and stats[2] == -1
    E_pot1 = float(S.energy.cpu()[0])
    ke1 = 0.5 * w.mass * float((S.vel[:, :3].double() ** 2).sum())
    mom1 = S.vel[:, :3].double().sum(0).cpu().numpy()
    assert np.abs(mom1 - mom0).max() <= 2e-5 * np.sqrt(w.n) * max(1.0, w.temperature) + 1e-3
    # velocity Verlet at these time steps: the oracle's own fp64 runs drift by 6.4e-5 (config 0, 100 steps),
    # 5.0e-5 / 2.5e-4 (N = 32k, T = 1 / T = 2) and 2.6e-5 (config 1) of |E|;
    # the bound is twice the largest of them for LJ and 1e-4 for the soft disks
    assert abs((ke1 + E_pot1) - (ke0 + E_pot0)) <= (1e-4 if w.kind == 1 else 5e-4) * abs(ke0 + E_pot0)
    # Newton's third law on the GPU forces (P5)
    F = S.force[:, :3].double()
    assert F.sum(0).abs().max().item() <= 1e-5 * F.norm(dim=1).mean().item() * np.sqrt(w.n)
    # snapshot -> oracle
    snap = dataclasses.replace(w, pos=unpermute(S, S.pos))
    diam = snap.pos[:, 3].astype(np.float64)
    idx_o, cnt_o, st_o = orc.neighbor_list(snap.pos, w.box, w.dim, w.r_cut, w.skin, w.capacity,
                                           predicate=1, method=1)
    f_o, e_o, E_o = orc.energy_force(snap.pos, diam, w.box, w.dim, w.kind, w.epsilon, w.sigma,
                                     float(np.float32(w.r_cut)), w.shift, idx_o, cnt_o)
    f = unpermute(S, S.force)
    assert force_error(f, f_o) <= FORCE_TOL
    assert abs(E_pot1 - E_o) <= ENERGY_TOL * abs(E_o)
    # the list in use is still valid: it contains every pair within r_cut of the snapshot
    rows, counts = gpu_rows_in_original_order(S)
    idx_c, cnt_c, _ = orc.neighbor_list(snap.pos, w.box, w.dim, float(np.float32(w.r_cut)) * (1 - 1e-6), 0.0,
                                        w.capacity, predicate=1, method=1)
    for i in range(0, w.n, max(1, w.n // 2000)):
        need = set(idx_c[i, : cnt_c[i]].tolist())
        have = set(rows[i, : counts[i]].tolist())
        assert need <= have
    # a fresh build on the snapshot is bit-exact against the oracle's canonical list
    S2 = B.System(snap)
    S2.build()
    check_list(S2, orc, snap, method=method)
    S2.close()
    rebuilds = int(stats[1])
    S.close()
    return rebuilds


def test_config1_snapshots(B, orc, W):
    """Config 1 over its own 1000 steps (BASELINE.json)."""
    w = W.config(1)
    rebuilds = snapshot_checks(B, orc, W, w, 1000)
    assert rebuilds >= 100


def test_config2_snapshots(B, orc, W):
    """Config 2 over its own 1000 steps."""
    w = W.config(2)
    rebuilds = snapshot_checks(B, orc, W, w, 1000)
    assert 80 <= rebuilds <= 200


def test_sanitizer_workout(B, W):
    """A short pass over every hot-path kernel on configs 0 and 1 -- both builders' part counts, the fused
    and the unfused step, graph and direct launches, a ragged last tile with an un-sorted system and a list
    buffer full of garbage -- cheap enough to run under a sanitizer or against a library built with
    -DMD_CHECKED (device-side index asserts; profiles/r2_sanitizer.md).  Here it checks that fused / unfused
    and graph / direct runs agree bit for bit."""
    ref = {}
    for ci in (0, 1):
        w = W.config(ci)
        for parts in (1, 2, 4):
            for fused, graph in ((1, 1), (0, 1), (1, 0)):
                S = B.System(w)
                B.md_set_option(S.sys, "builder_parts", parts)
                B.md_set_option(S.sys, "fused", fused)
                B.md_set_option(S.sys, "use_graph", graph)
                S.build(); S.compute_force()
                B.md_needs_rebuild(S.sys, S.pos, S.flag)
                S.step(41)
                torch.cuda.synchronize()
                st = S.stats.cpu().numpy()
                assert st[0] == 41 and st[1] >= 2 and st[2] == -1
                key = (ci, parts)             # the row order, hence the rounding, depends on the part count
                state = (S.pos.clone(), S.vel.clone(), S.id.clone())
                if key in ref:
                    assert all(torch.equal(a, b) for a, b in zip(state, ref[key]))
                else:
                    ref[key] = state
                S.close()
    # ragged last tile (n % 32 != 0), no physical re-sort, the list buffer pre-filled with garbage
    w = W.lj_fcc(0, 7, seed=5)
    w = dataclasses.replace(w, n=w.n - 5, pos=w.pos[:-5].copy(), vel=w.vel[:-5].copy())
    for resort in (0, 1):
        S = B.System(w, resort=resort)
        S.nbr_idx.fill_(0x7fffffff)
        S.build(); S.compute_force(); S.step(21)
        torch.cuda.synchronize()
        assert int(S.stats[0]) == 21 and int(S.stats[2]) == -1 and torch.isfinite(S.force).all()
        S.close()


# ------------------------- SURVEY 8(f) rows and the fast path at the sizes bench.py times ----

def state_force_parity(S, orc, w, alpha=None, species=None):
    """Force / energy of the GPU's CURRENT state against the oracle's list path (equal to all pairs by
    construction) on the same positions; returns the force error in units of the tolerance."""
    S.compute_force(want_energy=True)
    torch.cuda.synchronize()
    pos = unpermute(S, S.pos)
    diam = pos[:, 3].astype(np.float64) if species is None else species
    idx64, cnt64, _ = orc.neighbor_list(pos, w.box, w.dim, w.r_cut, w.skin, w.capacity, predicate=1, method=1)
    f_o, e_o, E_o = orc.energy_force(pos, diam, w.box, w.dim, w.kind, w.epsilon, w.sigma,
                                     float(np.float32(w.r_cut)), w.shift, idx64, cnt64, alpha=alpha)
    err = force_error(unpermute(S, S.force), f_o)
    E = float(S.energy.cpu()[0])
    assert err <= FORCE_TOL, err
    assert abs(E - E_o) <= ENERGY_TOL * abs(E_o), (E, E_o)
    return err / FORCE_TOL


@pytest.mark.parametrize("kind", ["morse", "buckingham", "species", "bks"])
def test_other_potentials_at_full_size(B, orc, W, kind):
    """SURVEY 8(f)-f2 at the geometry `bench.py --next-rows` times (config 3's 256,000 positions): at
    n >= 32,768 md_create selects the TMA-streamed force kernel (threads_per_particle = 0), which the
    small-system tests of these potentials never reach.  Force / energy against the oracle's list path."""
    base = W.config(3)
    f32 = lambda a: np.asarray(a, np.float32)
    d64 = lambda a: np.asarray(a, np.float64)
    pos = base.pos.copy()
    species = None
    alpha = None
    if kind == "morse":
        w = dataclasses.replace(base, kind=W.KIND_MORSE, epsilon=float(np.float32(0.9)), sigma=float(np.float32(1.12)), alpha=5.0)
        alpha = 5.0
    elif kind == "buckingham":
        w = dataclasses.replace(base, kind=W.KIND_BUCKINGHAM, epsilon=float(np.float32(9.02e5)),
                                sigma=float(np.float32(3.454)), alpha=12.5)
        alpha = 12.5
    else:
        pos[:, 3] = (np.arange(base.n) % 5 == 0).astype(np.float32)
        species = pos[:, 3].astype(np.float64)
        w = dataclasses.replace(base, kind=W.KIND_LJ_SPECIES if kind == "species" else W.KIND_BKS, pos=pos)
    S = B.System(w)
    if kind == "species":
        eps = f32([[1.0, 1.5], [1.5, 0.5]]); sig = f32([[1.0, 0.8], [0.8, 0.88]]); rc = f32(2.5 * sig)
        B.md_set_species_lj(S.sys, eps, sig, rc)
        orc.set_species_lj(d64(eps), d64(sig), d64(rc))
    if kind == "bks":
        Am = f32(9.02e5 * np.array([[1.0, 0.7], [0.7, 0.5]])); Bm = f32(12.5 * np.array([[1.0, 1.05], [1.05, 1.1]]))
        Cm = f32(3.454 * np.array([[1.0, 0.6], [0.6, 0.3]])); q = f32([0.6, -0.6])
        B.md_set_species_bks(S.sys, Am, Bm, Cm, q, float(np.float32(0.3)), 1.0)
        orc.set_species_bks(d64(Am), d64(Bm), d64(Cm), d64(q), float(np.float32(0.3)), 1.0)
    S.build()
    # Morse and Buckingham default to the fp32 fast path with fp64 re-evaluation (as LJ does);
    # "fast32" = 0 puts them on the fp64 kernels, which species LJ and BKS always use
    state_force_parity(S, orc, w, alpha=alpha, species=species)
    B.md_set_option(S.sys, "fast32", 0)
    state_force_parity(S, orc, w, alpha=alpha, species=species)
    # and the small-system kernel variant on the same state gives the same forces to rounding
    f_stream = S.force.clone()
    B.md_set_option(S.sys, "threads_per_particle", 1)
    S.compute_force()
    torch.cuda.synchronize()
    scale = f_stream[:, :3].norm(dim=1).clamp_min(1e-3)
    assert ((S.force[:, :3] - f_stream[:, :3]).norm(dim=1) / scale).max().item() <= 2e-6
    S.close()


@pytest.mark.parametrize("rule", ["langevin", "nose_hoover", "brownian", "fire"])
def test_update_rules_at_full_size(B, orc, W, rule):
    """SURVEY 8(f)-f3 at N = 256,000: 50 steps of the rule through its graph, then the state the GPU
    holds -- forces and energy at the final positions -- against the oracle, the list in use still
    complete, momentum / temperature where the rule fixes them."""
    w = W.config(3)
    if rule == "fire":
        w = dataclasses.replace(w, vel=np.zeros_like(w.vel))
    S = B.System(w)
    S.build(); S.compute_force()
    steps = 50
    dev = S.pos.device
    if rule == "langevin":
        B.md_langevin_step(S.sys, S.pot, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, w.dt, w.mass, 1.0, 1.0,
                           7, 0, steps, S.stats)
    elif rule == "nose_hoover":
        nh = torch.zeros(2, dtype=torch.float64, device=dev)
        B.md_nose_hoover_step(S.sys, S.pot, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, w.dt, w.mass, 1.0, 0.2,
                              nh, steps, S.stats)
    elif rule == "brownian":
        B.md_brownian_step(S.sys, S.pot, S.pos, S.force, S.id, S.nbr_idx, S.nbr_count, 1e-4, 1.0, 0.8, 7, 0, steps, S.stats)
    else:
        fs = torch.zeros(4, dtype=torch.float32, device=dev)
        fp = B.md_fire_params(0.002, 0.02, 5, 1.1, 0.5, 0.1, 0.99)
        B.md_fire_minimize(S.sys, S.pot, fp, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, fs, steps, S.stats)
    torch.cuda.synchronize()
    st = S.stats.cpu().numpy()
    assert st[0] == steps and st[2] == -1
    f_rule = S.force.clone()                              # the force the rule's last step left behind
    pos = unpermute(S, S.pos)
    idx64, cnt64, _ = orc.neighbor_list(pos, w.box, 3, w.r_cut, w.skin, w.capacity, predicate=1, method=1)
    f_o, e_o, E_o = orc.energy_force(pos, None, w.box, 3, w.kind, w.epsilon, w.sigma, float(np.float32(w.r_cut)),
                                     w.shift, idx64, cnt64)
    ids = S.id.cpu().numpy().astype(np.int64)
    f = np.empty((w.n, 4), np.float32); f[ids] = f_rule.cpu().numpy()
    assert force_error(f, f_o) <= FORCE_TOL
    # the list in use still holds every pair within r_cut of this state
    rows, counts = gpu_rows_in_original_order(S)
    idx_c, cnt_c, _ = orc.neighbor_list(pos, w.box, 3, float(np.float32(w.r_cut)) * (1 - 1e-6), 0.0, w.capacity,
                                        predicate=1, method=1)
    for i in range(0, w.n, 257):
        assert set(idx_c[i, : cnt_c[i]].tolist()) <= set(rows[i, : counts[i]].tolist())
    if rule in ("langevin", "nose_hoover"):
        T = w.mass * float((S.vel[:, :3].double() ** 2).sum()) / (3 * w.n)
        assert 0.6 < T < 1.2                              # from T = 1 on the lattice, thermostat at 1
    S.close()


def test_flocking_gradients_at_65536_boids(B, orc, W):
    """SURVEY 8(f)-f4 beyond the small flocks: one forward-Euler step of 65,536 boids (a jittered lattice,
    ~24 neighbors) against the oracle's all-pairs gradients, all three terms."""
    rng = np.random.default_rng(23)
    m = 256
    n = m * m
    L = np.float32(m * 1.26 + 0.37)
    box32 = np.array([L, L, 1.0], np.float32)
    g = (np.arange(m) + 0.5) * (float(L) / m)
    pos = np.zeros((n, 4), np.float32)
    pos[:, :2] = W.into_box_f32(np.stack(np.meshgrid(g, g, indexing="ij"), -1).reshape(-1, 2)
                                + rng.normal(0, 0.15, (n, 2)), box32)
    pos[:, 3] = rng.uniform(-np.pi, np.pi, n).astype(np.float32)
    speed, dt = 0.5, 0.01
    w = custom_workload(W, pos, box32, 2, 1, 3.0, 0.5, 64)
    th0 = pos[:, 3].astype(np.float64)
    par = (1.0, 3.0, 10.0, 1.0, 0.5, 3.0, 3.0)
    S = B.System(w)
    S.build()
    B.md_flock_step(S.sys, B.md_flock_params(*par, speed), S.pos, S.id, S.nbr_idx, S.nbr_count, dt, 1, S.stats)
    torch.cuda.synchronize()
    en, gR, gth = orc.flock_energy_grad(pos, th0, box32, par)
    one = unpermute(S, S.pos)
    d = one[:, :2].astype(np.float64) - pos[:, :2]
    d -= float(L) * np.round(d / float(L))
    want = dt * (speed * np.stack([np.cos(th0), np.sin(th0)], 1) - gR)
    # positions are fp32 at L = 323: half an ulp is 1.5e-5; the bulk of the comparison is the headings
    assert np.abs(d - want).max() <= 4e-5 * max(1.0, np.abs(want).max() / dt * dt)
    gth_scale = max(1.0, np.abs(gth).max())
    assert np.abs((one[:, 3].astype(np.float64) - th0) + dt * gth).max() <= 2e-6 * gth_scale
    S.close()


FAST32_STATES = [
    ("rho 0.5, jittered lattice", dict(rho=0.5), 0, {}),
    ("rho 0.5 after 200 steps", dict(rho=0.5), 200, {}),
    ("rho 1.0, jittered lattice", dict(rho=1.0), 0, {}),
    ("rho 1.0 after 200 steps", dict(rho=1.0), 200, {}),
    ("cold crystal, jitter 0.01", dict(jitter=0.01, temperature=0.01), 0, {}),
    ("cold crystal after 200 steps", dict(jitter=0.01, temperature=0.01), 200, {}),
    ("T = 4 liquid after 200 steps", dict(temperature=4.0), 200, dict(dt=0.002)),
    ("eps 0.3, sigma 1.7", dict(rho=0.8442 / 1.7 ** 3), 0, dict(epsilon=0.3, sigma=1.7, r_cut=4.25, skin=0.51)),
    ("eps 0.3, sigma 1.7 after 200 steps", dict(rho=0.8442 / 1.7 ** 3), 200, dict(epsilon=0.3, sigma=1.7, r_cut=4.25, skin=0.51, dt=0.01)),
]


@pytest.mark.parametrize("name,gen,steps,over", FAST32_STATES, ids=[s[0] for s in FAST32_STATES])
def test_fast32_estimator_away_from_its_calibration(B, orc, W, name, gen, steps, over):
    """The fp32 fast path's guarantee was calibrated on rho = 0.8442 states; here the same
    default est_thr on states it never saw -- other densities, a cold crystal, a hot liquid, other epsilon
    and sigma -- at N = 32,000 (the streaming dispatch): force / energy at the north_star tolerances."""
    w = W.lj_fcc(2, 20, seed=77, **gen)
    w = dataclasses.replace(w, **over)
    if "sigma" in over:                                   # the jitter scales with the lattice
        pass
    S = B.System(w)
    S.build(); S.compute_force()
    if steps:
        S.step(steps)
        torch.cuda.synchronize()
        assert int(S.stats[2]) == -1
    worst = state_force_parity(S, orc, w)
    cnt = torch.zeros(8, dtype=torch.int32, device=S.pos.device)
    B.md_counters(S.sys, cnt, reset=True); S.compute_force(); B.md_counters(S.sys, cnt)
    torch.cuda.synchronize()
    print(f"fast32 [{name}]: worst error {worst:.3f} x 1e-5, re-evaluated {int(cnt[0])} of {w.n}")
    S.close()


F2_STATES = [
    ("morse alpha 3, r0 1.0, rho 0.6 after 200 steps", "morse", dict(rho=0.6), 200, dict(epsilon=0.5, sigma=1.0, alpha=3.0, dt=0.002)),
    ("morse alpha 8, r0 1.2, jittered lattice", "morse", dict(), 0, dict(epsilon=2.0, sigma=1.2, alpha=8.0)),
    ("morse alpha 5, T = 3 after 200 steps", "morse", dict(temperature=3.0), 200, dict(epsilon=0.9, sigma=1.12, alpha=5.0, dt=0.002)),
    ("buckingham B 10, rho 0.6 after 200 steps", "buckingham", dict(rho=0.6), 200, dict(epsilon=1.0e5, sigma=2.0, alpha=10.0, dt=0.002)),
    ("buckingham B 15, rho 1.0, jittered lattice", "buckingham", dict(rho=1.0), 0, dict(epsilon=1.0e7, sigma=3.454, alpha=15.0)),
    ("buckingham B 12.5, cold crystal", "buckingham", dict(jitter=0.01, temperature=0.01), 0, dict(epsilon=9.02e5, sigma=3.454, alpha=12.5)),
]


@pytest.mark.parametrize("name,kind,gen,steps,over", F2_STATES, ids=[s[0] for s in F2_STATES])
def test_fast32_of_the_other_potentials_away_from_its_calibration(B, orc, W, name, kind, gen, steps, over):
    """As the test above for the Morse and Buckingham fast paths, whose estimate terms were scaled on
    config 3's positions with the parameters of test_other_potentials_at_full_size: other stiffnesses,
    densities and temperatures, at N = 32,000."""
    w = W.lj_fcc(2, 20, seed=78, **gen)
    over = {k: (float(np.float32(v)) if k in ("epsilon", "sigma") else v) for k, v in over.items()}
    kinds = {"morse": W.KIND_MORSE, "buckingham": W.KIND_BUCKINGHAM}
    w = dataclasses.replace(w, kind=kinds[kind], **over)
    S = B.System(w)
    S.build(); S.compute_force()
    if steps:
        S.step(steps)
        torch.cuda.synchronize()
        assert int(S.stats[2]) == -1
    worst = state_force_parity(S, orc, w, alpha=over.get("alpha"))
    cnt = torch.zeros(8, dtype=torch.int32, device=S.pos.device)
    B.md_counters(S.sys, cnt, reset=True); S.compute_force(); B.md_counters(S.sys, cnt)
    torch.cuda.synchronize()
    print(f"fast32 [{name}]: worst error {worst:.3f} x 1e-5, re-evaluated {int(cnt[0])} of {w.n}")
    assert int(cnt[0]) > 0                            # the fast path is the one that ran (the cutoff band alone flags some)
    S.close()


# ---------------------------------------------- full sizes, bench launch configuration ----

@pytest.mark.parametrize("ci,steps", [(3, 100), (4, 500)])
def test_full_size_configs(B, orc, W, ci, steps):
    """Configs 3 and 4 at BASELINE.json's full sizes, in the launch configuration bench.py
    times (re-sort on, CUDA graph, default threads per particle): bit-exact list and force /
    energy parity at step 0 against the oracle's cell-binned search, then snapshot parity."""
    w = W.config(ci)
    S = B.System(w)
    S.build()
    torch.cuda.synchronize()
    check_cells(S, orc, w)
    idx_o, cnt_o = check_list(S, orc, w, method=1)
    # oracle force over its own fp64 list (equal to all pairs by construction)
    idx64, cnt64, _ = orc.neighbor_list(w.pos, w.box, 3, w.r_cut, w.skin, w.capacity, predicate=1, method=1)
    check_force(S, orc, w, idx64, cnt64)
    S.close()
    del S
    torch.cuda.empty_cache()
    rebuilds = snapshot_checks(B, orc, W, w, steps)
    assert rebuilds >= 3


def test_config3_long_run(B, orc, W):
    """2000 MD steps of config 3 (twice the config's own run, ~260 rebuilds) through the fused graph:
    energy and momentum conserved, the list in use still complete, and force / energy / a fresh list
    of the final state against the oracle."""
    rebuilds = snapshot_checks(B, orc, W, W.config(3), 2000)
    assert rebuilds >= 200




def check_ranks_against_oracle(loops, orc, w):
    """The gathered final state of a split-list run against the ORACLE (not only against the one-GPU
    path): force and energy of the assembled ranges vs the definition on the final positions, and a
    fresh list build on every rank -- each rank's rows of its own range -- vs the oracle's canonical list."""
    S0 = loops[0].S
    snap = dataclasses.replace(w, pos=unpermute(S0, S0.pos))
    diam = snap.pos[:, 3].astype(np.float64)
    idx64, cnt64, _ = orc.neighbor_list(snap.pos, w.box, w.dim, w.r_cut, w.skin, w.capacity, predicate=1, method=1)
    f_o, e_o, E_o = orc.energy_force(snap.pos, diam, w.box, w.dim, w.kind, w.epsilon, w.sigma,
                                     float(np.float32(w.r_cut)), w.shift, idx64, cnt64,
                                     alpha=float(w.alpha) if w.kind == 2 else None)
    ids = S0.id.cpu().numpy().astype(np.int64)
    f = np.zeros((w.n, 4), np.float32)
    E = 0.0
    for lp in loops:                                  # every rank contributes the forces of its own range
        b, e = lp.range
        lp.S.compute_force(want_energy=True)
        torch.cuda.synchronize()
        f[ids[b:e]] = lp.S.force[b:e].cpu().numpy()
        E += float(lp.S.energy[0])
    tol = FORCE_TOL
    assert force_error(f, f_o) <= tol
    assert abs(E - E_o) <= ENERGY_TOL * abs(E_o)
    idx_o, cnt_o, st_o = orc.neighbor_list(snap.pos, w.box, w.dim, w.r_cut, w.skin, w.capacity, predicate=0, method=1)
    for lp in loops:
        lp.S.build()
        torch.cuda.synchronize()
        b, e = lp.range
        ids2 = lp.S.id.cpu().numpy().astype(np.int64)             # the build re-sorted: same order on every rank
        rows = lp.S.nbr_rows()[b:e].cpu().numpy().astype(np.int64)
        cnt = lp.S.nbr_count[b:e].cpu().numpy()
        lut = np.concatenate([ids2, [w.n]])
        mapped = np.sort(lut[rows], axis=1)
        assert np.array_equal(cnt, cnt_o[ids2[b:e]])
        assert np.array_equal(mapped, idx_o[ids2[b:e]])

@pytest.mark.parametrize("world,m,steps", [(2, 6, 100), (3, 6, 100), (3, 7, 80), (4, 12, 60)])      # m = 7: 1372 particles, a ragged last tile
def test_split_list_ranks_equal_one_gpu(B, orc, W, world, m, steps):
    """SURVEY §8f-f1 (replicated positions, split list; decomposition.py): `world` contexts in one
    process, each owning a range of list tiles, stepped in lockstep with the all-gather replaced by a
    stack -- positions, velocities, forces and ids after `steps` steps are bit-identical to md_nve_step
    on one context, with the same number of rebuilds; each rank's list holds rows of its range only."""
    from paper_1912_04232_b200 import decomposition as D
    w = W.lj_fcc(0, m, seed=3)
    one = B.System(w)
    one.build(); one.compute_force()
    one.step(steps)
    torch.cuda.synchronize()
    loops = []
    for r in range(world):
        S = B.System(w)
        loops.append(D.RankLoop(S, r, world))
    for lp in loops:
        lp.start()
    D.run_local(loops, steps)
    D.gather_state_local(loops)
    torch.cuda.synchronize()
    assert int(one.stats[1]) >= 3
    for lp in loops:
        assert lp.rebuilds == int(one.stats[1])
        assert torch.equal(lp.S.pos, one.pos) and torch.equal(lp.S.vel, one.vel) and torch.equal(lp.S.id, one.id)
        assert torch.equal(lp.S.force[:, :3], one.force[:, :3])
        b, e = lp.range
        assert torch.equal(lp.S.nbr_count[b:e], one.nbr_count[b:e])
    # the energy of the ranges adds up to the total
    one.compute_force()
    E = 0.0
    for lp in loops:
        lp.S.compute_force(want_energy=True)
        E += float(lp.S.energy[0])
    assert abs(E - float(one.energy[0])) <= 1e-12 * abs(float(one.energy[0]))
    # a range is not steppable from inside, and only tile-aligned ranges are accepted
    with pytest.raises(B.MdError):
        loops[0].S.step(1)
    with pytest.raises(B.MdError):
        B.md_set_range(loops[0].S.sys, 16, 64)
    check_ranks_against_oracle(loops, orc, w)
    # without the physical re-sort a range of the sorted order is not a range of particles: refused
    U = B.System(w, resort=0)
    with pytest.raises(B.MdError):
        B.md_set_range(U.sys, 0, 32)
    B.md_set_range(U.sys, 0, w.n)                    # the whole system is always a valid range
    with pytest.raises(ValueError):
        D.RankLoop(U, 0, world)
    U.close()
    for lp in loops:
        lp.S.close()
    one.close()


@pytest.mark.parametrize("which", ["soft2d", "morse3d", "lj64"])
def test_split_list_ranks_other_kernels(B, orc, W, which):
    """The range offset of the generic force kernels (fp64 pair chain, 2-D, threads-per-particle variants):
    three ranks in lockstep against one context, bit for bit."""
    from paper_1912_04232_b200 import decomposition as D
    if which == "soft2d":
        w = W.soft_disks(1, 3000)
        rng = np.random.default_rng(2)
        v = np.zeros_like(w.vel); v[:, :2] = rng.normal(0, 0.05, (w.n, 2)).astype(np.float32)
        w = dataclasses.replace(w, vel=v, dt=0.02)
        opts = {}
    elif which == "morse3d":
        w = dataclasses.replace(W.lj_fcc(0, 7, seed=5), kind=W.KIND_MORSE, sigma=1.12, alpha=5.0)
        opts = {"threads_per_particle": 2}
    else:
        w = W.lj_fcc(0, 7, seed=5)
        opts = {"fast32": 0, "threads_per_particle": 0}
    steps, world = 80, 3

    def make():
        S = B.System(w)
        for k, val in opts.items():
            B.md_set_option(S.sys, k, val)
        return S

    one = make()
    one.build(); one.compute_force()
    one.step(steps)
    torch.cuda.synchronize()
    loops = [D.RankLoop(make(), r, world) for r in range(world)]
    for lp in loops:
        lp.start()
    D.run_local(loops, steps)
    D.gather_state_local(loops)
    torch.cuda.synchronize()
    for lp in loops:
        assert lp.rebuilds == int(one.stats[1])
        assert torch.equal(lp.S.pos, one.pos) and torch.equal(lp.S.vel, one.vel) and torch.equal(lp.S.id, one.id)
        assert torch.equal(lp.S.force[:, :3], one.force[:, :3])
    check_ranks_against_oracle(loops, orc, w)
    for lp in loops:
        lp.S.close()
    one.close()
