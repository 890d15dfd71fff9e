"""Pins for the fp64 CPU oracle (oracle/md_oracle.c) -- CPU only.

Each test ties one oracle function to something OTHER than itself: a value
from tests/golden (cited), a textbook closed form, an invariant, a library
routine for a special case, or brute force on tiny inputs (SURVEY.md §8c "P").
A dropped term, wrong sign, wrong index or transposed operand in the oracle
fails at least one of them.
"""
import math

import numpy as np
import pytest
from scipy.spatial import cKDTree

from conftest import golden

LJ, SOFT = 0, 1
RHO = 0.8442


def fcc64(m):
    """fp64 perfect FCC lattice at rho = 0.8442 and its fp64 box."""
    from paper_1912_04232_b200.workloads import fcc_sites
    n = 4 * m ** 3
    L = (n / RHO) ** (1.0 / 3.0)
    return fcc_sites(m, L / m), np.array([L, L, L])


def rows_as_sets(idx, cnt, n):
    return [set(int(j) for j in idx[i, : min(cnt[i], idx.shape[1])] if j < n) for i in range(len(cnt))]


# ---------------------------------------------------------------- P2: FCC --

def test_fcc_shell_counts_and_lattice_sum(orc):
    g = golden("fcc_shells.txt")
    pos, box = fcc64(5)                        # L = 8.4 > 2 * 2.8
    n = pos.shape[0]
    a = box[0] / 5
    assert abs(a - g["lattice_constant"]) < 1e-9
    for R, key in [(2.8, "neighbors_within_2p8"), (2.7, "neighbors_within_2p7"),
                   (2.5, "neighbors_within_2p5")]:
        for method in (0, 1):
            idx, cnt, st = orc.neighbor_list(pos, box, 3, R, 0.0, 128, predicate=1, method=method)
            assert cnt.min() == cnt.max() == int(g[key]), (R, method)
            assert st[0] == 0 and st[1] == int(g[key])
    # independent lattice sum from the textbook FCC shells (multiplicity, k)
    shells = [(12, 1), (6, 2), (24, 3), (12, 4), (24, 5), (8, 6)]
    for (mult, k) in shells:
        assert abs(a * math.sqrt(k / 2) - g[f"shell_{k}_r"]) < 1e-6
    u = lambda r: 4.0 * (r ** -12 - r ** -6)
    uc = u(2.5)
    assert abs(uc - g["lj_u_cut_2p5"]) < 1e-12
    rs = [(mult, a * math.sqrt(k / 2)) for (mult, k) in shells if a * math.sqrt(k / 2) < 2.5]
    pe_unshifted = 0.5 * sum(mult * u(r) for mult, r in rs)
    pe_shifted = 0.5 * sum(mult * (u(r) - uc) for mult, r in rs)
    assert abs(pe_unshifted - g["pe_per_particle_unshifted"]) < 1e-9
    assert abs(pe_shifted - g["pe_per_particle_shifted"]) < 1e-9
    for shift, want in [(1, g["pe_per_particle_shifted"]), (0, g["pe_per_particle_unshifted"])]:
        f, e_i, E = orc.energy_force(pos, None, box, 3, LJ, 1.0, 1.0, 2.5, shift)
        assert abs(E / n - want) < 1e-10
        assert np.allclose(e_i, want, atol=1e-10)          # every site equivalent
        assert np.abs(f).max() < 1e-11                      # symmetry: F_i = 0
    # same over the list (smap.neighbors form)
    idx, cnt, st = orc.neighbor_list(pos, box, 3, 2.5, 0.3, 128, predicate=1, method=1)
    f, e_i, E = orc.energy_force(pos, None, box, 3, LJ, 1.0, 1.0, 2.5, 1, idx, cnt)
    assert abs(E / n - g["pe_per_particle_shifted"]) < 1e-10


# ------------------------------------------------- P3: two-body closed forms --

def two_body(r, axis=0, dim=3, box=20.0, diam=(1.0, 1.0), origin=(3.0, 4.0, 5.0)):
    pos = np.zeros((2, 3))
    pos[0, :dim] = origin[:dim]
    pos[1, :dim] = origin[:dim]
    pos[1, axis] += r
    return pos, np.array([box, box, box]), np.array(diam, dtype=np.float64)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_lj_two_body(orc, axis):
    eps, sig, rc = 1.7, 0.9, 2.5 * 0.9
    rmin = 2 ** (1 / 6) * sig
    # u(sigma) = 0 unshifted; u(rmin) = -eps; F(rmin) = 0
    pos, box, _ = two_body(sig, axis)
    f, e_i, E = orc.energy_force(pos, None, box, 3, LJ, eps, sig, rc, 0)
    assert abs(E) < 1e-12
    # at r = sigma the force is repulsive with magnitude 24 eps / sigma
    want = np.zeros(3); want[axis] = -24 * eps / sig      # particle 0 pushed to -axis
    assert np.allclose(f[0], want, rtol=1e-12) and np.allclose(f[1], -want, rtol=1e-12)
    pos, box, _ = two_body(rmin, axis)
    f, e_i, E = orc.energy_force(pos, None, box, 3, LJ, eps, sig, rc, 0)
    assert abs(E + eps) < 1e-12 and np.abs(f).max() < 1e-12
    assert np.allclose(e_i, [-eps / 2, -eps / 2])         # U = 1/2 sum_{i != j}: half each
    # general r: closed form, attractive beyond rmin (sign check)
    r = 1.5 * sig
    u = 4 * eps * ((sig / r) ** 12 - (sig / r) ** 6)
    du = 4 * eps * (-12 * sig ** 12 / r ** 13 + 6 * sig ** 6 / r ** 7)
    uc = 4 * eps * ((sig / rc) ** 12 - (sig / rc) ** 6)
    pos, box, _ = two_body(r, axis)
    f, e_i, E0 = orc.energy_force(pos, None, box, 3, LJ, eps, sig, rc, 0)
    _, _, E1 = orc.energy_force(pos, None, box, 3, LJ, eps, sig, rc, 1)
    assert abs(E0 - u) < 1e-13 and abs(E1 - (u - uc)) < 1e-13
    # F_0 = -dU/dr_0; r = x_1 - x_0 so dU/dx_0 = -u'(r)  =>  F_0 = +u'(r) e_axis
    assert abs(f[0, axis] - du) < 1e-12 and abs(f[1, axis] + du) < 1e-12
    assert du > 0 and f[0, axis] > 0                       # attraction pulls 0 toward 1
    # continuity at the cutoff when shifted; zero beyond
    pos, box, _ = two_body(rc * (1 - 1e-9), axis)
    _, _, E = orc.energy_force(pos, None, box, 3, LJ, eps, sig, rc, 1)
    assert abs(E) < 1e-8
    pos, box, _ = two_body(rc * (1 + 1e-9), axis)
    f, _, E = orc.energy_force(pos, None, box, 3, LJ, eps, sig, rc, 1)
    assert E == 0.0 and np.abs(f).max() == 0.0
    _, _, E = orc.energy_force(pos, None, box, 3, LJ, eps, sig, rc, 0)
    assert E == 0.0


@pytest.mark.parametrize("axis", [0, 2])
def test_morse_two_body(orc, axis):
    """Morse [75], u = D (1 - exp(-a (r - r0)))^2 - D: closed forms at r0, at
    r0 + ln(2)/a (where exp(..) = 1/2), on the repulsive side, and the shifted cutoff."""
    MORSE = 2
    D, r0, a, rc = 1.7, 1.1, 4.0, 2.6
    pos, box, _ = two_body(r0, axis)
    f, e_i, E = orc.energy_force(pos, None, box, 3, MORSE, D, r0, rc, 0, alpha=a)
    assert abs(E + D) < 1e-12 and np.abs(f).max() < 1e-12 and np.allclose(e_i, [-D / 2, -D / 2])
    r = r0 + np.log(2.0) / a
    pos, box, _ = two_body(r, axis)
    f, _, E = orc.energy_force(pos, None, box, 3, MORSE, D, r0, rc, 0, alpha=a)
    assert abs(E - (D * 0.25 - D)) < 1e-12
    du = 2 * D * a * 0.5 * 0.5                              # u'(r) > 0: attraction
    assert abs(f[0, axis] - du) < 1e-12 and abs(f[1, axis] + du) < 1e-12
    r = 0.8 * r0
    x = np.exp(-a * (r - r0))
    pos, box, _ = two_body(r, axis)
    f, _, E0 = orc.energy_force(pos, None, box, 3, MORSE, D, r0, rc, 0, alpha=a)
    _, _, E1 = orc.energy_force(pos, None, box, 3, MORSE, D, r0, rc, 1, alpha=a)
    uc = D * (1 - np.exp(-a * (rc - r0))) ** 2 - D
    assert abs(E0 - (D * (1 - x) ** 2 - D)) < 1e-12 and abs(E1 - (E0 - uc)) < 1e-12
    assert f[0, axis] < 0 and abs(f[0, axis] - 2 * D * a * x * (1 - x)) < 1e-10   # repulsion
    pos, box, _ = two_body(rc * (1 - 1e-9), axis)
    assert abs(orc.energy_force(pos, None, box, 3, MORSE, D, r0, rc, 1, alpha=a)[2]) < 1e-7
    pos, box, _ = two_body(rc * (1 + 1e-9), axis)
    f, _, E = orc.energy_force(pos, None, box, 3, MORSE, D, r0, rc, 1, alpha=a)
    assert E == 0.0 and np.abs(f).max() == 0.0


def test_morse_gradient_and_newton(orc, W):
    """Morse forces are -grad E (central differences) and sum to zero."""
    MORSE = 2
    w = W.lj_fcc(0, 3, seed=12)
    pos, box = w.pos[:, :3].astype(np.float64), w.box.astype(np.float64)
    args = (MORSE, 1.0, 1.12, 2.5, 1)
    f, _, _ = orc.energy_force(pos, None, box, 3, *args, alpha=5.0)
    assert np.abs(f.sum(0)).max() < 1e-10 * np.abs(f).sum()
    rng = np.random.default_rng(3)
    h, worst = 1e-5, 0.0
    for i in rng.choice(pos.shape[0], 8, replace=False):
        for q in range(3):
            pp = pos.copy(); pp[i, q] += h
            pm = pos.copy(); pm[i, q] -= h
            fd = -(orc.energy_force(pp, None, box, 3, *args, alpha=5.0)[2]
                   - orc.energy_force(pm, None, box, 3, *args, alpha=5.0)[2]) / (2 * h)
            worst = max(worst, abs(fd - f[i, q]) / max(1.0, np.abs(f[i]).max()))
    assert worst < 1e-6, worst


@pytest.mark.parametrize("dim", [2, 3])
def test_soft_two_body(orc, dim):
    eps = 1.3
    # equal disks, r = d/2: u = eps/8, |F| = eps/(2d)
    d = 1.4
    pos, box, diam = two_body(d / 2, axis=1, dim=dim, diam=(d, d))
    f, e_i, E = orc.energy_force(pos, diam, box, dim, SOFT, eps, 1.0, 1.4, 0)
    assert abs(E - eps / 8) < 1e-14
    assert abs(np.linalg.norm(f[0]) - eps / (2 * d)) < 1e-14
    assert f[0, 1] < 0 < f[1, 1]                           # repulsive
    # mixed pair: d_ij = (1.0 + 1.4)/2 = 1.2
    pos, box, diam = two_body(1.19, axis=0, dim=dim, diam=(1.0, 1.4))
    _, _, E = orc.energy_force(pos, diam, box, dim, SOFT, eps, 1.0, 1.4, 0)
    assert abs(E - 0.5 * eps * (1 - 1.19 / 1.2) ** 2) < 1e-15
    pos, box, diam = two_body(1.2000001, axis=0, dim=dim, diam=(1.0, 1.4))
    f, _, E = orc.energy_force(pos, diam, box, dim, SOFT, eps, 1.0, 1.4, 0)
    assert E == 0.0 and np.abs(f).max() == 0.0
    # r = 0: energy eps/2, zero force
    pos, box, diam = two_body(0.0, axis=0, dim=dim, diam=(1.0, 1.0))
    f, _, E = orc.energy_force(pos, diam, box, dim, SOFT, eps, 1.0, 1.4, 0)
    assert abs(E - eps / 2) < 1e-15 and np.abs(f).max() == 0.0


def test_two_body_across_periodic_boundary(orc):
    """Nearest image: a pair straddling x = 0 / x = L."""
    L = 12.0
    pos = np.array([[0.3, 5.0, 5.0], [L - 0.9, 5.0, 5.0]])   # separation 1.2 through the wall
    box = np.array([L, L, L])
    f, _, E = orc.energy_force(pos, None, box, 3, LJ, 1.0, 1.0, 2.5, 0)
    r = 1.2
    assert abs(E - 4 * (r ** -12 - r ** -6)) < 1e-13
    du = 4 * (-12 / r ** 13 + 6 / r ** 7)                  # > 0: attraction
    # particle 0 is at +1.2 from particle 1's image => pulled toward -x
    assert abs(f[0, 0] + du) < 1e-12 and abs(f[1, 0] - du) < 1e-12
    idx, cnt, _ = orc.neighbor_list(pos, box, 3, 2.5, 0.3, 8, predicate=0, method=0)
    assert list(cnt) == [1, 1] and idx[0, 0] == 1 and idx[1, 0] == 0


# -------------------------------------------------- P4: finite differences --

@pytest.mark.parametrize("kind,dim", [(LJ, 3), (SOFT, 2), (SOFT, 3), (LJ, 2)])
def test_force_is_minus_gradient(orc, W, kind, dim):
    """force = -grad U by central differences of the oracle's E."""
    rng = np.random.default_rng(5)
    if kind == LJ:
        # jittered lattice so that no pair sits on the repulsive wall
        m = 3
        if dim == 3:
            w = W.lj_fcc(0, m, seed=11)
            pos, box = w.pos[:, :3].astype(np.float64), w.box.astype(np.float64)
        else:
            g = np.arange(8.0)
            pos = np.zeros((64, 3))
            pos[:, :2] = np.stack(np.meshgrid(g, g, indexing="ij"), -1).reshape(-1, 2) * 1.15
            pos[:, :2] += rng.normal(0, 0.05, (64, 2))
            box = np.array([8 * 1.15, 8 * 1.15, 1.0])
        diam = None
        args = (kind, 1.0, 1.0, 2.5, 1)
    else:
        p4, box32 = W.random_box(3, 200, dim, [9.0] * dim, diam=(1.0, 1.4))
        pos, box, diam = p4[:, :3].astype(np.float64), box32.astype(np.float64), p4[:, 3].astype(np.float64)
        args = (kind, 1.0, 1.0, 1.4, 0)
    f, _, _ = orc.energy_force(pos, diam, box, dim, *args)
    h = 1e-5
    worst = 0.0
    for i in rng.choice(pos.shape[0], 12, replace=False):
        for q in range(dim):
            pp = pos.copy(); pp[i, q] += h
            pm = pos.copy(); pm[i, q] -= h
            Ep = orc.energy_force(pp, diam, box, dim, *args)[2]
            Em = orc.energy_force(pm, diam, box, dim, *args)[2]
            fd = -(Ep - Em) / (2 * h)
            worst = max(worst, abs(fd - f[i, q]) / max(1.0, np.abs(f[i]).max()))
    assert worst < 1e-6, worst
    if dim == 2:
        assert np.abs(f[:, 2]).max() == 0.0


# ------------------------------------------- P5/P6: Newton 3, translations --

def test_newton_third_law_and_translation_invariance(orc, W):
    for w in (W.config(0), W.soft_disks(1, 2048)):
        pos = w.pos[:, :3].astype(np.float64); box = w.box.astype(np.float64)
        diam = w.pos[:, 3].astype(np.float64)
        args = (w.dim, w.kind, w.epsilon, w.sigma, w.r_cut, w.shift)
        f, e_i, E = orc.energy_force(pos, diam, box, *args)
        assert np.abs(f.sum(0)).max() <= 1e-10 * np.linalg.norm(f, axis=1).sum()
        t = np.array([0.37, -11.3, 4.21 if w.dim == 3 else 0.0])
        pos_t = np.mod(pos + t, box)
        if w.dim == 2:
            pos_t[:, 2] = 0.0
        f2, e2, E2 = orc.energy_force(pos_t, diam, box, *args)
        assert abs(E2 - E) <= 1e-10 * abs(E)
        assert np.abs(f2 - f).max() <= 1e-9 * np.abs(f).max()
        # neighbor sets under the fp64 predicate are translation invariant
        a = orc.neighbor_list(pos, box, w.dim, w.r_cut, w.skin, w.capacity, predicate=1, method=1)
        b = orc.neighbor_list(pos_t, box, w.dim, w.r_cut, w.skin, w.capacity, predicate=1, method=1)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
        # the list is symmetric: j in S_i <=> i in S_j  (full list)
        sets = rows_as_sets(a[0], a[1], w.n)
        for i in range(0, w.n, 37):
            for j in sets[i]:
                assert i in sets[j]
        # list-based energy/force == all-pairs definition (PAPER.md:L78 vs L80)
        f3, e3, E3 = orc.energy_force(pos, diam, box, *args, a[0], a[1])
        assert abs(E3 - E) <= 1e-12 * abs(E) and np.abs(f3 - f).max() <= 1e-11 * np.abs(f).max()


# -------------------------------------------------- P1: neighbor sets -------

def edge_case_positions(W, seed, n, dim, box):
    """Uniform random + particles on cell faces, at 0 and just below L."""
    pos, box32 = W.random_box(seed, n, dim, box)
    R = np.float32(np.float32(1.0) + np.float32(0.25))
    for k in range(dim):
        L = box32[k]
        nk = int(math.floor(float(L) / float(R)))
        below = np.nextafter(L, np.float32(0.0), dtype=np.float32)
        specials = [np.float32(0.0), below]
        for c in range(1, nk):
            face = np.float32(c * float(L) / nk)
            specials += [face, np.nextafter(face, np.float32(0), dtype=np.float32),
                         np.nextafter(face, np.float32(1e9), dtype=np.float32)]
        for s, x in enumerate(specials):
            pos[(7 * s + 3 * k) % n, k] = x
    return pos, box32


@pytest.mark.parametrize("dim,box", [(3, [3.9, 5.2, 6.4]), (2, [3.8, 6.3]), (3, [5.01, 5.01, 5.01]),
                                     (2, [13.0, 4.0]), (3, [2.6, 3.0, 4.4])])
def test_neighbor_brute_vs_cells_vs_kdtree(orc, W, dim, box):
    n = 500 if dim == 3 else 300
    pos, box32 = edge_case_positions(W, 17 + dim, n, dim, box)
    r_cut, skin, cap = 1.0, 0.25, 192
    for predicate in (0, 1):
        a = orc.neighbor_list(pos, box32, dim, r_cut, skin, cap, predicate=predicate, method=0)
        b = orc.neighbor_list(pos, box32, dim, r_cut, skin, cap, predicate=predicate, method=1)
        assert a[2][0] == 0
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
        # rows ascending, padded with n
        for i in range(n):
            row = a[0][i]
            assert np.all(np.diff(row[: a[1][i]]) > 0) and np.all(row[a[1][i]:] == n)
    # library pin: scipy's periodic kd-tree, fp64 ball query
    p64 = pos[:, :dim].astype(np.float64)
    R = float(np.float32(np.float32(r_cut) + np.float32(skin)))
    tree = cKDTree(p64, boxsize=box32[:dim].astype(np.float64))
    pairs = tree.query_pairs(R, output_type="ndarray")
    want = [set() for _ in range(n)]
    for i, j in pairs:
        want[i].add(int(j)); want[j].add(int(i))
    got = rows_as_sets(*orc.neighbor_list(pos, box32, dim, r_cut, skin, cap, predicate=1, method=0)[:2], n)
    # kd-tree uses <=; a pair at exactly R would differ -- none here
    assert got == want
    # canonical fp32 predicate differs from fp64 only inside a 4e-6 R band (P11)
    nd, band, closest = orc.predicate_band(pos, box32, dim, r_cut, skin, method=0)
    assert band < 4e-6
    got32 = rows_as_sets(*orc.neighbor_list(pos, box32, dim, r_cut, skin, cap, predicate=0, method=0)[:2], n)
    ndiff = sum(len(x ^ y) for x, y in zip(got, got32))
    assert ndiff == nd


def test_canonical_predicate_by_hand(orc):
    """SURVEY §8c-A2/A3 retyped in NumPy fp32 on a tiny system (brute force)."""
    rng = np.random.default_rng(3)
    n, L = 60, np.float32(6.0)
    x = (rng.uniform(0, 1, (n, 3)) * 6.0).astype(np.float32)
    x[0] = [0.0, 0.0, 0.0]; x[1] = [np.nextafter(L, np.float32(0)), 0.1, 5.9]
    r_cut, skin = np.float32(1.5), np.float32(0.3)
    R = np.float32(r_cut + skin); R2 = np.float32(R * R); h = np.float32(L / np.float32(2))
    want = []
    for i in range(n):
        s = []
        for j in range(n):
            if i == j:
                continue
            d = []
            for k in range(3):
                a, b = x[i, k], x[j, k]
                dd = np.float32(a - b)
                if dd > h:
                    dd = np.float32(np.float32(a - L) - b)
                elif dd < -h:
                    dd = np.float32(a - np.float32(b - L))
                d.append(dd)
            r2 = np.float32(d[0] * d[0])
            r2 = np.float32(np.float64(d[1]) * np.float64(d[1]) + np.float64(r2))   # fmaf: one rounding
            r2 = np.float32(np.float64(d[2]) * np.float64(d[2]) + np.float64(r2))
            if r2 < R2:
                s.append(j)
        want.append(s)
    idx, cnt, st = orc.neighbor_list(x, np.array([L, L, L]), 3, 1.5, 0.3, 64, predicate=0, method=0)
    for i in range(n):
        assert list(idx[i, : cnt[i]]) == want[i]
    assert st[1] == max(len(s) for s in want)


def test_overflow_convention(orc, W):
    """P10: capacity 64 on config 0 overflows (static shapes)."""
    w = W.config(0)
    idx, cnt, st = orc.neighbor_list(w.pos, w.box, 3, w.r_cut, w.skin, 64)
    assert st[0] == 1 and st[1] == cnt.max() and 64 < st[1] < 128
    idx2, cnt2, st2 = orc.neighbor_list(w.pos, w.box, 3, w.r_cut, w.skin, 128)
    assert st2[0] == 0 and st2[1] == st[1] and np.array_equal(cnt, cnt2)
    assert 70 <= cnt2.min() and cnt2.max() <= 90 and abs(cnt2.mean() - 77.9) < 0.3


def test_predicate_band_on_configs(orc, W):
    """P11: fp32 vs fp64 predicate on the configs' initial states."""
    for w in (W.config(0), W.config(2)):
        nd, band, closest = orc.predicate_band(w.pos, w.box, w.dim, w.r_cut, w.skin, method=1)
        assert band < 4e-6
        assert nd <= 2


# ------------------------------------------------------- O2: cell list ------

def test_cell_list(orc, W):
    pos, box32 = edge_case_positions(W, 5, 400, 3, [3.9, 5.2, 6.4])
    ncell, cell_of, cell_start, members = orc.cell_list(pos, box32, 3, 1.0, 0.25)
    assert list(ncell) == [3, 4, 5]
    cells = 60
    assert cell_start[0] == 0 and cell_start[cells] == 400 and np.all(np.diff(cell_start) >= 0)
    assert sorted(members.tolist()) == list(range(400))
    for c in range(cells):
        seg = members[cell_start[c]: cell_start[c + 1]]
        assert np.all(cell_of[seg] == c) and np.all(np.diff(seg) > 0)
    # geometric meaning: the particle lies inside its cell (up to one fp32 ulp)
    side = box32.astype(np.float64) / ncell
    cx = cell_of % 3; cy = (cell_of // 3) % 4; cz = cell_of // 12
    for k, ck in enumerate((cx, cy, cz)):
        x = pos[:, k].astype(np.float64)
        assert np.all(x >= ck * side[k] - 1e-6) and np.all(x <= (ck + 1) * side[k] + 1e-6)
    # hand cases: x = 0 -> cell 0; largest float below L -> last cell
    p = np.zeros((2, 4), dtype=np.float32)
    p[1, :3] = np.nextafter(box32, np.float32(0), dtype=np.float32)
    _, cof, _, _ = orc.cell_list(p, box32, 3, 1.0, 0.25)
    assert cof[0] == 0 and cof[1] == cells - 1
    # 2-D: linear index cy*nx + cx
    p2, b2 = W.random_box(9, 100, 2, [13.0, 4.0])
    nc2, cof2, cs2, mem2 = orc.cell_list(p2, b2, 2, 1.0, 0.25)
    assert list(nc2) == [10, 3, 1]
    want = np.minimum((p2[:, 1] * np.float32(3 / 4.0)).astype(np.int32), 2) * 10 + \
        np.minimum((p2[:, 0] * (np.float32(10) / np.float32(13.0))).astype(np.int32), 9)
    assert np.array_equal(cof2, want)


# --------------------------------------------------- P9: rebuild test -------

def test_needs_rebuild_constructed(orc, W):
    w = W.config(0)
    ref = w.pos.copy()
    half = w.skin / 2
    u = np.array([1.0, 2.0, -2.0]) / 3.0
    for scale, want in [(1 - 1e-3, 0), (1 + 1e-3, 1)]:
        pos = ref.astype(np.float64).copy()
        pos[100, :3] = np.mod(pos[100, :3] + u * half * scale, w.box)
        flag, m = orc.needs_rebuild(pos, ref, w.box, 3, w.skin)
        assert flag == want and abs(math.sqrt(m) - half * scale) < 1e-9
    # crossing the periodic boundary by 0.01 is a 0.01 displacement, not ~L
    ref2 = ref.astype(np.float64).copy(); ref2[5, 0] = 0.004
    pos2 = ref2.copy(); pos2[5, 0] = float(w.box[0]) - 0.006
    flag, m = orc.needs_rebuild(pos2, ref2, w.box, 3, w.skin)
    assert flag == 0 and abs(math.sqrt(m) - 0.01) < 1e-6
    # 2-D ignores z
    p = np.zeros((4, 3)); r = np.zeros((4, 3)); r[:, 2] = 5.0
    assert orc.needs_rebuild(p, r, np.array([10.0, 10.0, 1.0]), 2, 0.1)[0] == 0


# --------------------------------------------------- P7/P8: integrator ------

def test_nve_invariants_config0(orc, W):
    w = W.config(0)
    box = w.box.astype(np.float64)
    args = (None, box, 3, LJ, 1.0, 1.0, 2.5, 1)
    f0, _, E0 = orc.energy_force(w.pos, None, box, 3, LJ, 1.0, 1.0, 2.5, 1)
    p, v, f, en, st = orc.nve_run(w.pos, w.vel, f0, *args, 0.005, 1.0, 100)
    tot = en.sum(1)
    drift = np.abs(tot / tot[0] - 1).max()
    assert drift < 2e-4                                   # symplectic: bounded, small
    assert abs(en[0, 1] - E0) < 1e-9
    # temperature bookkeeping of the generator: KE = 3(N-1)/2 T
    assert abs(en[0, 0] - 1.5 * (w.n - 1)) < 1e-3 * w.n
    # total momentum conserved (Newton 3)
    mom0 = w.vel[:, :3].astype(np.float64).sum(0)
    assert np.abs(v.sum(0) - mom0).max() < 1e-10
    # second order: halving dt shrinks the energy excursion ~4x
    p2, v2, f2, en2, _ = orc.nve_run(w.pos, w.vel, f0, *args, 0.0025, 1.0, 200)
    tot2 = en2.sum(1)
    ratio = drift / np.abs(tot2 / tot2[0] - 1).max()
    assert 3.0 < ratio < 5.5, ratio
    # time reversal: negate v, run back, recover the start
    pb, vb, fb, _, _ = orc.nve_run(p, -v, f, *args, 0.005, 1.0, 100, want_energies=False)
    d = pb - w.pos[:, :3].astype(np.float64)
    d -= box * np.round(d / box)
    assert np.abs(d).max() < 1e-8
    assert np.abs(vb + w.vel[:, :3].astype(np.float64)).max() < 1e-8
    # list-based loop with half-skin rebuilds gives the same trajectory
    # (a valid list changes nothing) and does rebuild
    pl, vl, fl, enl, stl = orc.nve_run(w.pos, w.vel, f0, *args, 0.005, 1.0, 100, use_list=1,
                                       skin=0.3, capacity=128)
    assert np.abs(pl - p).max() < 1e-10 and 5 <= stl[0] <= 20 and stl[1] == 0
    # positions stay in [0, L)
    assert p.min() >= 0 and np.all(p < box)


def test_velocity_verlet_harmonic_oscillator(orc):
    """P8: two overlapping equal soft disks = harmonic oscillator in the
    relative coordinate x = r - d with omega^2 = 2 eps / (m d^2); velocity
    Verlet reproduces it with cos(omega' dt) = 1 - (omega dt)^2 / 2 exactly."""
    eps, m, d, dt, nsteps = 1.0, 1.0, 1.0, 0.05, 20
    x0 = -0.05                                           # overlap 0.05, at rest
    box = np.array([10.0, 10.0, 1.0])
    pos = np.array([[4.0, 5.0, 0.0], [4.0 + d + x0, 5.0, 0.0]])
    vel = np.zeros((2, 3))
    diam = np.array([d, d])
    f0, _, _ = orc.energy_force(pos, diam, box, 2, SOFT, eps, 1.0, 1.4, 0)
    omega = math.sqrt(2 * eps / (m * d * d))
    omega_p = math.acos(1 - (omega * dt) ** 2 / 2) / dt
    # the spring is one-sided (u = 0 for r >= d): stay inside the first quarter
    # period pi/(2 omega) = 1.11 = 22 steps, while the disks still overlap
    for k in (1, 5, 13, nsteps):
        p, v, f, en, _ = orc.nve_run(pos, vel, f0, diam, box, 2, SOFT, eps, 1.0, 1.4, 0, dt, m, k)
        x = (p[1, 0] - p[0, 0]) - d
        assert x < 0
        assert abs(x - x0 * math.cos(omega_p * k * dt)) < 1e-12
        assert abs((p[0, 0] + p[1, 0]) - (pos[0, 0] + pos[1, 0])) < 1e-12   # centre of mass at rest
    # the continuous-time frequency would be off by a visible phase: the test discriminates
    assert abs(x0 * math.cos(omega * nsteps * dt) - x0 * math.cos(omega_p * nsteps * dt)) > 1e-6


def test_wrap_convention(orc):
    """mu(r, dr) keeps 0 <= x < L: free flight through the wall."""
    box = np.array([5.0, 5.0, 5.0])
    pos = np.array([[4.99, 0.01, 2.5], [1.0, 1.0, 1.0]])
    vel = np.array([[1.0, -1.0, 0.0], [0.0, 0.0, 0.0]])
    f0 = np.zeros((2, 3))
    # sigma tiny => no interaction; 5 steps of dt = 0.01 moves by 0.05
    p, v, f, _, _ = orc.nve_run(pos, vel, f0, None, box, 3, LJ, 1.0, 1e-3, 2.5e-3, 1, 0.01, 1.0, 5,
                                want_energies=False)
    assert np.allclose(p[0], [0.04, 4.96, 2.5], atol=1e-12)
    assert np.all(p >= 0) and np.all(p < box)


# ------------------------------------------------------------------ FIRE --

def test_fire_schedule_closed_form(orc):
    """While P = F.v > 0 the FIRE bookkeeping is a closed form: n_pos = k, and from the (n_min+1)-th
    step on dt grows by f_inc (capped at dt_max) and alpha shrinks by f_alpha.  Two overlapping
    soft disks released from rest roll downhill for the whole run."""
    d = 1.0
    box = np.array([10.0, 10.0, 1.0])
    pos = np.array([[4.0, 5.0, 0.0], [4.3, 5.0, 0.0]])          # overlap: r = 0.3 d
    vel = np.zeros((2, 3))
    par = (1e-3, 4e-3, 5, 1.1, 0.5, 0.1, 0.99)
    for k in (1, 5, 6, 12, 30):
        _, v, f, en, st = orc.fire_run(pos, vel, np.array([d, d]), box, 2, SOFT, 1.0, 1.0, 1.0, 0, k, par=par)
        grow = max(0, k - 5)
        assert st[2] == k
        assert abs(st[0] - min(1e-3 * 1.1 ** grow, 4e-3)) < 1e-15
        assert abs(st[1] - 0.1 * 0.99 ** grow) < 1e-15
        assert en[-1] < en[0] and v[0, 0] < 0 < v[1, 0]          # moving apart, energy released


def test_fire_uphill_start_is_reset(orc):
    """Velocities pointing up the energy gradient: P < 0 on the first step, so v = 0, dt is cut by
    f_dec, alpha returns to alpha_start and n_pos to 0."""
    box = np.array([10.0, 10.0, 1.0])
    pos = np.array([[4.0, 5.0, 0.0], [4.6, 5.0, 0.0]])
    vel = np.array([[0.5, 0.0, 0.0], [-0.5, 0.0, 0.0]])          # approaching: against the repulsion
    par = (1e-3, 4e-3, 5, 1.1, 0.5, 0.1, 0.99)
    _, v, _, _, st = orc.fire_run(pos, vel, np.array([1.0, 1.0]), box, 2, SOFT, 1.0, 1.0, 1.0, 0, 1, par=par)
    assert np.abs(v).max() == 0.0 and st[2] == 0 and abs(st[0] - 5e-4) < 1e-18 and st[1] == 0.1


def test_fire_without_mixing_is_velocity_verlet(orc, W):
    """alpha_start = 0, f_inc = 1: the mixing and the schedule are switched off and, as long as
    P > 0, FIRE is plain velocity Verlet -- the oracle's NVE loop (P7, P8 pin that one)."""
    w = W.soft_disks(1, 256)
    diam = w.pos[:, 3].astype(np.float64)
    par = (2e-3, 2e-3, 5, 1.0, 0.5, 0.0, 1.0)
    p, v, f, en, st = orc.fire_run(w.pos, w.vel, diam, w.box, 2, SOFT, 1.0, 1.0, 1.4, 0, 25, par=par)
    assert st[2] == 25                                            # P > 0 throughout (released from rest)
    f0, _, _ = orc.energy_force(w.pos, diam, w.box, 2, SOFT, 1.0, 1.0, 1.4, 0)
    p2, v2, f2, _, _ = orc.nve_run(w.pos, w.vel, f0, diam, w.box, 2, SOFT, 1.0, 1.0, 1.4, 0, 2e-3, 1.0, 25,
                                   want_energies=False)
    assert np.abs(p - p2).max() < 1e-13 and np.abs(v - v2).max() < 1e-13


def test_fire_relaxes_a_packing(orc, W):
    """Section 4.2's use: the bidisperse soft-disk packing relaxes -- the energy
    falls by more than an order of magnitude and the largest force with it."""
    w = W.soft_disks(1, 512)
    diam = w.pos[:, 3].astype(np.float64)
    f0, _, E0 = orc.energy_force(w.pos, diam, w.box, 2, SOFT, 1.0, 1.0, 1.4, 0)
    p, v, f, en, st = orc.fire_run(w.pos, w.vel, diam, w.box, 2, SOFT, 1.0, 1.0, 1.4, 0, 300)
    assert en[0] == E0 and en[-1] < 0.05 * E0
    assert np.abs(f).max() < 0.1 * np.abs(f0).max()
    assert ((p[:, :2] >= 0) & (p[:, :2] < w.box[:2])).all()


# ------------------------------------- Brownian / gradient descent --

def test_counter_based_normals(orc):
    """The generator both sides implement: standard-normal moments, no correlation between
    components, steps or neighbors, and a pure function of (seed, step, id)."""
    n = 200000
    g = orc.normals(11, 5, n, 3)
    assert np.abs(g.mean(0)).max() < 5 / np.sqrt(n)
    assert np.abs(g.var(0) - 1).max() < 5 * np.sqrt(2 / n)
    assert np.abs((g ** 4).mean(0) - 3).max() < 0.1
    c = np.corrcoef(g.T)
    assert np.abs(c - np.eye(3)).max() < 5 / np.sqrt(n)
    g2 = orc.normals(11, 6, n, 3)
    assert abs(np.corrcoef(g[:, 0], g2[:, 0])[0, 1]) < 5 / np.sqrt(n)
    assert abs(np.corrcoef(g[:-1, 0], g[1:, 0])[0, 1]) < 5 / np.sqrt(n)
    assert np.array_equal(g, orc.normals(11, 5, n, 3)) and not np.array_equal(g, orc.normals(12, 5, n, 3))
    assert np.array_equal(orc.normals(11, 5, 10, 2)[:, 2], np.zeros(10))
    assert np.array_equal(orc.normals(11, 5, 10, 2)[:, :2], g[:10, :2])


def test_brownian_free_diffusion(orc):
    """No forces (particles farther apart than r_cut): <|dr|^2> = 2 dim (kT/gamma) t."""
    m = 16
    g = np.arange(m, dtype=np.float64)
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3) * 3.0 + 1.0
    box = np.array([3.0 * m] * 3)
    dt, gamma, kT, steps = 1e-3, 2.0, 0.7, 40
    p, f, en = orc.brownian_run(pos, None, box, 3, LJ, 1.0, 1.0, 1.2, 1, dt, gamma, kT, 3, steps)
    assert np.abs(f).max() == 0.0 and np.abs(en).max() == 0.0
    d = p - pos
    d -= box * np.round(d / box)
    msd = (d ** 2).sum(1).mean()
    want = 2 * 3 * (kT / gamma) * steps * dt
    assert abs(msd / want - 1) < 5 * np.sqrt(2.0 / (3 * pos.shape[0]))      # chi-square spread
    # the increments are exactly the generator's normals
    p1, _, _ = orc.brownian_run(pos, None, box, 3, LJ, 1.0, 1.0, 1.2, 1, dt, gamma, kT, 3, 1, step0=9)
    assert np.allclose(p1 - pos, np.sqrt(2 * kT * dt / gamma) * orc.normals(3, 9, pos.shape[0], 3), atol=1e-13)


def test_gradient_descent_is_brownian_at_zero_temperature(orc, W):
    """kT = 0: r += (dt/gamma) F ("Gradient Descent").  One step by hand; two
    overlapping soft disks close their overlap geometrically; a packing's energy only falls."""
    w = W.soft_disks(1, 512)
    diam = w.pos[:, 3].astype(np.float64)
    pos = w.pos[:, :3].astype(np.float64); box = w.box.astype(np.float64)
    f0, _, E0 = orc.energy_force(pos, diam, box, 2, SOFT, 1.0, 1.0, 1.4, 0)
    p, f, en = orc.brownian_run(pos, diam, box, 2, SOFT, 1.0, 1.0, 1.4, 0, 0.05, 2.0, 0.0, 1, 1)
    want = pos + 0.025 * f0
    want[:, :2] -= box[:2] * np.floor(want[:, :2] / box[:2])
    assert np.abs(p - want).max() < 1e-13 and en[0] == E0
    p, f, en = orc.brownian_run(pos, diam, box, 2, SOFT, 1.0, 1.0, 1.4, 0, 0.05, 2.0, 0.0, 1, 60)
    assert np.all(np.diff(en) <= 0) and en[-1] < 0.5 * en[0]
    # dimer: overlap delta = d - r obeys delta' = delta (1 - 2 mu eps / d^2)
    d, mu = 1.0, 0.01
    box2 = np.array([10.0, 10.0, 1.0])
    pp = np.array([[4.0, 5.0, 0.0], [4.6, 5.0, 0.0]])
    q, _, _ = orc.brownian_run(pp, np.array([d, d]), box2, 2, SOFT, 1.0, 1.0, 1.0, 0, mu, 1.0, 0.0, 1, 25)
    delta = d - (q[1, 0] - q[0, 0])
    assert abs(delta - 0.4 * (1 - 2 * mu / d ** 2) ** 25) < 1e-13


# ---------------------------------------------------------- Langevin --

def test_langevin_without_bath_is_velocity_verlet(orc, W):
    """gamma = 0: c1 = 1, c2 = 0 and BAOAB is kick-drift-kick velocity Verlet (the NVE oracle)."""
    w = W.lj_fcc(0, 3, seed=4)
    f0, _, _ = orc.energy_force(w.pos, None, w.box, 3, LJ, 1.0, 1.0, 2.5, 1)
    p, v, f = orc.langevin_run(w.pos, w.vel, f0, None, w.box, 3, LJ, 1.0, 1.0, 2.5, 1, 0.004, 1.0, 0.0, 0.7, 5, 30)
    p2, v2, f2, _, _ = orc.nve_run(w.pos, w.vel, f0, None, w.box, 3, LJ, 1.0, 1.0, 2.5, 1, 0.004, 1.0, 30,
                                   want_energies=False)
    assert np.abs(p - p2).max() < 1e-12 and np.abs(v - v2).max() < 1e-11


def test_langevin_free_particles(orc):
    """No forces.  kT = 0: v_n = v_0 exp(-gamma dt)^n exactly.  kT > 0: the O step keeps the
    Maxwell-Boltzmann variance kT/m stationary, and from rest <v^2> = kT/m (1 - c1^(2n))."""
    m_ = 16
    g = np.arange(m_, dtype=np.float64)
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3) * 3.0 + 1.0
    box = np.array([3.0 * m_] * 3)
    n = pos.shape[0]
    f0 = np.zeros((n, 3))
    rng = np.random.default_rng(2)
    v0 = rng.normal(0, 1.0, (n, 3))
    dt, mass, gamma, steps = 5e-3, 2.0, 3.0, 40
    _, v, f = orc.langevin_run(pos, v0, f0, None, box, 3, LJ, 1.0, 1.0, 1.2, 1, dt, mass, gamma, 0.0, 1, steps)
    assert np.abs(f).max() == 0.0
    assert np.abs(v - v0 * np.exp(-gamma * dt) ** steps).max() < 1e-13
    kT = 0.9
    _, v, _ = orc.langevin_run(pos, np.zeros((n, 3)), f0, None, box, 3, LJ, 1.0, 1.0, 1.2, 1, dt, mass, gamma, kT, 1, steps)
    want = kT / mass * (1 - np.exp(-2 * gamma * dt * steps))
    assert abs((v ** 2).mean() / want - 1) < 5 * np.sqrt(2.0 / (3 * n))
    # one O step from rest is c2 * xi
    _, v1, _ = orc.langevin_run(pos, np.zeros((n, 3)), f0, None, box, 3, LJ, 1.0, 1.0, 1.2, 1, dt, mass, gamma, kT, 1, 1, step0=4)
    c1 = np.exp(-gamma * dt)
    assert np.allclose(v1, np.sqrt(kT / mass * (1 - c1 * c1)) * orc.normals(1, 4, n, 3), atol=1e-14)


# ------------------------------------------------------- Nose-Hoover --

def test_nose_hoover_decoupled_is_nve(orc, W):
    """tau -> infinity: Q -> infinity, the thermostat never moves and the step is velocity Verlet."""
    w = W.lj_fcc(0, 3, seed=6)
    f0, _, _ = orc.energy_force(w.pos, None, w.box, 3, LJ, 1.0, 1.0, 2.5, 1)
    p, v, f, cons, st = orc.nose_hoover_run(w.pos, w.vel, None, w.box, 3, LJ, 1.0, 1.0, 2.5, 1, 0.004, 1.0, 0.5, 1e9, 30)
    p2, v2, _, _, _ = orc.nve_run(w.pos, w.vel, f0, None, w.box, 3, LJ, 1.0, 1.0, 2.5, 1, 0.004, 1.0, 30,
                                  want_energies=False)
    assert np.abs(p - p2).max() < 1e-10 and np.abs(v - v2).max() < 1e-10 and abs(st[1]) < 1e-12


def test_nose_hoover_conserved_quantity_and_temperature(orc, W):
    """H' = K + U + Q v_xi^2/2 + dof kT xi is conserved to second order in dt (halving dt cuts its
    excursion ~4x), and the thermostat drives the kinetic temperature toward kT: started at T = 1
    with target 0.4 the time-averaged temperature of the second half lies near the target."""
    w = W.lj_fcc(0, 3, seed=8)                      # 108 particles, T = 1
    kT, tau = 0.4, 0.1
    out = {}
    for dt, steps in ((0.004, 400), (0.002, 800)):
        p, v, f, cons, st = orc.nose_hoover_run(w.pos, w.vel, None, w.box, 3, LJ, 1.0, 1.0, 2.5, 1, dt, 1.0, kT, tau, steps)
        out[dt] = np.abs(cons - cons[0]).max()
    assert out[0.004] < 2e-3 * abs(cons[0]) + 0.05
    assert 2.5 < out[0.004] / out[0.002] < 6.0
    # temperature: run in chunks and average the second half
    state, pos, vel, temps = None, w.pos, w.vel, []
    for chunk in range(40):
        pos4 = np.zeros((w.n, 4), np.float32); pos4[:, :3] = pos[:, :3]
        p, v, f, cons, state = orc.nose_hoover_run(pos, vel, None, w.box, 3, LJ, 1.0, 1.0, 2.5, 1, 0.004, 1.0, kT, tau, 25, state=state)
        temps.append((v ** 2).sum() / (3 * w.n))
        pos, vel = p, v
    assert abs(np.mean(temps[20:]) - kT) < 0.1 * kT


def test_nose_hoover_chain(orc, W):
    """Chains of thermostats ([67] is Martyna, Klein and Tuckerman's chain paper).
    (a) H' = K + U + sum Q_j v_j^2/2 + dof kT xi_1 + kT sum_{j>=2} xi_j is conserved to second order
        in dt for M = 3 (halving dt cuts the excursion ~4x) -- a wrong mass, sign or coupling in any
        link shows up here;
    (b) the splitting is symmetric: run forward, flip the signs of all velocities (particles' and
        thermostats'), run the same number of steps: the start comes back;
    (c) the second link moves as its equation says: starting from rest, after one small step
        v_2 ~ dt (Q_1 v_1^2 - kT)/Q_2 with v_1 ~ dt (2K - dof kT)/Q_1;
    (d) M = 1 through the chain code is the single thermostat (first two pins above still hold), and
        the far end of a long chain started at rest stays nearly at rest over a short run;
    (e) the temperature is driven to kT with M = 3 as well."""
    w = W.lj_fcc(0, 3, seed=8)
    kT, tau, M = 0.4, 0.1, 3
    run = lambda pos, vel, dt, steps, state=None, chain=M: orc.nose_hoover_run(
        pos, vel, None, w.box, 3, LJ, 1.0, 1.0, 2.5, 1, dt, 1.0, kT, tau, steps, state=state, chain=chain)
    out = {}
    for dt, steps in ((0.004, 300), (0.002, 600)):
        p, v, f, cons, st = run(w.pos, w.vel, dt, steps)
        out[dt] = np.abs(cons - cons[0]).max()
        assert np.abs(st[M:]).max() > 1e-3 and np.abs(st[1:M]).max() > 1e-6        # every link moved
    assert out[0.004] < 2e-3 * abs(cons[0]) + 0.05
    assert 2.5 < out[0.004] / out[0.002] < 6.0, out
    # (b)
    p, v, f, cons, st = run(w.pos, w.vel, 0.004, 60)
    st_back = st.copy(); st_back[M:] *= -1
    p2, v2, f2, cons2, st2 = run(p, -v, 0.004, 60, state=st_back)
    d = p2 - w.pos[:, :3].astype(np.float64); d -= w.box * np.round(d / w.box)
    assert np.abs(d).max() < 1e-9 and np.abs(v2 + w.vel[:, :3]).max() < 1e-9
    assert np.abs(st2[:M]).max() < 1e-7 and np.abs(st2[M:]).max() < 1e-7      # rounding, amplified by the small Q_j
    # (c)
    dt = 1e-5
    p, v, f, cons, st = run(w.pos, w.vel, dt, 1)
    dof = 3 * w.n
    K2 = (w.vel[:, :3].astype(np.float64) ** 2).sum()
    Q1, Q2 = dof * kT * tau ** 2, kT * tau ** 2
    v1 = dt * (K2 - dof * kT) / Q1
    assert abs(st[M] - v1) < 1e-3 * abs(v1)
    # v_2' = (Q_1 v_1(t)^2 - kT)/Q_2 with v_1(t) ~ v1 t/dt: v_2(dt) = dt (Q_1 v1^2/3 - kT)/Q_2 to leading order
    assert abs(st[M + 1] - dt * (Q1 * v1 ** 2 / 3 - kT) / Q2) < 2e-2 * abs(dt * kT / Q2)
    # (d)
    a = run(w.pos, w.vel, 0.004, 25, chain=1)
    b = orc.nose_hoover_run(w.pos, w.vel, None, w.box, 3, LJ, 1.0, 1.0, 2.5, 1, 0.004, 1.0, kT, tau, 25)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[4], b[4])
    # (e)
    state, pos, vel, temps = None, w.pos, w.vel, []
    for chunk in range(40):
        p, v, f, cons, state = run(pos, vel, 0.004, 25, state=state)
        temps.append((v ** 2).sum() / (3 * w.n))
        pos, vel = p, v
    assert abs(np.mean(temps[20:]) - kT) < 0.1 * kT


# ------------------------------------------------- Buckingham --

def test_buckingham_two_body_and_gradient(orc, W):
    """u = A exp(-B r) - C / r^6 (PAPER.md:L104 [71-73]): closed form at one distance, the force as
    -u'(r) with its sign, shifted cutoff, and -grad E by central differences on a lattice."""
    BUCK = 3
    A, Bc, Cc, rc = 1000.0, 9.0, 1.5, 2.5
    r = 1.3
    pos, box, _ = two_body(r, 0)
    f, e_i, E0 = orc.energy_force(pos, None, box, 3, BUCK, A, Cc, rc, 0, alpha=Bc)
    u = A * np.exp(-Bc * r) - Cc / r ** 6
    du = -A * Bc * np.exp(-Bc * r) + 6 * Cc / r ** 7
    assert abs(E0 - u) < 1e-13 and abs(f[0, 0] - du) < 1e-12 and abs(f[1, 0] + du) < 1e-12
    _, _, E1 = orc.energy_force(pos, None, box, 3, BUCK, A, Cc, rc, 1, alpha=Bc)
    assert abs(E1 - (u - (A * np.exp(-Bc * rc) - Cc / rc ** 6))) < 1e-13
    pos, box, _ = two_body(rc * (1 + 1e-9), 0)
    assert orc.energy_force(pos, None, box, 3, BUCK, A, Cc, rc, 1, alpha=Bc)[2] == 0.0
    w = W.lj_fcc(0, 3, seed=13)
    pos, box = w.pos[:, :3].astype(np.float64), w.box.astype(np.float64)
    args = (BUCK, A, Cc, rc, 1)
    f, _, _ = orc.energy_force(pos, None, box, 3, *args, alpha=Bc)
    assert np.abs(f.sum(0)).max() < 1e-10 * np.abs(f).sum()
    rng = np.random.default_rng(4)
    h, worst = 1e-5, 0.0
    for i in rng.choice(pos.shape[0], 6, replace=False):
        for q in range(3):
            pp = pos.copy(); pp[i, q] += h
            pm = pos.copy(); pm[i, q] -= h
            fd = -(orc.energy_force(pp, None, box, 3, *args, alpha=Bc)[2]
                   - orc.energy_force(pm, None, box, 3, *args, alpha=Bc)[2]) / (2 * h)
            worst = max(worst, abs(fd - f[i, q]) / max(1.0, np.abs(f[i]).max()))
    assert worst < 1e-6, worst


# ------------------------------------------- species x species LJ --

KA_EPS = np.array([[1.0, 1.5], [1.5, 0.5]])
KA_SIG = np.array([[1.0, 0.8], [0.8, 0.88]])


def test_species_lj_reduces_to_lj_and_mixed_pair_closed_form(orc, W):
    """Kind 4: identical species tables give plain LJ (the pinned kind 0); a mixed A-B pair of the
    Kob-Andersen tables follows the closed form with eps_AB, sigma_AB and its own cutoff; forces are
    -grad E and sum to zero on a binary mixture."""
    SPEC = 4
    w = W.lj_fcc(0, 3, seed=21)
    pos, box = w.pos[:, :3].astype(np.float64), w.box.astype(np.float64)
    one = np.ones((2, 2))
    orc.set_species_lj(one, one, 2.5 * one)
    sp = (np.arange(w.n) % 5 == 0).astype(np.float64)             # 20 % species 1
    f4, e4, E4 = orc.energy_force(pos, sp, box, 3, SPEC, 0.0, 0.0, 0.0, 1)
    f0, e0, E0 = orc.energy_force(pos, None, box, 3, LJ, 1.0, 1.0, 2.5, 1)
    assert np.array_equal(f4, f0) and np.array_equal(e4, e0) and E4 == E0
    orc.set_species_lj(KA_EPS, KA_SIG, 2.5 * KA_SIG)
    r = 0.95
    p2, b2, _ = two_body(r, 1)
    f, _, E = orc.energy_force(p2, np.array([0.0, 1.0]), b2, 3, SPEC, 0.0, 0.0, 0.0, 1)
    eps, sig, rc = 1.5, 0.8, 2.0
    u = 4 * eps * ((sig / r) ** 12 - (sig / r) ** 6) - 4 * eps * ((sig / rc) ** 12 - (sig / rc) ** 6)
    du = 4 * eps * (-12 * sig ** 12 / r ** 13 + 6 * sig ** 6 / r ** 7)
    assert abs(E - u) < 1e-13 and abs(f[0, 1] - du) < 1e-12 and abs(f[1, 1] + du) < 1e-12
    p2, b2, _ = two_body(2.0 * (1 + 1e-9), 1)                     # beyond rc_AB = 2.0 but inside rc_AA = 2.5
    assert orc.energy_force(p2, np.array([0.0, 1.0]), b2, 3, SPEC, 0.0, 0.0, 0.0, 1)[2] == 0.0
    assert orc.energy_force(p2, np.array([0.0, 0.0]), b2, 3, SPEC, 0.0, 0.0, 0.0, 1)[2] != 0.0
    f, _, _ = orc.energy_force(pos, sp, box, 3, SPEC, 0.0, 0.0, 0.0, 1)
    assert np.abs(f.sum(0)).max() < 1e-10 * np.abs(f).sum()
    rng = np.random.default_rng(6)
    h, worst = 1e-5, 0.0
    for i in rng.choice(pos.shape[0], 6, replace=False):
        for q in range(3):
            pp = pos.copy(); pp[i, q] += h
            pm = pos.copy(); pm[i, q] -= h
            fd = -(orc.energy_force(pp, sp, box, 3, SPEC, 0.0, 0.0, 0.0, 1)[2]
                   - orc.energy_force(pm, sp, box, 3, SPEC, 0.0, 0.0, 0.0, 1)[2]) / (2 * h)
            worst = max(worst, abs(fd - f[i, q]) / max(1.0, np.abs(f[i]).max()))
    assert worst < 1e-6, worst


# ----------------------------------------------------------- flocking --

FLOCK_PAR = (1.0, 3.0, 25.0, 1.5, 0.5, 4.0, 3.0)      # J_al, R_al, J_av, R_av, J_co, R_co, alpha


def test_flocking_two_boid_closed_forms(orc):
    """Eqs. (6)-(10) of PAPER.md App. B on a pair: rho, the alignment, avoidance and cohesion energies
    and their gradients written out by hand (reading A25 of DESIGN.md)."""
    Jal, Ral, Jav, Rav, Jco, Rco, al = FLOCK_PAR
    box = np.array([50.0, 50.0, 1.0])
    r, t0, t1 = 1.2, 0.3, 1.1
    pos = np.array([[10.0, 10.0, 0.0], [10.0 + r, 10.0, 0.0]])
    th = np.array([t0, t1])
    en, gR, gth = orc.flock_energy_grad(pos, th, box, FLOCK_PAR)
    rho = lambda x, Rc: (1 - x / Rc) ** al / al if x < Rc else 0.0
    drho = lambda x, Rc: -(1 - x / Rc) ** (al - 1) / Rc if x < Rc else 0.0
    c = np.cos(t0 - t1)
    assert abs(en[0] - Jal * rho(r, Ral) * (1 - c) ** 2) < 1e-14            # one pair, counted once
    assert abs(en[1] - Jav * rho(r, Rav)) < 1e-14
    # cohesion: boid 0 sees boid 1 along +x, boid 1 sees boid 0 along -x
    e0 = 0.5 * Jco * (1 - np.cos(t0)) ** 2
    e1 = 0.5 * Jco * (1 + np.cos(t1)) ** 2
    assert abs(en[2] - (e0 + e1)) < 1e-14
    # avoidance pushes apart: grad_R0 E_avoid = J rho'(r) * (R0 - R1)/r = -J rho' along +x ... boid 0 sits at smaller x
    ga = Jav * drho(r, Rav) * (-1.0)
    # cohesion gradient in x vanishes for a pair (D only changes length along the line of centres)
    assert abs(gR[0, 0] - ga) < 1e-12 and abs(gR[1, 0] + ga) < 1e-12
    # theta gradients
    g0 = Jal * rho(r, Ral) * 2 * (1 - c) * np.sin(t0 - t1) + Jco * (1 - np.cos(t0)) * np.sin(t0)
    assert abs(gth[0] - g0) < 1e-12
    # beyond every range: nothing
    pos[1, 0] = 10.0 + 4.5
    en, gR, gth = orc.flock_energy_grad(pos, th, box, FLOCK_PAR)
    assert np.abs(en).max() == 0.0 and np.abs(gR).max() == 0.0 and np.abs(gth).max() == 0.0


def test_flocking_gradients_and_invariances(orc):
    """grad_theta E and grad_R (E_avoid + E_cohesion) by central differences (the alignment term has
    no R gradient: stop-gradient, PAPER.md B.2.2); E is invariant under a rigid rotation of
    positions and headings and under a translation across the periodic boundary."""
    rng = np.random.default_rng(1)
    n, L = 150, 18.0
    pos = np.zeros((n, 3)); pos[:, :2] = rng.uniform(0, L, (n, 2))
    th = rng.uniform(-np.pi, np.pi, n)
    box = np.array([L, L, 1.0])
    en, gR, gth = orc.flock_energy_grad(pos, th, box, FLOCK_PAR)
    h, worst = 1e-6, 0.0
    for i in rng.choice(n, 8, replace=False):
        tp = th.copy(); tp[i] += h
        tm = th.copy(); tm[i] -= h
        fd = (orc.flock_energy_grad(pos, tp, box, FLOCK_PAR)[0].sum() - orc.flock_energy_grad(pos, tm, box, FLOCK_PAR)[0].sum()) / (2 * h)
        worst = max(worst, abs(fd - gth[i]))
        for q in range(2):
            pp = pos.copy(); pp[i, q] += h
            pm = pos.copy(); pm[i, q] -= h
            fd = (orc.flock_energy_grad(pp, th, box, FLOCK_PAR)[0][1:].sum()
                  - orc.flock_energy_grad(pm, th, box, FLOCK_PAR)[0][1:].sum()) / (2 * h)
            worst = max(worst, abs(fd - gR[i, q]))
    assert worst < 1e-6, worst
    shift = np.array([7.3, -4.1, 0.0])
    p2 = pos + shift; p2[:, :2] -= L * np.floor(p2[:, :2] / L)
    en2, gR2, gth2 = orc.flock_energy_grad(p2, th, box, FLOCK_PAR)
    assert np.abs(en2 - en).max() < 1e-10 and np.abs(gR2 - gR).max() < 1e-10
    # rotation about the centre of a cluster that does not touch the boundary
    big = np.array([200.0, 200.0, 1.0])
    c = pos[:, :2] + 90.0
    phi = 0.7
    Rm = np.array([[np.cos(phi), -np.sin(phi)], [np.sin(phi), np.cos(phi)]])
    p3 = np.zeros((n, 3)); p3[:, :2] = (c - 100.0) @ Rm.T + 100.0
    pc = np.zeros((n, 3)); pc[:, :2] = c
    e_a = orc.flock_energy_grad(pc, th, big, FLOCK_PAR)[0]
    e_b = orc.flock_energy_grad(p3, th + phi, big, FLOCK_PAR)[0]
    assert np.abs(e_a - e_b).max() < 1e-9


def test_flocking_forward_euler(orc):
    """Eqs. (4)-(5): a lone boid swims straight at speed v; two boids within R_al only (avoidance and
    cohesion switched off) turn toward each other's heading by the alignment gradient."""
    box = np.array([30.0, 30.0, 1.0])
    p, th = orc.flock_run(np.array([[5.0, 5.0, 0.0]]), np.array([0.5]), box, FLOCK_PAR, 0.8, 0.1, 10)
    assert abs(p[0, 0] - (5 + 0.8 * np.cos(0.5))) < 1e-12 and abs(p[0, 1] - (5 + 0.8 * np.sin(0.5))) < 1e-12 and th[0] == 0.5
    par = (1.0, 3.0, 0.0, 1.5, 0.0, 4.0, 3.0)
    pos = np.array([[5.0, 5.0, 0.0], [6.0, 5.0, 0.0]])
    th0 = np.array([0.2, 1.4])
    p, th = orc.flock_run(pos, th0, box, par, 0.0, 0.05, 1)
    g = (1 - 1.0 / 3.0) ** 3 / 3 * 2 * (1 - np.cos(-1.2)) * np.sin(-1.2)
    assert abs(th[0] - (0.2 - 0.05 * g)) < 1e-13 and abs(th[1] - (1.4 + 0.05 * g)) < 1e-13
    assert np.array_equal(p[:, :2], pos[:, :2])                       # speed 0, no R gradient from alignment
    p, th = orc.flock_run(pos, th0, box, par, 0.0, 0.05, 200)
    assert abs(th[0] - th[1]) < abs(th0[0] - th0[1]) * 0.7


def test_flocking_obstacles(orc):
    """Eq. (11) (A26).  Closed forms for one boid and one disk: heading
    straight at the centre e = 4 J rho, straight away e = 0 with zero gradients, sideways e = J rho;
    nothing outside the disk; gradients by central differences; the disk acts across the periodic
    boundary; a boid inside a disk and heading away from it is left alone by the Euler step while one
    heading at it is turned and pushed out."""
    box = np.array([20.0, 20.0, 1.0])
    J, D, al = 2.0, 3.0, 3.0
    cen = np.array([[10.0, 10.0]])
    rho = lambda r: (1 - r / D) ** al / al
    at = lambda x, y: np.array([[x, y, 0.0]])
    # boid at distance 1.2 to the left of the centre: R_io = (+1.2, 0), u = (1, 0)
    e, gR, gth = orc.flock_obstacle_energy_grad(at(8.8, 10.0), [0.0], box, cen, [D], J, al)     # heading at it
    assert abs(e - 4 * J * rho(1.2)) < 1e-14 and abs(gth[0]) < 1e-14
    e, gR, gth = orc.flock_obstacle_energy_grad(at(8.8, 10.0), [np.pi], box, cen, [D], J, al)   # heading away
    assert abs(e) < 1e-28 and np.abs(gR).max() < 1e-13 and abs(gth[0]) < 1e-13
    e, gR, gth = orc.flock_obstacle_energy_grad(at(8.8, 10.0), [np.pi / 2], box, cen, [D], J, al)
    assert abs(e - J * rho(1.2)) < 1e-14
    assert abs(gth[0] - 2 * J * rho(1.2) * (-1.0)) < 1e-13              # d/dtheta (1 + cos theta)^2 at pi/2
    e, gR, gth = orc.flock_obstacle_energy_grad(at(6.9, 10.0), [0.0], box, cen, [D], J, al)     # r = 3.1 > D
    assert e == 0.0 and not gR.any() and not gth.any()
    # across the boundary: disk at x = 0.5, boid at x = 19.5 (distance 1)
    e, _, _ = orc.flock_obstacle_energy_grad(at(19.5, 4.0), [0.0], box, [[0.5, 4.0]], [D], J, al)
    assert abs(e - 4 * J * rho(1.0)) < 1e-13
    # central differences, several boids and disks
    rng = np.random.default_rng(3)
    n = 40
    pos = np.zeros((n, 3)); pos[:, :2] = rng.uniform(0, 20, (n, 2))
    th = rng.uniform(-np.pi, np.pi, n)
    cens = rng.uniform(0, 20, (5, 2)); rad = rng.uniform(2.0, 5.0, 5)
    e0, gR, gth = orc.flock_obstacle_energy_grad(pos, th, box, cens, rad, J, 2.5)
    assert e0 > 0
    E = lambda p, t: orc.flock_obstacle_energy_grad(p, t, box, cens, rad, J, 2.5)[0]
    h, worst = 1e-6, 0.0
    for i in range(n):
        tp = th.copy(); tp[i] += h; tm = th.copy(); tm[i] -= h
        worst = max(worst, abs((E(pos, tp) - E(pos, tm)) / (2 * h) - gth[i]))
        for q in range(2):
            pp = pos.copy(); pp[i, q] += h; pm = pos.copy(); pm[i, q] -= h
            worst = max(worst, abs((E(pp, th) - E(pm, th)) / (2 * h) - gR[i, q]))
    assert worst < 2e-7, worst
    # forward Euler with the obstacle switched on, all boid-boid terms off
    par0 = (0.0, 3.0, 0.0, 1.5, 0.0, 4.0, al)
    orc.flock_set_obstacles(cen, [D], J)
    try:
        p, t = orc.flock_run(at(8.8, 10.0), [np.pi], box, par0, 0.5, 0.1, 5)
        assert abs(p[0, 0] - (8.8 - 0.25)) < 1e-12 and abs(t[0] - np.pi) < 1e-12     # swims away undisturbed
        p, t = orc.flock_run(at(8.8, 10.2), [0.1], box, par0, 0.0, 0.05, 40)
        r0 = np.hypot(1.2, 0.2); r1 = np.hypot(10.0 - p[0, 0], 10.0 - p[0, 1])
        assert r1 > r0                                                               # pushed outward
        u = np.array([10.0 - p[0, 0], 10.0 - p[0, 1]]) / r1
        assert np.cos(t[0]) * u[0] + np.sin(t[0]) * u[1] < np.cos(0.1) * 1.2 / r0 + np.sin(0.1) * (-0.2) / r0   # turned away
    finally:
        orc.flock_set_obstacles()
    p, t = orc.flock_run(at(8.8, 10.0), [0.0], box, par0, 0.5, 0.1, 1)               # obstacles cleared
    assert abs(p[0, 0] - 8.85) < 1e-12


def test_bks_type_potential(orc):
    """Kind 5 ("Buckingham / BKS" [71-73]; A27): exp-6 per species pair plus damped
    shifted-force Coulomb.
    (a) the rock-salt lattice: energy per ion plus the Wolf self term reproduces the Madelung constant
        1.747565 (exact lattice sum) to 1e-5, forces vanish by symmetry;
    (b) no damping: the textbook shifted-force Coulomb q q'(1/r - 1/rc + (r - rc)/rc^2), and bare q q'/r as
        rc -> infinity; energy and force both vanish at the cutoff; like charges repel;
    (c) zero charges: kind 3 (Buckingham, pinned on its own) with the same A, B, C;
    (d) forces are minus the central differences of the energy for a random binary configuration."""
    from math import erfc, sqrt, pi
    m, rc, a = 6, 5.9, 0.6
    g = np.stack(np.meshgrid(*[np.arange(2 * m)] * 3, indexing="ij"), -1).reshape(-1, 3)
    pos = g.astype(np.float64) + 0.25
    sp = (g.sum(1) % 2).astype(np.float64)
    box = np.array([2.0 * m] * 3)
    z = np.zeros((2, 2))
    orc.set_species_bks(z, z + 1.0, z, [1.0, -1.0], a, 1.0)
    f, e, E = orc.energy_force(pos, sp, box, 3, 5, 0.0, 0.0, rc, 0)
    per_ion = E / len(pos) - (erfc(a * rc) / (2 * rc) + a / sqrt(pi))
    assert abs(per_ion - (-1.747565 / 2)) < 1e-5, per_ion
    assert np.abs(f).max() < 1e-12
    # (b)
    big = np.array([400.0, 400.0, 400.0])
    two = lambda r: np.array([[100.0, 100.0, 100.0], [100.0 + r, 100.0, 100.0]])
    orc.set_species_bks(z, z + 1.0, z, [2.0, -0.5], 0.0, 3.0)
    for r in (0.8, 1.7, 2.9):
        f, e, E = orc.energy_force(two(r), [0.0, 1.0], big, 3, 5, 0.0, 0.0, 3.0, 0)
        qq = 3.0 * 2.0 * -0.5
        assert abs(E - qq * (1 / r - 1 / 3.0 + (r - 3.0) / 9.0)) < 1e-13
        assert abs(f[0, 0] - (-qq * (1 / r**2 - 1 / 9.0))) < 1e-13 and f[0, 0] > 0      # attracted toward +x
        assert np.allclose(f[0], -f[1], atol=1e-15)
    f, e, E = orc.energy_force(two(1.3), [0.0, 0.0], big, 3, 5, 0.0, 0.0, 3.0, 0)
    assert E > 0 and f[0, 0] < 0                                                         # like charges repel
    f, e, E = orc.energy_force(two(2.0), [0.0, 1.0], big, 3, 5, 0.0, 0.0, 150.0, 0)
    assert abs(E - (-3.0 / 2.0)) < 0.05                                                  # 2 q q' / rc away from bare Coulomb
    orc.set_species_bks(z, z + 1.0, z, [1.0, -1.0], 0.35, 1.0)
    f, e, E = orc.energy_force(two(3.0 - 1e-7), [0.0, 1.0], big, 3, 5, 0.0, 0.0, 3.0, 0)
    assert abs(E) < 1e-13 and np.abs(f).max() < 1e-7
    f, e, E = orc.energy_force(two(3.0 + 1e-7), [0.0, 1.0], big, 3, 5, 0.0, 0.0, 3.0, 0)
    assert E == 0.0 and not f.any()
    # (c)
    rng = np.random.default_rng(2)
    n, L = 200, 9.0
    gq = (np.arange(6) + 0.5) * (L / 6)
    p = np.stack(np.meshgrid(gq, gq, gq, indexing="ij"), -1).reshape(-1, 3)[:n] + rng.normal(0, 0.08, (n, 3))
    bx = np.array([L, L, L])
    A, Bq, Cq = 9.02e5, 12.5, 3.454
    one = np.ones((2, 2))
    spc = (np.arange(n) % 2).astype(np.float64)
    orc.set_species_bks(A * one, Bq * one, Cq * one, [0.0, 0.0], 0.3, 1.0)
    f5, e5, E5 = orc.energy_force(p, spc, bx, 3, 5, 0.0, 0.0, 2.5, 1)
    f3, e3, E3 = orc.energy_force(p, None, bx, 3, 3, A, Cq, 2.5, 1, alpha=Bq)
    assert np.abs(f5 - f3).max() < 1e-12 * np.abs(f3).max() and abs(E5 - E3) < 1e-12 * abs(E3)
    # (d) distinct tables per pair, charges on
    Am = A * np.array([[1.0, 0.7], [0.7, 0.5]]); Bm = Bq * np.array([[1.0, 1.05], [1.05, 1.1]])
    Cm = Cq * np.array([[1.0, 0.6], [0.6, 0.3]])
    orc.set_species_bks(Am, Bm, Cm, [0.6, -0.6], 0.3, 1.0)
    f, e, E = orc.energy_force(p, spc, bx, 3, 5, 0.0, 0.0, 2.5, 1)
    h, worst = 1e-6, 0.0
    for i in rng.choice(n, 6, replace=False):
        for q in range(3):
            pp = p.copy(); pp[i, q] += h; pm = p.copy(); pm[i, q] -= h
            fd = -(orc.energy_force(pp, spc, bx, 3, 5, 0.0, 0.0, 2.5, 1)[2]
                   - orc.energy_force(pm, spc, bx, 3, 5, 0.0, 0.0, 2.5, 1)[2]) / (2 * h)
            worst = max(worst, abs(fd - f[i, q]))
    assert worst < 1e-6 * max(1.0, np.abs(f).max()), worst
    assert np.abs(f.sum(0)).max() < 1e-10 * np.abs(f).max()                              # Newton's third law


def test_flocking_predators(orc):
    """Eqs. (12)-(13) (A28).  The chase term: a predator beside a clump of
    boids has e = J/2 (1 - cos phi)^2, phi the angle between its heading and the direction of the clump's
    centre of mass; nothing in range gives zero; gradients by central differences (clump well inside the
    range, so the set is fixed).  Dynamics: the predator turns toward and closes in on the clump; boids
    within R_flee of a predator end up farther from it than the same boids without predators; with no
    predators the run is orc_flock_run."""
    box = np.array([40.0, 40.0, 1.0])
    rng = np.random.default_rng(4)
    clump = np.zeros((30, 3)); clump[:, :2] = np.array([20.0, 20.0]) + rng.normal(0, 0.5, (30, 2))
    com = clump[:, :2].mean(0)
    ppos = np.array([[16.0, 18.5]])
    u = (com - ppos[0]) / np.linalg.norm(com - ppos[0])
    J, R = 3.0, 8.0
    for th in (-2.0, 0.3, 1.9):
        e, gR, gth = orc.predator_energy_grad(clump, box, ppos, [th], J, R)
        cphi = np.cos(th) * u[0] + np.sin(th) * u[1]
        assert abs(e - 0.5 * J * (1 - cphi) ** 2) < 1e-13
    e, gR, gth = orc.predator_energy_grad(clump, box, [[2.0, 2.0]], [0.3], J, R)
    assert e == 0.0 and not gR.any() and not gth.any()
    th = 1.9
    e0, gR, gth = orc.predator_energy_grad(clump, box, ppos, [th], J, R)
    h = 1e-6
    E = lambda pp, t: orc.predator_energy_grad(clump, box, pp, [t], J, R)[0]
    assert abs((E(ppos, th + h) - E(ppos, th - h)) / (2 * h) - gth[0]) < 1e-8
    for q in range(2):
        a = ppos.copy(); a[0, q] += h; b = ppos.copy(); b[0, q] -= h
        assert abs((E(a, th) - E(b, th)) / (2 * h) - gR[0, q]) < 1e-8
    # two predators, one across the periodic boundary from its prey
    far = np.zeros((5, 3)); far[:, :2] = np.array([39.0, 5.0]) + rng.normal(0, 0.3, (5, 2))
    both = np.concatenate([clump, far])
    e2, gR2, gth2 = orc.predator_energy_grad(both, box, [[16.0, 18.5], [1.5, 5.0]], [th, 0.0], J, R)
    assert abs(gth2[0] - gth[0]) < 1e-14 and e2 > e0          # the second predator looks away from its prey (at -x)
    # dynamics
    par = (1.0, 3.0, 10.0, 1.5, 0.0, 4.0, 3.0)
    ppar = (5.0, 4.0, 3.0, 8.0, 0.6)
    th_b = rng.uniform(-np.pi, np.pi, 30)
    p1, t1, pp1, pt1 = orc.flock_run_predators(clump, th_b, box, par, 0.2, 0.02, 150, ppos, [1.9], ppar)
    d0 = np.linalg.norm(com - ppos[0]); d1 = np.linalg.norm(p1[:, :2].mean(0) - pp1[0])
    u1 = (p1[:, :2].mean(0) - pp1[0]) / d1
    assert np.cos(pt1[0]) * u1[0] + np.sin(pt1[0]) * u1[1] > np.cos(1.9) * u[0] + np.sin(1.9) * u[1]   # turned toward
    assert d1 < d0                                                                                      # closed in
    near = np.zeros((12, 3)); near[:, :2] = np.array([10.0, 30.0]) + rng.normal(0, 1.2, (12, 2))
    th_n = rng.uniform(-np.pi, np.pi, 12)
    hunter = np.array([[10.0, 30.0]])
    pa, _, ppa, _ = orc.flock_run_predators(near, th_n, box, par, 0.0, 0.02, 100, hunter, [0.0], (5.0, 4.0, 0.0, 8.0, 0.0))
    pb, _ = orc.flock_run(near, th_n, box, par, 0.0, 0.02, 100)
    ra = np.linalg.norm(pa[:, :2] - hunter[0], axis=1).mean(); rb = np.linalg.norm(pb[:, :2] - hunter[0], axis=1).mean()
    assert np.array_equal(ppa, hunter) and ra > rb + 0.05
    pc, tc, _, _ = orc.flock_run_predators(near, th_n, box, par, 0.3, 0.02, 20, np.zeros((0, 2)), [], ppar)
    pd_, td = orc.flock_run(near, th_n, box, par, 0.3, 0.02, 20)
    assert np.array_equal(pc, pd_) and np.array_equal(tc, td)
