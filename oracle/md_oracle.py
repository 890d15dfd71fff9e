"""ctypes loader for the fp64 CPU oracle ``md_oracle.c``.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl
reference`` legs may import this.  It imports nothing from the CUDA package.
Argument marshalling only; every formula lives in ``md_oracle.c`` with its
PAPER.md citation.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "md_oracle.c")
_LIB = os.path.join(_HERE, "libmd_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile md_oracle.c with gcc (no implicit FMA, OpenMP over particles)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
               "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(t: int) -> None:
    lib().orc_set_num_threads(int(t))


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _pd(a):
    return _p(a, C.c_double) if a is not None else None


def _pi(a):
    return _p(a, C.c_int32) if a is not None else None


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed: {rc}")


def pos3(pos) -> np.ndarray:
    """float32[N,4] or any [N,>=3]/[N,2] array -> exact fp64 [N,3]."""
    a = np.asarray(pos)
    out = np.zeros((a.shape[0], 3), dtype=np.float64)
    k = min(3, a.shape[1])
    out[:, :k] = a[:, :k].astype(np.float64)
    return out


def cell_list(pos, box, dim, r_cut, skin):
    p = _d(pos3(pos)); b = _d(box)
    n = p.shape[0]
    ncell = np.zeros(3, dtype=np.int32)
    cell_of = np.zeros(n, dtype=np.int32)
    # first call sizes the arrays
    _check(lib().orc_cell_list(n, dim, _pd(p), _pd(b), C.c_float(r_cut), C.c_float(skin),
                               _pi(ncell), _pi(cell_of), None, None), "cell_list")
    cells = int(ncell[0]) * int(ncell[1]) * int(ncell[2])
    cell_start = np.zeros(cells + 1, dtype=np.int32)
    members = np.zeros(n, dtype=np.int32)
    _check(lib().orc_cell_list(n, dim, _pd(p), _pd(b), C.c_float(r_cut), C.c_float(skin),
                               _pi(ncell), _pi(cell_of), _pi(cell_start), _pi(members)), "cell_list")
    return ncell, cell_of, cell_start, members


def neighbor_list(pos, box, dim, r_cut, skin, capacity, predicate=0, method=0):
    p = _d(pos3(pos)); b = _d(box)
    n = p.shape[0]
    idx = np.empty((n, capacity), dtype=np.int32)
    cnt = np.empty(n, dtype=np.int32)
    status = np.zeros(2, dtype=np.int32)
    _check(lib().orc_neighbor_list(n, dim, _pd(p), _pd(b), C.c_float(r_cut), C.c_float(skin),
                                   capacity, predicate, method, _pi(idx), _pi(cnt), _pi(status)),
           "neighbor_list")
    return idx, cnt, status


def predicate_band(pos, box, dim, r_cut, skin, method=1):
    p = _d(pos3(pos)); b = _d(box)
    nd = C.c_int64(0); band = C.c_double(0); close = C.c_double(0)
    _check(lib().orc_predicate_band(p.shape[0], dim, _pd(p), _pd(b), C.c_float(r_cut),
                                    C.c_float(skin), method, C.byref(nd), C.byref(band),
                                    C.byref(close)), "predicate_band")
    return int(nd.value), float(band.value), float(close.value)


class Params(C.Structure):
    """orc_params of md_oracle.c: the parameters of kinds 2-5 and the Nose-Hoover chain length.  They travel
    with every call; the C library keeps no state.  A fresh object is in the UNSET state (alpha = NaN, no
    species tables), in which a call that needs one of them fails."""
    _fields_ = [("morse_alpha", C.c_double), ("ns", C.c_int32), ("bks_ns", C.c_int32), ("nh_chain", C.c_int32),
                ("pad_", C.c_int32), ("sp_eps", C.c_double * 16), ("sp_sig", C.c_double * 16),
                ("sp_rc", C.c_double * 16), ("bks_A", C.c_double * 16), ("bks_B", C.c_double * 16),
                ("bks_C", C.c_double * 16), ("bks_q", C.c_double * 4), ("bks_a", C.c_double), ("bks_k", C.c_double)]

    def __init__(self):
        super().__init__()
        assert C.sizeof(Params) == lib().orc_params_size()
        self.reset()

    def reset(self):
        lib().orc_params_reset(C.byref(self))

    def species_lj(self, eps, sigma, rc):
        e = _d(eps); sg = _d(sigma); r = _d(rc)
        _check(lib().orc_params_species_lj(C.byref(self), e.shape[0], _pd(e.reshape(-1).copy()),
                                           _pd(sg.reshape(-1).copy()), _pd(r.reshape(-1).copy())), "species_lj")

    def species_bks(self, A, B, Cc, q, coulomb_alpha, k_e=1.0):
        A = _d(A); B = _d(B); Cc = _d(Cc); q = _d(q)
        ns = q.shape[0]
        assert A.shape == (ns, ns) and B.shape == (ns, ns) and Cc.shape == (ns, ns)
        _check(lib().orc_params_species_bks(C.byref(self), ns, _pd(A), _pd(B), _pd(Cc), _pd(q),
                                            C.c_double(coulomb_alpha), C.c_double(k_e)), "species_bks")


_DEFAULT = None


def default_params() -> Params:
    """The Params object the functions below pass when the caller gives none (`params=None`); the set_*
    functions write into it.  tests/conftest.py resets it before every test."""
    global _DEFAULT
    if _DEFAULT is None:
        _DEFAULT = Params()
    return _DEFAULT


def _par(params):
    return C.byref(default_params() if params is None else params)


def set_species_lj(eps, sigma, rc) -> None:
    """Tables of kind 4 (species x species LJ): square arrays eps_ab, sigma_ab, rc_ab."""
    default_params().species_lj(eps, sigma, rc)


def set_species_bks(A, B, Cc, q, coulomb_alpha, k_e=1.0):
    """Tables of kind 5 (BKS-type): square arrays A_ab, B_ab, C_ab, charges q_a, DSF damping, Coulomb constant."""
    default_params().species_bks(A, B, Cc, q, coulomb_alpha, k_e)


def reset_params() -> None:
    """Put the default Params back into the unset state (Morse / Buckingham alpha, species tables, chain length):
    a later call that needs one fails until it is set again.  tests/conftest.py does this before every test."""
    default_params().reset()


def set_morse_alpha(alpha: float) -> None:
    """alpha of kind 2 (Morse) / B of kind 3 for the following calls that pass the default Params."""
    default_params().morse_alpha = float(alpha)


def energy_force(pos, diam, box, dim, kind, eps, sigma, r_cut, shift,
                 nbr_idx=None, nbr_count=None, alpha=None, params=None):
    if alpha is not None:
        (default_params() if params is None else params).morse_alpha = float(alpha)
    p = _d(pos3(pos)); b = _d(box)
    n = p.shape[0]
    dm = _d(diam) if diam is not None else None
    f = np.zeros((n, 3), dtype=np.float64)
    e_i = np.zeros(n, dtype=np.float64)
    E = C.c_double(0)
    cap = 0
    if nbr_idx is not None:
        nbr_idx = np.ascontiguousarray(nbr_idx, dtype=np.int32)
        nbr_count = np.ascontiguousarray(nbr_count, dtype=np.int32)
        cap = nbr_idx.shape[1]
    _check(lib().orc_energy_force(n, dim, _pd(p), _pd(dm), _pd(b), kind, C.c_double(eps),
                                  C.c_double(sigma), C.c_double(r_cut), shift, _pi(nbr_idx),
                                  _pi(nbr_count), cap, _pd(f), _pd(e_i), C.byref(E), _par(params)),
           "energy_force")
    return f, e_i, float(E.value)


def needs_rebuild(pos, ref, box, dim, skin):
    p = _d(pos3(pos)); r = _d(pos3(ref)); b = _d(box)
    flag = C.c_int32(0); m = C.c_double(0)
    _check(lib().orc_needs_rebuild(p.shape[0], dim, _pd(p), _pd(r), _pd(b), C.c_double(skin),
                                   C.byref(flag), C.byref(m)), "needs_rebuild")
    return int(flag.value), float(m.value)


def nve_run(pos, vel, force, diam, box, dim, kind, eps, sigma, r_cut, shift, dt, mass,
            nsteps, use_list=0, skin=0.0, capacity=128, want_energies=True, alpha=None, params=None):
    """Returns (pos, vel, force, energies[(nsteps+1),2] or None, stats[3])."""
    if alpha is not None:
        (default_params() if params is None else params).morse_alpha = float(alpha)
    p = _d(pos3(pos)).copy(); v = _d(pos3(vel)).copy(); f = _d(pos3(force)).copy()
    b = _d(box)
    dm = _d(diam) if diam is not None else None
    en = np.zeros((nsteps + 1, 2), dtype=np.float64) if want_energies else None
    stats = np.zeros(3, dtype=np.int32)
    _check(lib().orc_nve_run(p.shape[0], dim, _pd(p), _pd(v), _pd(f), _pd(dm), _pd(b), kind,
                             C.c_double(eps), C.c_double(sigma), C.c_double(r_cut), shift,
                             C.c_double(dt), C.c_double(mass), nsteps, use_list,
                             C.c_float(skin), capacity, _pd(en), _pi(stats), _par(params)), "nve_run")
    return p, v, f, en, stats


FIRE_DEFAULT = (0.01, 0.1, 5, 1.1, 0.5, 0.1, 0.99)   # dt_start, dt_max, n_min, f_inc, f_dec, alpha_start, f_alpha


def fire_run(pos, vel, diam, box, dim, kind, eps, sigma, r_cut, shift, nsteps, par=FIRE_DEFAULT,
             state=None, alpha_morse=None, params=None):
    """Returns (pos, vel, force, energies[nsteps+1], state[3] = (dt, alpha, n_pos))."""
    if alpha_morse is not None:
        (default_params() if params is None else params).morse_alpha = float(alpha_morse)
    p = _d(pos3(pos)).copy(); v = _d(pos3(vel)).copy(); f = np.zeros_like(p)
    b = _d(box)
    dm = _d(diam) if diam is not None else None
    pr = _d(par)
    st = _d(state) if state is not None else np.zeros(3, dtype=np.float64)
    st = st.copy()
    en = np.zeros(nsteps + 1, dtype=np.float64)
    _check(lib().orc_fire_run(p.shape[0], dim, _pd(p), _pd(v), _pd(f), _pd(dm), _pd(b), kind,
                              C.c_double(eps), C.c_double(sigma), C.c_double(r_cut), shift,
                              _pd(pr), _pd(st), nsteps, _pd(en), _par(params)), "fire_run")
    return p, v, f, en, st


def normals(seed, step, n, dim):
    """The counter-based standard normals of step `step` for particles 0..n-1, float64[n,3]."""
    out = np.zeros((n, 3), dtype=np.float64)
    lib().orc_normals(C.c_uint32(seed), C.c_uint32(step), n, dim, _pd(out))
    return out


def brownian_run(pos, diam, box, dim, kind, eps, sigma, r_cut, shift, dt, gamma, kT, seed, nsteps,
                 step0=0, alpha_morse=None, params=None):
    """Returns (pos, force, energies[nsteps+1])."""
    if alpha_morse is not None:
        (default_params() if params is None else params).morse_alpha = float(alpha_morse)
    p = _d(pos3(pos)).copy(); f = np.zeros_like(p)
    b = _d(box)
    dm = _d(diam) if diam is not None else None
    en = np.zeros(nsteps + 1, dtype=np.float64)
    _check(lib().orc_brownian_run(p.shape[0], dim, _pd(p), _pd(f), _pd(dm), _pd(b), kind, C.c_double(eps),
                                  C.c_double(sigma), C.c_double(r_cut), shift, C.c_double(dt),
                                  C.c_double(gamma), C.c_double(kT), C.c_uint32(seed), C.c_uint32(step0),
                                  nsteps, _pd(en), _par(params)), "brownian_run")
    return p, f, en


def langevin_run(pos, vel, force, diam, box, dim, kind, eps, sigma, r_cut, shift, dt, mass, gamma, kT,
                 seed, nsteps, step0=0, params=None):
    """BAOAB Langevin; returns (pos, vel, force)."""
    p = _d(pos3(pos)).copy(); v = _d(pos3(vel)).copy(); f = _d(pos3(force)).copy()
    b = _d(box)
    dm = _d(diam) if diam is not None else None
    _check(lib().orc_langevin_run(p.shape[0], dim, _pd(p), _pd(v), _pd(f), _pd(dm), _pd(b), kind,
                                  C.c_double(eps), C.c_double(sigma), C.c_double(r_cut), shift,
                                  C.c_double(dt), C.c_double(mass), C.c_double(gamma), C.c_double(kT),
                                  C.c_uint32(seed), C.c_uint32(step0), nsteps, _par(params)), "langevin_run")
    return p, v, f


def nose_hoover_run(pos, vel, diam, box, dim, kind, eps, sigma, r_cut, shift, dt, mass, kT, tau, nsteps,
                    state=None, chain=1, params=None):
    """Returns (pos, vel, force, conserved[nsteps+1], state[2*chain] = (xi_1.., v_xi_1..))."""
    p = _d(pos3(pos)).copy(); v = _d(pos3(vel)).copy(); f = np.zeros_like(p)
    b = _d(box)
    dm = _d(diam) if diam is not None else None
    st = (_d(state) if state is not None else np.zeros(2 * chain, dtype=np.float64)).copy()
    assert st.shape == (2 * chain,)
    cons = np.zeros(nsteps + 1, dtype=np.float64)
    (default_params() if params is None else params).nh_chain = int(chain)
    _check(lib().orc_nose_hoover_run(p.shape[0], dim, _pd(p), _pd(v), _pd(f), _pd(dm), _pd(b), kind,
                                     C.c_double(eps), C.c_double(sigma), C.c_double(r_cut), shift,
                                     C.c_double(dt), C.c_double(mass), C.c_double(kT), C.c_double(tau),
                                     _pd(st), nsteps, _pd(cons), _par(params)), "nose_hoover_run")
    return p, v, f, cons, st


def flock_energy_grad(pos, theta, box, par):
    """par = (J_al, R_al, J_av, R_av, J_co, R_co, alpha). Returns (energies[3], gR[n,2], gtheta[n])."""
    p = _d(pos3(pos)); th = _d(theta); b = _d(box); pr = _d(par)
    n = p.shape[0]
    en = np.zeros(3); gR = np.zeros((n, 2)); gth = np.zeros(n)
    _check(lib().orc_flock_energy_grad(n, _pd(p), _pd(th), _pd(b), _pd(pr), _pd(en), _pd(gR), _pd(gth)),
           "flock_energy_grad")
    return en, gR, gth


def flock_obstacle_energy_grad(pos, theta, box, centre, radius, J, alpha):
    """Eq. 11 alone: returns (energy, gR[n,2], gtheta[n]) of the obstacle term."""
    p = _d(pos3(pos)); th = _d(theta); b = _d(box)
    c = _d(np.asarray(centre, np.float64).reshape(-1, 2)); r = _d(radius)
    n = p.shape[0]
    en = np.zeros(1); gR = np.zeros((n, 2)); gth = np.zeros(n)
    _check(lib().orc_flock_obstacle_energy_grad(n, _pd(p), _pd(th), _pd(b), int(c.shape[0]), _pd(c), _pd(r),
                                                C.c_double(J), C.c_double(alpha), _pd(en), _pd(gR), _pd(gth)),
           "flock_obstacle_energy_grad")
    return float(en[0]), gR, gth


def flock_set_obstacles(centre=(), radius=(), J=0.0):
    """Obstacles seen by flock_run from now on (none: call without arguments)."""
    c = _d(np.asarray(centre, np.float64).reshape(-1, 2)); r = _d(np.asarray(radius, np.float64).reshape(-1))
    _check(lib().orc_flock_set_obstacles(int(c.shape[0]), _pd(c), _pd(r), C.c_double(J)), "flock_set_obstacles")


def predator_energy_grad(pos, box, ppos, pth, J, R):
    """The predators' chase term (eq. 13): returns (energy, gR[np,2], gtheta[np])."""
    p = _d(pos3(pos)); b = _d(box)
    pp = _d(np.asarray(ppos, np.float64).reshape(-1, 2)); pt = _d(pth)
    k = pp.shape[0]
    en = np.zeros(1); gR = np.zeros((k, 2)); gth = np.zeros(k)
    _check(lib().orc_predator_energy_grad(p.shape[0], _pd(p), _pd(b), k, _pd(pp), _pd(pt), C.c_double(J),
                                          C.c_double(R), _pd(en), _pd(gR), _pd(gth)), "predator_energy_grad")
    return float(en[0]), gR, gth


def flock_run_predators(pos, theta, box, par, speed, dt, nsteps, ppos, pth, ppar):
    """Boids and predators together; ppar = (J_flee, R_flee, J_chase, R_chase, speed_pred).
    Returns (pos, theta, ppos, ptheta)."""
    p = _d(pos3(pos)).copy(); th = _d(theta).copy(); b = _d(box); pr = _d(par)
    pp = _d(np.asarray(ppos, np.float64).reshape(-1, 2)).copy(); pt = _d(pth).copy(); pq = _d(ppar)
    _check(lib().orc_flock_run_predators(p.shape[0], _pd(p), _pd(th), _pd(b), _pd(pr), C.c_double(speed),
                                         C.c_double(dt), nsteps, pp.shape[0], _pd(pp), _pd(pt), _pd(pq)),
           "flock_run_predators")
    return p, th, pp, pt


def flock_run(pos, theta, box, par, speed, dt, nsteps):
    p = _d(pos3(pos)).copy(); th = _d(theta).copy(); b = _d(box); pr = _d(par)
    _check(lib().orc_flock_run(p.shape[0], _pd(p), _pd(th), _pd(b), _pd(pr), C.c_double(speed), C.c_double(dt),
                               nsteps), "flock_run")
    return p, th
