"""Thin ctypes binding over libmd_b200.so -- same names as include/md.h.

Argument marshalling only: every step of the path runs in the CUDA kernels
behind the C ABI.  PyTorch is used for device memory and streams.  There is no
CPU fallback: if the library is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

MD_OK, MD_EINVAL, MD_EBOX, MD_EWORKSPACE, MD_ECUDA = 0, -1, -2, -3, -4
MD_KIND_LJ, MD_KIND_SOFT, MD_KIND_MORSE, MD_KIND_BUCKINGHAM, MD_KIND_LJ_SPECIES, MD_KIND_BKS = 0, 1, 2, 3, 4, 5

SYMBOLS = [
    "md_last_error", "md_workspace_bytes", "md_create", "md_destroy", "md_set_option",
    "md_num_cells", "md_nbr_layout", "md_cell_list_build", "md_neighbor_list_build",
    "md_cell_list_static", "md_get_option", "md_needs_rebuild", "md_pair_energy_force", "md_nve_step", "md_nve_run_host", "md_counters",
    "md_nve_run_host_release", "md_fire_minimize", "md_brownian_step",
    "md_langevin_step", "md_nose_hoover_step", "md_set_species_lj",
    "md_flock_step", "md_flock_obstacles", "md_set_species_bks", "md_flock_predators",
    "md_set_range", "md_kick_drift", "md_half_kick", "md_force_half_kick",
    "md_slab_kick_drift", "md_slab_convert", "md_slab_pack", "md_slab_unpack",
    "md_slab_force_half_kick", "md_slab_step_open", "md_slab_step_close", "md_slab_split", "md_slab_append", "md_slab_border", "md_slab_load", "md_slab_plan",
]


class md_config(C.Structure):
    _fields_ = [("dim", C.c_int), ("box", C.c_float * 3), ("r_cut", C.c_float),
                ("skin", C.c_float), ("capacity", C.c_int), ("resort", C.c_int)]


class md_potential(C.Structure):
    _fields_ = [("kind", C.c_int), ("epsilon", C.c_float), ("sigma", C.c_float),
                ("r_cut", C.c_float), ("shift", C.c_int), ("alpha", C.c_float)]


class md_fire_params(C.Structure):
    _fields_ = [("dt_start", C.c_float), ("dt_max", C.c_float), ("n_min", C.c_int),
                ("f_inc", C.c_float), ("f_dec", C.c_float), ("alpha_start", C.c_float),
                ("f_alpha", C.c_float)]


class md_flock_params(C.Structure):
    _fields_ = [("J_align", C.c_float), ("R_align", C.c_float), ("J_avoid", C.c_float), ("R_avoid", C.c_float),
                ("J_cohesion", C.c_float), ("R_cohesion", C.c_float), ("alpha", C.c_float), ("speed", C.c_float)]


class md_slab_frame(C.Structure):
    _fields_ = [("kind", C.c_int), ("T", C.c_float), ("Lx", C.c_float), ("L", C.c_float),
                ("g2l_thr", C.c_float), ("l2g_thr", C.c_float)]


class md_predator_params(C.Structure):
    _fields_ = [("J_flee", C.c_float), ("R_flee", C.c_float), ("J_chase", C.c_float), ("R_chase", C.c_float),
                ("speed", C.c_float)]


class MdError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"libmd_b200 error {code}: {text}")
        self.code = code


_lib = None


def lib():
    """Load libmd_b200.so (built in-tree by build.py); raise if it is not there."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if not os.path.exists(path):
            raise RuntimeError(
                f"{path} is missing: build it with `python -m paper_1912_04232_b200.build` "
                "(nvcc, sm_100a). There is no CPU fallback.")
        L = C.CDLL(path)
        L.md_last_error.restype = C.c_char_p
        for name in SYMBOLS:
            getattr(L, name)           # AttributeError if the ABI lost a symbol
        vp, ip = C.c_void_p, C.c_void_p
        L.md_workspace_bytes.argtypes = [C.POINTER(md_config), C.c_int, C.POINTER(C.c_size_t)]
        L.md_create.argtypes = [C.POINTER(md_config), C.c_int, vp, C.c_size_t, C.POINTER(vp)]
        L.md_destroy.argtypes = [vp]
        L.md_set_option.argtypes = [vp, C.c_char_p, C.c_double]
        L.md_get_option.argtypes = [vp, C.c_char_p, C.POINTER(C.c_double)]
        L.md_counters.argtypes = [vp, ip, C.c_int, vp]
        L.md_set_species_lj.argtypes = [vp, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.md_brownian_step.argtypes = [vp, C.POINTER(md_potential), vp, vp, ip, ip, ip, C.c_float, C.c_float,
                                       C.c_float, C.c_uint32, C.c_uint32, C.c_int, ip, vp]
        L.md_langevin_step.argtypes = [vp, C.POINTER(md_potential), vp, vp, vp, ip, ip, ip, C.c_float, C.c_float,
                                       C.c_float, C.c_float, C.c_uint32, C.c_uint32, C.c_int, ip, vp]
        L.md_nose_hoover_step.argtypes = [vp, C.POINTER(md_potential), vp, vp, vp, ip, ip, ip, C.c_float,
                                          C.c_float, C.c_float, C.c_float, vp, C.c_int, ip, vp]
        L.md_set_species_bks.argtypes = [vp, C.c_int] + [C.POINTER(C.c_float)] * 4 + [C.c_float, C.c_float]
        L.md_set_range.argtypes = [vp, C.c_int, C.c_int]
        L.md_kick_drift.argtypes = [vp, vp, vp, vp, C.c_float, C.c_float, ip, vp]
        L.md_force_half_kick.argtypes = [vp, C.POINTER(md_potential), vp, ip, ip, vp, vp, C.c_float, C.c_float, vp]
        L.md_half_kick.argtypes = [vp, vp, vp, C.c_float, C.c_float, vp]
        L.md_slab_kick_drift.argtypes = [vp, C.POINTER(md_slab_frame), vp, vp, vp, ip, C.c_float, C.c_float, ip, ip, vp]
        L.md_slab_force_half_kick.argtypes = [vp, C.POINTER(md_potential), vp, ip, ip, vp, vp, C.c_float, C.c_float,
                                              ip, ip, ip, vp]
        L.md_slab_convert.argtypes = [C.POINTER(md_slab_frame), vp, C.c_int, C.c_int, vp]
        L.md_slab_pack.argtypes = [C.POINTER(md_slab_frame), vp, ip, C.c_int, vp, vp]
        L.md_slab_unpack.argtypes = [C.POINTER(md_slab_frame), vp, ip, C.c_int, vp, vp]
        L.md_slab_step_open.argtypes = [vp, C.POINTER(md_slab_frame), vp, vp, vp, ip, C.c_float, C.c_float, ip, ip,
                                        ip, C.c_int, vp, ip, C.c_int, vp, vp]
        L.md_slab_step_close.argtypes = [vp, C.POINTER(md_slab_frame), C.POINTER(md_potential), vp, ip, C.c_int, vp, ip,
                                         C.c_int, vp, ip, ip, vp, vp, C.c_float, C.c_float, ip, ip, ip, vp]
        L.md_slab_split.argtypes = [C.POINTER(md_slab_frame), C.c_float, C.c_float, vp, vp, ip, C.c_int, vp, vp, ip,
                                    vp, ip, vp, ip, C.c_int, ip, vp]
        L.md_slab_append.argtypes = [vp, ip, C.c_int, C.c_float, C.c_float, vp, vp, ip, C.c_int, ip, vp]
        L.md_slab_border.argtypes = [C.c_float, C.c_float, vp, ip, C.c_int, vp, ip, vp, ip, C.c_int, ip, ip, ip, vp]
        L.md_slab_load.argtypes = [C.POINTER(md_slab_frame), vp, vp, ip, C.c_int, vp, ip, C.c_int, vp, ip, C.c_int,
                                   vp, vp, ip, ip, vp]
        L.md_slab_plan.argtypes = [ip, C.c_int, ip, ip, ip, ip, ip, ip, ip, vp]
        L.md_flock_predators.argtypes = [vp, C.c_int, vp, C.POINTER(md_predator_params)]
        L.md_flock_obstacles.argtypes = [vp, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_float), C.c_float]
        L.md_flock_step.argtypes = [vp, C.POINTER(md_flock_params), vp, ip, ip, ip, C.c_float, C.c_int, ip, vp]
        L.md_fire_minimize.argtypes = [vp, C.POINTER(md_potential), C.POINTER(md_fire_params), vp, vp, vp,
                                       ip, ip, ip, vp, C.c_int, ip, vp]
        L.md_num_cells.argtypes = [vp, C.POINTER(C.c_int * 3)]
        L.md_nbr_layout.argtypes = [vp] + [C.POINTER(C.c_long)] * 5
        L.md_cell_list_build.argtypes = [vp, vp, vp, ip, ip, ip, vp]
        L.md_cell_list_static.argtypes = [C.POINTER(md_config), C.c_int, vp, ip, ip, vp, vp]
        L.md_neighbor_list_build.argtypes = [vp, vp, ip, ip, ip, ip, ip, vp]
        L.md_needs_rebuild.argtypes = [vp, vp, ip, vp]
        L.md_pair_energy_force.argtypes = [vp, C.POINTER(md_potential), vp, ip, ip, vp, vp, vp]
        L.md_nve_step.argtypes = [vp, C.POINTER(md_potential), vp, vp, vp, ip, ip, ip,
                                  C.c_float, C.c_float, C.c_int, ip, vp]
        L.md_nve_run_host.argtypes = [C.POINTER(md_config), C.POINTER(md_potential), C.c_int, vp,
                                      vp, vp, C.POINTER(C.c_double), C.c_float, C.c_float, C.c_int,
                                      vp]
        _lib = L
    return _lib


def _check(rc):
    if rc != MD_OK:
        raise MdError(rc, md_last_error())


def _ptr(t):
    """Device (or host, for *_host calls) address of a tensor / array, or NULL."""
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        assert t.is_contiguous()
        return t.data_ptr()
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    return int(t)


def _stream(stream):
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream
    return int(stream)


def make_config(dim, box, r_cut, skin, capacity, resort=1) -> md_config:
    b = [float(x) for x in box] + [1.0] * (3 - len(box))
    return md_config(int(dim), (C.c_float * 3)(*b[:3]), float(r_cut), float(skin), int(capacity),
                     int(resort))


def make_potential(kind, epsilon=1.0, sigma=1.0, r_cut=2.5, shift=1, alpha=0.0) -> md_potential:
    return md_potential(int(kind), float(epsilon), float(sigma), float(r_cut), int(shift), float(alpha))


# ------------------------------------------------------------ the C ABI, same names ----

def md_last_error() -> str:
    return lib().md_last_error().decode()


def md_workspace_bytes(cfg: md_config, n: int) -> int:
    out = C.c_size_t(0)
    _check(lib().md_workspace_bytes(C.byref(cfg), n, C.byref(out)))
    return int(out.value)


def md_create(cfg: md_config, n: int, workspace: torch.Tensor):
    h = C.c_void_p(None)
    _check(lib().md_create(C.byref(cfg), n, _ptr(workspace), workspace.numel() * workspace.element_size(),
                           C.byref(h)))
    return h


def md_destroy(sys) -> None:
    _check(lib().md_destroy(sys))


def md_set_option(sys, name: str, value: float) -> None:
    _check(lib().md_set_option(sys, name.encode(), float(value)))


def md_get_option(sys, name: str) -> float:
    v = C.c_double(0.0)
    _check(lib().md_get_option(sys, name.encode(), C.byref(v)))
    return float(v.value)


def md_brownian_step(sys, pot: md_potential, pos, force, id, nbr_idx, nbr_count, dt, gamma, kT, seed, step0,
                     nsteps, stats, stream=None) -> None:
    _check(lib().md_brownian_step(sys, C.byref(pot), _ptr(pos), _ptr(force), _ptr(id), _ptr(nbr_idx),
                                  _ptr(nbr_count), float(dt), float(gamma), float(kT), int(seed), int(step0),
                                  int(nsteps), _ptr(stats), _stream(stream)))


def md_langevin_step(sys, pot: md_potential, pos, vel, force, id, nbr_idx, nbr_count, dt, mass, gamma, kT,
                     seed, step0, nsteps, stats, stream=None) -> None:
    _check(lib().md_langevin_step(sys, C.byref(pot), _ptr(pos), _ptr(vel), _ptr(force), _ptr(id),
                                  _ptr(nbr_idx), _ptr(nbr_count), float(dt), float(mass), float(gamma),
                                  float(kT), int(seed), int(step0), int(nsteps), _ptr(stats), _stream(stream)))


def md_nose_hoover_step(sys, pot: md_potential, pos, vel, force, id, nbr_idx, nbr_count, dt, mass, kT, tau,
                        nh_state, nsteps, stats, stream=None) -> None:
    _check(lib().md_nose_hoover_step(sys, C.byref(pot), _ptr(pos), _ptr(vel), _ptr(force), _ptr(id),
                                     _ptr(nbr_idx), _ptr(nbr_count), float(dt), float(mass), float(kT),
                                     float(tau), _ptr(nh_state), int(nsteps), _ptr(stats), _stream(stream)))


def md_flock_obstacles(sys, centre=(), radius=(), J=0.0) -> None:
    import numpy as np
    c = np.ascontiguousarray(np.asarray(centre, np.float32).reshape(-1, 2))
    r = np.ascontiguousarray(np.asarray(radius, np.float32).reshape(-1))
    if c.shape[0] != r.shape[0]:
        raise ValueError("one radius per centre")
    fp = C.POINTER(C.c_float)
    _check(lib().md_flock_obstacles(sys, int(r.shape[0]), c.ctypes.data_as(fp), r.ctypes.data_as(fp), float(J)))


def md_flock_predators(sys, pred=None, par: md_predator_params | None = None) -> None:
    """pred: device float32[npred, 4] tensor (x, y, 0, theta), kept by pointer; None removes the predators."""
    if pred is None:
        _check(lib().md_flock_predators(sys, 0, None, None))
    else:
        _check(lib().md_flock_predators(sys, int(pred.shape[0]), _ptr(pred), C.byref(par)))


def md_flock_step(sys, par: md_flock_params, pos, id, nbr_idx, nbr_count, dt, nsteps, stats, stream=None) -> None:
    _check(lib().md_flock_step(sys, C.byref(par), _ptr(pos), _ptr(id), _ptr(nbr_idx), _ptr(nbr_count), float(dt),
                               int(nsteps), _ptr(stats), _stream(stream)))


def md_fire_minimize(sys, pot: md_potential, par: md_fire_params, pos, vel, force, id, nbr_idx, nbr_count,
                     fire_state, nsteps, stats, stream=None) -> None:
    _check(lib().md_fire_minimize(sys, C.byref(pot), C.byref(par), _ptr(pos), _ptr(vel), _ptr(force),
                                  _ptr(id), _ptr(nbr_idx), _ptr(nbr_count), _ptr(fire_state), int(nsteps),
                                  _ptr(stats), _stream(stream)))


def md_nve_run_host_release() -> None:
    _check(lib().md_nve_run_host_release())


def md_set_species_lj(sys, epsilon, sigma, r_cut) -> None:
    """Square host arrays eps_ab, sigma_ab, rc_ab (up to 4 x 4)."""
    import numpy as np
    e = np.ascontiguousarray(epsilon, dtype=np.float32); sg = np.ascontiguousarray(sigma, dtype=np.float32)
    r = np.ascontiguousarray(r_cut, dtype=np.float32)
    fp = C.POINTER(C.c_float)
    _check(lib().md_set_species_lj(sys, int(e.shape[0]), e.ctypes.data_as(fp), sg.ctypes.data_as(fp),
                                   r.ctypes.data_as(fp)))


def md_set_species_bks(sys, A, B, Cc, charge, coulomb_alpha, k_e=1.0) -> None:
    import numpy as np
    q = np.ascontiguousarray(np.asarray(charge, np.float32).reshape(-1))
    ns = q.shape[0]
    tabs = [np.ascontiguousarray(np.asarray(t, np.float32).reshape(ns * ns)) for t in (A, B, Cc)]
    fp = C.POINTER(C.c_float)
    _check(lib().md_set_species_bks(sys, ns, *[t.ctypes.data_as(fp) for t in tabs], q.ctypes.data_as(fp),
                                    float(coulomb_alpha), float(k_e)))


def md_set_range(sys, begin: int, end: int) -> None:
    _check(lib().md_set_range(sys, int(begin), int(end)))


def md_kick_drift(sys, pos, vel, force, dt, mass, flag, stream=None) -> None:
    _check(lib().md_kick_drift(sys, _ptr(pos), _ptr(vel), _ptr(force), float(dt), float(mass), _ptr(flag),
                               _stream(stream)))


def md_force_half_kick(sys, pot: md_potential, pos, nbr_idx, nbr_count, force, vel, dt, mass, stream=None) -> None:
    _check(lib().md_force_half_kick(sys, C.byref(pot), _ptr(pos), _ptr(nbr_idx), _ptr(nbr_count), _ptr(force),
                                    _ptr(vel), float(dt), float(mass), _stream(stream)))


def md_slab_kick_drift(sys, frame: md_slab_frame, pos, vel, force, id, dt, mass, flag, stop=None, stream=None) -> None:
    _check(lib().md_slab_kick_drift(sys, C.byref(frame), _ptr(pos), _ptr(vel), _ptr(force), _ptr(id), float(dt), float(mass),
                                    _ptr(flag), _ptr(stop), _stream(stream)))


def md_slab_force_half_kick(sys, pot, pos, nbr_idx, nbr_count, force, vel, dt, mass, flag, stop, done,
                            stream=None) -> None:
    _check(lib().md_slab_force_half_kick(sys, C.byref(pot), _ptr(pos), _ptr(nbr_idx), _ptr(nbr_count), _ptr(force),
                                         _ptr(vel), float(dt), float(mass), _ptr(flag), _ptr(stop), _ptr(done),
                                         _stream(stream)))


def md_slab_convert(frame: md_slab_frame, pos, n, to_local, stream=None) -> None:
    _check(lib().md_slab_convert(C.byref(frame), _ptr(pos), int(n), int(to_local), _stream(stream)))


def md_slab_pack(frame: md_slab_frame, pos, slots, rows_out, stream=None) -> None:
    _check(lib().md_slab_pack(C.byref(frame), _ptr(pos), _ptr(slots), int(slots.numel()), _ptr(rows_out), _stream(stream)))


def md_slab_unpack(frame: md_slab_frame, rows, slots, pos, stream=None) -> None:
    _check(lib().md_slab_unpack(C.byref(frame), _ptr(rows), _ptr(slots), int(slots.numel()), _ptr(pos), _stream(stream)))


def md_slab_step_open(sys, frame: md_slab_frame, pos, vel, force, id, dt, mass, flag, stop, border_prev, rows_prev,
                      border_next, rows_next, stream=None) -> None:
    _check(lib().md_slab_step_open(sys, C.byref(frame), _ptr(pos), _ptr(vel), _ptr(force), _ptr(id), float(dt),
                                   float(mass), _ptr(flag), _ptr(stop), _ptr(border_prev), int(border_prev.numel()),
                                   _ptr(rows_prev), _ptr(border_next), int(border_next.numel()), _ptr(rows_next),
                                   _stream(stream)))


def md_slab_step_close(sys, frame: md_slab_frame, pot, rows_prev, halo_prev, rows_next, halo_next, pos, nbr_idx,
                       nbr_count, force, vel, dt, mass, flag, stop, done, stream=None) -> None:
    _check(lib().md_slab_step_close(sys, C.byref(frame), C.byref(pot), _ptr(rows_prev), _ptr(halo_prev),
                                    int(halo_prev.numel()), _ptr(rows_next), _ptr(halo_next), int(halo_next.numel()),
                                    _ptr(pos), _ptr(nbr_idx), _ptr(nbr_count), _ptr(force), _ptr(vel), float(dt),
                                    float(mass), _ptr(flag), _ptr(stop), _ptr(done), _stream(stream)))


def md_slab_split(frame: md_slab_frame, lo, hi, pos, vel, id, n, own_pos, own_vel, own_id, prev_rows, prev_ids,
                  next_rows, next_ids, cap_rows, counts, stream=None) -> None:
    _check(lib().md_slab_split(C.byref(frame), float(lo), float(hi), _ptr(pos), _ptr(vel), _ptr(id), int(n),
                               _ptr(own_pos), _ptr(own_vel), _ptr(own_id), _ptr(prev_rows), _ptr(prev_ids),
                               _ptr(next_rows), _ptr(next_ids), int(cap_rows), _ptr(counts), _stream(stream)))


def md_slab_append(rows, ids, m, lo, hi, own_pos, own_vel, own_id, offset, errors, stream=None) -> None:
    _check(lib().md_slab_append(_ptr(rows), _ptr(ids), int(m), float(lo), float(hi), _ptr(own_pos), _ptr(own_vel),
                                _ptr(own_id), int(offset), _ptr(errors), _stream(stream)))


def md_slab_border(lo_edge, hi_edge, own_pos, own_id, n_own, prev_rows, prev_ids, next_rows, next_ids, cap_rows,
                   map_prev, map_next, counts, stream=None) -> None:
    _check(lib().md_slab_border(float(lo_edge), float(hi_edge), _ptr(own_pos), _ptr(own_id), int(n_own),
                                _ptr(prev_rows), _ptr(prev_ids), _ptr(next_rows), _ptr(next_ids), int(cap_rows),
                                _ptr(map_prev), _ptr(map_next), _ptr(counts), _stream(stream)))


def md_slab_load(frame: md_slab_frame, own_pos, own_vel, own_id, n_own, hp_rows, hp_ids, h_prev, hn_rows, hn_ids,
                 h_next, pos, vel, id, map_halo, stream=None) -> None:
    _check(lib().md_slab_load(C.byref(frame), _ptr(own_pos), _ptr(own_vel), _ptr(own_id), int(n_own), _ptr(hp_rows),
                              _ptr(hp_ids), int(h_prev), _ptr(hn_rows), _ptr(hn_ids), int(h_next), _ptr(pos),
                              _ptr(vel), _ptr(id), _ptr(map_halo), _stream(stream)))


def md_slab_plan(id, n, nbr_count, map_prev, map_next, map_halo, border_prev, border_next, halo_slots,
                 stream=None) -> None:
    _check(lib().md_slab_plan(_ptr(id), int(n), _ptr(nbr_count), _ptr(map_prev), _ptr(map_next), _ptr(map_halo),
                              _ptr(border_prev), _ptr(border_next), _ptr(halo_slots), _stream(stream)))


def md_half_kick(sys, vel, force, dt, mass, stream=None) -> None:
    _check(lib().md_half_kick(sys, _ptr(vel), _ptr(force), float(dt), float(mass), _stream(stream)))


def md_counters(sys, out, reset=False, stream=None) -> None:
    _check(lib().md_counters(sys, _ptr(out), int(reset), _stream(stream)))


def md_num_cells(sys):
    out = (C.c_int * 3)()
    _check(lib().md_num_cells(sys, C.byref(out)))
    return [int(out[0]), int(out[1]), int(out[2])]


def md_nbr_layout(sys):
    """(tile, tile_stride, particle_stride, slot_stride, length), see include/md.h."""
    v = [C.c_long(0) for _ in range(5)]
    _check(lib().md_nbr_layout(sys, *[C.byref(x) for x in v]))
    return tuple(int(x.value) for x in v)


def nbr_offsets(layout, n, capacity, device=None):
    """int64[n, capacity] offsets of entry (i, k) in a list buffer (index marshalling only)."""
    tile, tile_stride, p_stride, s_stride, _ = layout
    i = torch.arange(n, dtype=torch.int64, device=device)[:, None]
    k = torch.arange(capacity, dtype=torch.int64, device=device)[None, :]
    return (i // tile) * tile_stride + (i % tile) * p_stride + k * s_stride


def md_cell_list_build(sys, pos, vel, id, cell_start, perm, stream=None) -> None:
    _check(lib().md_cell_list_build(sys, _ptr(pos), _ptr(vel), _ptr(id), _ptr(cell_start), _ptr(perm),
                                    _stream(stream)))


MD_STATIC_MAX_N, MD_STATIC_MAX_CELLS = 65536, 16384      # md.h


def md_cell_list_static(cfg: md_config, n, pos, cell_start, perm, pos_sorted, stream=None) -> None:
    """The cell list without a md_system, a workspace or any allocation (md.h): scratch is static in the library."""
    _check(lib().md_cell_list_static(C.byref(cfg), int(n), _ptr(pos), _ptr(cell_start), _ptr(perm),
                                     _ptr(pos_sorted), _stream(stream)))


def md_neighbor_list_build(sys, pos, cell_start, perm, nbr_idx, nbr_count, status, stream=None) -> None:
    _check(lib().md_neighbor_list_build(sys, _ptr(pos), _ptr(cell_start), _ptr(perm), _ptr(nbr_idx),
                                        _ptr(nbr_count), _ptr(status), _stream(stream)))


def md_needs_rebuild(sys, pos, flag, stream=None) -> None:
    _check(lib().md_needs_rebuild(sys, _ptr(pos), _ptr(flag), _stream(stream)))


def md_pair_energy_force(sys, pot: md_potential, pos, nbr_idx, nbr_count, force, energy_total=None,
                         stream=None) -> None:
    _check(lib().md_pair_energy_force(sys, C.byref(pot), _ptr(pos), _ptr(nbr_idx), _ptr(nbr_count),
                                      _ptr(force), _ptr(energy_total), _stream(stream)))


def md_nve_step(sys, pot: md_potential, pos, vel, force, id, nbr_idx, nbr_count, dt, mass, nsteps,
                stats, stream=None) -> None:
    _check(lib().md_nve_step(sys, C.byref(pot), _ptr(pos), _ptr(vel), _ptr(force), _ptr(id),
                             _ptr(nbr_idx), _ptr(nbr_count), float(dt), float(mass), int(nsteps),
                             _ptr(stats), _stream(stream)))


def md_nve_run_host(cfg: md_config, pot: md_potential, pos_host, vel_host, force_host, dt, mass,
                    nsteps, stats_host=None, want_energy=True):
    """HOST buffers in/out (numpy float32[n,4] or pinned CPU tensors). Returns the final
    potential energy (or None)."""
    n = pos_host.shape[0]
    e = C.c_double(0.0)
    _check(lib().md_nve_run_host(C.byref(cfg), C.byref(pot), n, _ptr(pos_host), _ptr(vel_host),
                                 _ptr(force_host), C.byref(e) if want_energy else None, float(dt),
                                 float(mass), int(nsteps), _ptr(stats_host)))
    return float(e.value) if want_energy else None


# -------------------------------------------------- device buffers for one system ------

class System:
    """Owns the torch tensors one simulation needs (allocation only; no arithmetic)."""

    def __init__(self, w, device="cuda:0", resort=None, capacity=None):
        self.w = w
        self.device = torch.device(device)
        self.cfg = make_config(w.dim, w.box, w.r_cut, w.skin, capacity or w.capacity,
                               w.resort if resort is None else resort)
        self.pot = make_potential(w.kind, w.epsilon, w.sigma, w.r_cut, w.shift, getattr(w, "alpha", 0.0))
        n, cap = w.n, self.cfg.capacity
        self.n, self.capacity = n, cap
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(md_workspace_bytes(self.cfg, n), dtype=torch.uint8,
                                         device=self.device)
            self.sys = md_create(self.cfg, n, self.workspace)
        ncell = md_num_cells(self.sys)
        self.cells = ncell[0] * ncell[1] * ncell[2]
        dev = self.device
        self.pos = torch.from_numpy(w.pos).to(dev)
        self.vel = torch.from_numpy(w.vel).to(dev)
        self.force = torch.zeros(n, 4, dtype=torch.float32, device=dev)
        self.id = torch.arange(n, dtype=torch.int32, device=dev)
        self.cell_start = torch.zeros(self.cells + 1, dtype=torch.int32, device=dev)
        self.perm = torch.zeros(n, dtype=torch.int32, device=dev)
        self.layout = md_nbr_layout(self.sys)
        self.nbr_idx = torch.full((self.layout[4],), -1, dtype=torch.int32, device=dev)
        self.nbr_count = torch.zeros(n, dtype=torch.int32, device=dev)
        self.status = torch.zeros(2, dtype=torch.int32, device=dev)
        self.flag = torch.zeros(1, dtype=torch.int32, device=dev)
        self.stats = torch.zeros(4, dtype=torch.int32, device=dev)
        self.energy = torch.zeros(1, dtype=torch.float64, device=dev)

    def nbr_rows(self):
        """The list as a dense int32[n, capacity] tensor (row i = neighbors of particle i)."""
        return self.nbr_idx[nbr_offsets(self.layout, self.n, self.capacity, self.device)]

    def set_nbr_rows(self, rows, counts):
        """Load a dense int32[n, capacity] list (e.g. one built elsewhere) into the layout."""
        off = nbr_offsets(self.layout, self.n, self.capacity, self.device)
        self.nbr_idx[off.reshape(-1)] = torch.as_tensor(rows, dtype=torch.int32, device=self.device).reshape(-1)
        self.nbr_count.copy_(torch.as_tensor(counts, dtype=torch.int32))

    def reset(self):
        self.pos.copy_(torch.from_numpy(self.w.pos))
        self.vel.copy_(torch.from_numpy(self.w.vel))
        self.id.copy_(torch.arange(self.n, dtype=torch.int32))

    def build(self, stream=None):
        md_cell_list_build(self.sys, self.pos, self.vel, self.id, self.cell_start, self.perm, stream)
        md_neighbor_list_build(self.sys, self.pos, self.cell_start, self.perm, self.nbr_idx,
                               self.nbr_count, self.status, stream)

    def compute_force(self, want_energy=True, stream=None):
        md_pair_energy_force(self.sys, self.pot, self.pos, self.nbr_idx, self.nbr_count, self.force,
                             self.energy if want_energy else None, stream)

    def step(self, nsteps, stream=None):
        md_nve_step(self.sys, self.pot, self.pos, self.vel, self.force, self.id, self.nbr_idx,
                    self.nbr_count, self.w.dt, self.w.mass, nsteps, self.stats, stream)

    def close(self):
        if self.sys is not None:
            torch.cuda.synchronize(self.device)
            md_destroy(self.sys)
            self.sys = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
