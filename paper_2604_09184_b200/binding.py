"""Thin ctypes face of libnbkick.so (include/nbkick.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch is used for device memory and
streams only: tensors are passed as raw device pointers.  There is no CPU fallback; if the shared
library is missing or cannot be loaded this module raises at import of the first call.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

from . import build as _build

NB_OK = 0
NB_E_NULL, NB_E_BADN, NB_E_BADARG, NB_E_WORKSPACE, NB_E_CUDA = -1, -2, -3, -4, -5
CHANGEOVER_RATIONAL, CHANGEOVER_QUINTIC = 0, 1
FORCE_AUTO, FORCE_TILES, FORCE_SYMMETRIC = 0, 1, 2
PRECISION_F64, PRECISION_MIXED = 0, 1

# every symbol include/nbkick.h declares (tests check the library exports each of them)
SYMBOLS = (
    "nb_default_config", "nb_configure", "nb_workspace_bytes", "nb_rcrit", "nb_kick", "nb_kick_static_setup", "nb_kick_static", "nb_shift",
    "nb_drift_kepler", "nb_midpoint_drag", "nb_step", "nb_groups", "nb_encounter", "nb_encounter_collide", "nb_encounter_levels", "nb_merge", "nb_kick_host", "nb_step_host", "nb_status", "nb_status_reset",
    "nb_last_force_ms", "nb_force_time", "nb_force_time_reset", "nb_force_geometry", "nb_fp64_peak", "nb_release", "nb_last_error", "nb_version",
)


class NbConfig(C.Structure):
    _fields_ = [
        ("stream", C.c_void_p),
        ("workspace", C.c_void_p),
        ("workspace_bytes", C.c_size_t),
        ("pair_capacity", C.c_int64),
        ("n_active", C.c_int64),
        ("G", C.c_double),
        ("n1", C.c_double),
        ("n2", C.c_double),
        ("changeover_kind", C.c_int),
        ("i_per_thread", C.c_int),
        ("j_splits", C.c_int),
        ("use_graph", C.c_int),
        ("reuse_acc", C.c_int),
        ("time_force", C.c_int),
        ("force_kernel", C.c_int),
        ("sym_block", C.c_int),
        ("resolve_encounters", C.c_int),
        ("bs_tol", C.c_double),
        ("radius_factor", C.c_double),
        ("sort_staging", C.c_int),
        ("levels", C.c_int),
        ("drag_gamma", C.c_double),
        ("drag_eta", C.c_double),
        ("drag_power", C.c_int),
        ("midpoint_iters", C.c_int),
        ("midpoint_tol", C.c_double),
        ("precision", C.c_int),
        ("slot_bytes_max", C.c_int64),
        ("collide_radius", C.c_void_p),
        ("collide_absorbed_by", C.c_void_p),
    ]


class NbError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libnbkick error {code}: {msg}")
        self.code = code


_lib = None


def lib_path() -> str:
    return _build.LIB


def load():
    """Load libnbkick.so (built in-tree by paper_2604_09184_b200/build.py).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -m paper_2604_09184_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(path)
    vp, dbl, i64, sz = C.c_void_p, C.c_double, C.c_int64, C.c_size_t
    lib.nb_default_config.argtypes = [C.POINTER(NbConfig)]
    lib.nb_default_config.restype = None
    lib.nb_configure.argtypes = [C.POINTER(NbConfig)]
    lib.nb_workspace_bytes.argtypes = [i64]
    lib.nb_workspace_bytes.restype = sz
    lib.nb_rcrit.argtypes = [vp, vp, vp, dbl, i64, dbl, vp]
    lib.nb_kick.argtypes = [vp, vp, vp, dbl, i64, dbl, vp, vp, vp, vp]
    lib.nb_kick_static.argtypes = [vp, vp, vp, dbl, i64, dbl, vp, vp, vp, vp, vp]
    lib.nb_kick_static_setup.argtypes = []
    lib.nb_shift.argtypes = [vp, vp, vp, dbl, i64, dbl]
    lib.nb_drift_kepler.argtypes = [vp, vp, dbl, i64, dbl]
    lib.nb_midpoint_drag.argtypes = [vp, vp, dbl, i64, dbl]
    lib.nb_step.argtypes = [vp, vp, vp, dbl, i64, dbl, vp, vp, vp, vp, i64]
    lib.nb_groups.argtypes = [vp, vp, i64, vp, vp, vp, vp]
    lib.nb_encounter.argtypes = [vp, vp, vp, vp, dbl, i64, dbl, vp, vp, vp]
    lib.nb_encounter_collide.argtypes = [vp, vp, vp, vp, vp, dbl, i64, dbl, vp, vp, vp, vp]
    lib.nb_encounter_levels.argtypes = [vp, vp, vp, vp, vp, dbl, i64, dbl, vp, vp]
    lib.nb_merge.argtypes = [vp, vp, vp, vp, i64, vp, vp, vp, vp]
    lib.nb_kick_host.argtypes = [vp, vp, vp, dbl, i64, dbl, vp, vp, vp, vp]
    lib.nb_step_host.argtypes = [vp, vp, vp, dbl, i64, dbl, vp, vp, vp, vp, i64]
    lib.nb_status.argtypes = [C.POINTER(C.c_int64)]
    lib.nb_status_reset.argtypes = []
    lib.nb_last_force_ms.argtypes = []
    lib.nb_last_force_ms.restype = dbl
    lib.nb_force_time.argtypes = [C.POINTER(C.c_int64), C.POINTER(dbl)]
    lib.nb_force_time_reset.argtypes = []
    lib.nb_force_geometry.argtypes = [i64, C.POINTER(C.c_int64)]
    lib.nb_fp64_peak.argtypes = [i64, C.POINTER(dbl), C.POINTER(dbl)]
    lib.nb_release.argtypes = []
    lib.nb_release.restype = None
    lib.nb_last_error.restype = C.c_char_p
    lib.nb_version.restype = C.c_char_p
    _lib = lib
    return lib


def _check(rc: int):
    if rc != NB_OK:
        raise NbError(rc, load().nb_last_error().decode())


def _dev(t, n_elem=None, dtype=None):
    """Raw device pointer of a contiguous CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    if n_elem is not None and t.numel() < n_elem:
        raise ValueError(f"tensor has {t.numel()} elements, need {n_elem}")
    return C.c_void_p(t.data_ptr())


def _host(a, n_elem=None, dtype=np.float64):
    if a is None:
        return None
    if not (isinstance(a, np.ndarray) and a.flags.c_contiguous and a.dtype == dtype):
        raise TypeError(f"expected a C-contiguous numpy array of {dtype}")
    if n_elem is not None and a.size < n_elem:
        raise ValueError("host array too small")
    return C.c_void_p(a.ctypes.data)


@dataclass
class Geometry:
    i_per_thread: int
    i_blocks: int
    j_splits: int
    threads: int
    tile_j: int


_state = dict(cfg=None, workspace=None)


def default_config() -> NbConfig:
    cfg = NbConfig()
    load().nb_default_config(C.byref(cfg))
    return cfg


def configure(N=None, *, stream=None, pair_capacity=0, n_active=0, G=None, n1=3.0, n2=0.4, changeover_kind=0,
              i_per_thread=0, j_splits=0, use_graph=True, reuse_acc=False, time_force=False,
              force_kernel=0, sym_block=0, resolve_encounters=False, bs_tol=1e-12, radius_factor=1.0, sort_staging=0, levels=0, drag_gamma=0.0, drag_eta=0.0, drag_power=0,
              midpoint_iters=50, midpoint_tol=1e-14, precision=0, slot_bytes_max=0, collide_radius=None, collide_absorbed_by=None,
              workspace_bytes=None,
              device="cuda"):
    """nb_configure with a torch-allocated workspace sized for N bodies (N=None: no workspace,
    enough for the _host calls; workspace_bytes: explicit size, e.g. the head that the O(N) calls
    need).  Keeps the workspace tensor alive."""
    lib = load()
    cfg = default_config()
    if G is not None:
        cfg.G = float(G)
    cfg.n1, cfg.n2 = float(n1), float(n2)
    cfg.pair_capacity = int(pair_capacity)
    cfg.n_active = int(n_active)
    cfg.changeover_kind = int(changeover_kind)
    cfg.i_per_thread, cfg.j_splits = int(i_per_thread), int(j_splits)
    cfg.use_graph = 1 if use_graph else 0
    cfg.reuse_acc = 1 if reuse_acc else 0
    cfg.time_force = 1 if time_force else 0
    cfg.force_kernel, cfg.sym_block = int(force_kernel), int(sym_block)
    cfg.resolve_encounters, cfg.bs_tol = (1 if resolve_encounters else 0), float(bs_tol)
    cfg.radius_factor = float(radius_factor)
    cfg.sort_staging = int(sort_staging)
    cfg.levels = int(levels)
    cfg.drag_gamma, cfg.drag_eta, cfg.drag_power = float(drag_gamma), float(drag_eta), int(drag_power)
    cfg.midpoint_iters, cfg.midpoint_tol = int(midpoint_iters), float(midpoint_tol)
    cfg.precision = int(precision)
    cfg.slot_bytes_max = int(slot_bytes_max)
    cfg.collide_radius = _dev(collide_radius, None, None)
    cfg.collide_absorbed_by = _dev(collide_absorbed_by, None, None)
    _state["collide"] = (collide_radius, collide_absorbed_by)   # keep the tensors alive
    if N is not None:
        import torch
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        cfg.stream = C.c_void_p(int(stream)) if stream else None
        _check(lib.nb_configure(C.byref(cfg)))  # tuning first: the workspace size depends on it
        nbytes = int(lib.nb_workspace_bytes(int(N))) if workspace_bytes is None else int(workspace_bytes)
        ws = torch.zeros(nbytes + 256, dtype=torch.uint8, device=device)
        off = (-ws.data_ptr()) % 256
        cfg.workspace = C.c_void_p(ws.data_ptr() + off)
        cfg.workspace_bytes = nbytes
        _state["workspace"] = ws
    else:
        cfg.stream = C.c_void_p(int(stream)) if stream else None
        _state["workspace"] = None
    _check(lib.nb_configure(C.byref(cfg)))
    _state["cfg"] = cfg
    return cfg


def workspace_bytes(N: int) -> int:
    return int(load().nb_workspace_bytes(int(N)))


def force_geometry(N: int) -> Geometry:
    out = (C.c_int64 * 5)()
    _check(load().nb_force_geometry(int(N), out))
    return Geometry(*[int(v) for v in out])


def nb_rcrit(x, v, m, M_star, dt, rcrit):
    import torch
    N = m.numel()
    _check(load().nb_rcrit(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), _dev(m, N, torch.float64),
                           float(M_star), N, float(dt), _dev(rcrit, N, torch.float64)))


def nb_kick(x, v, m, M_star, dt, rcrit, acc, pairs=None, npairs=None):
    import torch
    N = m.numel()
    _check(load().nb_kick(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), _dev(m, N, torch.float64),
                          float(M_star), N, float(dt), _dev(rcrit, N, torch.float64), _dev(acc, 3 * N, torch.float64),
                          _dev(pairs, None, torch.int32), _dev(npairs, 1, torch.int64)))


def nb_kick_static(x, v, m, M_star, dt, rcrit, acc, pairs=None, npairs=None, status8=None):
    """nb_kick with the scratch in the library's static device array (include/nbkick.h): allocates nothing."""
    import torch
    N = m.numel()
    _check(load().nb_kick_static(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), _dev(m, N, torch.float64),
                                 float(M_star), N, float(dt), _dev(rcrit, N, torch.float64), _dev(acc, 3 * N, torch.float64),
                                 _dev(pairs, None, torch.int32), _dev(npairs, 1, torch.int64), _dev(status8, 8, torch.int64)))


def nb_kick_static_setup():
    _check(load().nb_kick_static_setup())


def nb_shift(x, v, m, M_star, dt):
    import torch
    N = m.numel()
    _check(load().nb_shift(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), _dev(m, N, torch.float64),
                           float(M_star), N, float(dt)))


def nb_drift_kepler(x, v, M_star, dt):
    import torch
    N = x.numel() // 3
    _check(load().nb_drift_kepler(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), float(M_star), N,
                                  float(dt)))


def nb_midpoint_drag(x, v, M_star, dt):
    import torch
    N = x.numel() // 3
    _check(load().nb_midpoint_drag(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), float(M_star), N, float(dt)))


def nb_step(x, v, m, M_star, dt, rcrit, acc, pairs=None, npairs=None, nsteps=1):
    import torch
    N = m.numel()
    _check(load().nb_step(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), _dev(m, N, torch.float64),
                          float(M_star), N, float(dt), _dev(rcrit, N, torch.float64), _dev(acc, 3 * N, torch.float64),
                          _dev(pairs, None, torch.int32), _dev(npairs, 1, torch.int64), int(nsteps)))


def nb_groups(pairs, npairs, N, label, members, gstart, gstat):
    import torch
    _check(load().nb_groups(_dev(pairs, None, torch.int32), _dev(npairs, 1, torch.int64), int(N),
                            _dev(label, N, torch.int32), _dev(members, N, torch.int32),
                            _dev(gstart, N // 2 + 2, torch.int32), _dev(gstat, 4, torch.int64)))


def nb_encounter(x, v, m, rcrit, M_star, dt, members, gstart, gstat):
    import torch
    N = m.numel()
    _check(load().nb_encounter(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), _dev(m, N, torch.float64),
                               _dev(rcrit, N, torch.float64), float(M_star), N, float(dt), _dev(members, N, torch.int32),
                               _dev(gstart, N // 2 + 2, torch.int32), _dev(gstat, 4, torch.int64)))


def nb_encounter_collide(x, v, m, radius, rcrit, M_star, dt, members, gstart, gstat, absorbed_by):
    import torch
    N = m.numel()
    _check(load().nb_encounter_collide(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), _dev(m, N, torch.float64),
                                       _dev(radius, N, torch.float64), _dev(rcrit, N, torch.float64), float(M_star), N, float(dt),
                                       _dev(members, N, torch.int32), _dev(gstart, N // 2 + 2, torch.int32),
                                       _dev(gstat, 4, torch.int64), _dev(absorbed_by, N, torch.int32)))


def nb_encounter_levels(x, v, m, rc_hill, rc_vel, M_star, dt, pairs, npairs):
    import torch
    N = m.numel()
    _check(load().nb_encounter_levels(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), _dev(m, N, torch.float64),
                                      _dev(rc_hill, N, torch.float64), _dev(rc_vel, N, torch.float64), float(M_star), N,
                                      float(dt), _dev(pairs, None, torch.int32), _dev(npairs, 1, torch.int64)))


def nb_merge(x, v, m, radius, pairs, npairs, survivor_of, mstat):
    import torch
    N = m.numel()
    _check(load().nb_merge(_dev(x, 3 * N, torch.float64), _dev(v, 3 * N, torch.float64), _dev(m, N, torch.float64),
                           _dev(radius, N, torch.float64), N, _dev(pairs, None, torch.int32), _dev(npairs, 1, torch.int64),
                           _dev(survivor_of, N, torch.int32), _dev(mstat, 4, torch.int64)))


def nb_kick_host(x, v, m, M_star, dt, rcrit, acc, pairs=None, npairs=None):
    N = m.size
    _check(load().nb_kick_host(_host(x, 3 * N), _host(v, 3 * N), _host(m, N), float(M_star), N, float(dt),
                               _host(rcrit, N), _host(acc, 3 * N), _host(pairs, None, np.int32),
                               _host(npairs, 1, np.int64)))


def nb_step_host(x, v, m, M_star, dt, rcrit, acc, pairs=None, npairs=None, nsteps=1):
    N = m.size
    _check(load().nb_step_host(_host(x, 3 * N), _host(v, 3 * N), _host(m, N), float(M_star), N, float(dt),
                               _host(rcrit, N), _host(acc, 3 * N), _host(pairs, None, np.int32),
                               _host(npairs, 1, np.int64), int(nsteps)))


def nb_status() -> dict:
    f = (C.c_int64 * 8)()
    _check(load().nb_status(f))
    return dict(pairs_dropped=int(f[0]), kepler_fail=int(f[1]), nonfinite=int(f[2]), singular=int(f[3]),
                groups_skipped=int(f[4]), bs_fail=int(f[5]), midpoint_fail=int(f[6]), absorbed=int(f[7]))


def nb_status_reset():
    _check(load().nb_status_reset())


def nb_last_force_ms() -> float:
    return float(load().nb_last_force_ms())


def nb_force_time():
    """(launches, total_ms) of the force-tile launches recorded since nb_force_time_reset."""
    n, ms = C.c_int64(0), C.c_double(0.0)
    _check(load().nb_force_time(C.byref(n), C.byref(ms)))
    return int(n.value), float(ms.value)


def nb_force_time_reset():
    _check(load().nb_force_time_reset())


def set_flags(**kw):
    """Re-issue nb_configure with some fields of the current config changed (same workspace)."""
    cfg = _state["cfg"]
    if cfg is None:
        raise RuntimeError("configure() first")
    for k, v in kw.items():
        setattr(cfg, k, int(v) if isinstance(v, bool) else v)
    _check(load().nb_configure(C.byref(cfg)))


def nb_fp64_peak(iters: int = 0):
    """(TFLOP/s, ms) of a register-only fp64 FMA chain on every SM."""
    t, ms = C.c_double(0.0), C.c_double(0.0)
    _check(load().nb_fp64_peak(int(iters), C.byref(t), C.byref(ms)))
    return float(t.value), float(ms.value)


def nb_release():
    load().nb_release()
    _state["workspace"] = None


def nb_version() -> str:
    return load().nb_version().decode()
