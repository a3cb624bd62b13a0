"""ctypes face of the CPU oracle (oracle/nb_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2604_09184_b200/ (the CUDA path), and the
CUDA path never imports it.  Every function takes and returns numpy float64 host arrays.
Citations are in nb_oracle.c next to each function.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nb_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

# -ffp-contract=off: the oracle states r^2 = (dx*dx + dy*dy) + dz*dz without fused multiply-adds.
_CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *_CFLAGS, "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        dp, ip, lp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
        i64, dbl, i32 = C.c_int64, C.c_double, C.c_int
        lib.oracle_num_threads.restype = i32
        lib.oracle_long_double_digits.restype = i32
        lib.oracle_encounter_rhs.argtypes = [dp, i32, dp, dp, i32, dbl, i32, dp]
        lib.oracle_level_kick.argtypes = [dp, dp, dp, i64, dbl, i32, ip, i64, dp, i64, dbl]
        lib.oracle_set_num_threads.argtypes = [i32]
        lib.oracle_changeover.restype = dbl
        lib.oracle_changeover.argtypes = [dbl, dbl, i32]
        lib.oracle_rcrit.argtypes = [dp, dp, dp, dbl, i64, dbl, dbl, dbl, dbl, dp]
        lib.oracle_accel.argtypes = [dp, dp, dp, i64, i64, dbl, i32, lp, i64, dp, dp, lp]
        lib.oracle_kick.argtypes = [dp, dp, dp, i64, i64, dbl, dp, dbl, i32, dp]
        lib.oracle_pairs.argtypes = [dp, dp, i64, i64, dbl, lp, i64, ip, i64, lp, ip, i64, lp]
        lib.oracle_shift.argtypes = [dp, dp, dp, dbl, i64, dbl]
        lib.oracle_kepler_elliptic.restype = i32
        lib.oracle_kepler_elliptic.argtypes = [dp, dp, dbl, dbl]
        lib.oracle_kepler_universal.restype = i32
        lib.oracle_kepler_universal.argtypes = [dp, dp, dbl, dbl]
        lib.oracle_drift_kepler.restype = i64
        lib.oracle_drift_kepler.argtypes = [dp, dp, dbl, i64, dbl, dbl, i32]
        lib.oracle_step.restype = i64
        lib.oracle_step.argtypes = [dp, dp, dp, dbl, i64, i64, dbl, dbl, dbl, dbl, i32, dp, dp, i64]
        lib.oracle_diagnostics.argtypes = [dp, dp, dp, dbl, i64, dbl, dp]
        lib.oracle_encounter.argtypes = [dp, dp, dp, dp, i64, i64, dbl, dbl, dbl, i32, dbl, ip, ip, i64, i64, lp]
        lib.oracle_encounter_collide.argtypes = [dp, dp, dp, dp, dp, i64, i64, dbl, dbl, dbl, i32, dbl, dbl, ip, ip, i64, i64, ip, lp]
        lib.oracle_encounter_split.argtypes = [dp, dp, dp, dp, i64, i64, dbl, dbl, dbl, i32, dbl, ip, ip, i64, i64, i64, lp]
        lib.oracle_midpoint_drag.restype = i64
        lib.oracle_midpoint_drag.argtypes = [dp, dp, i64, dbl, dbl, dbl, i32, dbl, dbl, i64, lp]
        lib.oracle_step_drag.restype = i64
        lib.oracle_step_drag.argtypes = [dp, dp, dp, dbl, i64, i64, dbl, dbl, dbl, dbl, i32, dp, dp, i64, dbl, i32, dbl, dbl, i64]
        lib.oracle_groups.restype = i32
        lib.oracle_groups.argtypes = [ip, i64, i64, ip, ip, ip, lp]
        _lib = lib
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _rows(rows):
    if rows is None:
        return None, None, 0
    r = np.ascontiguousarray(rows, dtype=np.int64)
    return r, r.ctypes.data_as(C.POINTER(C.c_int64)), r.shape[0]


def num_threads() -> int:
    return int(_L().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _L().oracle_set_num_threads(int(n))


def long_double_digits() -> int:
    """Significand bits of the type oracle_accel sums in (64 on x86-64; see the header of nb_oracle.c)."""
    return int(_L().oracle_long_double_digits())


def changeover(r: float, rc: float, kind: int = 0) -> float:
    return float(_L().oracle_changeover(float(r), float(rc), int(kind)))


def rcrit(x, v, m, M_star, dt, G, n1=3.0, n2=0.4):
    x, px = _d(x); v, pv = _d(v); m, pm = _d(m)
    N = m.shape[0]
    out = np.empty(N)
    _L().oracle_rcrit(px, pv, pm, M_star, N, dt, G, n1, n2, out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def accel(x, m, rcrit_, G, n_active=0, kind=0, rows=None, want_abs=False):
    """a_i (and optionally sum_j |term|).  Returns (acc, abs_sum or None, n_singular)."""
    x, px = _d(x); m, pm = _d(m)
    N = m.shape[0]
    if rcrit_ is None:
        prc = None
    else:
        rcrit_, prc = _d(rcrit_)
    r, pr, nr = _rows(rows)
    n_out = nr if rows is not None else N
    acc = np.empty((n_out, 3))
    ab = np.empty((n_out, 3)) if want_abs else None
    ns = C.c_int64(0)
    _L().oracle_accel(px, pm, prc, N, n_active, G, kind, pr, nr,
                      acc.ctypes.data_as(C.POINTER(C.c_double)),
                      ab.ctypes.data_as(C.POINTER(C.c_double)) if want_abs else None, C.byref(ns))
    return acc, ab, int(ns.value)


def kick(x, v, m, dt, rcrit_, G, n_active=0, kind=0):
    """Returns (v_new, acc)."""
    x, px = _d(x); m, pm = _d(m)
    v = np.array(v, dtype=np.float64, order="C", copy=True)
    N = m.shape[0]
    if rcrit_ is None:
        prc = None
    else:
        rcrit_, prc = _d(rcrit_)
    acc = np.empty((N, 3))
    _L().oracle_kick(px, v.ctypes.data_as(C.POINTER(C.c_double)), pm, N, n_active, dt, prc, G, kind,
                     acc.ctypes.data_as(C.POINTER(C.c_double)))
    return v, acc


def _canon(p):
    """Canonical pair order: unique rows sorted by (min, max) (reading S12)."""
    if p.shape[0] == 0:
        return p.reshape(0, 2)
    return np.unique(p, axis=0)


def pairs(x, rcrit_, n_active=0, tol2=2e-12, rows=None, cap=1 << 22):
    """Returns (sure[ns,2], borderline[nb,2]) int32, canonically sorted, de-duplicated."""
    x, px = _d(x); rcrit_, prc = _d(rcrit_)
    N = rcrit_.shape[0]
    r, pr, nr = _rows(rows)
    while True:
        sure = np.empty((cap, 2), dtype=np.int32)
        bord = np.empty((cap, 2), dtype=np.int32)
        ns, nb = C.c_int64(0), C.c_int64(0)
        _L().oracle_pairs(px, prc, N, n_active, tol2, pr, nr,
                          sure.ctypes.data_as(C.POINTER(C.c_int32)), cap, C.byref(ns),
                          bord.ctypes.data_as(C.POINTER(C.c_int32)), cap, C.byref(nb))
        if ns.value <= cap and nb.value <= cap:
            break
        cap = int(max(ns.value, nb.value))
    return _canon(sure[: ns.value]), _canon(bord[: nb.value])


def shift(x, v, m, M_star, dt):
    x = np.array(x, dtype=np.float64, order="C", copy=True)
    v, pv = _d(v); m, pm = _d(m)
    _L().oracle_shift(x.ctypes.data_as(C.POINTER(C.c_double)), pv, pm, M_star, m.shape[0], dt)
    return x


def kepler_one(x, v, mu, h, solver="elliptic"):
    """Advance ONE body.  Returns (x, v, code)."""
    x = np.array(x, dtype=np.float64, copy=True).reshape(3)
    v = np.array(v, dtype=np.float64, copy=True).reshape(3)
    fn = _L().oracle_kepler_elliptic if solver == "elliptic" else _L().oracle_kepler_universal
    code = fn(x.ctypes.data_as(C.POINTER(C.c_double)), v.ctypes.data_as(C.POINTER(C.c_double)), mu, h)
    return x, v, int(code)


def drift_kepler(x, v, M_star, dt, G, solver=0):
    """Returns (x_new, v_new, n_fail)."""
    x = np.array(x, dtype=np.float64, order="C", copy=True)
    v = np.array(v, dtype=np.float64, order="C", copy=True)
    N = x.shape[0]
    nf = _L().oracle_drift_kepler(x.ctypes.data_as(C.POINTER(C.c_double)),
                                  v.ctypes.data_as(C.POINTER(C.c_double)), M_star, N, dt, G, solver)
    return x, v, int(nf)


def step(x, v, m, M_star, dt, G, nsteps, n_active=0, n1=3.0, n2=0.0, kind=0, rcrit_=None):
    """nsteps steps B(dt/2)C(dt/2)A(dt)C(dt/2)B(dt/2).  Returns dict(x, v, acc, rcrit, n_fail)."""
    x = np.array(x, dtype=np.float64, order="C", copy=True)
    v = np.array(v, dtype=np.float64, order="C", copy=True)
    m, pm = _d(m)
    N = m.shape[0]
    rc = np.zeros(N) if rcrit_ is None else np.array(rcrit_, dtype=np.float64, copy=True)
    acc = np.empty((N, 3))
    P = C.POINTER(C.c_double)
    nf = _L().oracle_step(x.ctypes.data_as(P), v.ctypes.data_as(P), pm, M_star, N, n_active, dt, G,
                          n1, n2, kind, rc.ctypes.data_as(P), acc.ctypes.data_as(P), nsteps)
    return dict(x=x, v=v, acc=acc, rcrit=rc, n_fail=int(nf))


def midpoint_drag(x, v, mu, dt, gamma, power=0, eta=0.0, tol=1e-14, max_iter=50):
    """Implicit midpoint (Eq. 8) for the drag a_f = -gamma |u|^p u, u = v - (1 - eta) v_circ(R) e_phi
    (reading S24).  Returns (v_new, n_not_converged, most iterations used)."""
    x, px = _d(x)
    v = np.array(v, dtype=np.float64, order="C", copy=True)
    N = v.shape[0]
    it = C.c_int64(0)
    nf = _L().oracle_midpoint_drag(px, v.ctypes.data_as(C.POINTER(C.c_double)), N, float(mu), float(dt), float(gamma), int(power),
                                   float(eta), float(tol), int(max_iter), C.byref(it))
    return v, int(nf), int(it.value)


def step_drag(x, v, m, M_star, dt, G, nsteps, gamma, power=0, eta=0.0, tol=1e-14, max_iter=50, n_active=0, n1=3.0, n2=0.0,
              kind=0, rcrit_=None):
    """nsteps of D(dt/2) B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2) D(dt/2) (reading S24).  Returns dict(x, v, acc, rcrit, n_fail)."""
    x = np.array(x, dtype=np.float64, order="C", copy=True)
    v = np.array(v, dtype=np.float64, order="C", copy=True)
    m, pm = _d(m)
    N = m.shape[0]
    rc = np.zeros(N) if rcrit_ is None else np.array(rcrit_, dtype=np.float64, copy=True)
    acc = np.empty((N, 3))
    P = C.POINTER(C.c_double)
    nf = _L().oracle_step_drag(x.ctypes.data_as(P), v.ctypes.data_as(P), pm, M_star, N, n_active, dt, G, n1, n2, kind,
                               rc.ctypes.data_as(P), acc.ctypes.data_as(P), nsteps, float(gamma), int(power), float(eta),
                               float(tol), int(max_iter))
    return dict(x=x, v=v, acc=acc, rcrit=rc, n_fail=int(nf))


def diagnostics(x, v, m, M_star, G):
    """dict(E, L[3], T, T_star, U_star, U_mutual) -- PAPER.md:84-92 with the K terms cancelling."""
    x, px = _d(x); v, pv = _d(v); m, pm = _d(m)
    out = np.empty(8)
    _L().oracle_diagnostics(px, pv, pm, M_star, m.shape[0], G, out.ctypes.data_as(C.POINTER(C.c_double)))
    return dict(E=out[0], L=out[1:4].copy(), T=out[4], T_star=out[5], U_star=out[6], U_mutual=out[7])


def groups(pairs_, N):
    """Independent encounter groups = connected components of the pair graph.
    Returns dict(label[N], members[nmembers], gstart[ngroups+1], ngroups, nmembers, largest)."""
    p = np.ascontiguousarray(np.asarray(pairs_, dtype=np.int32).reshape(-1, 2))
    N = int(N)
    label = np.empty(N, dtype=np.int32)
    members = np.empty(max(N, 1), dtype=np.int32)
    gstart = np.empty(N // 2 + 2, dtype=np.int32)
    gstat = np.zeros(4, dtype=np.int64)
    ip, lp = C.POINTER(C.c_int32), C.POINTER(C.c_int64)
    rc = _L().oracle_groups(p.ctypes.data_as(ip), p.shape[0], N, label.ctypes.data_as(ip), members.ctypes.data_as(ip),
                            gstart.ctypes.data_as(ip), gstat.ctypes.data_as(lp))
    if rc != 0:
        raise ValueError("oracle.groups: a pair holds an index outside [0, N) or i == j")
    ng, nm = int(gstat[0]), int(gstat[1])
    return dict(label=label, members=members[:nm].copy(), gstart=gstart[:ng + 1].copy(), ngroups=ng, nmembers=nm,
                largest=int(gstat[2]))


def encounter_rhs(x, v, gm, rc, mu, kind=0):
    """Right-hand side of the group equations of motion (Eq. 4): returns (dx/dt, dv/dt) of the n bodies
    of ONE group, dv/dt = -mu x/r^3 + sum_j gm_j [1 - W(r_ij; max(rc_i, rc_j))] (x_j - x_i)/r_ij^3.  rc may be [nlev, n]
    (multi-level scheme: the pair term carries the product of the levels' [1 - W_k])."""
    x = np.ascontiguousarray(x, dtype=np.float64); v = np.ascontiguousarray(v, dtype=np.float64)
    n = x.shape[0]
    y = np.concatenate([x.reshape(-1), v.reshape(-1)])
    gm = np.ascontiguousarray(gm, dtype=np.float64); rc = np.ascontiguousarray(rc, dtype=np.float64).reshape(-1, n)
    f = np.empty(6 * n)
    dp = C.POINTER(C.c_double)
    _L().oracle_encounter_rhs(y.ctypes.data_as(dp), n, gm.ctypes.data_as(dp), rc.ctypes.data_as(dp), rc.shape[0], float(mu),
                              int(kind), f.ctypes.data_as(dp))
    return f[:3 * n].reshape(n, 3), f[3 * n:].reshape(n, 3)


def encounter(x, v, m, rcrit_, M_star, dt, G, grp, kind=0, tol=1e-12, max_group=1024, n_active=0, split_max_core=-1,
              radius=None, radius_factor=1.0, absorbed_by=None):
    """H_A with encounters (Eq. 4, 98, 106): the members of every group of `grp` (a dict from
    groups()) are advanced by dt with the Bulirsch-Stoer integrator; returns (x, v, stats) with
    stats = dict(integrated, skipped, failed, steps).  Semi-active mode (0 < n_active < N, reading S22): every
    group that has test particles is split into its active core and independent {core + particle} problems;
    split_max_core >= 0 restricts the splitting to cores of at most that many members (what an implementation
    with a bounded core size does; the tests pass the CUDA path's bound).
    radius given (fully active case): collisions are examined inside the solver after every accepted step and the
    colliding members merged at once (reading S26); stats then also holds m, radius (new arrays),
    absorbed_by (int32[N]: the body an absorbed body sits on, -1 otherwise; continues the array passed in) and absorbed."""
    x = np.array(x, dtype=np.float64, order="C"); v = np.array(v, dtype=np.float64, order="C")
    m = np.ascontiguousarray(m, dtype=np.float64)
    N = m.shape[0]
    rc = np.ascontiguousarray(rcrit_, dtype=np.float64).reshape(-1, N)     # [nlev, N]; nlev = 1: the plain hybrid scheme
    nlev = rc.shape[0]
    members = np.ascontiguousarray(grp["members"], dtype=np.int32)
    gstart = np.ascontiguousarray(grp["gstart"], dtype=np.int32)
    stats = np.zeros(5, dtype=np.int64)
    dp, ip, lp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
    if radius is not None:
        if 0 < int(n_active) < N:
            raise ValueError("collisions inside the solver are defined for the fully active case (reading S26)")
        m2 = np.array(m, dtype=np.float64); R2 = np.array(radius, dtype=np.float64)
        ab = np.full(N, -1, dtype=np.int32) if absorbed_by is None else np.array(absorbed_by, dtype=np.int32)
        _L().oracle_encounter_collide(x.ctypes.data_as(dp), v.ctypes.data_as(dp), m2.ctypes.data_as(dp), R2.ctypes.data_as(dp),
                                      rc.ctypes.data_as(dp), nlev, N, float(M_star), float(G), float(dt), int(kind), float(tol),
                                      float(radius_factor), members.ctypes.data_as(ip), gstart.ctypes.data_as(ip),
                                      int(grp["ngroups"]), int(max_group), ab.ctypes.data_as(ip), stats.ctypes.data_as(lp))
        return x, v, dict(integrated=int(stats[0]), skipped=int(stats[1]), failed=int(stats[2]), steps=int(stats[3]),
                          absorbed=int(stats[4]), m=m2, radius=R2, absorbed_by=ab)
    if 0 < int(n_active) < N:
        if nlev != 1:
            raise ValueError("the multi-level scheme is defined for the fully active case only")
        # semi-active mode: cores and test particles are integrated separately (oracle_encounter_split)
        _L().oracle_encounter_split(x.ctypes.data_as(dp), v.ctypes.data_as(dp), m.ctypes.data_as(dp), rc.ctypes.data_as(dp),
                                    N, int(n_active), float(M_star), float(G), float(dt), int(kind), float(tol),
                                    members.ctypes.data_as(ip), gstart.ctypes.data_as(ip), int(grp["ngroups"]),
                                    int(max_group), int(split_max_core), stats.ctypes.data_as(lp))
    else:
        _L().oracle_encounter(x.ctypes.data_as(dp), v.ctypes.data_as(dp), m.ctypes.data_as(dp), rc.ctypes.data_as(dp), nlev, N,
                              float(M_star), float(G), float(dt), int(kind), float(tol), members.ctypes.data_as(ip),
                              gstart.ctypes.data_as(ip), int(grp["ngroups"]), int(max_group), stats.ctypes.data_as(lp))
    return x, v, dict(integrated=int(stats[0]), skipped=int(stats[1]), failed=int(stats[2]), steps=int(stats[3]))


def step_enc(x, v, m, M_star, dt, G, nsteps, n1=3.0, n2=0.4, kind=0, tol=1e-12, max_group=1024, n_active=0, split_max_core=-1,
             radius=None, radius_factor=1.0):
    """nsteps of B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2) with close encounters resolved:
    in A the members of the encounter groups of the step's opening pair list (groups of at most max_group
    bodies) are propagated by encounter(), every other body by the Kepler drift.  Composed of the pinned
    pieces above; rcrit is recomputed before every force evaluation (S17) and held through the step.  With
    n_active (semi-active mode) only the first n_active bodies exert force and every pair has an active member.
    radius given: collisions inside the solver (reading S26) -- m and radius change from step to step (an absorbed body
    stays in the arrays with m = 0, R = 0 on top of its survivor until merge() compacts them) and are returned too.
    Returns dict(x, v, acc, rcrit, pairs, stats [, m, radius, absorbed_by])."""
    x = np.array(x, dtype=np.float64, order="C"); v = np.array(v, dtype=np.float64, order="C")
    m = np.array(m, dtype=np.float64)
    N = m.shape[0]
    tot = dict(integrated=0, skipped=0, failed=0, steps=0, border=0, absorbed=0)
    R = None if radius is None else np.array(radius, dtype=np.float64)
    ab = np.full(N, -1, dtype=np.int32)

    def evaluate(x, v):
        rc = rcrit(x, v, m, M_star, dt, G, n1, n2)
        acc, _, _ = accel(x, m, rc, G, n_active=n_active, kind=kind)
        sure, border = pairs(x, rc, n_active=n_active)
        tot["border"] += border.shape[0]
        return rc, acc, sure

    rc, acc, pr = evaluate(x, v)
    for _ in range(int(nsteps)):
        v = v + (0.5 * dt) * acc
        x = shift(x, v, m, M_star, 0.5 * dt)
        grp = groups(pr, N)
        xk, vk, nfail = drift_kepler(x, v, M_star, dt, G)
        xe, ve, st = encounter(x, v, m, rc, M_star, dt, G, grp, kind=kind, tol=tol, max_group=max_group, n_active=n_active,
                               split_max_core=split_max_core, radius=R, radius_factor=radius_factor, absorbed_by=ab)
        if R is not None:
            m, R, ab = st["m"], st["radius"], st["absorbed_by"]
            tot["absorbed"] += st["absorbed"]
        moved = np.zeros(N, dtype=bool)
        for g in range(grp["ngroups"]):
            seg = grp["members"][grp["gstart"][g]:grp["gstart"][g + 1]]
            size = seg.shape[0]
            if 0 < n_active < N:
                nc = int(np.count_nonzero(seg < n_active))
                if nc < size and (split_max_core < 0 or nc <= split_max_core):
                    size = nc                      # split group: only the core counts against max_group
            if size <= max_group:
                moved[seg] = True
        x = np.where(moved[:, None], xe, xk)
        v = np.where(moved[:, None], ve, vk)
        for k in ("integrated", "skipped", "failed", "steps"):
            tot[k] += st[k]
        x = shift(x, v, m, M_star, 0.5 * dt)
        rc, acc, pr = evaluate(x, v)
        v = v + (0.5 * dt) * acc
    out = dict(x=x, v=v, acc=acc, rcrit=rc, pairs=pr, stats=tot)
    if R is not None:
        out.update(m=m, radius=R, absorbed_by=ab)
    return out


# ---------------------------------------------------------------------------------------------------------------------
# Multi-level changeover (reading S23).  The statement of the recursion; the arithmetic pieces
# are the C functions above (oracle_level_kick, oracle_drift_kepler, oracle_encounter with level radii, oracle_groups).
# ---------------------------------------------------------------------------------------------------------------------
def level_rcrit(x, v, m, M_star, dt, G, n1, n2, nlev, rcrit0=None):
    """Critical radii of the levels 0 .. nlev-1, [nlev, N]: Eq. 7 evaluated with the level's own time step
    dt / 2^l -- "a second term is used to increase the critical radius in situations where too few steps are used
    through the changeover function", so the velocity term shrinks with the step while the Hill term
    stays.  n1 == n2 == 0 (caller's radii, rcrit0): rc_l = rcrit0 / 2^l."""
    if n1 == 0.0 and n2 == 0.0:
        return np.stack([np.asarray(rcrit0, dtype=np.float64) / 2.0 ** l for l in range(nlev)])
    return np.stack([rcrit(x, v, m, M_star, dt / 2.0 ** l, G, n1, n2) for l in range(nlev)])


def level_weights(r, rcs, kind=0):
    """Share of the Newtonian pair force each operator carries at separation r, for pairwise level radii rcs[0..L]:
    [W_0, Omega_0 W_1, ..., Omega_{L-1} W_L, Omega_L] (L + 2 numbers: the outer kick, the L level kicks, the direct
    solver).  They sum to 1 at every r."""
    out, om = [], 1.0
    for rc in rcs:
        W = changeover(r, rc, kind)
        out.append(om * W)
        om = om * (1.0 - W)
    out.append(om)
    return out


def level_kick(x, v, m, G, pairs_, rcl, level, h, kind=0):
    """v_i += h sum_{j: {i,j} listed} G m_j Omega_level W_{level+1} (x_j - x_i)/r^3; returns the new v."""
    x, px = _d(x); m, pm = _d(m)
    v = np.array(v, dtype=np.float64, order="C", copy=True)
    N = m.shape[0]
    p = np.ascontiguousarray(np.asarray(pairs_, dtype=np.int32).reshape(-1, 2))
    rcl = np.ascontiguousarray(rcl, dtype=np.float64).reshape(-1, N)
    if rcl.shape[0] < level + 2:
        raise ValueError("level_kick needs the radii of levels 0 .. level + 1")
    dp = C.POINTER(C.c_double)
    _L().oracle_level_kick(px, v.ctypes.data_as(dp), pm, N, float(G), int(kind), p.ctypes.data_as(C.POINTER(C.c_int32)),
                           p.shape[0], rcl.ctypes.data_as(dp), int(level), float(h))
    return v


def _pairs_within(x, p, rc_level):
    """Rows of the pair list p whose bodies are closer than max(rc_i, rc_j) of the given level (strict, fp64 on r^2 with
    the definition's expression), in the order of p."""
    if p.shape[0] == 0:
        return p
    i, j = p[:, 0], p[:, 1]
    dx = x[j] - x[i]
    r2 = (dx[:, 0] * dx[:, 0] + dx[:, 1] * dx[:, 1]) + dx[:, 2] * dx[:, 2]
    rc = np.maximum(rc_level[i], rc_level[j])
    return p[r2 < rc * rc]


def encounter_ml(x, v, m, rcl, M_star, dt, G, pairs0, kind=0, tol=1e-12, max_group=1024, radius=None, radius_factor=1.0,
                 absorbed_by=None):
    """H_A over dt for the bodies of the pair list pairs0 with L = len(rcl) - 1 intermediate levels (reading S23).

        advance(l, P, tau):                      # Kepler + sum_{pairs in P} (pair force) Omega_l, for the bodies of P
            if l == L:  Bulirsch-Stoer over tau for the groups of P, pair weight Omega_L         (the direct solver)
            else twice, with h = tau / 2:
                P' = pairs of P closer than rc_{l+1} now
                kick  h/2 with weight Omega_l W_{l+1} over P
                bodies of P not in P': Kepler drift h;   advance(l + 1, P', h)
                kick  h/2 with weight Omega_l W_{l+1} over P

    L = 0 is oracle.encounter on the groups of pairs0.  Bodies outside pairs0 are not touched (the caller drifts them).
    radius given: the direct solver of the innermost level examines collisions (reading S26); the masses then change on
    the way -- the level kicks that follow use the merged masses -- and stats also holds m, radius, absorbed_by, absorbed.
    Returns (x, v, stats) with stats = dict(integrated, skipped, failed, steps, kicks, level_pairs[L+1])."""
    x = np.array(x, dtype=np.float64, order="C"); v = np.array(v, dtype=np.float64, order="C")
    m = np.array(m, dtype=np.float64)
    N = m.shape[0]
    R = None if radius is None else np.array(radius, dtype=np.float64)
    ab = None if radius is None else (np.full(N, -1, dtype=np.int32) if absorbed_by is None else np.array(absorbed_by, dtype=np.int32))
    rcl = np.ascontiguousarray(rcl, dtype=np.float64).reshape(-1, N)
    L = rcl.shape[0] - 1
    stats = dict(integrated=0, skipped=0, failed=0, steps=0, kicks=0, absorbed=0, level_pairs=[0] * (L + 1))
    P0 = _canon(np.asarray(pairs0, dtype=np.int32).reshape(-1, 2))

    def bodies(P):
        return np.unique(P.reshape(-1)) if P.shape[0] else np.zeros(0, dtype=np.int64)

    def advance(l, P, tau):
        nonlocal x, v, m, R, ab
        stats["level_pairs"][l] += int(P.shape[0])
        if P.shape[0] == 0:
            return
        if l == L:
            grp = groups(P, N)
            xe, ve, st = encounter(x, v, m, rcl, M_star, tau, G, grp, kind=kind, tol=tol, max_group=max_group,
                                   radius=R, radius_factor=radius_factor, absorbed_by=ab)
            if R is not None:
                m, R, ab = st["m"], st["radius"], st["absorbed_by"]
                stats["absorbed"] += st["absorbed"]
            # groups beyond max_group are left to the Kepler drift (counted), as in step_enc
            big = np.zeros(N, dtype=bool)
            for g in range(grp["ngroups"]):
                seg = grp["members"][grp["gstart"][g]:grp["gstart"][g + 1]]
                if seg.shape[0] > max_group:
                    big[seg] = True
            if big.any():
                idx = np.flatnonzero(big)
                xk, vk, _ = drift_kepler(x[idx], v[idx], M_star, tau, G)
                xe[idx] = xk; ve[idx] = vk
            x, v = xe, ve
            for k in ("integrated", "skipped", "failed", "steps"):
                stats[k] += st[k]
            return
        h = 0.5 * tau
        for _ in range(2):
            Pn = _pairs_within(x, P, rcl[l + 1])
            v = level_kick(x, v, m, G, P, rcl, l, 0.5 * h, kind)
            outer = np.setdiff1d(bodies(P), bodies(Pn))
            if outer.size:
                xk, vk, nf = drift_kepler(x[outer], v[outer], M_star, h, G)
                stats["failed"] += nf
                x[outer] = xk; v[outer] = vk
            advance(l + 1, Pn, h)
            v = level_kick(x, v, m, G, P, rcl, l, 0.5 * h, kind)
            stats["kicks"] += 2

    advance(0, P0, dt)
    if R is not None:
        stats.update(m=m, radius=R, absorbed_by=ab)
    return x, v, stats


def step_ml(x, v, m, M_star, dt, G, nsteps, nlev, n1=3.0, n2=0.4, kind=0, tol=1e-12, max_group=1024, rcrit0=None,
            radius=None, radius_factor=1.0):
    """nsteps of B(dt/2) C(dt/2) A(dt) C(dt/2) B(dt/2) with the close encounters of A resolved through nlev - 1 intermediate
    levels (encounter_ml); nlev = 1 is step_enc.  Level radii by level_rcrit from the state at each force evaluation
    (S17), held through the step.  radius given: collisions inside the innermost solver (reading S26), as in step_enc.
    Returns dict(x, v, acc, rcrit [nlev, N], pairs, stats [, m, radius, absorbed_by])."""
    x = np.array(x, dtype=np.float64, order="C"); v = np.array(v, dtype=np.float64, order="C")
    m = np.array(m, dtype=np.float64)
    N = m.shape[0]
    tot = dict(integrated=0, skipped=0, failed=0, steps=0, kicks=0, border=0, absorbed=0, level_pairs=[0] * nlev)
    R = None if radius is None else np.array(radius, dtype=np.float64)
    ab = np.full(N, -1, dtype=np.int32)

    def evaluate(x, v):
        rcl = level_rcrit(x, v, m, M_star, dt, G, n1, n2, nlev, rcrit0)
        acc, _, _ = accel(x, m, rcl[0], G, kind=kind)
        sure, border = pairs(x, rcl[0])
        tot["border"] += border.shape[0]
        return rcl, acc, sure

    rcl, acc, pr = evaluate(x, v)
    for _ in range(int(nsteps)):
        v = v + (0.5 * dt) * acc
        x = shift(x, v, m, M_star, 0.5 * dt)
        inside = np.zeros(N, dtype=bool)
        inside[pr.reshape(-1)] = True
        free = np.flatnonzero(~inside)
        xe, ve, st = encounter_ml(x, v, m, rcl, M_star, dt, G, pr, kind=kind, tol=tol, max_group=max_group,
                                  radius=R, radius_factor=radius_factor, absorbed_by=ab)
        if R is not None:
            m, R, ab = st["m"], st["radius"], st["absorbed_by"]
            tot["absorbed"] += st["absorbed"]
        if free.size:
            xk, vk, nf = drift_kepler(x[free], v[free], M_star, dt, G)
            xe[free] = xk; ve[free] = vk
            tot["failed"] += nf
        x, v = xe, ve
        for k in ("integrated", "skipped", "failed", "steps", "kicks"):
            tot[k] += st[k]
        tot["level_pairs"] = [a + b for a, b in zip(tot["level_pairs"], st["level_pairs"])]
        x = shift(x, v, m, M_star, 0.5 * dt)
        rcl, acc, pr = evaluate(x, v)
        v = v + (0.5 * dt) * acc
    out = dict(x=x, v=v, acc=acc, rcrit=rcl, pairs=pr, stats=tot)
    if R is not None:
        out.update(m=m, radius=R, absorbed_by=ab)
    return out


def merge(x, v, m, radius, pairs_, f=1.0):
    """Perfect merging ("N-body simulations often treat collisions as perfect mergers"; PAPER.md:168:
    radii may be inflated by a constant factor f).  DESIGN.md reading S21:
      * two bodies of a listed pair collide iff r_ij < f (R_i + R_j) (strict, decided in fp64 on r^2);
      * colliding bodies that are linked by a chain of collisions merge into ONE body, the one with the smallest
        index: m <- sum m_k, x <- sum m_k x_k / sum m_k, v <- sum m_k v_k / sum m_k (mass and momentum of the
        democratic coordinates conserved; members in index order), R <- (sum R_k^3)^(1/3) (volume conserved);
        if all masses are zero the survivor keeps its x, v;
      * every other member is removed; the arrays are then compacted in index order (a stable partition, so a
        semi-active ordering survives).
    Returns dict(x, v, m, radius, N, alive[N_old] bool, survivor_of[N_old] int32 (label of the merged body, own
    index for untouched bodies), n_collisions (colliding pair rows), n_merged (bodies removed))."""
    x = np.array(x, dtype=np.float64, order="C"); v = np.array(v, dtype=np.float64, order="C")
    m = np.array(m, dtype=np.float64); R = np.array(radius, dtype=np.float64)
    N = m.shape[0]
    p = np.asarray(pairs_, dtype=np.int32).reshape(-1, 2)
    hits = []
    for i, j in p:
        dx = x[j] - x[i]
        r2 = (dx[0] * dx[0] + dx[1] * dx[1]) + dx[2] * dx[2]
        s = f * (R[i] + R[j])
        if r2 < s * s:
            hits.append((i, j))
    hits = np.array(hits, dtype=np.int32).reshape(-1, 2)
    g = groups(hits, N)
    alive = np.ones(N, dtype=bool)
    for k in range(g["ngroups"]):
        seg = g["members"][g["gstart"][k]:g["gstart"][k + 1]]
        s = int(seg[0])
        mt = 0.0; mx = np.zeros(3); mv = np.zeros(3); vol = 0.0
        for b in seg:                      # index order
            mt = mt + m[b]
            mx = mx + m[b] * x[b]
            mv = mv + m[b] * v[b]
            vol = vol + R[b] * R[b] * R[b]
        if mt > 0.0:
            x[s] = mx / mt
            v[s] = mv / mt
        m[s] = mt
        R[s] = np.cbrt(vol)
        alive[seg[1:]] = False
    keep = np.flatnonzero(alive)
    return dict(x=x[keep].copy(), v=v[keep].copy(), m=m[keep].copy(), radius=R[keep].copy(), N=int(keep.shape[0]),
                alive=alive, survivor_of=g["label"].copy(), n_collisions=int(hits.shape[0]),
                n_merged=int(N - keep.shape[0]))
