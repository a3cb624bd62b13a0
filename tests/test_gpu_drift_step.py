"""-m gpu parity: nb_drift_kepler and nb_step (C ABI, CUDA path) against the CPU oracle."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import ENERGY_TOL, GpuState, assert_acc_close, assert_pairs_match, to_dev

pytestmark = pytest.mark.gpu


def _random_orbits(n, seed, emax=0.9, hyperbolic_frac=0.0):
    rng = np.random.default_rng(seed)
    a = rng.uniform(0.3, 6.0, n)
    e = rng.uniform(0.0, emax, n)
    inc = rng.uniform(0.0, 0.5, n)
    w, O, M = (rng.uniform(0.0, 2 * np.pi, n) for _ in range(3))
    x, v = nb_inputs.elements_to_cartesian(a, e, inc, w, O, M, G_GAUSS)
    nh = int(hyperbolic_frac * n)
    if nh:
        v[:nh] *= rng.uniform(1.5, 3.0, nh)[:, None]  # beyond escape speed => universal-variable branch
    return np.ascontiguousarray(x), np.ascontiguousarray(v)


def _drift_gpu(x, v, dt, M_star=1.0):
    import paper_2604_09184_b200 as nb
    import torch
    N = x.shape[0]
    nb.configure(N, G=G_GAUSS)
    nb.nb_status_reset()
    xd, vd = to_dev(x), to_dev(v)
    nb.nb_drift_kepler(xd, vd, M_star, dt)
    torch.cuda.synchronize()
    return xd.cpu().numpy(), vd.cpu().numpy(), nb.nb_status()


@pytest.mark.parametrize("dt", [6.0, 3.0, -6.0, 400.0, 5000.0])
def test_drift_random_orbits(dt):
    # 10 % of the bodies are unbound (1.5 .. 3 x their orbital speed) at every step length: the CUDA path takes
    # them through its universal-variable Laguerre-Conway solver, the oracle through its safeguarded Newton
    x, v = _random_orbits(5000, seed=int(abs(dt)) + 1, hyperbolic_frac=0.1)
    xg, vg, status = _drift_gpu(x, v, dt)
    xr, vr, nfail = oracle.drift_kepler(x, v, 1.0, dt, G_GAUSS)
    assert nfail == 0 and status["kepler_fail"] == 0
    # the error of the Kepler map grows with the number of radians travelled: n |dt| eps / (1 - e)
    nmax = np.sqrt(G_GAUSS / 0.3 ** 3)
    tol = 1e-13 + 40 * 2.2e-16 * nmax * abs(dt) / (1 - 0.9)
    scale_x = np.linalg.norm(xr, axis=1, keepdims=True)
    scale_v = np.linalg.norm(vr, axis=1, keepdims=True)
    assert np.max(np.abs(xg - xr) / scale_x) <= tol
    assert np.max(np.abs(vg - vr) / scale_v) <= tol


def test_drift_unbound_near_parabolic_and_non_finite_bodies():
    """Everything the fast bound-orbit path declines: strongly hyperbolic bodies over long intervals, bodies within
    rounding of the parabola (alpha = O(eps), where elliptic elements are meaningless), high-e orbits near pericentre
    (r0/a < 0.05), against the oracle (whose own solvers are pinned by closed forms and by numerical integration);
    non-finite rows are counted and left alone -- the call returns (no endless loop) and the other bodies are right."""
    rng = np.random.default_rng(99)
    n = 512
    r0 = rng.uniform(0.3, 3.0, n)
    ang = rng.uniform(0, 2 * np.pi, n)
    x = np.stack([r0 * np.cos(ang), r0 * np.sin(ang), 0.05 * r0 * rng.standard_normal(n)], axis=1)
    rn = np.linalg.norm(x, axis=1)
    vesc = np.sqrt(2 * G_GAUSS / rn)
    fac = np.concatenate([np.full(64, 1.0), 1.0 + rng.uniform(-1e-12, 1e-12, 64), rng.uniform(0.98, 1.02, 128),
                          rng.uniform(1.0, 10.0, 128), rng.uniform(0.97, 0.9999, 128)])
    th = rng.uniform(0.2, 2.9, n)
    rad = x / rn[:, None]
    tang = np.cross(np.array([0.0, 0.0, 1.0]), rad); tang /= np.linalg.norm(tang, axis=1, keepdims=True)
    v = (fac * vesc)[:, None] * (np.sin(th)[:, None] * tang + np.cos(th)[:, None] * rad)
    x = np.ascontiguousarray(x); v = np.ascontiguousarray(v)
    for dt in (6.0, -40.0, 400.0, 2000.0):
        xg, vg, status = _drift_gpu(x, v, dt)
        xr, vr, nfail = oracle.drift_kepler(x, v, 1.0, dt, G_GAUSS)
        assert nfail == 0 and status["kepler_fail"] == 0, (dt, nfail, status)
        ex = np.max(np.abs(xg - xr) / np.linalg.norm(xr, axis=1, keepdims=True))
        ev = np.max(np.abs(vg - vr) / np.linalg.norm(vr, axis=1, keepdims=True))
        print(f"unbound / near-parabolic drift dt={dt}: rel dx {ex:.2e} dv {ev:.2e}")
        # f x + g v cancels by up to ~exp(hyperbolic anomaly) ~ 1e3 on the long hyperbolic arcs, on both sides
        assert ex <= 2e-12 and ev <= 2e-12
    # non-finite rows: counted, unchanged, and nobody else is disturbed
    xb, vb = x.copy(), v.copy()
    vb[3] = np.inf; vb[10, 1] = np.nan; xb[20] = np.inf; xb[33] = 0.0
    bad = np.array([3, 10, 20, 33])
    xg, vg, status = _drift_gpu(xb, vb, 6.0)
    assert status["kepler_fail"] == bad.size
    good = np.setdiff1d(np.arange(n), bad)
    xr, vr, _ = oracle.drift_kepler(x[good], v[good], 1.0, 6.0, G_GAUSS)
    assert np.max(np.abs(xg[good] - xr)) <= 1e-12 and np.max(np.abs(vg[good] - vr)) <= 1e-12 * np.max(np.abs(vr))
    for b in bad:
        assert np.array_equal(xg[b], xb[b], equal_nan=True) and np.array_equal(vg[b], vb[b], equal_nan=True)


def test_drift_config_like_and_edge_cases():
    d = nb_inputs.make_config(0, n_override=2048)
    xg, vg, status = _drift_gpu(d.x, d.v, d.dt)
    xr, vr, nfail = oracle.drift_kepler(d.x, d.v, 1.0, d.dt, G_GAUSS)
    assert status["kepler_fail"] == 0 and nfail == 0
    assert np.max(np.abs(xg - xr)) <= 1e-13 * np.max(np.abs(xr))
    assert np.max(np.abs(vg - vr)) <= 1e-13 * np.max(np.abs(vr))
    # circular orbit over exactly one period returns to the start (2 pi reduction); dt = 0 is the identity
    a = 1.3
    x0 = np.array([[a, 0.0, 0.0]]); v0 = np.array([[0.0, np.sqrt(G_GAUSS / a), 0.0]])
    P = 2 * np.pi * np.sqrt(a ** 3 / G_GAUSS)
    xg, vg, _ = _drift_gpu(x0, v0, P)
    assert np.max(np.abs(xg - x0)) <= 1e-13 and np.max(np.abs(vg - v0)) <= 1e-14
    xg, vg, _ = _drift_gpu(x0, v0, 0.0)
    assert np.array_equal(xg, x0) and np.array_equal(vg, v0)
    xq = a * np.array([[np.cos(1.0), np.sin(1.0), 0.0]])
    xg, vg, _ = _drift_gpu(x0, v0, P / (2 * np.pi))  # one radian
    assert np.max(np.abs(xg - xq)) <= 1e-14


def _step_compare(d, nsteps, n1, n2, *, what, x_tol, use_graph=True, **tune):
    na = d.n_active if d.n_active < d.N else 0
    ref = oracle.step(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, nsteps, n_active=na, n1=n1, n2=n2)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n_active=na, n1=n1, n2=n2, use_graph=use_graph, **tune)
    st.step(d.dt, nsteps)
    xg, vg, accg, rcg = st.host()
    status = st.nb.nb_status()
    assert status["kepler_fail"] == 0 and ref["n_fail"] == 0
    assert np.max(np.abs(rcg - ref["rcrit"]) / ref["rcrit"].clip(1e-300)) <= 1e-9
    ex = np.max(np.abs(xg - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(vg - ref["v"])) / np.max(np.abs(ref["v"]))
    assert ex <= x_tol and ev <= x_tol, f"{what}: state differs from the oracle run: x {ex:.3g}, v {ev:.3g}"
    # energy error of both runs from the same CPU diagnostic (reading S16)
    E0 = oracle.diagnostics(d.x, d.v, d.m, d.M_star, G_GAUSS)
    Eg = oracle.diagnostics(xg, vg, d.m, d.M_star, G_GAUSS)
    Er = oracle.diagnostics(ref["x"], ref["v"], d.m, d.M_star, G_GAUSS)
    de_g = (Eg["E"] - E0["E"]) / E0["E"]
    de_r = (Er["E"] - E0["E"]) / E0["E"]
    assert abs(de_g - de_r) <= ENERGY_TOL, f"{what}: energy error gpu {de_g:.3e} vs oracle {de_r:.3e}"
    dL = np.linalg.norm(Eg["L"] - E0["L"]) / np.linalg.norm(E0["L"])
    assert dL <= 1e-12, f"{what}: angular momentum drift {dL:.3e}"
    # last evaluation: accelerations and pair list at the final positions, from the GPU's own final state
    acc_ref, ab, _ = oracle.accel(xg, d.m, rcg, G_GAUSS, n_active=na, want_abs=True)
    assert_acc_close(accg, acc_ref, what + " final acc", ab)
    sure, border = oracle.pairs(xg, rcg, n_active=na)
    gp, n = st.get_pairs()
    assert_pairs_match(gp, n, sure, border, what + " final pairs")
    return dict(ex=ex, ev=ev, de_g=de_g, de_r=de_r, dL=dL)


def test_step_zero_steps_is_one_evaluation():
    d = nb_inputs.make_config(0, n_override=777)
    st = GpuState(d.x, d.v, d.m, G=G_GAUSS, n1=3.0, n2=0.4)
    st.step(d.dt, 0)
    xg, vg, accg, rcg = st.host()
    assert np.array_equal(xg, d.x) and np.array_equal(vg, d.v)
    rc_ref = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, 0.4)
    acc_ref, ab, _ = oracle.accel(d.x, d.m, rc_ref, G_GAUSS, want_abs=True)
    assert_acc_close(accg, acc_ref, "nsteps=0", ab)


@pytest.mark.parametrize("use_graph", [True, False])
def test_step_config1_100_steps(use_graph):
    """BASELINE.json:configs[0] in full: N = 2048, dt = 6 d, 100 steps, rcrit = 3 Hill radii."""
    d = nb_inputs.make_config(0)
    r = _step_compare(d, d.nsteps, 3.0, 0.0, what="config1 x100", x_tol=1e-9, use_graph=use_graph)
    print("config1:", r)


def test_step_one_and_two_steps_tight():
    d = nb_inputs.make_config(1, n_override=1200)
    _step_compare(d, 1, 3.0, 0.4, what="config2-shape x1", x_tol=1e-13)
    _step_compare(d, 2, 3.0, 0.4, what="config2-shape x2", x_tol=1e-13)
    _step_compare(d, 3, 3.0, 0.4, what="config2-shape x3 I=4", x_tol=1e-13, i_per_thread=4, j_splits=2)


def test_step_giants_1000_steps_energy():
    """north_star: after 1000 steps the relative energy error stays within 1e-9 of the oracle run
    (config-2 shape with both giants, planetesimal count reduced so the oracle run takes ~1 min)."""
    d = nb_inputs.make_config(1, n_override=1022)
    r = _step_compare(d, 1000, 3.0, 0.0, what="config2-shape x1000", x_tol=1e-7)
    print("giants x1000:", r)


def test_step_semi_active_and_ring():
    d = nb_inputs.make_config(3, n_override=4096)  # 32 active embryos + test masses
    _step_compare(d, 20, 3.0, 0.4, what="semi-active x20", x_tol=1e-10)
    d = nb_inputs.make_config(2, n_override=3000)  # encounter-dense ring, power-law masses
    _step_compare(d, 20, 3.0, 0.4, what="ring x20", x_tol=1e-10)


def test_step_reversible_on_gpu():
    d = nb_inputs.make_config(0, n_override=600)
    st = GpuState(d.x, d.v, d.m, G=G_GAUSS, n1=3.0, n2=0.0)
    st.step(d.dt, 5, with_pairs=False)
    st.step(-d.dt, 5, with_pairs=False)
    xg, vg, _, _ = st.host()
    assert np.max(np.abs(xg - d.x)) <= 1e-11 * np.max(np.abs(d.x))
    assert np.max(np.abs(vg - d.v)) <= 1e-11 * np.max(np.abs(d.v))
