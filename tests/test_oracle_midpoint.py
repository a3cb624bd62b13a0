"""-m "not gpu": pins of the oracle's implicit-midpoint wrapper for velocity-dependent forces (Eq. 8)
with the one force that stands in for the paper's list (drag against a gas disk; reading S24):
  * linear drag: Eq. 8 is linear in v^{t+dt} and has the closed form v' = [v (1 - g/2) + g v_gas] / (1 + g/2), g = gamma dt;
  * quadratic drag in one dimension: Eq. 8 is a quadratic equation for the midpoint speed, solved in closed form;
  * the implicit midpoint rule is symmetric: a step back from the result returns the start;
  * it is second order: against dv/dt = -gamma v |v|, v(t) = v0 / (1 + gamma v0 t);
  * "needs some iterations to converge": the iteration count is reported, divergence (gamma dt / 2 > 1) is counted;
  * in the step: gamma = 0 is the plain step bit for bit; a body on a circular orbit in sub-Keplerian gas spirals in at
    da/dt = -2 gamma eta a (headwind eta v_c; textbook drag migration)."""
import math

import numpy as np

import nb_inputs as nbi
import oracle

G = nbi.G_GAUSS


def test_linear_drag_closed_form():
    rng = np.random.default_rng(2)
    x = rng.uniform(-2, 2, (50, 3)); v = rng.uniform(-0.02, 0.02, (50, 3))
    for gamma, dt, eta in ((0.05, 3.0, 1.0), (0.01, 6.0, 0.0), (0.2, 1.5, 0.005), (0.3, -2.0, 0.1)):
        g = gamma * dt
        R = np.hypot(x[:, 0], x[:, 1])
        vc = (1 - eta) * np.sqrt(G / R)
        vg = np.stack([-vc * x[:, 1] / R, vc * x[:, 0] / R, np.zeros(50)], axis=1)
        v1, nf, it = oracle.midpoint_drag(x, v, G, dt, gamma, power=0, eta=eta, tol=1e-15, max_iter=200)
        ref = (v * (1 - g / 2) + g * vg) / (1 + g / 2)
        assert nf == 0 and 2 <= it <= 200
        np.testing.assert_allclose(v1, ref, rtol=0, atol=2e-15 * max(np.abs(ref).max(), np.abs(vg).max()))
    # gamma dt / 2 > 1: the fixed-point iteration of Eq. 8 does not converge -- counted, not hidden
    v1, nf, it = oracle.midpoint_drag(x, v, G, 10.0, 0.3, power=0, eta=1.0, tol=1e-14, max_iter=40)
    assert nf == 50 and it == 40


def test_quadratic_drag_closed_form_symmetry_and_order():
    gamma, dt = 3.0, 2.0
    # one dimension, gas at rest (eta = 1): dt gamma s^2 + 2 s - 2 v = 0 for the midpoint speed s
    x = np.array([[1.0, 0.0, 0.0]])
    for v0 in (0.02, 0.1, -0.05):
        v = np.array([[0.0, 0.0, v0]])          # along z: no gas component there
        v1, nf, it = oracle.midpoint_drag(x, v, G, dt, gamma, power=1, eta=1.0, tol=1e-15, max_iter=200)
        s = (-1 + math.sqrt(1 + 2 * gamma * dt * abs(v0))) / (gamma * dt)
        assert nf == 0 and abs(v1[0, 2] - math.copysign(2 * s - abs(v0), v0)) <= 1e-15
    # symmetric (time-reversible): a step of -dt from the result returns the start, with gas, in 3-D
    rng = np.random.default_rng(4)
    x = rng.uniform(0.5, 2, (40, 3)); v = rng.uniform(-0.02, 0.02, (40, 3))
    for power, gam in ((0, 0.5), (1, 15.0)):
        v1, nf, _ = oracle.midpoint_drag(x, v, G, 1.5, gam, power=power, eta=0.01, tol=1e-15, max_iter=300)
        v2, nf2, _ = oracle.midpoint_drag(x, v1, G, -1.5, gam, power=power, eta=0.01, tol=1e-15, max_iter=300)
        assert nf == 0 and nf2 == 0 and np.max(np.abs(v2 - v)) <= 2e-16 * 300
        assert np.max(np.abs(v1 - v)) > 1e-4
    # second order against the exact solution of dv/dt = -gamma v |v|
    v0, T = 0.1, 8.0
    exact = v0 / (1 + gamma * v0 * T)
    errs = []
    for n in (8, 16, 32):
        v = np.array([[0.0, 0.0, v0]])
        for _ in range(n):
            v, nf, _ = oracle.midpoint_drag(x, v, G, T / n, gamma, power=1, eta=1.0, tol=1e-15, max_iter=300)
        errs.append(abs(v[0, 2] - exact))
    assert 3.6 <= errs[0] / errs[1] <= 4.4 and 3.8 <= errs[1] / errs[2] <= 4.2, errs


def test_step_with_drag():
    d = nbi.make_config(0, n_override=300)
    a = oracle.step(d.x, d.v, d.m, d.M_star, d.dt, G, 3, n1=3.0, n2=0.4)
    b = oracle.step_drag(d.x, d.v, d.m, d.M_star, d.dt, G, 3, 0.0, n1=3.0, n2=0.4)
    assert b["n_fail"] == 0
    for k in ("x", "v", "acc", "rcrit"):
        assert np.array_equal(a[k], b[k])                    # gamma = 0: the plain step, bit for bit
    # one massless body on a circular orbit in sub-Keplerian gas: da/dt = -2 gamma eta a
    a0, gamma, eta = 1.0, 2e-3, 0.02
    x = np.array([[a0, 0.0, 0.0]]); v = np.array([[0.0, math.sqrt(G / a0), 0.0]]); m = np.zeros(1)
    nsteps, dt = 400, 2.0
    r = oracle.step_drag(x, v, m, 1.0, dt, G, nsteps, gamma, power=0, eta=eta, n1=3.0, n2=0.0)
    assert r["n_fail"] == 0
    rr = np.linalg.norm(r["x"][0]); vv = r["v"][0] @ r["v"][0]
    a1 = 1.0 / (2.0 / rr - vv / G)
    expect = a0 * math.exp(-2 * gamma * eta * nsteps * dt)
    assert a1 < a0 and abs((a1 - a0) / (expect - a0) - 1.0) < 0.05
    # co-rotating gas (eta = 0) leaves a circular orbit alone
    r0 = oracle.step_drag(x, v, m, 1.0, dt, G, 50, gamma, power=1, eta=0.0, n1=3.0, n2=0.0)
    assert abs(np.linalg.norm(r0["x"][0]) - a0) < 1e-12
