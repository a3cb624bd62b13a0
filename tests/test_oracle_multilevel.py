"""-m "not gpu": pins of the oracle's multi-level changeover (reading S23) against what the
paper's statement and the mathematics fix:
  * the levels' weights are a partition of unity at every separation (H = H_A + H_B must stay the Newtonian pair force
    however many "higher-level changeover functions" are introduced) -- closed form through the pinned W (P1);
  * one level kick of one pair is Omega_l W_{l+1} G m_j / r^2 along the line of centres; all operators together give
    G m_j / r^2 (the sum rule that ties oracle_level_kick and the level product of the direct solver's right-hand side
    to Eq. 4 + Eq. 5);
  * no intermediate level (nlev = 1) is the plain hybrid step, bit for bit;
  * every operator is a sum of central pair forces or a Kepler flow: total momentum of a group and the angular momentum
    are conserved to rounding;
  * the intermediate levels are a second-order symplectic approximation of the flow the direct solver integrates: the
    difference to a tight Bulirsch-Stoer solution of the same Hamiltonian falls by 4 when the step is halved;
  * the regime the paper describes ("every particle is in a close encounter ... the single group of close encounters that
    contain all particles"): with the full Eq. 7 radius a dense ring is one group beyond the direct solver's cap -- the
    levels shrink the groups until nothing is skipped, and the energy error drops."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

G = G_GAUSS


@pytest.mark.parametrize("kind", [0, 1])
def test_level_weights_are_a_partition_of_unity(kind):
    rng = np.random.default_rng(3)
    for _ in range(50):
        L = int(rng.integers(0, 5))
        rcs = np.sort(rng.uniform(1e-3, 1.0, L + 1))[::-1]
        if rng.uniform() < 0.3:
            rng.shuffle(rcs)                                   # not even nested: the identity is algebraic
        for r in np.concatenate([rng.uniform(0, 1.2, 40), 0.1 * rcs, rcs, 0.55 * rcs]):
            w = oracle.level_weights(float(r), rcs, kind)
            assert len(w) == L + 2 and all(0.0 <= t <= 1.0 for t in w)
            assert abs(sum(w) - 1.0) <= 4e-16 * (L + 2)
    rcs = [0.8, 0.4, 0.2]
    assert oracle.level_weights(0.8, rcs, kind) == [1.0, 0.0, 0.0, 0.0]            # beyond rc_0: all in the outer kick
    assert oracle.level_weights(0.02, rcs, kind) == [0.0, 0.0, 0.0, 1.0]           # inside 0.1 rc_L: all in the direct solver
    w = oracle.level_weights(0.44, rcs, kind)                                      # = 0.55 rc_0, beyond rc_1
    assert abs(w[0] - 0.5) < 1e-15 and abs(w[1] - 0.5) < 1e-15 and w[2] == 0.0 and w[3] == 0.0
    w = oracle.level_weights(0.22, rcs, kind)                                      # = 0.55 rc_1, inside the shell of rc_0, beyond rc_2
    W0 = oracle.changeover(0.22, 0.8, kind)
    assert w[0] == W0 and abs(w[1] - 0.5 * (1 - W0)) < 1e-15 and abs(w[2] - 0.5 * (1 - W0)) < 1e-15 and w[3] == 0.0


@pytest.mark.parametrize("kind", [0, 1])
def test_level_kick_of_one_pair_and_the_sum_rule(kind):
    m = np.array([2e-3, 5e-4, 1e-3])
    d = np.array([0.36, -0.48, 0.8])
    rc0 = np.array([0.04, 0.012, 0.0]); rcl = np.stack([rc0, 0.5 * rc0, 0.25 * rc0])    # L = 2
    for frac in (0.05, 0.15, 0.22, 0.3, 0.45, 0.7, 0.95, 1.2):
        x = np.stack([np.array([1.0, 0.3, -0.2]), np.array([1.0, 0.3, -0.2]) + frac * 0.04 * d, np.array([1.0, 0.3, -0.2]) - 0.001 * d])
        r = float(np.linalg.norm(x[1] - x[0])); u = (x[1] - x[0]) / r
        v0 = np.array([[1e-3, -2e-3, 5e-4], [3e-3, 1e-3, -1e-3], [0.0, 1e-3, 0.0]])
        w = oracle.level_weights(r, [0.04, 0.02, 0.01], kind)
        full = G * m / r ** 2
        total = np.zeros((2, 3))
        for level in (0, 1):
            h = 0.7
            v1 = oracle.level_kick(x, v0, m, G, [[0, 1]], rcl, level, h, kind)
            dv = (v1 - v0) / h
            np.testing.assert_allclose(dv[0], w[level + 1] * full[1] * u, rtol=1e-11, atol=1e-13 * full[1])
            np.testing.assert_allclose(dv[1], -w[level + 1] * full[0] * u, rtol=1e-11, atol=1e-13 * full[0])
            assert np.array_equal(v1[2], v0[2])                                    # body 2 is in no listed pair
            p0, p1 = (m[:, None] * v0).sum(0), (m[:, None] * v1).sum(0)
            assert np.max(np.abs(p1 - p0)) <= 1e-15 * np.abs(m[:, None] * v0).sum()
            total += dv[:2]
        # outer kick (Eq. 5) + level kicks + direct solver's pair term (Eq. 4 at the innermost level) = Newton
        acc, _, _ = oracle.accel(x[:2], m[:2], rcl[0][:2], G, kind=kind)
        _, vd = oracle.encounter_rhs(x[:2], v0[:2], G * m[:2], rcl[:, :2], 0.0, kind)
        np.testing.assert_allclose(acc[0], w[0] * full[1] * u, rtol=2e-14, atol=4e-16 * full[1])
        np.testing.assert_allclose(vd[0], w[3] * full[1] * u, rtol=2e-14, atol=4e-16 * full[1])
        np.testing.assert_allclose(acc[0] + total[0] + vd[0], full[1] * u, rtol=1e-11)
        np.testing.assert_allclose(acc[1] + total[1] + vd[1], -full[0] * u, rtol=1e-11)
    # a massless body pulls on nobody; an empty list is the identity
    m0 = np.array([1e-3, 0.0])
    x = np.array([[1.0, 0, 0], [1.0, 0.01, 0]]); v0 = np.zeros((2, 3))
    v1 = oracle.level_kick(x, v0, m0, G, [[0, 1]], np.full((2, 2), 0.05) * np.array([[1.0], [0.5]]), 0, 1.0, kind)
    assert np.array_equal(v1[0], v0[0]) and v1[1][1] < 0.0
    assert np.array_equal(oracle.level_kick(x, v0, m0, G, np.zeros((0, 2)), np.full((2, 2), 0.05), 0, 1.0, kind), v0)


def test_no_intermediate_level_is_the_plain_hybrid_step():
    d = nb_inputs.make_config(2, n_override=700)
    a = oracle.step_enc(d.x, d.v, d.m, d.M_star, d.dt, G, 4, n1=3.0, n2=0.4)
    b = oracle.step_ml(d.x, d.v, d.m, d.M_star, d.dt, G, 4, 1, n1=3.0, n2=0.4)
    assert a["stats"]["integrated"] > 0
    assert np.array_equal(a["x"], b["x"]) and np.array_equal(a["v"], b["v"]) and np.array_equal(a["acc"], b["acc"])
    assert np.array_equal(a["pairs"], b["pairs"]) and np.array_equal(a["rcrit"], b["rcrit"][0])
    assert b["stats"]["integrated"] == a["stats"]["integrated"] and b["stats"]["kicks"] == 0


def test_level_radii_follow_eq7_with_the_level_time_step():
    d = nb_inputs.make_config(0, n_override=200)
    rcl = oracle.level_rcrit(d.x, d.v, d.m, d.M_star, d.dt, G, 3.0, 0.4, 4)
    hill = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G, 3.0, 0.0)
    vel = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G, 0.0, 0.4)
    for l in range(4):
        assert np.array_equal(rcl[l], np.maximum(hill, vel / 2 ** l))             # the Hill term is the floor
    assert np.all(rcl[0] >= rcl[1]) and np.mean(rcl[0] > rcl[1]) > 0.5 and np.all(rcl[3] >= hill)
    r0 = np.linspace(0.01, 0.02, 200)
    assert np.array_equal(oracle.level_rcrit(d.x, d.v, d.m, d.M_star, d.dt, G, 0.0, 0.0, 3, rcrit0=r0), np.stack([r0, r0 / 2, r0 / 4]))


def _clump(n, seed, spacing=2.5e-3, mass=(2e-7, 6e-7)):
    rng = np.random.default_rng(seed)
    side = int(np.ceil(np.sqrt(n)))
    cell = rng.permutation(side * side)[:n]
    gi, gj = np.divmod(cell, side)
    a = 1.0 + spacing * (gi - side / 2) + rng.uniform(-3e-4, 3e-4, n)
    M = 0.4 + spacing * (gj - side / 2) + rng.uniform(-3e-4, 3e-4, n)
    x, v = nb_inputs.elements_to_cartesian(a, rng.uniform(0, 2e-3, n), rng.uniform(0, 1e-3, n), np.zeros(n), np.zeros(n), M, G)
    return np.ascontiguousarray(x), np.ascontiguousarray(v), rng.uniform(*mass, n)


def test_levels_conserve_momentum_and_angular_momentum():
    x, v, m = _clump(12, 4)
    rc0 = np.full(12, 0.03)
    rcl = oracle.level_rcrit(x, v, m, 1.0, 4.0, G, 0.0, 0.0, 4, rcrit0=rc0)
    sure, _ = oracle.pairs(x, rc0)
    assert sure.shape[0] > 20
    L0 = (m[:, None] * np.cross(x, v)).sum(0)
    xe, ve, st = oracle.encounter_ml(x, v, m, rcl, 1.0, 4.0, G, sure, tol=1e-13)
    assert st["failed"] == 0 and st["skipped"] == 0 and st["kicks"] > 0 and st["level_pairs"][3] > 0
    L1 = (m[:, None] * np.cross(xe, ve)).sum(0)
    assert np.linalg.norm(L1 - L0) <= 2e-14 * np.linalg.norm(L0)
    assert np.max(np.abs(xe - x)) > 1e-3


def test_levels_are_second_order_accurate_for_the_flow_of_H_A():
    """Fixed Hamiltonian: Kepler + listed pair terms weighted by Omega_0 (level radii rc / 2^l, caller's rc).  Reference:
    the direct solver alone (L = 0) at tol 1e-14.  The two-level scheme over the same total time in n outer intervals:
    error ~ 1/n^2."""
    x, v, m = _clump(6, 8, spacing=4e-3, mass=(1e-6, 3e-6))
    rc0 = np.full(6, 0.05)
    sure, _ = oracle.pairs(x, rc0)
    assert sure.shape[0] == 15
    T = 2.0
    xr, vr, _ = oracle.encounter_ml(x, v, m, rc0[None], 1.0, T, G, sure, tol=1e-14)
    rcl = np.stack([rc0, rc0 / 2, rc0 / 4])
    errs = []
    for n in (2, 4, 8):
        xa, va = x.copy(), v.copy()
        for _ in range(n):
            xa, va, st = oracle.encounter_ml(xa, va, m, rcl, 1.0, T / n, G, sure, tol=1e-14)
            assert st["failed"] == 0
        errs.append(np.max(np.abs(xa - xr)))
    print("levels vs direct solver:", errs)
    assert errs[0] > 1e-11                                     # the intermediate levels really are a different integrator
    assert 3.0 <= errs[0] / errs[1] <= 5.0 and 3.0 <= errs[1] / errs[2] <= 5.0


def test_close_approach_energy_with_levels():
    """The two embryos of the L = 0 physics pin (tests/test_oracle_encounter.py), full Eq. 7 radius: resolving the
    encounter through 2 or 3 intermediate levels conserves the energy as well as handing the whole encounter to the
    direct solver, and far better than the plain Kepler drift."""
    m = np.array([3e-6, 3e-6])
    x, v = nb_inputs.elements_to_cartesian(np.array([1.0, 1.004]), np.array([0.0, 0.004]), np.array([0.0, 0.001]),
                                           np.array([0.0, 0.2]), np.array([0.0, 0.0]), np.array([0.0, -0.208]), G)
    x = np.ascontiguousarray(x); v = np.ascontiguousarray(v)
    v -= np.sum(m[:, None] * v, axis=0) / (1.0 + m.sum())
    dt, nsteps = 2.0, 60
    E0 = oracle.diagnostics(x, v, m, 1.0, G)["E"]
    plain = oracle.step(x, v, m, 1.0, dt, G, nsteps, n1=3.0, n2=0.4)
    dE = {0: abs((oracle.diagnostics(plain["x"], plain["v"], m, 1.0, G)["E"] - E0) / E0)}
    for nlev in (1, 3, 4):
        r = oracle.step_ml(x, v, m, 1.0, dt, G, nsteps, nlev, n1=3.0, n2=0.4)
        assert r["stats"]["failed"] == 0 and r["stats"]["integrated"] >= 1
        dE[nlev] = abs((oracle.diagnostics(r["x"], r["v"], m, 1.0, G)["E"] - E0) / E0)
        if nlev > 1:
            assert r["stats"]["kicks"] > 0
    print("dE/E: plain", dE[0], "nlev=1", dE[1], "nlev=3", dE[3], "nlev=4", dE[4])
    assert dE[3] < 0.05 * dE[0] and dE[4] < 0.05 * dE[0]
    assert dE[3] < 5.0 * dE[1] and dE[4] < 5.0 * dE[1]


def test_levels_dissolve_the_giant_group_of_a_dense_ring():
    """bodies "too tightly packed, such that every particle is in a close encounter with another particle
    ... the single group of close encounters that contain all particles".  The config-3 ring at N = 8192 with the full
    Eq. 7 radius is one group of ~8100 bodies, beyond the direct solver's cap of 1024: without levels it is skipped (left
    to the Kepler drift); with 3 intermediate levels the groups that reach the direct solver fit, nothing is skipped, and
    the energy error drops by orders of magnitude."""
    d = nb_inputs.make_config(2, n_override=8192)
    E0 = oracle.diagnostics(d.x, d.v, d.m, d.M_star, G)["E"]
    out = {}
    for nlev in (1, 4):
        r = oracle.step_ml(d.x, d.v, d.m, d.M_star, d.dt, G, 3, nlev, n1=3.0, n2=0.4)
        out[nlev] = (r["stats"], abs((oracle.diagnostics(r["x"], r["v"], d.m, d.M_star, G)["E"] - E0) / E0))
        print(nlev, out[nlev])
    assert out[1][0]["skipped"] > 0
    assert out[4][0]["skipped"] == 0 and out[4][0]["failed"] == 0
    lp = out[4][0]["level_pairs"]
    assert lp[0] > lp[1] / 2 > lp[2] / 4 > lp[3] / 8 > 0      # fewer pairs per visit, level by level (level l is visited 2^l times)
    assert out[4][1] < 0.01 * out[1][1]
