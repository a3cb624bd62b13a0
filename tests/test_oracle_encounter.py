"""-m "not gpu": pins of the oracle's close-encounter integrator (oracle_encounter; Eq. 4,
PAPER.md:98, 106) against what the mathematics fixes:
  * with the pair term switched off (rc = 0 => 1 - W = 0) H_A is a set of Kepler problems: the result
    must equal the analytic Kepler drift (oracle.drift_kepler, itself pinned by closed forms);
  * deep inside the changeover (1 - W = 1) around a star of negligible mass the relative motion of a
    pair is a Kepler problem in the relative coordinates with mu = G (m1 + m2) and the barycentre moves
    uniformly: checked with the oracle's Kepler solver (an independent route);
  * the flow of H_A conserves H_A's own energy and the angular momentum, and is reversible;
  * the error follows the tolerance;
  * bodies outside groups, and groups beyond max_group, are left untouched."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS


def _grp(pairs, N):
    return oracle.groups(np.asarray(pairs, dtype=np.int32), N)


def test_no_pair_term_reduces_to_kepler_drift():
    x, v = nb_inputs.elements_to_cartesian(np.array([1.0, 1.3, 2.2, 0.7]), np.array([0.1, 0.3, 0.0, 0.6]),
                                           np.array([0.0, 0.1, 0.2, 0.05]), np.array([0.3, 1.0, 2.0, 4.0]),
                                           np.array([0.0, 2.0, 1.0, 3.0]), np.array([0.5, 3.0, 6.0, 0.1]), G_GAUSS)
    m = np.array([1e-6, 3e-6, 1e-7, 2e-6]); rc = np.zeros(4)
    for dt in (6.0, -6.0, 40.0):
        xe, ve, st = oracle.encounter(x, v, m, rc, 1.0, dt, G_GAUSS, _grp([[0, 1], [1, 2]], 4), tol=1e-13)
        xk, vk, nfail = oracle.drift_kepler(x, v, 1.0, dt, G_GAUSS)
        assert nfail == 0 and st["integrated"] == 1 and st["failed"] == 0
        assert np.max(np.abs(xe[:3] - xk[:3])) <= 2e-12 and np.max(np.abs(ve[:3] - vk[:3])) <= 2e-12 * np.max(np.abs(vk))
        assert np.array_equal(xe[3], x[3]) and np.array_equal(ve[3], v[3])       # body 3 is in no group


def test_isolated_pair_is_a_relative_kepler_problem():
    G = G_GAUSS
    m = np.array([3e-6, 1e-6]); M_star = 1e-30                                    # star switched off
    # relative orbit: a = 0.01 AU, e = 0.4 about the pair's barycentre, which drifts uniformly
    mu_rel = G * m.sum()
    xr, vr = nb_inputs.elements_to_cartesian(np.array([0.01]), np.array([0.4]), np.array([0.3]), np.array([1.0]),
                                             np.array([2.0]), np.array([0.7]), mu_rel)
    xb, vb = np.array([1.0, -0.5, 0.2]), np.array([1e-3, 2e-3, -5e-4])
    x = np.stack([xb - m[1] / m.sum() * xr[0], xb + m[0] / m.sum() * xr[0]])
    v = np.stack([vb - m[1] / m.sum() * vr[0], vb + m[0] / m.sum() * vr[0]])
    rc = np.full(2, 10.0)                                                          # r << 0.1 rc: 1 - W = 1 throughout
    P = 2 * np.pi * np.sqrt(0.01 ** 3 / mu_rel)
    for dt in (0.3 * P, 1.7 * P):
        xe, ve, st = oracle.encounter(x, v, m, rc, M_star, dt, G, _grp([[0, 1]], 2), tol=1e-13)
        xk, vk, code = oracle.kepler_one(xr[0], vr[0], mu_rel, dt)
        assert code == 0
        rel_x, rel_v = xe[1] - xe[0], ve[1] - ve[0]
        assert np.max(np.abs(rel_x - xk)) <= 1e-10 * 0.01, (rel_x, xk)
        assert np.max(np.abs(rel_v - vk)) <= 1e-10 * np.linalg.norm(vk)
        bary_x = (m[0] * xe[0] + m[1] * xe[1]) / m.sum()
        assert np.max(np.abs(bary_x - (xb + dt * vb))) <= 1e-13
        assert st["steps"] >= 2


def _energy_HA(x, v, m, M_star, G):
    """H_A with 1 - W = 1 for every pair (Eq. 4 inside the changeover)."""
    E = np.sum(0.5 * m * np.sum(v * v, axis=1)) - np.sum(G * M_star * m / np.linalg.norm(x, axis=1))
    for i in range(len(m)):
        for j in range(i + 1, len(m)):
            E -= G * m[i] * m[j] / np.linalg.norm(x[i] - x[j])
    return E


def test_conservation_reversibility_and_tolerance():
    G = G_GAUSS
    rng = np.random.default_rng(5)
    n = 5
    m = rng.uniform(1e-6, 1e-5, n)
    a = 1.0 + rng.uniform(-1e-2, 1e-2, n)
    x, v = nb_inputs.elements_to_cartesian(a, rng.uniform(0, 0.01, n), rng.uniform(0, 0.005, n), np.full(n, 1.0),
                                           np.full(n, 2.0), 0.3 + rng.uniform(-1e-2, 1e-2, n), G)
    rc = np.full(n, 1.0)                                    # every pair far inside 0.1 rc
    grp = _grp([[0, 1], [1, 2], [2, 3], [3, 4]], n)
    dt = 6.0
    E0 = _energy_HA(x, v, m, 1.0, G); L0 = np.sum(m[:, None] * np.cross(x, v), axis=0)
    xe, ve, st = oracle.encounter(x, v, m, rc, 1.0, dt, G, grp, tol=1e-13)
    E1 = _energy_HA(xe, ve, m, 1.0, G); L1 = np.sum(m[:, None] * np.cross(xe, ve), axis=0)
    def pair_energy(xx):
        return -sum(G * m[i] * m[j] / np.linalg.norm(xx[i] - xx[j]) for i in range(n) for j in range(i + 1, n))
    assert abs((pair_energy(xe) - pair_energy(x)) / E0) >= 1e-7       # the pair terms really exchange energy
    assert abs((E1 - E0) / E0) <= 1e-11
    assert np.linalg.norm(L1 - L0) <= 1e-13 * np.linalg.norm(L0)
    xb, vb, _ = oracle.encounter(xe, ve, m, rc, 1.0, -dt, G, grp, tol=1e-13)
    assert np.max(np.abs(xb - x)) <= 1e-11 and np.max(np.abs(vb - v)) <= 1e-11 * np.max(np.abs(v))
    # the error follows the tolerance
    xl, vl, stl = oracle.encounter(x, v, m, rc, 1.0, dt, G, grp, tol=1e-8)
    xt, vt, stt = oracle.encounter(x, v, m, rc, 1.0, dt, G, grp, tol=1e-11)
    e_loose, e_tight = np.max(np.abs(xl - xe)), np.max(np.abs(xt - xe))
    assert e_tight <= 1e-9 and e_loose <= 1e-5 and e_tight < e_loose
    # quintic weight: same invariants inside the shell where both shapes give 1 - W = 1
    xq, vq, _ = oracle.encounter(x, v, m, rc, 1.0, dt, G, grp, kind=1, tol=1e-13)
    assert np.max(np.abs(xq - xe)) <= 1e-12


def test_transition_shell_and_group_cap():
    """Inside the transition shell the pair force is a fraction 0 < 1 - W < 1 of the Newtonian one: the
    result lies strictly between the pure Kepler drift (1 - W = 0) and the full pair force (1 - W = 1);
    a group beyond max_group is skipped and reported."""
    G = G_GAUSS
    m = np.array([1e-4, 1e-4])
    x, v = nb_inputs.elements_to_cartesian(np.array([1.0, 1.0]), np.zeros(2), np.zeros(2), np.zeros(2), np.zeros(2),
                                           np.array([0.0, 0.004]), G)
    sep = np.linalg.norm(x[1] - x[0])
    grp = _grp([[0, 1]], 2)
    res = {}
    for name, rcv in (("none", 0.0), ("half", sep / 0.55), ("full", 100.0)):
        res[name] = oracle.encounter(x, v, m, np.full(2, rcv), 1.0, 3.0, G, grp, tol=1e-13)[0]
    d_half = np.linalg.norm(res["half"][1] - res["half"][0])
    d_none = np.linalg.norm(res["none"][1] - res["none"][0])
    d_full = np.linalg.norm(res["full"][1] - res["full"][0])
    assert d_full < d_half < d_none or d_full > d_half > d_none
    xs, vs, st = oracle.encounter(x, v, m, np.full(2, 100.0), 1.0, 3.0, G, grp, max_group=1)
    assert st["skipped"] == 1 and st["integrated"] == 0 and np.array_equal(xs, x) and np.array_equal(vs, v)


def test_resolving_encounters_restores_energy_conservation():
    """Two embryos on crossing orbits that pass within a fraction of a Hill radius: with the pure Kepler
    drift in A the part [1 - W] of their attraction is simply missing while they are close, and the total
    energy jumps; with the direct solver (step_enc) it is conserved orders of magnitude better -- the
    reason the hybrid scheme exists."""
    G = G_GAUSS
    m = np.array([3e-6, 3e-6])
    x, v = nb_inputs.elements_to_cartesian(np.array([1.0, 1.004]), np.array([0.0, 0.004]), np.array([0.0, 0.001]),
                                           np.array([0.0, 0.2]), np.array([0.0, 0.0]), np.array([0.0, -0.208]), G)
    x = np.ascontiguousarray(x); v = np.ascontiguousarray(v)
    v -= np.sum(m[:, None] * v, axis=0) / (1.0 + m.sum())
    dt, nsteps = 2.0, 60
    E0 = oracle.diagnostics(x, v, m, 1.0, G)["E"]
    plain = oracle.step(x, v, m, 1.0, dt, G, nsteps, n1=3.0, n2=0.4)
    res = oracle.step_enc(x, v, m, 1.0, dt, G, nsteps, n1=3.0, n2=0.4)
    dmin = np.linalg.norm(x[1] - x[0])
    assert res["stats"]["integrated"] >= 3 and res["stats"]["failed"] == 0       # the pair really was a group
    dE_plain = abs((oracle.diagnostics(plain["x"], plain["v"], m, 1.0, G)["E"] - E0) / E0)
    dE_enc = abs((oracle.diagnostics(res["x"], res["v"], m, 1.0, G)["E"] - E0) / E0)
    print("dE/E plain", dE_plain, "with encounters", dE_enc, "initial separation", dmin)
    assert dE_enc < 0.05 * dE_plain
    # no encounter => the two schemes coincide exactly (nothing is in a group)
    far_x, far_v = nb_inputs.elements_to_cartesian(np.array([1.0, 2.0]), np.zeros(2), np.zeros(2), np.zeros(2),
                                                   np.zeros(2), np.array([0.0, 2.0]), G)
    a = oracle.step(far_x, far_v, m, 1.0, dt, G, 5, n1=3.0, n2=0.4)
    b = oracle.step_enc(far_x, far_v, m, 1.0, dt, G, 5, n1=3.0, n2=0.4)
    assert np.array_equal(a["x"], b["x"]) and np.array_equal(a["v"], b["v"]) and b["stats"]["integrated"] == 0


def test_semi_active_groups_are_split_into_core_and_independent_test_particles():
    """Semi-active mode (reading S22): test particles pull on nobody, so the core of a group must move exactly as
    if they were absent, every test particle exactly as in the problem {core + that particle}, and a single
    embryo with a test particle deep inside its changeover radius around a negligible star is a Kepler problem
    about the embryo."""
    G = G_GAUSS
    rng = np.random.default_rng(9)
    n_act, n_sat = 3, 12
    N = n_act + n_sat + 2
    # embryos and test particles on a jittered 4 x 4 lattice (spacing 3e-3): close, but nobody on top of anybody
    gi, gj = np.divmod(rng.permutation(16)[: n_act + n_sat], 4)
    a = np.concatenate([1.0 + 3e-3 * (gi - 1.5) + rng.uniform(-5e-4, 5e-4, n_act + n_sat), [2.0, 2.5]])
    M = np.concatenate([0.4 + 3e-3 * (gj - 1.5) + rng.uniform(-5e-4, 5e-4, n_act + n_sat), [1.0, 3.0]])
    x, v = nb_inputs.elements_to_cartesian(a, np.full(N, 1e-3), np.full(N, 5e-4), np.zeros(N), np.zeros(N), M, G)
    x = np.ascontiguousarray(x); v = np.ascontiguousarray(v)
    m = np.zeros(N); m[:n_act] = [2e-7, 1e-7, 3e-7]
    rc = np.full(N, 0.05)
    pairs = [[0, 1], [1, 2]] + [[int(rng.integers(0, n_act)), k] for k in range(n_act, n_act + n_sat)]
    grp = oracle.groups(np.array(pairs, dtype=np.int32), N)
    assert grp["ngroups"] == 1 and grp["largest"] == n_act + n_sat
    xs, vs, st = oracle.encounter(x, v, m, rc, 1.0, 3.0, G, grp, n_active=n_act, tol=1e-13)
    assert st["integrated"] == 1 and st["failed"] == 0
    # core: identical to the core integrated alone (bit for bit: it IS that integration)
    core = oracle.groups(np.array([[0, 1], [1, 2]], dtype=np.int32), N)
    xc, vc, _ = oracle.encounter(x, v, m, rc, 1.0, 3.0, G, core, tol=1e-13)
    assert np.array_equal(xs[:n_act], xc[:n_act]) and np.array_equal(vs[:n_act], vc[:n_act])
    # every test particle: identical to the problem {core + particle}
    for k in (n_act, n_act + 7, n_act + n_sat - 1):
        one = oracle.groups(np.array([[0, 1], [1, 2], [0, k]], dtype=np.int32), N)
        xo, vo, _ = oracle.encounter(x, v, m, rc, 1.0, 3.0, G, one, tol=1e-13)
        assert np.array_equal(xs[k], xo[k]) and np.array_equal(vs[k], vo[k])
    # bodies outside the group untouched; the unsplit treatment agrees to the tolerance (same physics)
    assert np.array_equal(xs[-2:], x[-2:])
    xu, vu, _ = oracle.encounter(x, v, m, rc, 1.0, 3.0, G, grp, tol=1e-13)
    assert np.max(np.abs(xu[:n_act] - xs[:n_act])) <= 1e-11 and np.median(np.abs(xu - xs)) <= 1e-11
    # closed form: embryo + test particle, star switched off => Kepler orbit of the particle about the embryo
    m2 = np.array([3e-6, 0.0]); mu = G * m2[0]
    xr, vr = nb_inputs.elements_to_cartesian(np.array([0.01]), np.array([0.3]), np.array([0.2]), np.array([1.0]),
                                             np.array([2.0]), np.array([0.5]), mu)
    x2 = np.stack([np.array([1.0, 0.2, 0.0]), np.array([1.0, 0.2, 0.0]) + xr[0]]); v2 = np.stack([np.array([0.0, 1e-3, 0.0]), np.array([0.0, 1e-3, 0.0]) + vr[0]])
    P = 2 * np.pi * np.sqrt(0.01 ** 3 / mu)
    xe, ve, _ = oracle.encounter(x2, v2, m2, np.full(2, 10.0), 1e-30, 0.8 * P, G, oracle.groups(np.array([[0, 1]]), 2), n_active=1, tol=1e-13)
    xk, vk, code = oracle.kepler_one(xr[0], vr[0], mu, 0.8 * P)
    assert code == 0 and np.max(np.abs((xe[1] - xe[0]) - xk)) <= 1e-10 * 0.01
    assert np.max(np.abs(xe[0] - (x2[0] + 0.8 * P * v2[0]))) <= 1e-13      # the embryo does not feel the particle


@pytest.mark.parametrize("kind", [0, 1])
def test_pair_term_inside_the_transition_shell_is_one_minus_W(kind):
    """Pin of the [1 - W] factor BETWEEN its end values (Eq. 4 carries [1 - K], Eq. 5 carries K):
    for a pair at r/rc in {0.15, 0.3, 0.7, 0.95} (all off the symmetric point 0.55, so W and 1 - W differ)
      (i)  the group right-hand side gives exactly (1 - oracle.changeover(r, rc)) G m_j / r^2 along the line
           (oracle.changeover is pinned on its own by P1: end points, midpoint, monotone, W(y) + W(1-y) = 1);
      (ii) the kick acceleration (oracle.accel, weight W) plus the encounter acceleration is the full Newtonian
           G m_j / r^2 -- the two Hamiltonians share one pair force (Eq. 4 [1 - K] + Eq. 5 K);
      (iii) integrated: two bodies at relative rest around a star of negligible mass, tiny dt: dv/dt of each body
           equals that acceleration."""
    G = G_GAUSS
    m = np.array([2e-3, 5e-4])
    rcv = 0.04
    d = np.array([0.36, -0.48, 0.8])                                     # unit vector
    for frac in (0.15, 0.3, 0.7, 0.95):
        r = frac * rcv
        x = np.stack([np.array([1.0, 0.3, -0.2]), np.array([1.0, 0.3, -0.2]) + r * d])
        v = np.tile(np.array([1e-6, 2e-6, -1e-6]), (2, 1))             # common drift: fixes the velocity scale of the error test
        rc = np.array([rcv, 0.3 * rcv])                                   # max rule: rc_ij = rcv
        r = float(np.linalg.norm(x[1] - x[0])); d = (x[1] - x[0]) / r      # the separation as stored (x ~ 1 rounds r at 1e-14)
        W = oracle.changeover(r, rcv, kind)
        assert 0.0 < W < 1.0 and abs(W - 0.5) > 0.05
        # (i) right-hand side, star switched off
        xd, vd = oracle.encounter_rhs(x, v, G * m, rc, 0.0, kind)
        assert np.array_equal(xd, v)
        # (1 - W formed here from the pinned W loses eps/(1 - W) to cancellation: allow eps of the FULL force on top)
        full = G * m / r ** 2
        np.testing.assert_allclose(vd[0], (1.0 - W) * full[1] * d, rtol=2e-14, atol=4e-16 * full[1])
        np.testing.assert_allclose(vd[1], -(1.0 - W) * full[0] * d, rtol=2e-14, atol=4e-16 * full[0])
        # (ii) sum rule with the kick
        acc, _, _ = oracle.accel(x, m, rc, G, kind=kind)
        np.testing.assert_allclose(acc[0] + vd[0], G * m[1] / r ** 2 * d, rtol=2e-14)
        np.testing.assert_allclose(acc[1] + vd[1], -G * m[0] / r ** 2 * d, rtol=2e-14)
        # (iii) through the integrator: dv = a dt + O(dt^3) (relative rest => no dt^2 term); a dt^2 / r ~ 1e-10
        dt = 1e-5
        xe, ve, st = oracle.encounter(x, v, m, rc, 1e-30, dt, G, _grp([[0, 1]], 2), kind=kind, tol=1e-14)
        assert st["integrated"] == 1 and st["failed"] == 0
        for b, sign, mj in ((0, 1.0, m[1]), (1, -1.0, m[0])):
            a_num = (ve[b] - v[b]) / dt
            a_ref = sign * (1.0 - W) * G * mj / r ** 2 * d
            assert np.linalg.norm(a_num - a_ref) <= 1e-8 * np.linalg.norm(a_ref), (frac, kind, a_num, a_ref)
    # outside rc the pair term vanishes, inside 0.1 rc it is the full force
    for frac, w1 in ((1.2, 0.0), (0.05, 1.0)):
        x = np.stack([np.zeros(3) + [1, 0, 0], np.array([1.0, 0, 0]) + frac * rcv * d])
        r = float(np.linalg.norm(x[1] - x[0])); d = (x[1] - x[0]) / r
        _, vd = oracle.encounter_rhs(x, np.zeros((2, 3)), G * m, np.full(2, rcv), 0.0, kind)
        np.testing.assert_allclose(vd[0], w1 * G * m[1] / r ** 2 * d, rtol=2e-14, atol=0)


def test_split_threshold_is_an_argument_not_a_constant():
    """Reading S22: the definition splits EVERY group that has test particles; an implementation may stop splitting at
    some core size (split_max_core).  Both treatments describe the same motion: they agree to the Bulirsch-Stoer
    tolerance; with the threshold below the core size nothing is split (identical to the fully active routine)."""
    G = G_GAUSS
    rng = np.random.default_rng(12)
    n_act, n_sat = 4, 6
    N = n_act + n_sat
    a = 1.0 + 3e-3 * rng.permutation(N) + rng.uniform(-3e-4, 3e-4, N)
    M = 0.4 + 3e-3 * rng.permutation(N) + rng.uniform(-3e-4, 3e-4, N)
    x, v = nb_inputs.elements_to_cartesian(a, np.full(N, 1e-3), np.full(N, 5e-4), np.zeros(N), np.zeros(N), M, G)
    x = np.ascontiguousarray(x); v = np.ascontiguousarray(v)
    m = np.zeros(N); m[:n_act] = rng.uniform(1e-7, 3e-7, n_act)
    rc = np.full(N, 0.05)
    grp = oracle.groups(np.array([[i, i + 1] for i in range(N - 1)], dtype=np.int32), N)
    always = oracle.encounter(x, v, m, rc, 1.0, 3.0, G, grp, n_active=n_act, tol=1e-13)
    wide = oracle.encounter(x, v, m, rc, 1.0, 3.0, G, grp, n_active=n_act, tol=1e-13, split_max_core=n_act)
    never = oracle.encounter(x, v, m, rc, 1.0, 3.0, G, grp, n_active=n_act, tol=1e-13, split_max_core=n_act - 1)
    plain = oracle.encounter(x, v, m, rc, 1.0, 3.0, G, grp, tol=1e-13)
    assert np.array_equal(always[0], wide[0]) and np.array_equal(always[1], wide[1])
    assert np.array_equal(never[0], plain[0]) and np.array_equal(never[1], plain[1])
    assert np.max(np.abs(always[0] - never[0])) <= 1e-11 and np.max(np.abs(always[1] - never[1])) <= 1e-11 * np.max(np.abs(v))
