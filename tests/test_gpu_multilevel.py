"""-m gpu parity of the multi-level changeover (reading S23): nb_encounter_levels and nb_step
with levels > 0 against the CPU oracle (oracle.encounter_ml / oracle.step_ml, pinned in tests/test_oracle_multilevel.py).

Tolerance.  The level kicks and Kepler drifts are deterministic fp64 maps that agree with the oracle's to a few ulp per
operation; the innermost level is the Bulirsch-Stoer solver, for which both sides carry a local error <= bs_tol per step
(tests/test_gpu_encounter.py: ENC_TOL = 1e-9 is what the arithmetic guarantees, ~1e-13 is what is observed).  A listing
decision r^2 < rc_{l+1}^2 that falls differently at a 1-ulp edge moves a pair between two levels at a separation where
the deeper level's weight is still 0 to rounding, so it changes nothing beyond that tolerance."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import ENERGY_TOL, GpuState, assert_acc_close, assert_pairs_match, to_dev, torch_mod

pytestmark = pytest.mark.gpu

ENC_TOL = 1e-9


def _clump(n, seed, spacing=2.5e-3, mass=(2e-7, 6e-7), extra=10):
    rng = np.random.default_rng(seed)
    side = int(np.ceil(np.sqrt(n)))
    cell = rng.permutation(side * side)[:n]
    gi, gj = np.divmod(cell, side)
    a = np.concatenate([1.0 + spacing * (gi - side / 2) + rng.uniform(-3e-4, 3e-4, n), rng.uniform(2.0, 3.0, extra)])
    M = np.concatenate([0.4 + spacing * (gj - side / 2) + rng.uniform(-3e-4, 3e-4, n), rng.uniform(0, 6, extra)])
    N = n + extra
    x, v = nb_inputs.elements_to_cartesian(a, rng.uniform(0, 2e-3, N), rng.uniform(0, 1e-3, N), np.zeros(N), np.zeros(N), M, G_GAUSS)
    return np.ascontiguousarray(x), np.ascontiguousarray(v), rng.uniform(*mass, N)


def _gpu_levels(x, v, m, hill, vel, M_star, dt, pairs, levels, kind=0, cap=None):
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    N = m.shape[0]
    p = np.ascontiguousarray(np.asarray(pairs, dtype=np.int32).reshape(-1, 2))
    cap = max(16, p.shape[0]) if cap is None else cap
    nb.configure(N, G=G_GAUSS, changeover_kind=kind, bs_tol=1e-12, pair_capacity=cap, levels=levels)
    nb.nb_status_reset()
    xd, vd, md = to_dev(x), to_dev(v), to_dev(m)
    pd = torch.full((cap, 2), -1, dtype=torch.int32, device="cuda")
    pd[: p.shape[0]] = to_dev(p)
    npd = torch.tensor([p.shape[0]], dtype=torch.int64, device="cuda")
    nb.nb_encounter_levels(xd, vd, md, to_dev(hill), to_dev(vel), M_star, dt, pd, npd)
    torch.cuda.synchronize()
    return xd.cpu().numpy(), vd.cpu().numpy(), nb.nb_status()


@pytest.mark.parametrize("kind", [0, 1])
@pytest.mark.parametrize("levels", [1, 2, 4])
def test_encounter_levels_clump_against_oracle(levels, kind):
    x, v, m = _clump(40, 6)
    N = m.shape[0]
    rc0 = np.full(N, 0.03)
    sure, _ = oracle.pairs(x, rc0)
    rng = np.random.default_rng(1)
    shuffled = sure[rng.permutation(sure.shape[0])]                 # the CUDA list arrives in any order
    shuffled[::3] = shuffled[::3, ::-1]                              # and either orientation
    assert sure.shape[0] > 100
    rcl = oracle.level_rcrit(x, v, m, 1.0, 4.0, G_GAUSS, 0.0, 0.0, levels + 1, rcrit0=rc0)
    for dt in (4.0, -4.0):
        xr, vr, st = oracle.encounter_ml(x, v, m, rcl, 1.0, dt, G_GAUSS, sure, kind=kind, tol=1e-12)
        xg, vg, status = _gpu_levels(x, v, m, np.zeros(N), rc0, 1.0, dt, shuffled, levels, kind=kind)
        assert st["failed"] == 0 and st["skipped"] == 0 and status["bs_fail"] == 0 and status["groups_skipped"] == 0
        assert status["kepler_fail"] == 0 and st["level_pairs"][levels] > 0
        listed = np.zeros(N, dtype=bool); listed[sure.reshape(-1)] = True
        assert np.array_equal(xg[~listed], x[~listed]) and np.array_equal(vg[~listed], v[~listed])
        ex = np.max(np.abs(xg[listed] - xr[listed]) / np.linalg.norm(xr[listed], axis=1, keepdims=True))
        ev = np.max(np.abs(vg[listed] - vr[listed]) / np.linalg.norm(vr[listed], axis=1, keepdims=True))
        print(f"levels={levels} kind={kind} dt={dt}: level pairs {st['level_pairs']}, BS steps {st['steps']}, rel dx {ex:.2e} dv {ev:.2e}")
        assert ex <= ENC_TOL and ev <= ENC_TOL
        assert np.max(np.abs(xr[listed] - x[listed])) > 1e-3
    # bit-reproducible whatever the order of the list
    xg2, vg2, _ = _gpu_levels(x, v, m, np.zeros(N), rc0, 1.0, -4.0, sure, levels, kind=kind)
    assert np.array_equal(xg, xg2) and np.array_equal(vg, vg2)


def test_encounter_levels_eq7_radii_hill_floor_and_big_group():
    """Radii as Eq. 7 gives them (Hill floor + velocity term halving per level) on a ring; a direct-solver cap that is
    exceeded at the innermost level: those bodies take the Kepler drift there and are counted."""
    d = nb_inputs.make_config(2, n_override=2500)
    hill = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, 0.0)
    vel = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 0.0, 0.4)
    L = 3
    rcl = oracle.level_rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, 0.4, L + 1)
    sure, _ = oracle.pairs(d.x, rcl[0])
    assert sure.shape[0] > 2000
    xr, vr, st = oracle.encounter_ml(d.x, d.v, d.m, rcl, d.M_star, d.dt, G_GAUSS, sure, tol=1e-12)
    xg, vg, status = _gpu_levels(d.x, d.v, d.m, hill, vel, d.M_star, d.dt, sure, L)
    assert st["failed"] == 0 and status["bs_fail"] == 0 and status["kepler_fail"] == 0
    assert status["groups_skipped"] == st["skipped"] == 0
    listed = np.zeros(d.N, dtype=bool); listed[sure.reshape(-1)] = True
    ex = np.max(np.abs(xg[listed] - xr[listed]) / np.linalg.norm(xr[listed], axis=1, keepdims=True))
    ev = np.max(np.abs(vg[listed] - vr[listed]) / np.linalg.norm(vr[listed], axis=1, keepdims=True))
    print(f"ring N={d.N} L={L}: level pairs {st['level_pairs']}, groups integrated {st['integrated']}, rel dx {ex:.2e} dv {ev:.2e}")
    assert ex <= ENC_TOL and ev <= ENC_TOL
    assert np.array_equal(xg[~listed], d.x[~listed])


@pytest.mark.parametrize("levels,nsteps", [(3, 1), (3, 5), (2, 20)])
def test_step_with_levels_matches_oracle(levels, nsteps):
    d = nb_inputs.make_config(2, n_override=2000)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, resolve_encounters=True, levels=levels, pair_capacity=1 << 16)
    st.step(d.dt, nsteps)
    xg, vg, ag, rcg = st.host()
    ref = oracle.step_ml(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, nsteps, levels + 1, n1=3.0, n2=0.4)
    status = st.nb.nb_status()
    assert ref["stats"]["failed"] == 0 and ref["stats"]["border"] == 0 and ref["stats"]["kicks"] > 0
    assert status["bs_fail"] == 0 and status["kepler_fail"] == 0 and status["groups_skipped"] == ref["stats"]["skipped"]
    ex = np.max(np.abs(xg - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(vg - ref["v"])) / np.max(np.abs(ref["v"]))
    print(f"step_ml levels={levels} x{nsteps}: level pairs {ref['stats']['level_pairs']}, rel dx {ex:.2e} dv {ev:.2e}")
    tol = 1e-10 if nsteps <= 5 else 1e-8
    assert ex <= tol and ev <= tol
    assert np.max(np.abs(rcg - ref["rcrit"][0]) / ref["rcrit"][0]) <= 1e-12
    acc_ref, ab, _ = oracle.accel(xg, d.m, rcg, G_GAUSS, want_abs=True)
    assert_acc_close(ag, acc_ref, "step_ml final acc", ab)
    sure, border = oracle.pairs(xg, rcg)
    gp, n = st.get_pairs()
    assert_pairs_match(gp, n, sure, border, "step_ml final pairs")


def test_levels_dissolve_the_giant_group_on_the_gpu():
    """The oracle's regime pin on the CUDA path: the N = 8192 ring with the full Eq. 7 radius is one group of ~8100 bodies.
    levels = 0: skipped every step; levels = 3: nothing skipped, energy error orders of magnitude smaller and within 1e-9
    of the oracle run (north_star's energy criterion, S16); graph replay and plain launches agree bit for bit."""
    d = nb_inputs.make_config(2, n_override=8192)
    E0 = oracle.diagnostics(d.x, d.v, d.m, d.M_star, G_GAUSS)["E"]
    out = {}
    for levels, use_graph in ((0, True), (3, True), (3, False)):
        st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, resolve_encounters=True, levels=levels,
                      pair_capacity=1 << 18, use_graph=use_graph)
        st.step(d.dt, 3)
        xg, vg, _, _ = st.host()
        status = st.nb.nb_status()
        out[(levels, use_graph)] = (xg, vg, status, (oracle.diagnostics(xg, vg, d.m, d.M_star, G_GAUSS)["E"] - E0) / E0)
        assert status["bs_fail"] == 0 and status["kepler_fail"] == 0 and status["pairs_dropped"] == 0
    assert out[(0, True)][2]["groups_skipped"] == 3
    assert out[(3, True)][2]["groups_skipped"] == 0
    assert np.array_equal(out[(3, True)][0], out[(3, False)][0]) and np.array_equal(out[(3, True)][1], out[(3, False)][1])
    ref = oracle.step_ml(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3, 4, n1=3.0, n2=0.4)
    de_ref = (oracle.diagnostics(ref["x"], ref["v"], d.m, d.M_star, G_GAUSS)["E"] - E0) / E0
    print("dE/E: levels=0", out[(0, True)][3], "levels=3", out[(3, True)][3], "oracle levels=3", de_ref)
    assert abs(out[(3, True)][3] - de_ref) <= ENERGY_TOL
    assert abs(out[(3, True)][3]) < 0.01 * abs(out[(0, True)][3])
    ex = np.max(np.abs(out[(3, True)][0] - ref["x"])) / np.max(np.abs(ref["x"]))
    assert ex <= 1e-9


def test_levels_need_the_fully_active_case_and_validate():
    import paper_2604_09184_b200 as nb
    d = nb_inputs.make_config(3, n_override=1024)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n_active=d.n_active, resolve_encounters=True, levels=2)
    with pytest.raises(nb.NbError) as e:
        st.step(d.dt, 1)
    assert e.value.code == nb.binding.NB_E_BADARG
    with pytest.raises(nb.NbError):
        nb.configure(100, levels=9)


@pytest.mark.slow
def test_config3_full_eq7_radius_200_steps_with_levels():
    """SURVEY 8(f) NEXT-3 at full size: BASELINE.json:configs[2] (N = 65536 ring, dt = 3 d, 200 steps) with the FULL Eq. 7
    radius, where the plain hybrid scheme finds one group of ~65000 bodies every step.  With 4 intermediate levels the
    direct solver skips nothing; L is conserved to rounding, the energy error is reported (gpurun_out/parity_r2.jsonl)."""
    from test_gpu_acceptance import record
    d = nb_inputs.make_config(2)
    D0 = oracle.diagnostics(d.x, d.v, d.m, d.M_star, G_GAUSS)
    res = {}
    for levels, nsteps in ((0, 20), (4, d.nsteps)):
        st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, resolve_encounters=True, levels=levels, pair_capacity=1 << 23)
        st.step(d.dt, nsteps)
        xg, vg, _, _ = st.host()
        status = st.nb.nb_status()
        D1 = oracle.diagnostics(xg, vg, d.m, d.M_star, G_GAUSS)
        res[levels] = dict(nsteps=nsteps, status=status, dE=(D1["E"] - D0["E"]) / D0["E"],
                           dL=float(np.linalg.norm(D1["L"] - D0["L"]) / np.linalg.norm(D0["L"])), npairs=int(st.npairs.item()))
        assert status["pairs_dropped"] == 0 and status["bs_fail"] == 0 and status["kepler_fail"] == 0
    record(check="config3_eq7_levels", N=d.N, plain=res[0], levels4=res[4])
    assert res[0]["status"]["groups_skipped"] >= 20            # one giant group per step without levels
    assert res[4]["status"]["groups_skipped"] == 0
    assert res[4]["dL"] <= 1e-12
    assert abs(res[4]["dE"]) < 1e-7
