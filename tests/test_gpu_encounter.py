"""-m gpu parity of the direct solver of close encounters (nb_encounter) and of nb_step with
resolve_encounters against the CPU oracle (oracle.encounter / oracle.step_enc).

Tolerance.  Both sides run the same Bulirsch-Stoer algorithm with relative tolerance bs_tol = 1e-12, but
their accelerations differ in the last bits (fused multiply-adds, order of the pair sum), so an accept /
reject decision that sits exactly at the tolerance can fall differently; each side then still carries a
local error <= bs_tol per step.  Two integrations that both approximate the exact flow to ~n_steps * bs_tol
(amplified by the encounter itself) agree to ENC_TOL = 1e-9 relative; observed agreement is printed and is
typically 1e-13.  Bodies outside the integrated groups must come back bit-identical."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import GpuState, assert_acc_close, assert_pairs_match, to_dev, torch_mod

pytestmark = pytest.mark.gpu

ENC_TOL = 1e-9


def _gpu_encounter(x, v, m, rc, M_star, dt, grp, kind=0, tol=1e-12, n_active=0):
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    N = m.shape[0]
    nb.configure(N, G=G_GAUSS, changeover_kind=kind, bs_tol=tol, pair_capacity=16, n_active=n_active)
    nb.nb_status_reset()
    xd, vd, md, rcd = to_dev(x), to_dev(v), to_dev(m), to_dev(rc)
    members = torch.full((N,), -1, dtype=torch.int32, device="cuda")
    gstart = torch.full((N // 2 + 2,), -1, dtype=torch.int32, device="cuda")
    members[: grp["nmembers"]] = to_dev(grp["members"])
    gstart[: grp["ngroups"] + 1] = to_dev(grp["gstart"])
    gstat = torch.tensor([grp["ngroups"], grp["nmembers"], grp["largest"], 0], dtype=torch.int64, device="cuda")
    nb.nb_encounter(xd, vd, md, rcd, M_star, dt, members, gstart, gstat)
    torch.cuda.synchronize()
    return xd.cpu().numpy(), vd.cpu().numpy(), nb.nb_status()


def _compare(x, v, m, rc, M_star, dt, grp, what, kind=0, max_group=1024):
    xg, vg, status = _gpu_encounter(x, v, m, rc, M_star, dt, grp, kind=kind)
    xr, vr, st = oracle.encounter(x, v, m, rc, M_star, dt, G_GAUSS, grp, kind=kind, tol=1e-12, max_group=max_group)
    assert status["bs_fail"] == st["failed"] == 0 and status["groups_skipped"] == st["skipped"]
    moved = np.zeros(m.shape[0], dtype=bool)
    for g in range(grp["ngroups"]):
        seg = grp["members"][grp["gstart"][g]:grp["gstart"][g + 1]]
        if seg.shape[0] <= max_group:
            moved[seg] = True
    assert np.array_equal(xg[~moved], x[~moved]) and np.array_equal(vg[~moved], v[~moved]), f"{what}: a body outside the groups moved"
    if moved.any():
        ex = np.max(np.abs(xg[moved] - xr[moved]) / np.linalg.norm(xr[moved], axis=1, keepdims=True))
        ev = np.max(np.abs(vg[moved] - vr[moved]) / np.linalg.norm(vr[moved], axis=1, keepdims=True))
        print(f"{what}: groups {st['integrated']} (largest {grp['largest']}), BS steps {st['steps']}, max rel dx {ex:.2e} dv {ev:.2e}")
        assert ex <= ENC_TOL and ev <= ENC_TOL, f"{what}: GPU and oracle differ by {ex:.3g} / {ev:.3g}"
        assert np.max(np.abs(xr[moved] - x[moved])) > 0
    return st


@pytest.mark.parametrize("kind", [0, 1])
@pytest.mark.parametrize("cfg,n_override,n1,n2", [(0, 2048, 30.0, 0.0), (1, 3000, 3.0, 0.4), (2, 2500, 10.0, 0.0)])
def test_encounter_groups_of_disk_pair_lists(cfg, n_override, n1, n2, kind):
    d = nb_inputs.make_config(cfg, n_override=n_override)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, n1, n2)
    sure, border = oracle.pairs(d.x, rc)
    grp = oracle.groups(sure, d.N)
    assert grp["ngroups"] > 5
    st = _compare(d.x, d.v, d.m, rc, d.M_star, d.dt, grp, f"{d.name} n1={n1} n2={n2} kind={kind}", kind=kind)
    assert st["integrated"] == grp["ngroups"] - st["skipped"]


def test_encounter_sizes_around_the_warp_and_cta_limits():
    """Groups of exactly 2, 32, 33, 200 and 1024 members (one warp / one CTA per group), a group of 1025
    (skipped and counted), negative dt, deep and shallow encounters mixed."""
    rng = np.random.default_rng(21)
    sizes = [2, 32, 33, 200, 1024, 1025, 3]
    N = sum(sizes) + 50
    a = np.empty(N); M = np.empty(N)
    pairs = []
    pos = 0
    for k, n in enumerate(sizes):
        # jittered lattice in (a, M) with 4e-3 spacing: neighbours sit inside each other's transition shells,
        # nobody comes so close that the step count explodes (the oracle is O(n^2) per right-hand side)
        side = int(np.ceil(np.sqrt(n)))
        gi, gj = np.divmod(np.arange(n), side)
        a[pos:pos + n] = 0.8 + 0.3 * k + 4e-3 * (gi - side / 2) + rng.uniform(-5e-4, 5e-4, n)
        M[pos:pos + n] = 0.5 * k + 4e-3 * (gj - side / 2) + rng.uniform(-5e-4, 5e-4, n)
        pairs += [[pos + i, pos + i + 1] for i in range(n - 1)]
        pos += n
    a[pos:] = rng.uniform(3.0, 4.0, N - pos); M[pos:] = rng.uniform(0, 6, N - pos)
    x, v = nb_inputs.elements_to_cartesian(a, rng.uniform(0, 5e-4, N), rng.uniform(0, 2e-4, N), np.zeros(N), np.zeros(N), M, G_GAUSS)
    x = np.ascontiguousarray(x); v = np.ascontiguousarray(v)
    m = rng.uniform(1e-10, 1e-8, N)
    rc = rng.uniform(2e-3, 2e-2, N)
    grp = oracle.groups(np.array(pairs, dtype=np.int32), N)
    assert sorted(np.diff(grp["gstart"]).tolist()) == sorted(sizes)
    for dt in (3.0, -3.0):
        st = _compare(x, v, m, rc, 1.0, dt, grp, f"group sizes dt={dt}")
        assert st["skipped"] == 1 and st["integrated"] == len(sizes) - 1


@pytest.mark.parametrize("nsteps", [1, 3, 40])
def test_step_with_encounters_matches_oracle(nsteps):
    d = nb_inputs.make_config(1, n_override=900)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, resolve_encounters=True, pair_capacity=1 << 16)
    st.step(d.dt, nsteps)
    xg, vg, ag, rcg = st.host()
    ref = oracle.step_enc(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, nsteps, n1=3.0, n2=0.4)
    assert ref["stats"]["border"] == 0 and ref["stats"]["integrated"] > 0 and ref["stats"]["failed"] == 0
    status = st.nb.nb_status()
    assert status["bs_fail"] == 0 and status["kepler_fail"] == 0 and status["groups_skipped"] == ref["stats"]["skipped"]
    tol = 1e-10 if nsteps <= 3 else 1e-8  # a few Bulirsch-Stoer steps at bs_tol = 1e-12 on each side (module docstring)
    ex = np.max(np.abs(xg - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(vg - ref["v"])) / np.max(np.abs(ref["v"]))
    print(f"step_enc x{nsteps}: groups integrated {ref['stats']['integrated']}, rel dx {ex:.2e} dv {ev:.2e}")
    assert ex <= tol and ev <= tol
    acc_ref, ab, _ = oracle.accel(xg, d.m, rcg, G_GAUSS, want_abs=True)
    assert_acc_close(ag, acc_ref, f"step_enc x{nsteps}: final acc", ab)
    sure, border = oracle.pairs(xg, rcg)
    gp, n = st.get_pairs()
    assert_pairs_match(gp, n, sure, border, f"step_enc x{nsteps}")


def test_step_with_encounters_conserves_energy_through_a_close_approach():
    """The oracle's physics pin (tests/test_oracle_encounter.py) on the CUDA path: same two embryos."""
    G = G_GAUSS
    m = np.array([3e-6, 3e-6])
    x, v = nb_inputs.elements_to_cartesian(np.array([1.0, 1.004]), np.array([0.0, 0.004]), np.array([0.0, 0.001]),
                                           np.array([0.0, 0.2]), np.array([0.0, 0.0]), np.array([0.0, -0.208]), G)
    x = np.ascontiguousarray(x); v = np.ascontiguousarray(v)
    v -= np.sum(m[:, None] * v, axis=0) / (1.0 + m.sum())
    dt, nsteps = 2.0, 60
    E0 = oracle.diagnostics(x, v, m, 1.0, G)["E"]
    out = {}
    for enc in (False, True):
        st = GpuState(x, v, m, 1.0, G=G, n1=3.0, n2=0.4, resolve_encounters=enc, pair_capacity=64)
        st.step(dt, nsteps)
        xg, vg, _, _ = st.host()
        out[enc] = (xg, vg, abs((oracle.diagnostics(xg, vg, m, 1.0, G)["E"] - E0) / E0))
    ref = oracle.step_enc(x, v, m, 1.0, dt, G, nsteps, n1=3.0, n2=0.4)
    print("dE/E: Kepler drift only", out[False][2], "with encounters", out[True][2])
    assert out[True][2] < 0.05 * out[False][2]
    dE_ref = (oracle.diagnostics(ref["x"], ref["v"], m, 1.0, G)["E"] - E0) / E0
    dE_gpu = (oracle.diagnostics(out[True][0], out[True][1], m, 1.0, G)["E"] - E0) / E0
    assert abs(dE_gpu - dE_ref) <= 1e-9       # north_star's energy criterion, with encounters resolved
    assert np.max(np.abs(out[True][0] - ref["x"])) <= 1e-9


def test_resolve_encounters_needs_the_pair_list():
    import paper_2604_09184_b200 as nb
    d = nb_inputs.make_config(0, n_override=300)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, resolve_encounters=True)
    with pytest.raises(nb.NbError) as e:
        nb.nb_step(st.x, st.v, st.m, d.M_star, d.dt, st.rcrit, st.acc, None, None, 1)
    assert e.value.code == nb.binding.NB_E_BADARG


def test_step_with_encounters_is_bitwise_reproducible():
    """Groups (unique labels, ordered member lists), the direct solver (fixed summation order inside a group) and
    the Newton-III force kernel (fixed partial slots) leave nothing to thread timing: two runs agree bit for bit."""
    d = nb_inputs.make_config(2, n_override=3000)
    out = []
    for _ in range(2):
        st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=10.0, n2=0.0, resolve_encounters=True, pair_capacity=1 << 16,
                      force_kernel=2, sym_block=256)
        st.step(d.dt, 5)
        xg, vg, ag, _ = st.host()
        gp, n = st.get_pairs()
        out.append((xg.copy(), vg.copy(), ag.copy(), {tuple(p) for p in gp.tolist()}))
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert np.array_equal(out[0][2], out[1][2]) and out[0][3] == out[1][3]


def test_step_with_encounters_semi_active():
    """Semi-active mode with encounters resolved: test-mass planetesimals that meet an embryo join its group (they
    feel the [1 - W] part of the embryo's pull in the direct solver, and exert nothing)."""
    d = nb_inputs.make_config(3, n_override=3000)
    assert 0 < d.n_active < d.N
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n_active=d.n_active, n1=3.0, n2=0.4, resolve_encounters=True,
                  pair_capacity=1 << 16)
    st.step(d.dt, 10)
    xg, vg, ag, rcg = st.host()
    ref = oracle.step_enc(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 10, n1=3.0, n2=0.4, n_active=d.n_active)
    assert ref["stats"]["integrated"] > 0 and ref["stats"]["border"] == 0
    status = st.nb.nb_status()
    assert status["bs_fail"] == 0 and status["kepler_fail"] == 0 and status["groups_skipped"] == ref["stats"]["skipped"]
    ex = np.max(np.abs(xg - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(vg - ref["v"])) / np.max(np.abs(ref["v"]))
    print(f"semi-active step_enc x10: groups integrated {ref['stats']['integrated']}, rel dx {ex:.2e} dv {ev:.2e}")
    assert ex <= 1e-9 and ev <= 1e-9
    sure, border = oracle.pairs(xg, rcg, n_active=d.n_active)
    gp, n = st.get_pairs()
    assert_pairs_match(gp, n, sure, border, "semi-active step_enc")


def test_encounter_semi_active_split_groups():
    """Semi-active mode (reading S22): star-shaped groups -- a few embryos, each with many test particles, one group far
    beyond NB_MAX_GROUP bodies whose core is two embryos -- are split into the core and independent test particles."""
    rng = np.random.default_rng(31)
    n_act = 6
    sat_per = [1500, 40, 3, 0, 25, 1]                      # embryo 0 and 1 share a group: 1540 + 2 bodies
    N = n_act + sum(sat_per) + 30
    a = np.empty(N); M = np.empty(N)
    a[:n_act] = 1.0 + 0.2 * np.arange(n_act); M[:n_act] = 0.7 * np.arange(n_act)
    a[1] = a[0] + 1.5e-3; M[1] = M[0] + 1.5e-3             # embryos 0 and 1 in encounter (mid-way between lattice cells)
    pairs = [[0, 1]]
    pos = n_act
    for e, ns in enumerate(sat_per):
        # test particles on a jittered lattice around their embryo, never closer than ~1e-3
        side = int(np.ceil(np.sqrt(ns + 1))) | 1
        cells = [(i, j) for i in range(side) for j in range(side) if (i, j) != (side // 2, side // 2)][:ns]
        for (i, j) in cells:
            a[pos] = a[e] + 3e-3 * (i - side // 2) + rng.uniform(-4e-4, 4e-4)
            M[pos] = M[e] + 3e-3 * (j - side // 2) + rng.uniform(-4e-4, 4e-4)
            pairs.append([e, pos]); pos += 1
    a[pos:] = rng.uniform(3.0, 4.0, N - pos); M[pos:] = rng.uniform(0, 6, N - pos)
    x, v = nb_inputs.elements_to_cartesian(a, rng.uniform(0, 1e-4, N), rng.uniform(0, 5e-5, N), np.zeros(N), np.zeros(N), M, G_GAUSS)
    x = np.ascontiguousarray(x); v = np.ascontiguousarray(v)
    m = np.zeros(N); m[:n_act] = rng.uniform(1e-9, 1e-8, n_act)       # Hill radii ~1e-3: no deep fly-by in 3 days
    rc = np.full(N, 0.2)
    grp = oracle.groups(np.array(pairs, dtype=np.int32), N)
    assert grp["largest"] == 1542 and grp["ngroups"] == 4
    xg, vg, status = _gpu_encounter(x, v, m, rc, 1.0, 3.0, grp, n_active=n_act)
    xr, vr, st = oracle.encounter(x, v, m, rc, 1.0, 3.0, G_GAUSS, grp, tol=1e-12, n_active=n_act)
    assert st["skipped"] == 0 and st["failed"] == 0 and status["groups_skipped"] == 0 and status["bs_fail"] == 0
    moved = np.zeros(N, dtype=bool); moved[grp["members"]] = True
    assert np.array_equal(xg[~moved], x[~moved]) and np.array_equal(vg[~moved], v[~moved])
    ex = np.max(np.abs(xg[moved] - xr[moved]) / np.linalg.norm(xr[moved], axis=1, keepdims=True))
    ev = np.max(np.abs(vg[moved] - vr[moved]) / np.linalg.norm(vr[moved], axis=1, keepdims=True))
    print(f"semi-active split: {int(moved.sum())} bodies in {grp['ngroups']} groups, BS steps {st['steps']}, max rel dx {ex:.2e} dv {ev:.2e}")
    assert ex <= ENC_TOL and ev <= ENC_TOL
    assert np.max(np.abs(xr[moved] - x[moved])) > 0


def test_encounter_semi_active_core_beyond_one_warp_against_the_always_split_definition():
    """Reading S22: the definition (oracle default) splits EVERY semi-active group into its active core and independent
    {core + particle} problems.  The CUDA path splits only while core + particle fit one warp (core <= 31) and otherwise
    integrates the group as one problem -- the same motion, to the Bulirsch-Stoer tolerance.  A core of 36 embryos with 60
    test particles: CUDA (unsplit) against the always-split oracle at ENC_TOL; and a core of 31 (split on both sides)."""
    rng = np.random.default_rng(41)
    for n_act, n_sat in ((36, 60), (31, 40)):
        n = n_act + n_sat
        N = n + 20
        side = int(np.ceil(np.sqrt(n)))
        cell = rng.permutation(side * side)[:n]
        gi, gj = np.divmod(cell, side)
        a = np.concatenate([1.0 + 3e-3 * (gi - side / 2) + rng.uniform(-4e-4, 4e-4, n), rng.uniform(2.0, 3.0, N - n)])
        M = np.concatenate([0.4 + 3e-3 * (gj - side / 2) + rng.uniform(-4e-4, 4e-4, n), rng.uniform(0, 6, N - n)])
        x, v = nb_inputs.elements_to_cartesian(a, rng.uniform(0, 2e-4, N), rng.uniform(0, 1e-4, N), np.zeros(N), np.zeros(N), M, G_GAUSS)
        x = np.ascontiguousarray(x); v = np.ascontiguousarray(v)
        # semi-active ordering: the embryos first
        m = np.zeros(N); m[:n_act] = rng.uniform(1e-9, 1e-8, n_act)
        rc = np.full(N, 0.02)
        pairs = [[i, i + 1] for i in range(n_act - 1)] + [[int(rng.integers(0, n_act)), k] for k in range(n_act, n)]
        grp = oracle.groups(np.array(pairs, dtype=np.int32), N)
        assert grp["ngroups"] == 1 and grp["largest"] == n
        xg, vg, status = _gpu_encounter(x, v, m, rc, 1.0, 3.0, grp, n_active=n_act)
        xr, vr, st = oracle.encounter(x, v, m, rc, 1.0, 3.0, G_GAUSS, grp, tol=1e-12, n_active=n_act)   # always split
        assert st["failed"] == 0 and st["skipped"] == 0 and status["bs_fail"] == 0 and status["groups_skipped"] == 0
        mem = grp["members"]
        ex = np.max(np.abs(xg[mem] - xr[mem]) / np.linalg.norm(xr[mem], axis=1, keepdims=True))
        ev = np.max(np.abs(vg[mem] - vr[mem]) / np.linalg.norm(vr[mem], axis=1, keepdims=True))
        print(f"semi-active core of {n_act}: CUDA vs always-split oracle: max rel dx {ex:.2e} dv {ev:.2e}")
        assert ex <= ENC_TOL and ev <= ENC_TOL
        assert np.array_equal(xg[n:], x[n:]) and np.max(np.abs(xr[mem] - x[mem])) > 0
