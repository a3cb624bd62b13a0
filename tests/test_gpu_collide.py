"""-m gpu parity of nb_encounter_collide (collisions examined inside the direct solver: PAPER.md:98, 130, 168; DESIGN.md
reading S26) against oracle.encounter(radius=...), whose own pins are in tests/test_oracle_collide.py.

What is unique is compared exactly: who absorbed whom, the merged masses (the same unfused sums in index order on both
sides), zero mass / radius of the absorbed bodies, absorbed bodies sitting ON their survivors; merged radii to 2 ulp
(two cbrt routines); positions and velocities to the direct solver's ENC_TOL (tests/test_gpu_encounter.py)."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import to_dev, torch_mod

pytestmark = pytest.mark.gpu

ENC_TOL = 1e-9


def _grp_all(n):
    return dict(ngroups=1, members=np.arange(n, dtype=np.int32), gstart=np.array([0, n], dtype=np.int32),
                label=np.zeros(n, dtype=np.int32), nmembers=n, largest=n)


def _gpu_collide(x, v, m, rad, rc, M_star, dt, grp, f=1.0, absorbed_by=None):
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    N = m.shape[0]
    nb.configure(N, G=G_GAUSS, bs_tol=1e-12, pair_capacity=16, radius_factor=f)
    nb.nb_status_reset()
    xd, vd, md, Rd, rcd = to_dev(x), to_dev(v), to_dev(m), to_dev(rad), to_dev(rc)
    members = torch.full((N,), -1, dtype=torch.int32, device="cuda")
    gstart = torch.full((N // 2 + 2,), -1, dtype=torch.int32, device="cuda")
    nmem = int(grp["gstart"][grp["ngroups"]])
    members[:nmem] = to_dev(grp["members"][:nmem])
    gstart[: grp["ngroups"] + 1] = to_dev(grp["gstart"][: grp["ngroups"] + 1])
    gstat = torch.tensor([grp["ngroups"], nmem, 0, 0], dtype=torch.int64, device="cuda")
    ab = to_dev(np.full(N, -1, dtype=np.int32) if absorbed_by is None else absorbed_by)
    nb.nb_encounter_collide(xd, vd, md, Rd, rcd, M_star, dt, members, gstart, gstat, ab)
    torch.cuda.synchronize()
    return dict(x=xd.cpu().numpy(), v=vd.cpu().numpy(), m=md.cpu().numpy(), radius=Rd.cpu().numpy(),
                absorbed_by=ab.cpu().numpy(), status=nb.nb_status())


def _compare(x, v, m, rad, rc, M_star, dt, grp, what, f=1.0, absorbed_by=None, expect_absorbed=None):
    g = _gpu_collide(x, v, m, rad, rc, M_star, dt, grp, f=f, absorbed_by=absorbed_by)
    xr, vr, st = oracle.encounter(x, v, m, rc, M_star, dt, G_GAUSS, grp, radius=rad, radius_factor=f, absorbed_by=absorbed_by)
    assert g["status"]["bs_fail"] == st["failed"] == 0
    assert np.array_equal(g["absorbed_by"], st["absorbed_by"]), f"{what}: who absorbed whom differs"
    assert g["status"]["absorbed"] == st["absorbed"]
    if expect_absorbed is not None:
        assert st["absorbed"] == expect_absorbed, f"{what}: the case does not do what it was built for"
    assert np.array_equal(g["m"], st["m"]), f"{what}: merged masses differ"
    # two cbrt routines (glibc, CUDA), each within 1 ulp of the exact value: up to 2 ulp apart
    assert np.max(np.abs(g["radius"] - st["radius"])) <= 5e-16 * max(st["radius"].max(), 1e-300)
    assert np.array_equal(g["radius"] == 0.0, st["radius"] == 0.0)
    gone = np.flatnonzero(g["absorbed_by"] >= 0)
    assert np.array_equal(g["x"][gone], g["x"][g["absorbed_by"][gone]]) and np.array_equal(g["v"][gone], g["v"][g["absorbed_by"][gone]])
    ex = np.max(np.abs(g["x"] - xr)) / np.max(np.linalg.norm(xr, axis=1))
    ev = np.max(np.abs(g["v"] - vr)) / np.max(np.linalg.norm(vr, axis=1))
    print(f"{what}: absorbed {st['absorbed']}, BS steps {st['steps']}, max rel dx {ex:.2e} dv {ev:.2e}")
    assert ex <= ENC_TOL and ev <= ENC_TOL, f"{what}: GPU and oracle differ by {ex:.3g} / {ev:.3g}"
    return g, st


def test_free_fall_to_contact():
    m1, m2, d0, R = 3.0e-6, 1.0e-6, 1.0e-3, 5.0e-5
    x = np.array([[1.0, 0.0, 0.0], [1.0 + d0, 0.0, 0.0]]); v = np.tile(np.array([0.0, 1e-3, 0.0]), (2, 1))
    m = np.array([m1, m2]); rc = np.full(2, 1.0); rad = np.array([R, 2.0 * R])
    q = 1.5 * 3.0 * R / d0
    tc = np.sqrt(d0 ** 3 / (2.0 * G_GAUSS * (m1 + m2))) * (np.arccos(np.sqrt(q)) + np.sqrt(q * (1.0 - q)))
    _compare(x, v, m, rad, rc, 1e-30, 0.98 * tc, _grp_all(2), "free fall, before contact", f=1.5, expect_absorbed=0)
    g, _ = _compare(x, v, m, rad, rc, 1e-30, 1.02 * tc, _grp_all(2), "free fall, after contact", f=1.5, expect_absorbed=1)
    assert g["m"][0] == m1 + m2 and g["m"][1] == 0.0
    _compare(x, v, m, rad, rc, 1e-30, 1.02 * tc, _grp_all(2), "free fall, f = 1", f=1.0, expect_absorbed=0)


@pytest.mark.parametrize("seed,expect", [(3, 2), (4, 2), (7, 5), (6, 0)])
def test_clusters_of_two_three_and_all(seed, expect):
    rng = np.random.default_rng(seed)
    n = 6
    x = np.array([1.0, 0.0, 0.0]) + 2e-4 * rng.standard_normal((n, 3))
    v = np.array([0.0, np.sqrt(G_GAUSS), 0.0]) + 1e-4 * np.sqrt(G_GAUSS) * rng.standard_normal((n, 3))
    m = rng.uniform(1e-7, 3e-7, n); rc = np.full(n, 3e-3); rad = rng.uniform(0.9e-4, 1.6e-4, n)
    _compare(x, v, m, rad, rc, 1.0, 0.05, _grp_all(n), f"6 bodies, seed {seed}", expect_absorbed=expect)


def test_chain_then_a_second_call_with_the_absorbed_bodies_still_in_the_arrays():
    R = 1.0e-4
    x = np.array([[1.0, 0.0, 0.0], [1.0 + 1.8 * R, 0.0, 0.0], [1.0 + 3.6 * R, 0.0, 0.0], [1.0, 2.0e-3, 0.0]])
    v = np.tile(np.array([0.0, np.sqrt(G_GAUSS), 0.0]), (4, 1))
    m = np.array([1e-7, 2e-7, 3e-7, 1e-7]); rc = np.full(4, 5e-3); rad = np.full(4, R)
    g, st = _compare(x, v, m, rad, rc, 1.0, 1e-3, _grp_all(4), "chain", expect_absorbed=2)
    assert list(g["absorbed_by"]) == [-1, 0, 0, -1]
    g2, _ = _compare(g["x"], g["v"], g["m"], g["radius"], rc, 1.0, 0.5, _grp_all(4), "chain, next call",
                     absorbed_by=g["absorbed_by"], expect_absorbed=0)
    assert list(g2["absorbed_by"]) == [-1, 0, 0, -1] and np.array_equal(g2["m"], g["m"])


@pytest.mark.parametrize("n,scale,rmax", [(40, 4e-4, 1.2e-4), (200, 1.2e-3, 0.8e-4)])
def test_groups_beyond_one_warp(n, scale, rmax):
    """One group of 40 (the 128-thread kernel) and of 200 bodies (the 1024-thread kernel) with several contacts during dt."""
    rng = np.random.default_rng(100 + n)
    x = np.array([1.0, 0.0, 0.0]) + scale * rng.standard_normal((n, 3))
    v = np.array([0.0, np.sqrt(G_GAUSS), 0.0]) + 2e-4 * np.sqrt(G_GAUSS) * rng.standard_normal((n, 3))
    m = rng.uniform(1e-8, 3e-8, n); rc = np.full(n, 20 * scale); rad = rng.uniform(0.3 * rmax, rmax, n)
    g, st = _compare(x, v, m, rad, rc, 1.0, 0.5, _grp_all(n), f"group of {n}")
    assert 2 <= st["absorbed"] < n // 2


def test_disk_groups_with_inflated_radii():
    """The encounter groups of a ring's pair list (Eq. 7 radius), radii inflated by f = 400 so that some groups collide;
    bodies outside the groups come back bit-identical."""
    d = nb_inputs.make_config(2, n_override=2500)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, 0.4)
    sure, _ = oracle.pairs(d.x, rc)
    grp = oracle.groups(sure, d.N)
    assert grp["ngroups"] > 50
    g, st = _compare(d.x, d.v, d.m, d.radius, rc, d.M_star, d.dt, grp, "ring N=2500, f=400", f=400.0)
    assert st["absorbed"] >= 3
    inside = np.zeros(d.N, dtype=bool); inside[grp["members"][: grp["gstart"][grp["ngroups"]]]] = True
    assert np.array_equal(g["x"][~inside], d.x[~inside]) and np.array_equal(g["m"][~inside], d.m[~inside])
    # a second call with the absorbed bodies still in the arrays: they stay out of the encounter and follow their holders
    g2, st2 = _compare(g["x"], g["v"], g["m"], g["radius"], rc, d.M_star, d.dt, grp, "ring N=2500, f=400, second call", f=400.0,
                       absorbed_by=g["absorbed_by"])
    assert np.all(g2["absorbed_by"][g["absorbed_by"] >= 0] >= 0)
    g0, st0 = _compare(d.x, d.v, d.m, d.radius, rc, d.M_star, d.dt, grp, "ring N=2500, f=1", f=1.0, expect_absorbed=0)
    # nobody touches: the collision-free solver's result, bit for bit
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    xd, vd = to_dev(d.x), to_dev(d.v)
    members = torch.full((d.N,), -1, dtype=torch.int32, device="cuda"); gstart = torch.full((d.N // 2 + 2,), -1, dtype=torch.int32, device="cuda")
    nmem = int(grp["gstart"][grp["ngroups"]])
    members[:nmem] = to_dev(grp["members"][:nmem]); gstart[: grp["ngroups"] + 1] = to_dev(grp["gstart"][: grp["ngroups"] + 1])
    gstat = torch.tensor([grp["ngroups"], nmem, 0, 0], dtype=torch.int64, device="cuda")
    nb.nb_encounter(xd, vd, to_dev(d.m), to_dev(rc), d.M_star, d.dt, members, gstart, gstat)
    torch.cuda.synchronize()
    assert np.array_equal(xd.cpu().numpy(), g0["x"]) and np.array_equal(vd.cpu().numpy(), g0["v"])


def test_absorbed_bodies_follow_their_holder():
    """2 goes into 1 after the first accepted step, 0 absorbs 1 later in the same call: 2 moves on to 0 with its holder."""
    R, mass = 1e-4, 1e-5
    x = np.array([[1.0 - 20 * R, 0, 0], [1.0, 0, 0], [1.0 + 1.5 * R, 0, 0]])
    v = np.tile(np.array([0.0, np.sqrt(G_GAUSS), 0.0]), (3, 1)); v[0, 0] += 60 * R
    m = np.array([mass, mass, 0.5 * mass]); rc = np.full(3, 1e-2); rad = np.full(3, R)
    g, st = _compare(x, v, m, rad, rc, 1.0, 0.5, _grp_all(3), "sequential absorption", expect_absorbed=2)
    assert list(g["absorbed_by"]) == [-1, 0, 0]


@pytest.mark.parametrize("use_graph", [True, False])
def test_step_with_collisions_inside_the_solver(use_graph):
    """nb_step(resolve_encounters, collide_radius) against oracle.step_enc(radius=...): 4 steps of a ring with radii
    inflated by f = 400; the masses change from step to step, absorbed bodies stay in the arrays on their holders."""
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    d = nb_inputs.make_config(2, n_override=1500)
    nsteps, f = 4, 400.0
    ref = oracle.step_enc(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, nsteps, n1=3.0, n2=0.4, radius=d.radius, radius_factor=f)
    assert ref["stats"]["absorbed"] >= 3 and ref["stats"]["failed"] == 0 and ref["stats"]["border"] == 0
    x, v, m, R = to_dev(d.x), to_dev(d.v), to_dev(d.m), to_dev(d.radius)
    ab = torch.full((d.N,), -1, dtype=torch.int32, device="cuda")
    acc = torch.zeros_like(x); rcd = torch.zeros(d.N, dtype=torch.float64, device="cuda")
    cap = 1 << 16
    pairs = torch.zeros((cap, 2), dtype=torch.int32, device="cuda"); npairs = torch.zeros(1, dtype=torch.int64, device="cuda")
    nb.configure(d.N, G=G_GAUSS, n1=3.0, n2=0.4, pair_capacity=cap, resolve_encounters=True, radius_factor=f,
                 collide_radius=R, collide_absorbed_by=ab, use_graph=use_graph)
    nb.nb_status_reset()
    nb.nb_step(x, v, m, d.M_star, d.dt, rcd, acc, pairs, npairs, nsteps)
    torch.cuda.synchronize()
    st = nb.nb_status()
    assert st["bs_fail"] == 0 and st["groups_skipped"] == 0 and st["absorbed"] == ref["stats"]["absorbed"]
    assert np.array_equal(ab.cpu().numpy(), ref["absorbed_by"])
    assert np.array_equal(m.cpu().numpy(), ref["m"])
    assert np.max(np.abs(R.cpu().numpy() - ref["radius"])) <= 5e-16 * ref["radius"].max()
    ex = np.max(np.abs(x.cpu().numpy() - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(v.cpu().numpy() - ref["v"])) / np.max(np.abs(ref["v"]))
    print(f"step with collisions (graph {use_graph}): absorbed {st['absorbed']}, rel dx {ex:.2e} dv {ev:.2e}")
    assert ex <= ENC_TOL and ev <= ENC_TOL
    n = int(npairs.item())
    got = {tuple(p) for p in pairs[:n].cpu().numpy().tolist()}
    assert got == {tuple(p) for p in ref["pairs"].tolist()}
    # then the step-boundary merge removes the absorbed bodies: N shrinks by exactly their number
    surv = torch.zeros(d.N, dtype=torch.int32, device="cuda"); mstat = torch.zeros(4, dtype=torch.int64, device="cuda")
    nb.configure(d.N, G=G_GAUSS, pair_capacity=cap, radius_factor=1.0)
    nb.nb_merge(x, v, m, R, pairs, npairs, surv, mstat)
    torch.cuda.synchronize()
    assert int(mstat[0].item()) == d.N - st["absorbed"]
    assert float(m[: int(mstat[0].item())].min().item()) > 0.0


def test_error_codes_of_the_collision_calls():
    """Host-detectable misuse: semi-active mode, a missing absorbed_by array."""
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    d = nb_inputs.make_config(2, n_override=600)
    x, v, m, R = to_dev(d.x), to_dev(d.v), to_dev(d.m), to_dev(d.radius)
    rc = torch.zeros(d.N, dtype=torch.float64, device="cuda"); acc = torch.zeros_like(x)
    ab = torch.full((d.N,), -1, dtype=torch.int32, device="cuda")
    members = torch.zeros(d.N, dtype=torch.int32, device="cuda"); gstart = torch.zeros(d.N // 2 + 2, dtype=torch.int32, device="cuda")
    gstat = torch.zeros(4, dtype=torch.int64, device="cuda")
    pairs = torch.zeros((1024, 2), dtype=torch.int32, device="cuda"); npairs = torch.zeros(1, dtype=torch.int64, device="cuda")
    nb.configure(d.N, G=G_GAUSS, pair_capacity=1024, n_active=100)
    with pytest.raises(nb.NbError) as e:
        nb.nb_encounter_collide(x, v, m, R, rc, d.M_star, d.dt, members, gstart, gstat, ab)
    assert e.value.code == nb.binding.NB_E_BADARG
    nb.configure(d.N, G=G_GAUSS, pair_capacity=1024, resolve_encounters=True, collide_radius=R)
    with pytest.raises(nb.NbError) as e:
        nb.nb_step(x, v, m, d.M_star, d.dt, rc, acc, pairs, npairs, 1)
    assert e.value.code == nb.binding.NB_E_NULL
    nb.configure(d.N, G=G_GAUSS, pair_capacity=1024, resolve_encounters=True, n_active=100, collide_radius=R, collide_absorbed_by=ab)
    with pytest.raises(nb.NbError) as e:
        nb.nb_step(x, v, m, d.M_star, d.dt, rc, acc, pairs, npairs, 1)
    assert e.value.code == nb.binding.NB_E_BADARG
    torch.cuda.synchronize()
    assert np.array_equal(x.cpu().numpy(), d.x) and np.array_equal(m.cpu().numpy(), d.m)      # nothing ran
    # zero groups: a no-op that returns
    nb.configure(d.N, G=G_GAUSS, pair_capacity=1024)
    nb.nb_encounter_collide(x, v, m, R, rc, d.M_star, d.dt, members, gstart, gstat, ab)
    torch.cuda.synchronize()
    assert np.array_equal(x.cpu().numpy(), d.x) and int(ab.max().item()) == -1


def test_multilevel_step_with_collisions_inside_the_innermost_solver():
    """nb_step(levels = 2, collide_radius) against oracle.step_ml(nlev = 3, radius=...): the masses change inside the
    recursion and the level kicks that follow use them."""
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    d = nb_inputs.make_config(2, n_override=1200)
    nsteps, f, L = 2, 400.0, 2
    ref = oracle.step_ml(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, nsteps, L + 1, n1=3.0, n2=0.4, radius=d.radius, radius_factor=f)
    assert ref["stats"]["absorbed"] >= 3 and ref["stats"]["failed"] == 0 and ref["stats"]["border"] == 0
    x, v, m, R = to_dev(d.x), to_dev(d.v), to_dev(d.m), to_dev(d.radius)
    ab = torch.full((d.N,), -1, dtype=torch.int32, device="cuda")
    acc = torch.zeros_like(x); rcd = torch.zeros(d.N, dtype=torch.float64, device="cuda")
    cap = 1 << 16
    pairs = torch.zeros((cap, 2), dtype=torch.int32, device="cuda"); npairs = torch.zeros(1, dtype=torch.int64, device="cuda")
    nb.configure(d.N, G=G_GAUSS, n1=3.0, n2=0.4, pair_capacity=cap, resolve_encounters=True, levels=L, radius_factor=f,
                 collide_radius=R, collide_absorbed_by=ab)
    nb.nb_status_reset()
    nb.nb_step(x, v, m, d.M_star, d.dt, rcd, acc, pairs, npairs, nsteps)
    torch.cuda.synchronize()
    st = nb.nb_status()
    assert st["bs_fail"] == 0 and st["groups_skipped"] == 0 and st["absorbed"] == ref["stats"]["absorbed"]
    assert np.array_equal(ab.cpu().numpy(), ref["absorbed_by"]) and np.array_equal(m.cpu().numpy(), ref["m"])
    ex = np.max(np.abs(x.cpu().numpy() - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(v.cpu().numpy() - ref["v"])) / np.max(np.abs(ref["v"]))
    print(f"levels = {L} with collisions: absorbed {st['absorbed']}, rel dx {ex:.2e} dv {ev:.2e}")
    assert ex <= ENC_TOL and ev <= ENC_TOL
