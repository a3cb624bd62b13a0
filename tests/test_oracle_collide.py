"""Pins of the oracle's collisions INSIDE the direct solver ("propagates the involved bodies through the
close encounter phase", PAPER.md:130 perfect mergers, PAPER.md:168 radius factor f; reading S26) -- none of
them restates its loops: closed-form free fall to contact, the conserved barycentre, identity with the pinned
step-boundary merge (oracle.merge, reading S21) when the contact is found at the end of a single accepted step, exact
identity with the collision-free solver when nobody touches, chains of contacts, and what an absorbed body looks like."""
import numpy as np
import pytest

import oracle

G = 0.01720209895 ** 2


def _one_group(n):
    return dict(ngroups=1, members=np.arange(n, dtype=np.int32), gstart=np.array([0, n], dtype=np.int32),
                label=np.zeros(n, dtype=np.int32))


def _free_fall_time(d0, s, mu):
    """two bodies at rest, separation d0 -> s under mu = G (m1 + m2): the radial Kepler problem (e = 1, a = d0 / 2)"""
    q = s / d0
    return np.sqrt(d0 ** 3 / (2.0 * mu)) * (np.arccos(np.sqrt(q)) + np.sqrt(q * (1.0 - q)))


def test_free_fall_to_contact_closed_form():
    # a pair at rest around a star of negligible mass, deep inside 0.1 rc: the solver carries the full Newtonian pair force
    m1, m2, d0, R = 3.0e-6, 1.0e-6, 1.0e-3, 5.0e-5
    x = np.array([[1.0, 0.0, 0.0], [1.0 + d0, 0.0, 0.0]])
    v = np.zeros((2, 3))
    m = np.array([m1, m2]); rc = np.full(2, 1.0e3 * d0)
    rad = np.array([R, 2.0 * R])
    f = 1.5
    tc = _free_fall_time(d0, f * 3.0 * R, G * (m1 + m2))
    xb = (m1 * x[0] + m2 * x[1]) / (m1 + m2)
    # shortly before contact: nothing happens, and the result is the collision-free solver's, bit for bit
    xa, va, st = oracle.encounter(x, v, m, rc, 1e-30, 0.98 * tc, G, _one_group(2), radius=rad, radius_factor=f)
    x0, v0, st0 = oracle.encounter(x, v, m, rc, 1e-30, 0.98 * tc, G, _one_group(2))
    assert st["absorbed"] == 0 and np.array_equal(xa, x0) and np.array_equal(va, v0)
    assert np.array_equal(st["m"], m) and np.array_equal(st["radius"], rad) and np.all(st["absorbed_by"] == -1)
    sep = np.linalg.norm(xa[1] - xa[0])
    assert f * 3.0 * R < sep < 1.3 * f * 3.0 * R                 # the closed form really puts contact right behind
    # shortly after: one body of mass m1 + m2 at rest at the barycentre (which never moved), volume conserved
    xa, va, st = oracle.encounter(x, v, m, rc, 1e-30, 1.02 * tc, G, _one_group(2), radius=rad, radius_factor=f)
    assert st["absorbed"] == 1 and list(st["absorbed_by"]) == [-1, 0]
    assert st["m"][0] == m1 + m2 and st["m"][1] == 0.0 and st["radius"][1] == 0.0
    assert abs(st["radius"][0] - np.cbrt(9.0) * R) <= 1e-15 * R
    assert np.max(np.abs(xa[0] - xb)) <= 1e-10 * d0 and np.max(np.abs(va[0])) <= 1e-9 * np.sqrt(G * (m1 + m2) / d0)
    # the absorbed body sits on its survivor
    assert np.array_equal(xa[1], xa[0]) and np.array_equal(va[1], va[0])
    # with the inflation factor back at 1 the same interval ends before contact
    _, _, st = oracle.encounter(x, v, m, rc, 1e-30, 1.02 * tc, G, _one_group(2), radius=rad, radius_factor=1.0)
    assert st["absorbed"] == 0


@pytest.mark.parametrize("seed,expect", [(3, [-1, -1, -1, -1, 1, 1]), (4, [-1, -1, -1, 0, 2, -1]), (7, [-1, 0, 0, 0, 0, 0])])
def test_single_step_contact_equals_the_step_boundary_merge(seed, expect):
    """A short interval that Bulirsch-Stoer accepts in ONE step: the contact is then examined exactly once, at the state
    the collision-free solver ends in -- the result must be oracle.merge (reading S21, pinned by its own closed forms)
    applied to that state, bit for bit, with the removed bodies put on their survivors.  Seeds: one cluster of three,
    two clusters of two, everybody in one cluster."""
    rng = np.random.default_rng(seed)
    n = 6
    x = np.array([1.0, 0.0, 0.0]) + 2e-4 * rng.standard_normal((n, 3))
    v = np.array([0.0, np.sqrt(G), 0.0]) + 1e-4 * np.sqrt(G) * rng.standard_normal((n, 3))
    m = rng.uniform(1e-7, 3e-7, n)
    rc = np.full(n, 3e-3)
    rad = rng.uniform(0.9e-4, 1.6e-4, n)
    dt = 0.05
    x0, v0, st0 = oracle.encounter(x, v, m, rc, 1.0, dt, G, _one_group(n))
    assert st0["steps"] == 1
    allp = np.array([(i, j) for i in range(n) for j in range(i + 1, n)], dtype=np.int32)
    ref = oracle.merge(x0, v0, m, rad, allp, f=1.0)
    xa, va, st = oracle.encounter(x, v, m, rc, 1.0, dt, G, _one_group(n), radius=rad)
    assert st["steps"] == 1 and st["absorbed"] == ref["n_merged"] and list(st["absorbed_by"]) == expect
    keep = np.flatnonzero(ref["alive"])
    assert np.array_equal(xa[keep], ref["x"]) and np.array_equal(va[keep], ref["v"])
    assert np.array_equal(st["m"][keep], ref["m"])
    assert np.max(np.abs(st["radius"][keep] - ref["radius"])) <= 2.3e-16 * ref["radius"].max()   # two cbrt routines: 1 ulp
    gone = np.flatnonzero(~ref["alive"])
    assert np.array_equal(st["absorbed_by"][gone], ref["survivor_of"][gone]) and np.all(st["absorbed_by"][keep] == -1)
    assert np.all(st["m"][gone] == 0.0) and np.all(st["radius"][gone] == 0.0)
    assert np.array_equal(xa[gone], xa[ref["survivor_of"][gone]]) and np.array_equal(va[gone], va[ref["survivor_of"][gone]])
    # conservation through the merge: mass, momentum of the democratic velocities, volume
    assert abs(st["m"].sum() - m.sum()) <= 4e-16 * m.sum()
    p0 = (m[:, None] * v0).sum(axis=0); p1 = (st["m"][:, None] * va).sum(axis=0)
    assert np.max(np.abs(p1 - p0)) <= 1e-15 * np.linalg.norm(p0)
    assert abs((st["radius"] ** 3).sum() - (rad ** 3).sum()) <= 1e-15 * (rad ** 3).sum()


def test_chain_of_contacts_and_later_steps():
    """0-1 and 1-2 touch, 0-2 do not: all three end in body 0; a fourth body far away is untouched.  In the next call the
    absorbed bodies (m = 0, R = 0) are massless members that nobody tests again: nothing is absorbed twice and the
    survivor's mass stays."""
    R = 1.0e-4
    x = np.array([[1.0, 0.0, 0.0], [1.0 + 1.8 * R, 0.0, 0.0], [1.0 + 3.6 * R, 0.0, 0.0], [1.0, 2.0e-3, 0.0]])
    v = np.tile(np.array([0.0, np.sqrt(G), 0.0]), (4, 1))
    m = np.array([1e-7, 2e-7, 3e-7, 1e-7])
    rc = np.full(4, 5e-3)
    rad = np.full(4, R)
    xa, va, st = oracle.encounter(x, v, m, rc, 1.0, 1e-3, G, _one_group(4), radius=rad)
    assert list(st["absorbed_by"]) == [-1, 0, 0, -1] and st["absorbed"] == 2
    assert abs(st["m"][0] - 6e-7) <= 1e-22 and st["m"][3] == 1e-7
    assert abs(st["radius"][0] - np.cbrt(3.0) * R) <= 1e-15 * R
    xb, vb, st2 = oracle.encounter(xa, va, st["m"], rc, 1.0, 0.5, G, _one_group(4), radius=st["radius"],
                                   absorbed_by=st["absorbed_by"])
    assert st2["absorbed"] == 0 and np.array_equal(st2["m"], st["m"]) and list(st2["absorbed_by"]) == [-1, 0, 0, -1]
    assert np.array_equal(xb[1], xb[0]) and np.array_equal(xb[2], xb[0])


def test_step_enc_with_radii():
    """Whole steps: radii too small to touch => step_enc bit for bit; radii inflated by f => bodies are absorbed, the total
    mass stays, every absorbed body is massless and sits on a body that gained mass."""
    import nb_inputs
    d = nb_inputs.make_config(2, n_override=1500)
    rad = d.radius
    a = oracle.step_enc(d.x, d.v, d.m, d.M_star, d.dt, G, 3, n1=3.0, n2=0.4)
    b = oracle.step_enc(d.x, d.v, d.m, d.M_star, d.dt, G, 3, n1=3.0, n2=0.4, radius=rad, radius_factor=1.0)
    assert b["stats"]["absorbed"] == 0
    assert np.array_equal(a["x"], b["x"]) and np.array_equal(a["v"], b["v"]) and np.array_equal(b["m"], d.m)
    c = oracle.step_enc(d.x, d.v, d.m, d.M_star, d.dt, G, 3, n1=3.0, n2=0.4, radius=rad, radius_factor=400.0)
    nab = c["stats"]["absorbed"]
    assert nab > 0 and np.count_nonzero(c["absorbed_by"] >= 0) == nab
    assert abs(c["m"].sum() - d.m.sum()) <= 1e-15 * d.m.sum()
    gone = np.flatnonzero(c["absorbed_by"] >= 0)
    assert np.all(c["m"][gone] == 0.0) and np.all(c["radius"][gone] == 0.0)
    assert np.all(c["m"][c["absorbed_by"][gone]] > d.m[c["absorbed_by"][gone]])
    assert np.array_equal(c["x"][gone], c["x"][c["absorbed_by"][gone]])
    E0 = oracle.diagnostics(d.x, d.v, d.m, d.M_star, G); E1 = oracle.diagnostics(c["x"], c["v"], c["m"], d.M_star, G)
    # a perfect merger keeps mass and momentum; the pair's angular momentum about its own barycentre (reduced mass x
    # separation x relative speed: the merged body's spin) leaves the orbital budget -- tiny, and not zero
    assert 0.0 < np.linalg.norm(E1["L"] - E0["L"]) <= 1e-7 * np.linalg.norm(E0["L"])


def test_absorbed_bodies_follow_their_holder_when_it_is_absorbed_later():
    """1 and 2 touch at the start (2 goes into 1 after the first accepted step); 0 arrives later and absorbs 1.  An absorbed
    body takes no part in the encounter any more (it feels only the star) -- left to feel the pair terms it would be a
    massless particle at zero distance from a massive one with another critical radius: a singular encounter -- and
    ends on the body that holds it at the end, here body 0.  Pinned by the two-body problem {0, 1 + 2 merged}: same
    final state of body 0 and about as many steps."""
    R, mass = 1e-4, 1e-5
    x = np.array([[1.0 - 20 * R, 0, 0], [1.0, 0, 0], [1.0 + 1.5 * R, 0, 0]])
    v = np.tile(np.array([0.0, np.sqrt(G), 0.0]), (3, 1)); v[0, 0] += 60 * R
    m = np.array([mass, mass, 0.5 * mass]); rc = np.full(3, 1e-2); rad = np.full(3, R)
    xa, va, st = oracle.encounter(x, v, m, rc, 1.0, 0.5, G, _one_group(3), radius=rad)
    assert list(st["absorbed_by"]) == [-1, 0, 0] and st["m"][0] == mass + (mass + 0.5 * mass)
    assert np.array_equal(xa[1], xa[0]) and np.array_equal(xa[2], xa[0]) and np.array_equal(va[2], va[0])
    m12 = m[1] + m[2]
    x2 = np.array([x[0], (m[1] * x[1] + m[2] * x[2]) / m12]); v2 = np.array([v[0], (m[1] * v[1] + m[2] * v[2]) / m12])
    xb, vb, st2 = oracle.encounter(x2, v2, np.array([mass, m12]), rc[:2], 1.0, 0.5, G, _one_group(2), radius=np.array([R, np.cbrt(2.0) * R]))
    assert st2["absorbed"] == 1
    assert np.max(np.abs(xb[0] - xa[0])) <= 1e-12 and np.max(np.abs(vb[0] - va[0])) <= 1e-11 * np.sqrt(G)
    assert st["steps"] <= st2["steps"] + 10


def test_bodies_absorbed_in_an_earlier_call_stay_out_of_the_encounter():
    """The ring group that showed the problem: two members touch in the first half of the interval; in a second call over
    the other half the absorbed ones are still in the arrays (m = 0, R = 0, on their holders).  They must not be
    integrated against their holders: the second call converges in a step or two, does not fail and absorbs nothing."""
    import nb_inputs
    d = nb_inputs.make_config(2, n_override=2500)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G, 3.0, 0.4)
    sure, _ = oracle.pairs(d.x, rc)
    grp = oracle.groups(sure, d.N)
    seg = grp["members"][grp["gstart"][0]:grp["gstart"][1]]
    sub = dict(ngroups=1, members=seg.astype(np.int32), gstart=np.array([0, len(seg)], dtype=np.int32), label=None)
    x1, v1, s1 = oracle.encounter(d.x, d.v, d.m, rc, d.M_star, 1.5, G, sub, radius=d.radius, radius_factor=400.0)
    assert s1["failed"] == 0 and s1["absorbed"] == 2
    x2, v2, s2 = oracle.encounter(x1, v1, s1["m"], rc, d.M_star, 1.5, G, sub, radius=s1["radius"], radius_factor=400.0,
                                  absorbed_by=s1["absorbed_by"])
    assert s2["failed"] == 0 and s2["absorbed"] == 0 and s2["steps"] <= 3
    assert np.array_equal(s2["absorbed_by"], s1["absorbed_by"])
    gone = np.flatnonzero(s2["absorbed_by"] >= 0)
    assert np.array_equal(x2[gone], x2[s2["absorbed_by"][gone]]) and np.array_equal(v2[gone], v2[s2["absorbed_by"][gone]])
    # and in one call over the whole interval (the first trial step is rejected, the contact is found at t = dt / 2)
    x3, v3, s3 = oracle.encounter(d.x, d.v, d.m, rc, d.M_star, 3.0, G, sub, radius=d.radius, radius_factor=400.0)
    assert s3["failed"] == 0 and s3["absorbed"] == 2 and np.array_equal(s3["absorbed_by"], s1["absorbed_by"])
    live = s3["absorbed_by"][seg] < 0
    assert np.max(np.abs(x3[seg][live] - x2[seg][live])) <= 1e-11


def test_multilevel_steps_with_radii():
    """The multi-level scheme (reading S23) with collisions in its innermost solver: one level (nlev = 1) is step_enc with
    radii bit for bit; radii too small to touch => step_ml bit for bit; inflated radii => bodies absorbed, mass conserved,
    no failures, and about as many absorbed as the one-level scheme finds on the same input."""
    import nb_inputs
    d = nb_inputs.make_config(2, n_override=1200)
    a = oracle.step_enc(d.x, d.v, d.m, d.M_star, d.dt, G, 2, n1=3.0, n2=0.4, radius=d.radius, radius_factor=400.0)
    b = oracle.step_ml(d.x, d.v, d.m, d.M_star, d.dt, G, 2, 1, n1=3.0, n2=0.4, radius=d.radius, radius_factor=400.0)
    assert np.array_equal(a["x"], b["x"]) and np.array_equal(a["v"], b["v"]) and np.array_equal(a["m"], b["m"])
    assert np.array_equal(a["absorbed_by"], b["absorbed_by"]) and a["stats"]["absorbed"] == b["stats"]["absorbed"] > 0
    c0 = oracle.step_ml(d.x, d.v, d.m, d.M_star, d.dt, G, 2, 3, n1=3.0, n2=0.4)
    c1 = oracle.step_ml(d.x, d.v, d.m, d.M_star, d.dt, G, 2, 3, n1=3.0, n2=0.4, radius=d.radius, radius_factor=1.0)
    assert c1["stats"]["absorbed"] == 0 and np.array_equal(c0["x"], c1["x"]) and np.array_equal(c0["v"], c1["v"])
    c = oracle.step_ml(d.x, d.v, d.m, d.M_star, d.dt, G, 2, 3, n1=3.0, n2=0.4, radius=d.radius, radius_factor=400.0)
    assert c["stats"]["failed"] == 0 and c["stats"]["absorbed"] > 0
    assert abs(c["m"].sum() - d.m.sum()) <= 1e-15 * d.m.sum()
    assert abs(c["stats"]["absorbed"] - a["stats"]["absorbed"]) <= max(3, a["stats"]["absorbed"] // 2)
    gone = np.flatnonzero(c["absorbed_by"] >= 0)
    assert np.all(c["m"][gone] == 0.0) and np.all(c["m"][c["absorbed_by"][gone]] > 0.0)
