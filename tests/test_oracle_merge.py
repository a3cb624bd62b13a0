"""-m "not gpu": pins of the oracle's perfect-merging step (oracle.merge; reading S21): closed
forms, the conservation laws a perfect merger is defined by, invariances."""
import numpy as np

import oracle


def _rand(n, seed):
    rng = np.random.default_rng(seed)
    return rng.normal(size=(n, 3)), rng.normal(size=(n, 3)) * 0.01, rng.uniform(1e-7, 1e-5, n), rng.uniform(1e-4, 3e-4, n)


def test_two_body_closed_form_and_threshold():
    x = np.array([[1.0, 0, 0], [1.0 + 5e-4, 0, 0], [3.0, 0, 0]]); v = np.array([[0, 1.0, 0], [0, 3.0, 0], [0, 0, 1.0]])
    m = np.array([1.0, 3.0, 2.0]); R = np.array([2e-4, 2e-4, 1e-4])
    out = oracle.merge(x, v, m, R, [[0, 1], [1, 2]])
    assert out["N"] == 3 and out["n_collisions"] == 0                      # 5e-4 > 4e-4: no contact
    out = oracle.merge(x, v, m, R, [[0, 1], [1, 2]], f=1.5)                # inflated radii: 6e-4 > 5e-4
    assert out["N"] == 2 and out["n_merged"] == 1 and out["n_collisions"] == 1
    assert np.allclose(out["x"][0], [1.0 + 0.75 * 5e-4, 0, 0], rtol=0, atol=1e-16)
    assert np.array_equal(out["v"][0], [0, 2.5, 0]) and out["m"][0] == 4.0
    assert abs(out["radius"][0] - 2e-4 * 2 ** (1 / 3)) < 1e-19
    assert np.array_equal(out["x"][1], x[2]) and out["m"][1] == 2.0        # body 2 untouched, moved up one slot
    assert out["alive"].tolist() == [True, False, True] and out["survivor_of"].tolist() == [0, 0, 2]
    # strictness: exactly touching is not a collision
    x2 = np.array([[0.0, 0, 0], [4e-4, 0, 0]])
    assert oracle.merge(x2, v[:2], m[:2], R[:2], [[0, 1]])["N"] == 2
    # a pair that is not on the list is not examined
    assert oracle.merge(x, v, m, R, [[1, 2]], f=1.5)["N"] == 3


def test_conservation_and_chains():
    n = 400
    x, v, m, R = _rand(n, 3)
    x *= 0.004                                                             # crowded: many contacts, chains of them
    iu = np.triu_indices(n, 1)
    pairs = np.stack(iu, axis=1).astype(np.int32)
    out = oracle.merge(x, v, m, R, pairs)
    assert 0 < out["n_merged"] < n and out["N"] == n - out["n_merged"]
    assert abs(out["m"].sum() - m.sum()) <= 1e-15 * m.sum()
    assert np.max(np.abs((out["m"][:, None] * out["v"]).sum(0) - (m[:, None] * v).sum(0))) <= 1e-15 * np.abs(m[:, None] * v).sum()
    assert np.max(np.abs((out["m"][:, None] * out["x"]).sum(0) - (m[:, None] * x).sum(0))) <= 1e-15 * np.abs(m[:, None] * x).sum()
    assert abs((out["radius"] ** 3).sum() - (R ** 3).sum()) <= 1e-14 * (R ** 3).sum()
    # merged clusters = connected components of the contact graph (independent route: scipy)
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    d = np.linalg.norm(x[iu[0]] - x[iu[1]], axis=1)
    hit = d < (R[iu[0]] + R[iu[1]])
    ncomp, comp = connected_components(coo_matrix((np.ones(hit.sum()), (iu[0][hit], iu[1][hit])), shape=(n, n)), directed=False)
    assert out["N"] == ncomp and out["n_collisions"] == int(hit.sum())
    assert np.array_equal(out["alive"], np.array([i == np.flatnonzero(comp == comp[i])[0] for i in range(n)]))
    # order and orientation of the list do not matter; survivors keep index order
    rng = np.random.default_rng(1)
    out2 = oracle.merge(x, v, m, R, pairs[rng.permutation(pairs.shape[0])][:, ::-1])
    for k in ("x", "v", "m", "radius"):
        assert np.array_equal(out[k], out2[k])
    # massless bodies: a test particle hitting a massive one adds no mass and does not move it
    m0 = m.copy(); m0[1::2] = 0.0
    out3 = oracle.merge(x, v, m0, R, pairs)
    assert abs(out3["m"].sum() - m0.sum()) <= 1e-15 * m0.sum() and np.all(np.isfinite(out3["x"]))


def test_no_contact_is_the_identity():
    x, v, m, R = _rand(50, 5)
    out = oracle.merge(x, v, m, R, np.stack(np.triu_indices(50, 1), axis=1))
    assert out["N"] == 50 and out["n_merged"] == 0
    for k, a in (("x", x), ("v", v), ("m", m), ("radius", R)):
        assert np.array_equal(out[k], a)
