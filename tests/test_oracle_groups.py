"""-m "not gpu": pins of the oracle's encounter-group builder (oracle_groups) against what
the mathematics fixes: closed-form graphs, scipy's connected_components, brute-force label relaxation,
invariance under edge order / orientation / duplication."""
import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components

import oracle


def _check_structure(g, N, pairs):
    label, members, gstart = g["label"], g["members"], g["gstart"]
    assert label.shape == (N,) and np.all(label <= np.arange(N)) and np.all(label[label] == label)
    pairs = np.asarray(pairs).reshape(-1, 2)
    if pairs.size:
        assert np.all(label[pairs[:, 0]] == label[pairs[:, 1]])            # an edge never leaves its group
    sizes = np.bincount(label, minlength=N)
    leaders = np.flatnonzero(sizes >= 2)
    assert g["ngroups"] == leaders.size and g["nmembers"] == int(sizes[leaders].sum())
    assert g["largest"] == (int(sizes.max()) if leaders.size else 0)
    assert gstart[0] == 0 if g["ngroups"] else gstart.shape[0] == 1
    for k, lead in enumerate(leaders):                                       # groups in label order, members ascending
        seg = members[gstart[k]:gstart[k + 1]]
        assert np.array_equal(seg, np.flatnonzero(label == lead))


def test_closed_form_graphs():
    N = 50
    g = oracle.groups(np.zeros((0, 2), dtype=np.int32), N)                   # no pairs: every body alone
    assert np.array_equal(g["label"], np.arange(N)) and g["ngroups"] == 0 and g["members"].size == 0
    chain = np.stack([np.arange(N - 1), np.arange(1, N)], axis=1)            # a chain is one group
    g = oracle.groups(chain, N)
    assert np.all(g["label"] == 0) and g["ngroups"] == 1 and g["largest"] == N
    assert np.array_equal(g["members"], np.arange(N)) and np.array_equal(g["gstart"], [0, N])
    star = np.stack([np.full(9, 40), np.arange(10, 19)], axis=1)            # star centred on 40: label = 10
    g = oracle.groups(star, N)
    assert np.all(g["label"][10:19] == 10) and g["label"][40] == 10 and g["ngroups"] == 1 and g["largest"] == 10
    assert np.array_equal(g["members"], list(range(10, 19)) + [40])
    # k disjoint triangles on bodies 3k, 3k+1, 3k+2
    tri = np.array([[3 * k + a, 3 * k + b] for k in range(10) for a, b in ((0, 1), (1, 2), (0, 2))])
    g = oracle.groups(tri, N)
    assert g["ngroups"] == 10 and g["nmembers"] == 30 and g["largest"] == 3
    assert np.array_equal(g["label"][:30], np.repeat(np.arange(0, 30, 3), 3))
    assert np.array_equal(g["label"][30:], np.arange(30, N))
    assert np.array_equal(g["gstart"], np.arange(0, 31, 3))
    with pytest.raises(ValueError):
        oracle.groups(np.array([[1, 1]]), N)
    with pytest.raises(ValueError):
        oracle.groups(np.array([[1, N]]), N)


@pytest.mark.parametrize("N,E,seed", [(10, 4, 1), (200, 60, 2), (200, 400, 3), (5000, 2500, 4), (5000, 20000, 5)])
def test_against_scipy_and_brute_force(N, E, seed):
    rng = np.random.default_rng(seed)
    a = rng.integers(0, N, E); b = rng.integers(0, N, E)
    keep = a != b
    pairs = np.stack([a[keep], b[keep]], axis=1).astype(np.int32)
    g = oracle.groups(pairs, N)
    _check_structure(g, N, pairs)
    # scipy: same partition; the oracle's label is the smallest index of each part
    m = coo_matrix((np.ones(pairs.shape[0]), (pairs[:, 0], pairs[:, 1])), shape=(N, N))
    _, comp = connected_components(m, directed=False)
    mins = np.full(comp.max() + 1, N)
    np.minimum.at(mins, comp, np.arange(N))
    assert np.array_equal(g["label"], mins[comp])
    if N <= 200:
        # brute force: relax label[i] = min over neighbours until nothing changes
        lab = np.arange(N)
        changed = True
        while changed:
            changed = False
            for i, j in pairs:
                lo = min(lab[i], lab[j])
                if lab[i] != lo or lab[j] != lo:
                    lab[i] = lab[j] = lo
                    changed = True
        assert np.array_equal(g["label"], lab)


def test_invariances():
    rng = np.random.default_rng(7)
    N = 3000
    pairs = rng.integers(0, N, (2000, 2)).astype(np.int32)
    pairs = pairs[pairs[:, 0] != pairs[:, 1]]
    g0 = oracle.groups(pairs, N)
    for variant in (pairs[::-1], pairs[:, ::-1], np.concatenate([pairs, pairs[:500]]), pairs[rng.permutation(pairs.shape[0])]):
        g = oracle.groups(variant, N)
        assert np.array_equal(g["label"], g0["label"]) and np.array_equal(g["members"], g0["members"])
        assert np.array_equal(g["gstart"], g0["gstart"])


def test_groups_of_a_disk_pair_list():
    """Pair list of a reduced ring workload with an inflated critical radius: groups are consistent with
    the geometry (every listed pair inside one group, bodies without pairs alone)."""
    import nb_inputs
    from nb_inputs import G_GAUSS
    d = nb_inputs.make_config(2, n_override=3000)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 30.0, 0.0)
    sure, border = oracle.pairs(d.x, rc)
    assert sure.shape[0] > 100
    g = oracle.groups(sure, d.N)
    _check_structure(g, d.N, sure)
    alone = np.setdiff1d(np.arange(d.N), np.unique(sure))
    assert np.array_equal(g["label"][alone], alone)
