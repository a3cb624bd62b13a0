"""-m gpu parity of nb_groups (C ABI, CUDA path: lock-free union-find + scans) against the CPU oracle's
breadth-first search: integer work, so label / members / gstart / counts must be bit-exact."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import GpuState, to_dev, torch_mod

pytestmark = pytest.mark.gpu


def _gpu_groups(pairs, N, cap=None, npairs_claimed=None):
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    pairs = np.ascontiguousarray(np.asarray(pairs, dtype=np.int32).reshape(-1, 2))
    cap = int(cap if cap is not None else max(pairs.shape[0], 1))
    nb.configure(N, pair_capacity=cap, G=G_GAUSS)
    nb.nb_status_reset()
    buf = torch.full((cap, 2), -7, dtype=torch.int32, device="cuda")
    k = min(cap, pairs.shape[0])
    if k:
        buf[:k] = to_dev(pairs[:k])
    npd = torch.tensor([pairs.shape[0] if npairs_claimed is None else npairs_claimed], dtype=torch.int64, device="cuda")
    label = torch.full((N,), -5, dtype=torch.int32, device="cuda")
    members = torch.full((N,), -5, dtype=torch.int32, device="cuda")
    gstart = torch.full((N // 2 + 2,), -5, dtype=torch.int32, device="cuda")
    gstat = torch.full((4,), -5, dtype=torch.int64, device="cuda")
    nb.nb_groups(buf, npd, N, label, members, gstart, gstat)
    torch.cuda.synchronize()
    return label.cpu().numpy(), members.cpu().numpy(), gstart.cpu().numpy(), gstat.cpu().numpy(), nb.nb_status()


def _assert_same(pairs, N, what, **kw):
    label, members, gstart, gstat, status = _gpu_groups(pairs, N, **kw)
    used = np.asarray(pairs, dtype=np.int32).reshape(-1, 2)
    if "cap" in kw and kw["cap"] is not None:
        used = used[:kw["cap"]]
    ref = oracle.groups(used, N)
    assert np.array_equal(label, ref["label"]), f"{what}: labels differ"
    ng, nm = ref["ngroups"], ref["nmembers"]
    assert [int(v) for v in gstat] == [ng, nm, ref["largest"], used.shape[0]], f"{what}: counts {gstat} vs oracle"
    assert np.array_equal(members[:nm], ref["members"]), f"{what}: member list differs"
    assert np.all(members[nm:] == -1), f"{what}: tail of members is not -1"
    assert np.array_equal(gstart[:ng + 1], ref["gstart"]), f"{what}: group offsets differ"
    assert np.all(gstart[ng + 1:] == -1), f"{what}: tail of gstart is not -1"
    assert status["nonfinite"] == 0
    return ref


def test_groups_closed_forms_and_edges():
    N = 50
    ref = _assert_same(np.zeros((0, 2), dtype=np.int32), N, "no pairs")
    assert ref["ngroups"] == 0
    _assert_same(np.stack([np.arange(N - 1), np.arange(1, N)], axis=1), N, "chain")
    _assert_same(np.stack([np.full(9, 40), np.arange(10, 19)], axis=1), N, "star")
    _assert_same(np.array([[0, 1]]), 2, "two bodies")
    _assert_same(np.zeros((0, 2), dtype=np.int32), 1, "one body")


@pytest.mark.parametrize("N,E,seed", [(200, 60, 2), (200, 400, 3), (5000, 2500, 4), (5000, 20000, 5), (100003, 40000, 6),
                                      (100003, 300000, 7), (1 << 20, 400000, 8)])
def test_groups_random_graphs(N, E, seed):
    rng = np.random.default_rng(seed)
    a = rng.integers(0, N, E); b = rng.integers(0, N, E)
    keep = a != b
    pairs = np.stack([a[keep], b[keep]], axis=1).astype(np.int32)
    pairs = np.concatenate([pairs, pairs[: E // 10, ::-1]])  # duplicates, reversed orientation
    _assert_same(pairs, N, f"random N={N} E={E}")


def test_groups_giant_and_mixed_sizes():
    """One group beyond the indicator-scan threshold (a randomly ordered chain: deep union-find trees), many
    small ones, and a mid-size one just below the threshold."""
    rng = np.random.default_rng(11)
    N = 150000
    perm = rng.permutation(N)
    giant = perm[:60000]
    mid = perm[60000:62047]                      # 2047 members: rank-sorted
    edges = [np.stack([giant[:-1], giant[1:]], axis=1), np.stack([mid[:-1], mid[1:]], axis=1)]
    rest = perm[62047:]
    small = rest[: (rest.size // 3) * 3].reshape(-1, 3)[:20000]
    edges += [small[:, :2], small[:, 1:]]
    pairs = np.concatenate(edges).astype(np.int32)
    pairs = pairs[rng.permutation(pairs.shape[0])]
    ref = _assert_same(pairs, N, "giant + mixed")
    assert ref["largest"] == 60000 and ref["ngroups"] == 20002
    # every body in one group
    ring = np.stack([np.arange(N), (np.arange(N) + 1) % N], axis=1).astype(np.int32)
    ref = _assert_same(ring[rng.permutation(N)], N, "all in one group")
    assert ref["largest"] == N and ref["ngroups"] == 1


def test_groups_capacity_and_bad_rows():
    rng = np.random.default_rng(13)
    N = 4000
    pairs = rng.integers(0, N, (3000, 2)).astype(np.int32)
    pairs = pairs[pairs[:, 0] != pairs[:, 1]]
    # the device counter says more pairs than the buffer holds: only the first `capacity` rows exist
    _assert_same(pairs, N, "capacity", cap=1000, npairs_claimed=pairs.shape[0])
    bad = pairs[:100].copy()
    bad[3] = [5, 5]; bad[7] = [-1, 4]; bad[9] = [2, N]
    label, members, gstart, gstat, status = _gpu_groups(bad, N)
    good = np.delete(bad, [3, 7, 9], axis=0)
    ref = oracle.groups(good, N)
    assert np.array_equal(label, ref["label"]) and status["nonfinite"] == 3


@pytest.mark.parametrize("cfg,n_override,n1,n2", [(2, 8192, 3.0, 0.4), (2, 8192, 30.0, 0.0), (1, 6000, 3.0, 0.4), (0, 2048, 30.0, 0.0)])
def test_groups_from_the_kick_pair_list(cfg, n_override, n1, n2):
    """nb_kick's device pair list and counter fed straight into nb_groups; the oracle builds the groups of
    the oracle's own pair list -- the two lists are equal as sets, so the groups must be identical."""
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    d = nb_inputs.make_config(cfg, n_override=n_override)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=n1, n2=n2, pair_capacity=1 << 20)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, n1, n2)
    st.set_rcrit(rc)
    st.kick(0.0)
    N = d.N
    label = torch.empty(N, dtype=torch.int32, device="cuda"); members = torch.empty(N, dtype=torch.int32, device="cuda")
    gstart = torch.empty(N // 2 + 2, dtype=torch.int32, device="cuda"); gstat = torch.empty(4, dtype=torch.int64, device="cuda")
    nb.nb_groups(st.pairs, st.npairs, N, label, members, gstart, gstat)
    torch.cuda.synchronize()
    sure, border = oracle.pairs(d.x, rc)
    assert border.shape[0] == 0 and sure.shape[0] > 0
    ref = oracle.groups(sure, N)
    assert np.array_equal(label.cpu().numpy(), ref["label"])
    gs = gstat.cpu().numpy()
    assert [int(gs[0]), int(gs[1]), int(gs[2])] == [ref["ngroups"], ref["nmembers"], ref["largest"]]
    assert np.array_equal(members.cpu().numpy()[: ref["nmembers"]], ref["members"])
    assert np.array_equal(gstart.cpu().numpy()[: ref["ngroups"] + 1], ref["gstart"])
    print(d.name, "pairs", sure.shape[0], "groups", ref["ngroups"], "members", ref["nmembers"], "largest", ref["largest"])
