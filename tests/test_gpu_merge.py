"""-m gpu parity of nb_merge (perfect merging: contact test on the pair rows, clusters, momentum-conserving merger,
stable compaction) against oracle.merge.  The contact decision is taken in the same fp64 arithmetic on both sides
and the sums run in index order without fused multiply-adds, so x, v, m, the new N, the survivor map and the counts
are bit-exact; the merged radius goes through cbrt (1 ulp)."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import GpuState, to_dev, torch_mod

pytestmark = pytest.mark.gpu


def _gpu_merge(x, v, m, R, pairs, f=1.0, n_active=0, claimed=None):
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    N = m.shape[0]
    pairs = np.ascontiguousarray(np.asarray(pairs, dtype=np.int32).reshape(-1, 2))
    cap = max(pairs.shape[0], 1)
    nb.configure(N, pair_capacity=cap, G=G_GAUSS, radius_factor=f, n_active=n_active)
    nb.nb_status_reset()
    xd, vd, md, Rd = to_dev(x), to_dev(v), to_dev(m), to_dev(R)
    buf = torch.zeros((cap, 2), dtype=torch.int32, device="cuda")
    if pairs.shape[0]:
        buf[: pairs.shape[0]] = to_dev(pairs)
    npd = torch.tensor([pairs.shape[0] if claimed is None else claimed], dtype=torch.int64, device="cuda")
    surv = torch.full((N,), -3, dtype=torch.int32, device="cuda")
    mstat = torch.full((4,), -3, dtype=torch.int64, device="cuda")
    nb.nb_merge(xd, vd, md, Rd, buf, npd, surv, mstat)
    torch.cuda.synchronize()
    return xd.cpu().numpy(), vd.cpu().numpy(), md.cpu().numpy(), Rd.cpu().numpy(), surv.cpu().numpy(), [int(t) for t in mstat.cpu().tolist()]


def _assert_same(x, v, m, R, pairs, what, f=1.0, n_active=0):
    xg, vg, mg, Rg, surv, mstat = _gpu_merge(x, v, m, R, pairs, f=f, n_active=n_active)
    ref = oracle.merge(x, v, m, R, pairs, f=f)
    Nn = ref["N"]
    na_new = int(ref["alive"][: (n_active or m.shape[0])].sum())
    assert mstat == [Nn, ref["n_collisions"], ref["n_merged"], na_new], f"{what}: counts {mstat}"
    assert np.array_equal(surv, ref["survivor_of"]), f"{what}: survivor map differs"
    assert np.array_equal(xg[:Nn], ref["x"]) and np.array_equal(vg[:Nn], ref["v"]) and np.array_equal(mg[:Nn], ref["m"]), \
        f"{what}: merged state differs"
    assert np.max(np.abs(Rg[:Nn] - ref["radius"]) / ref["radius"]) <= 4e-16, f"{what}: radii differ"
    return ref


def test_merge_closed_form_and_identity():
    x = np.array([[1.0, 0, 0], [1.0 + 5e-4, 0, 0], [3.0, 0, 0]]); v = np.array([[0, 1.0, 0], [0, 3.0, 0], [0, 0, 1.0]])
    m = np.array([1.0, 3.0, 2.0]); R = np.array([2e-4, 2e-4, 1e-4])
    ref = _assert_same(x, v, m, R, [[0, 1], [1, 2]], "no contact")
    assert ref["N"] == 3
    ref = _assert_same(x, v, m, R, [[0, 1], [1, 2]], "inflated radii", f=1.5)
    assert ref["N"] == 2
    _assert_same(x, v, m, R, np.zeros((0, 2), dtype=np.int32), "empty list")


@pytest.mark.parametrize("n,scale,seed", [(400, 0.0015, 3), (5000, 0.005, 4), (20000, 0.01, 5)])
def test_merge_crowded_clusters(n, scale, seed):
    rng = np.random.default_rng(seed)
    x = rng.normal(size=(n, 3)) * scale; v = rng.normal(size=(n, 3)) * 0.01
    m = rng.uniform(1e-7, 1e-5, n); R = rng.uniform(1e-4, 3e-4, n)
    m[::5] = 0.0                                                 # test particles among them
    from scipy.spatial import cKDTree
    pairs = cKDTree(x).query_pairs(8e-4, output_type="ndarray").astype(np.int32)   # superset of all contacts
    pairs = pairs[rng.permutation(pairs.shape[0])]
    ref = _assert_same(x, v, m, R, pairs, f"crowded n={n}")
    assert ref["n_merged"] > n // 100
    print(f"n={n}: candidate rows {pairs.shape[0]}, contacts {ref['n_collisions']}, removed {ref['n_merged']}")


def test_merge_after_a_kick_on_a_disk_with_inflated_radii():
    """The kick's own pair list (rc = 3 R_Hill + velocity term) feeds the merger; radii from the bulk density of the
    configs (2 g/cm^3), inflated until a few hundred bodies touch; semi-active ordering survives the compaction."""
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    d = nb_inputs.make_config(3, n_override=6000)
    rho = 3.367443e6                                             # 2 g/cm^3 in M_sun / AU^3
    m_eff = np.where(d.m > 0, d.m, 1e-12)
    R = (3.0 * m_eff / (4.0 * np.pi * rho)) ** (1.0 / 3.0)
    f = 400.0
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n_active=d.n_active, n1=3.0, n2=0.4, pair_capacity=1 << 18, radius_factor=f)
    st.step(d.dt, 0)
    gp, n = st.get_pairs()
    Rd = to_dev(R)
    surv = torch.empty(d.N, dtype=torch.int32, device="cuda"); mstat = torch.zeros(4, dtype=torch.int64, device="cuda")
    nb.nb_merge(st.x, st.v, st.m, Rd, st.pairs, st.npairs, surv, mstat)
    torch.cuda.synchronize()
    ref = oracle.merge(d.x, d.v, d.m, R, gp, f=f)
    ms = [int(t) for t in mstat.cpu().tolist()]
    assert ref["n_merged"] > 0
    assert ms == [ref["N"], ref["n_collisions"], ref["n_merged"], int(ref["alive"][: d.n_active].sum())]
    Nn = ref["N"]
    assert np.array_equal(st.x.cpu().numpy()[:Nn], ref["x"]) and np.array_equal(st.m.cpu().numpy()[:Nn], ref["m"])
    # the survivors form a valid state: a force evaluation on the new N runs and matches the oracle
    xs, vs, msr = st.x[:Nn].contiguous(), st.v[:Nn].contiguous(), st.m[:Nn].contiguous()
    st2 = GpuState(xs.cpu().numpy(), vs.cpu().numpy(), msr.cpu().numpy(), d.M_star, G=G_GAUSS, n_active=ms[3], n1=3.0, n2=0.4)
    st2.step(d.dt, 0)
    acc_ref, ab, _ = oracle.accel(ref["x"], ref["m"], st2.rcrit.cpu().numpy(), G_GAUSS, n_active=ms[3], want_abs=True)
    from gpu_util import assert_acc_close
    assert_acc_close(st2.acc.cpu().numpy(), acc_ref, "after merge", ab)
    print("merged", ref["n_merged"], "of", d.N, "contacts", ref["n_collisions"], "new n_active", ms[3])
