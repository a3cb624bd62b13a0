"""-m gpu parity: nb_kick / nb_rcrit / nb_shift (C ABI, CUDA path) against the CPU oracle, element by
element on the same seeded inputs.  Sizes span several 128-body tiles and ragged tails."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import GpuState, assert_acc_close, assert_pairs_match

pytestmark = pytest.mark.gpu


def _kick_case(x, v, m, rc, *, G=G_GAUSS, n_active=0, kind=0, dt=0.0, what="", **tune):
    """One nb_kick against oracle.accel + oracle.pairs with a caller-supplied rcrit."""
    st = GpuState(x, v, m, G=G, n_active=n_active, kind=kind, **tune)
    st.set_rcrit(rc)
    st.kick(dt)
    _, v_gpu, acc_gpu, _ = st.host()
    acc_ref, ab, nsing = oracle.accel(x, m, rc, G, n_active=n_active, kind=kind, want_abs=True)
    ratio, lit = assert_acc_close(acc_gpu, acc_ref, what, ab)
    sure, border = oracle.pairs(x, rc, n_active=n_active)
    gp, n = st.get_pairs()
    info = assert_pairs_match(gp, n, sure, border, what)
    if dt != 0.0:
        v_ref, acc_k = oracle.kick(x, v, m, dt, rc, G, n_active=n_active, kind=kind)   # pinned by its two-body closed form
        assert np.array_equal(acc_k, acc_ref)
        assert np.max(np.abs(v_gpu - v_ref)) <= 1e-12 * np.max(np.abs(v_ref)) + 1e-300
    else:
        assert np.array_equal(v_gpu, np.asarray(v))
    status = st.nb.nb_status()
    assert status["singular"] == nsing
    assert status["pairs_dropped"] == 0 and status["nonfinite"] == 0
    return dict(ratio=ratio, lit=lit, **info)


def test_two_body_closed_form_and_oracle():
    x, v, m = nb_inputs.two_body(m1=1e-3, m2=2e-3, sep=0.01)
    rc = np.zeros(2)
    info = _kick_case(x, v, m, rc, what="two_body W=1")
    assert info["n_gpu"] == 0
    # inside the changeover shell
    rc = np.array([0.02, 0.015])
    info = _kick_case(x, v, m, rc, what="two_body changeover")
    assert info["n_gpu"] == 1


@pytest.mark.parametrize("ipt", [1, 2, 4])
@pytest.mark.parametrize("N", [1, 2, 127, 128, 129, 700])
def test_random_cluster_newtonian(N, ipt):
    x, v, m = nb_inputs.random_cluster(N, seed=100 + N)
    info = _kick_case(x, v, m, np.zeros(N), i_per_thread=ipt, what=f"cluster N={N} I={ipt}")
    assert info["n_gpu"] == 0


@pytest.mark.parametrize("kind", [0, 1])
@pytest.mark.parametrize("ipt,splits", [(1, 0), (2, 3), (4, 1), (4, 0)])
def test_random_cluster_with_changeover_and_pairs(kind, ipt, splits):
    N = 1000
    x, v, m = nb_inputs.random_cluster(N, seed=5, scale=0.2)
    rng = np.random.default_rng(9)
    rc = rng.uniform(0.0, 0.06, N)
    rc[::7] = 0.0
    info = _kick_case(x, v, m, rc, kind=kind, dt=0.37, i_per_thread=ipt, j_splits=splits,
                      what=f"cluster changeover kind={kind} I={ipt} splits={splits}")
    assert info["n_sure"] > 300  # the pair path really is exercised


def test_chain_and_lattice_pair_counts():
    # 1-D chain, spacing 1: rc = 1.5 => N-1 pairs; rc = 2.5 => 2N-3
    N = 300
    x, v, m = nb_inputs.chain_1d(N)
    for rcv, expect in ((1.5, N - 1), (2.5, 2 * N - 3)):
        info = _kick_case(x, v, m, np.full(N, rcv), G=1.0, what=f"chain rc={rcv}")
        assert info["n_gpu"] == expect
    x, v, m = nb_inputs.cubic_lattice(7)
    n = 7
    info = _kick_case(x, v, m, np.full(n ** 3, 1.2), G=1.0, what="lattice")
    assert info["n_gpu"] == 3 * n * n * (n - 1)


def test_coincident_bodies():
    # coincident with rc > 0: W = 0, contributes exactly 0, is a pair; with rc == 0: counted singular
    x, v, m = nb_inputs.random_cluster(40, seed=3)
    x[7] = x[21]
    rc = np.full(40, 0.01)
    info = _kick_case(x, v, m, rc, what="coincident rc>0")
    assert info["n_gpu"] >= 1
    _kick_case(x, v, m, np.zeros(40), what="coincident rc=0")


@pytest.mark.parametrize("cfg,n_override", [(0, 2048), (1, 3000), (2, 4096), (3, 8192), (4, 5000)])
@pytest.mark.parametrize("n1,n2", [(3.0, 0.0), (3.0, 0.4), (30.0, 0.0)])
def test_disk_configs_reduced(cfg, n_override, n1, n2):
    """The five workload shapes (BASELINE.json:configs) at sizes the oracle finishes in seconds:
    Hill-only headline radius, full Eq. 7 stress radius, and an inflated radius that makes pairs dense."""
    d = nb_inputs.make_config(cfg, n_override=n_override)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, n1, n2)
    na = d.n_active if d.n_active < d.N else 0
    info = _kick_case(d.x, d.v, d.m, rc, n_active=na, dt=0.5 * d.dt, what=f"{d.name} n1={n1} n2={n2}")
    if n1 == 30.0 or n2 > 0:
        assert info["n_sure"] > 0


def test_internal_rcrit_and_nb_rcrit():
    d = nb_inputs.make_config(1, n_override=1500)
    rc_ref = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, 0.4)
    st = GpuState(d.x, d.v, d.m, G=G_GAUSS, n1=3.0, n2=0.4)
    st.nb.nb_rcrit(st.x, st.v, st.m, d.M_star, d.dt, st.rcrit)
    rc_gpu = st.rcrit.cpu().numpy()
    assert np.max(np.abs(rc_gpu - rc_ref) / rc_ref) <= 1e-14
    # rcrit = NULL: nb_kick computes Eq. 7 internally from (x, v, m, M_star, dt)
    st.kick(d.dt, rcrit_given=False)
    acc_ref, ab, _ = oracle.accel(d.x, d.m, rc_ref, G_GAUSS, want_abs=True)
    assert_acc_close(st.acc.cpu().numpy(), acc_ref, "internal rcrit", ab)
    sure, border = oracle.pairs(d.x, rc_ref)
    gp, n = st.get_pairs()
    assert_pairs_match(gp, n, sure, border, "internal rcrit")


def test_pairs_null_skips_detection_and_overflow_counts():
    N = 600
    x, v, m = nb_inputs.random_cluster(N, seed=11, scale=0.1)
    rc = np.full(N, 0.05)
    sure, border = oracle.pairs(x, rc)
    acc_ref, ab, _ = oracle.accel(x, m, rc, G_GAUSS, want_abs=True)
    st = GpuState(x, v, m, G=G_GAUSS, pair_capacity=100)
    st.set_rcrit(rc)
    st.kick(0.0, with_pairs=False)
    assert_acc_close(st.acc.cpu().numpy(), acc_ref, "pairs=NULL", ab)
    st.kick(0.0, with_pairs=True)
    gp, n = st.get_pairs()
    assert sure.shape[0] <= n <= sure.shape[0] + border.shape[0]
    assert gp.shape[0] == 100  # only the first `capacity` rows are written, the count keeps counting
    assert st.nb.nb_status()["pairs_dropped"] == n - 100
    assert_acc_close(st.acc.cpu().numpy(), acc_ref, "overflow", ab)


def test_shift_parity():
    d = nb_inputs.make_config(1, n_override=3000)
    st = GpuState(d.x, d.v, d.m, G=G_GAUSS)
    st.nb.nb_shift(st.x, st.v, st.m, d.M_star, 0.5 * d.dt)
    x_ref = oracle.shift(d.x, d.v, d.m, d.M_star, 0.5 * d.dt)
    x_gpu = st.x.cpu().numpy()
    disp = np.max(np.abs(x_ref - d.x))
    assert disp > 0
    assert np.max(np.abs(x_gpu - x_ref)) <= 1e-15 * np.max(np.abs(x_ref)) + 1e-12 * disp


def test_error_codes():
    import paper_2604_09184_b200 as nb
    d = nb_inputs.make_config(0, n_override=256)
    st = GpuState(d.x, d.v, d.m, G=G_GAUSS)
    with pytest.raises(nb.NbError) as e:
        nb.nb_kick(st.x, st.v, st.m, -1.0, 0.0, st.rcrit, st.acc)
    assert e.value.code == nb.binding.NB_E_BADARG
    with pytest.raises(nb.NbError) as e:
        nb.nb_kick(st.x, st.v, st.m, 1.0, float("nan"), st.rcrit, st.acc)
    assert e.value.code == nb.binding.NB_E_BADARG
    with pytest.raises(nb.NbError) as e:
        nb.nb_kick(st.x, st.v, st.m, 1.0, 0.0, st.rcrit, None)
    assert e.value.code == nb.binding.NB_E_NULL
    # workspace too small for a bigger N
    cfg = nb.binding._state["cfg"]
    cfg.workspace_bytes = 1024
    import ctypes as C
    assert nb.load().nb_configure(C.byref(cfg)) == 0
    with pytest.raises(nb.NbError) as e:
        nb.nb_kick(st.x, st.v, st.m, 1.0, 0.0, st.rcrit, st.acc)
    assert e.value.code == nb.binding.NB_E_WORKSPACE
