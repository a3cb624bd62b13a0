"""-m gpu parity at BASELINE.json's full sizes, in the launch configuration bench.py times (automatic
tuning): sampled outputs the oracle can compute row by row, plus properties that hold at any size."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import GpuState, assert_acc_close, canon_pairs

pytestmark = pytest.mark.gpu

_SAMPLE_ROWS = {0: 2048, 1: 1024, 2: 512, 3: 1024, 4: 96}


def _check_full(cfg, n1, n2):
    d = nb_inputs.make_config(cfg)
    N = d.N
    na = d.n_active if d.n_active < N else 0
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, n1, n2)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n_active=na, n1=n1, n2=n2, pair_capacity=1 << 24)
    st.set_rcrit(rc)
    st.kick(0.0)
    acc = st.acc.cpu().numpy()
    gp, n = st.get_pairs()
    status = st.nb.nb_status()
    assert status["pairs_dropped"] == 0 and status["nonfinite"] == 0 and status["singular"] == 0
    assert n == gp.shape[0]

    # --- sampled rows against the oracle (always includes the first, last and any giant rows)
    rng = np.random.default_rng(4242 + cfg)
    k = min(_SAMPLE_ROWS[cfg], N)
    rows = np.unique(np.concatenate([rng.choice(N, size=k, replace=False), [0, N - 1, N - 2], np.arange(min(4, N))]))
    acc_ref, ab, _ = oracle.accel(d.x, d.m, rc, G_GAUSS, n_active=na, rows=rows, want_abs=True)
    ratio, lit = assert_acc_close(acc[rows], acc_ref, f"{d.name} sampled rows", ab)
    sure, border = oracle.pairs(d.x, rc, n_active=na, rows=rows)
    in_rows = np.zeros(N, dtype=bool)
    in_rows[rows] = True
    cg = canon_pairs(gp)
    assert cg.shape[0] == gp.shape[0], "duplicate pairs"
    touching = cg[in_rows[cg[:, 0]] | in_rows[cg[:, 1]]] if cg.shape[0] else cg
    key = lambda p: p[:, 0].astype(np.int64) * (1 << 32) + p[:, 1]
    ks, kb, kg = key(sure), key(border), key(touching)
    assert np.setdiff1d(ks, kg).size == 0, "sure pairs incident to the sampled rows are missing"
    assert np.setdiff1d(kg, np.union1d(ks, kb)).size == 0, "CUDA pairs incident to the sampled rows are not pairs"

    # --- properties at full size
    if cg.shape[0]:
        i, j = cg[:, 0], cg[:, 1]
        assert np.all(i < j)
        dx = d.x[j] - d.x[i]
        r2 = (dx[:, 0] * dx[:, 0] + dx[:, 1] * dx[:, 1]) + dx[:, 2] * dx[:, 2]
        rc2 = np.maximum(rc[i], rc[j]) ** 2
        assert np.all(r2 < rc2 * (1 + 2e-12)), "a listed pair is outside its critical radius"
        if na:
            assert np.all(i < na), "semi-active: a listed pair has no active member"
    if not na:
        # Newton III: sum m_i a_i = 0 (symmetric rc_ij)
        f = d.m[:, None] * acc
        assert np.linalg.norm(f.sum(axis=0)) <= 1e-12 * np.abs(f).sum()
    return dict(name=d.name, N=N, pairs=int(n), ratio=ratio, lit=lit)


@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_full_size_hill_only(cfg):
    print(_check_full(cfg, 3.0, 0.0))


@pytest.mark.parametrize("cfg", [1, 2])
def test_full_size_eq7_stress(cfg):
    print(_check_full(cfg, 3.0, 0.4))


@pytest.mark.slow
def test_full_size_config5():
    print(_check_full(4, 3.0, 0.0))


def test_full_size_steps_conserve_angular_momentum():
    """Every sub-step conserves L exactly (symmetric rc_ij): a whole-step invariant that holds at any
    size; config 2 in full (N = 16386 with both giants), 10 steps, diagnostics on the CPU."""
    d = nb_inputs.make_config(1)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.0)
    D0 = oracle.diagnostics(d.x, d.v, d.m, d.M_star, G_GAUSS)
    st.step(d.dt, 10)
    xg, vg, _, _ = st.host()
    D1 = oracle.diagnostics(xg, vg, d.m, d.M_star, G_GAUSS)
    assert st.nb.nb_status()["kepler_fail"] == 0
    dL = np.linalg.norm(D1["L"] - D0["L"]) / np.linalg.norm(D0["L"])
    dE = abs((D1["E"] - D0["E"]) / D0["E"])
    print("config2 x10: dL/L", dL, "dE/E", dE)
    assert dL <= 1e-13
    assert dE <= 1e-6
