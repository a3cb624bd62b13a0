"""-m gpu: the fused small-N step (step_small.cuh: all steps of nb_step in ONE cooperative launch for N <= 8192) against
the multi-launch path (bit for bit: same device functions on the same virtual blocks) and against the oracle."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import ENERGY_TOL, GpuState, assert_acc_close, assert_pairs_match

pytestmark = pytest.mark.gpu


def _run(d, nsteps, use_graph, with_pairs=True, n2=0.4, **tune):
    na = d.n_active if d.n_active < d.N else 0
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n_active=na, n1=3.0, n2=n2, use_graph=use_graph, pair_capacity=1 << 16, **tune)
    st.step(d.dt, nsteps, with_pairs=with_pairs)
    xg, vg, ag, rcg = st.host()
    gp, n = st.get_pairs() if with_pairs else (np.zeros((0, 2), dtype=np.int32), 0)
    return xg, vg, ag, rcg, gp, n, st.nb.nb_status()


@pytest.mark.parametrize("cfg,n_override,tune", [(0, 300, {}), (0, 2048, {}), (1, 5000, dict(force_kernel=1)), (3, 4096, {}),
                                                 (2, 8192, dict(i_per_thread=2, force_kernel=1)),    # one-sided kernel kept above the
                                                 (0, 1000, dict(i_per_thread=4, j_splits=2))])      # Newton-III threshold (N >= 4096)
@pytest.mark.parametrize("nsteps", [1, 2, 9])
def test_fused_small_step_is_the_multi_launch_step_bit_for_bit(cfg, n_override, tune, nsteps):
    d = nb_inputs.make_config(cfg, n_override=n_override)
    a = _run(d, nsteps, True, **tune)      # fused (one cooperative launch)
    b = _run(d, nsteps, False, **tune)     # five launches per step
    for k in range(4):
        assert np.array_equal(a[k], b[k]), f"array {k} differs"
    assert a[5] == b[5] and {tuple(p) for p in a[4].tolist()} == {tuple(p) for p in b[4].tolist()}
    assert a[6] == b[6]


def test_fused_small_step_against_oracle_config1_full():
    """BASELINE.json:configs[0] in full (N = 2048, dt = 6 d, 100 steps, 3 R_Hill) through the fused path."""
    d = nb_inputs.make_config(0)
    xg, vg, ag, rcg, gp, n, status = _run(d, d.nsteps, True, n2=0.0)
    ref = oracle.step(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, d.nsteps, n1=3.0, n2=0.0)
    assert status["kepler_fail"] == 0
    ex = np.max(np.abs(xg - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(vg - ref["v"])) / np.max(np.abs(ref["v"]))
    E0 = oracle.diagnostics(d.x, d.v, d.m, d.M_star, G_GAUSS)
    Eg = oracle.diagnostics(xg, vg, d.m, d.M_star, G_GAUSS)
    Er = oracle.diagnostics(ref["x"], ref["v"], d.m, d.M_star, G_GAUSS)
    print(f"fused config 1 x100: rel dx {ex:.2e} dv {ev:.2e}")
    assert ex <= 1e-9 and ev <= 1e-9
    assert abs((Eg["E"] - Er["E"]) / E0["E"]) <= ENERGY_TOL
    acc_ref, ab, _ = oracle.accel(xg, d.m, rcg, G_GAUSS, want_abs=True)
    assert_acc_close(ag, acc_ref, "fused final acc", ab)
    sure, border = oracle.pairs(xg, rcg)
    assert_pairs_match(gp, n, sure, border, "fused final pairs")


def test_fused_small_step_without_pairs_and_chunked():
    d = nb_inputs.make_config(0, n_override=1500)
    a = _run(d, 6, True, with_pairs=False)
    b = _run(d, 6, False, with_pairs=False)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    # chunked with the cached force: 2 + 4 steps equal 6
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, pair_capacity=1 << 16)
    st.step(d.dt, 2, with_pairs=False)
    st.nb.set_flags(reuse_acc=1)
    st.step(d.dt, 4, with_pairs=False)
    st.nb.set_flags(reuse_acc=0)
    xg, vg, _, _ = st.host()
    assert np.array_equal(xg, a[0]) and np.array_equal(vg, a[1])
