"""-m gpu parity of the implicit-midpoint extra force (Eq. 8; reading S24): nb_midpoint_drag and nb_step
with drag_gamma > 0 against the oracle (oracle.midpoint_drag / oracle.step_drag, pinned in tests/test_oracle_midpoint.py).
Both sides run the same fixed-point iteration to tol = 1e-14; a stopping decision that falls differently by one
iteration leaves a difference below tol |v|, so 1e-13 relative is what the arithmetic guarantees for one application."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import GpuState, to_dev, torch_mod

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("power,gamma,eta", [(0, 0.02, 0.0), (0, 0.05, 0.01), (1, 5.0, 0.005), (1, 4.0, 1.0)])  # gas at rest: gamma |v| dt <= 0.3, the iteration contracts (gamma = 20 does not: 802 bodies diverge in the oracle itself)
def test_midpoint_drag_against_oracle(power, gamma, eta):
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    d = nb_inputs.make_config(1, n_override=3000)
    for dt in (3.0, -3.0):
        nb.configure(d.N, G=G_GAUSS, drag_gamma=gamma, drag_eta=eta, drag_power=power, midpoint_tol=1e-14, midpoint_iters=100)
        nb.nb_status_reset()
        xd, vd = to_dev(d.x), to_dev(d.v)
        nb.nb_midpoint_drag(xd, vd, d.M_star, dt)
        torch.cuda.synchronize()
        vg = vd.cpu().numpy()
        vr, nf, it = oracle.midpoint_drag(d.x, d.v, G_GAUSS * d.M_star, dt, gamma, power=power, eta=eta, tol=1e-14, max_iter=100)
        assert nf == 0 and nb.nb_status()["midpoint_fail"] == 0
        err = np.max(np.abs(vg - vr)) / np.max(np.abs(vr))
        print(f"midpoint drag p={power} gamma={gamma} eta={eta} dt={dt}: oracle iterations <= {it}, rel dv {err:.2e}")
        assert err <= 1e-13
        assert np.max(np.abs(vr - d.v)) > 1e-6 * np.max(np.abs(d.v))
    # divergence is counted: gamma dt / 2 > 1
    nb.configure(d.N, G=G_GAUSS, drag_gamma=1.0, drag_power=0, drag_eta=1.0, midpoint_iters=20)
    nb.nb_status_reset()
    vd = to_dev(d.v)
    nb.nb_midpoint_drag(to_dev(d.x), vd, d.M_star, 6.0)
    torch.cuda.synchronize()
    assert nb.nb_status()["midpoint_fail"] == d.N


@pytest.mark.parametrize("use_graph", [True, False])
@pytest.mark.parametrize("nsteps", [1, 2, 25])
def test_step_with_drag_matches_oracle(nsteps, use_graph):
    d = nb_inputs.make_config(0, n_override=1500)
    gamma, eta = 2e-3, 0.01
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, drag_gamma=gamma, drag_eta=eta, drag_power=1,
                  use_graph=use_graph)
    st.step(d.dt, nsteps)
    xg, vg, ag, rcg = st.host()
    ref = oracle.step_drag(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, nsteps, gamma, power=1, eta=eta, n1=3.0, n2=0.4)
    plain = oracle.step(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, nsteps, n1=3.0, n2=0.4)
    status = st.nb.nb_status()
    assert ref["n_fail"] == 0 and status["midpoint_fail"] == 0 and status["kepler_fail"] == 0
    ex = np.max(np.abs(xg - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(vg - ref["v"])) / np.max(np.abs(ref["v"]))
    print(f"step_drag x{nsteps}: rel dx {ex:.2e} dv {ev:.2e}; drag moved v by {np.max(np.abs(ref['v'] - plain['v'])) / np.max(np.abs(plain['v'])):.2e}")
    tol = 1e-12 if nsteps <= 2 else 1e-10
    assert ex <= tol and ev <= tol
    assert np.max(np.abs(ref["v"] - plain["v"])) > 1e-9 * np.max(np.abs(plain["v"]))
    assert np.max(np.abs(rcg - ref["rcrit"]) / ref["rcrit"]) <= 1e-10
    # chunked stepping with the cached force: 1 + (nsteps - 1) equals nsteps
    if nsteps > 1:
        st2 = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, drag_gamma=gamma, drag_eta=eta, drag_power=1,
                       use_graph=use_graph)
        st2.step(d.dt, 1)
        st2.nb.set_flags(reuse_acc=1)
        st2.step(d.dt, nsteps - 1)
        st2.nb.set_flags(reuse_acc=0)
        x2, v2, _, _ = st2.host()
        assert np.array_equal(x2, xg) and np.array_equal(v2, vg)
