"""-m gpu: BASELINE.json:north_star's acceptance at FULL size -- "accelerations, pair lists and energy error all match the
oracle within the stated tolerances on all five configs" -- in the launch configuration bench.py times (automatic
tuning: Newton-III kernel with sorted staging where it applies, CUDA-graph replay).

  config 1 (N = 2048, 100 steps)        tests/test_gpu_drift_step.py::test_step_config1_100_steps (oracle re-run)
  config 2 (N = 16386, 1000 steps)      oracle re-run here (~5 min of host time: slow)
  config 3 (N = 65536, 200 steps)       tests/golden/config3_trajectory.txt (one 16-minute oracle run, oracle/make_golden.py)
  config 4 (N = 131072 / 1024, 100)     oracle re-run here (~15 s)
  config 5 (N = 524288, 10 steps)       tests/golden/config5_trajectory.txt (one ~1 h oracle run)

plus COMPLETE pair lists at full size (oracle.pairs on every row at N = 65536 for both radii; an independent
cKDTree route at N = 524288), the host-buffer entry points nb_kick_host / nb_step_host (the e2e leg of bench.py)
against the oracle, and the per-config parity record gpurun_out/parity_r2.jsonl (summarised in profiles/r2_parity.md).
"""
import hashlib
import json
import os

import numpy as np
import pytest
from scipy.spatial import cKDTree

import nb_inputs
import oracle
from nb_inputs import G_GAUSS
from oracle import make_golden

from gpu_util import ENERGY_TOL, GpuState, acc_error, assert_acc_close, assert_pairs_match, canon_pairs

pytestmark = pytest.mark.gpu

_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
_GOLDEN = os.path.join(_ROOT, "tests", "golden")


def record(**kw):
    """One JSON line per check into gpurun_out/parity_r2.jsonl (a scratch record; profiles/r2_parity.md is the
    committed summary)."""
    out = os.path.join(_ROOT, "gpurun_out")
    try:
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_r2.jsonl"), "a") as f:
            f.write(json.dumps(kw) + "\n")
    except OSError:
        pass
    print(kw)


def _acc_report(acc_gpu, acc_ref, ab):
    """The three readings of "1e-12 per component" side by side."""
    d = np.abs(acc_gpu - acc_ref)
    norm = np.linalg.norm(acc_ref, axis=1, keepdims=True)
    s9 = 1e-12 * np.maximum(np.abs(acc_ref), 1e-3 * norm)
    with np.errstate(divide="ignore", invalid="ignore"):
        lit = np.where(acc_ref != 0.0, d / np.abs(acc_ref), 0.0)
    ratio_full, _ = acc_error(acc_gpu, acc_ref, ab)
    return dict(ratio_with_backward_term=ratio_full, ratio_s9_only=float(np.max(d / np.where(s9 > 0, s9, 1e-300))),
                literal_max=float(np.max(lit)), literal_frac_over_1e12=float(np.mean(lit > 1e-12)),
                backward_max_eps=float(np.max(d / np.where(ab > 0, ab, 1e-300)) / 2.220446049250313e-16))


def _trajectory_vs_oracle(k, what, x_tol):
    d = nb_inputs.make_config(k)
    na = d.n_active if d.n_active < d.N else 0
    ref = oracle.step(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, d.nsteps, n_active=na, n1=3.0, n2=0.0)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n_active=na, n1=3.0, n2=0.0, pair_capacity=1 << 22)
    st.step(d.dt, d.nsteps)
    xg, vg, accg, rcg = st.host()
    status = st.nb.nb_status()
    assert status["kepler_fail"] == 0 and ref["n_fail"] == 0 and status["pairs_dropped"] == 0
    ex = np.max(np.abs(xg - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(vg - ref["v"])) / np.max(np.abs(ref["v"]))
    E0 = oracle.diagnostics(d.x, d.v, d.m, d.M_star, G_GAUSS)
    Eg = oracle.diagnostics(xg, vg, d.m, d.M_star, G_GAUSS)
    Er = oracle.diagnostics(ref["x"], ref["v"], d.m, d.M_star, G_GAUSS)
    de_g, de_r = (Eg["E"] - E0["E"]) / E0["E"], (Er["E"] - E0["E"]) / E0["E"]
    dL = np.linalg.norm(Eg["L"] - E0["L"]) / np.linalg.norm(E0["L"])
    # last evaluation at the GPU's own final state: every row, complete pair list
    acc_ref, ab, _ = oracle.accel(xg, d.m, rcg, G_GAUSS, n_active=na, want_abs=True)
    rep = _acc_report(accg, acc_ref, ab)
    sure, border = oracle.pairs(xg, rcg, n_active=na)
    gp, n = st.get_pairs()
    info = assert_pairs_match(gp, n, sure, border, what + " final pairs")
    record(check="trajectory_vs_oracle_rerun", config=k + 1, name=d.name, N=d.N, nsteps=d.nsteps, rel_dx=ex, rel_dv=ev,
           dE_gpu=de_g, dE_oracle=de_r, dE_diff=abs(de_g - de_r), dL=dL, pairs=info, acc=rep,
           geometry=str(st.nb.force_geometry(d.N)))
    assert ex <= x_tol and ev <= x_tol, f"{what}: state differs from the oracle run: x {ex:.3g}, v {ev:.3g}"
    assert abs(de_g - de_r) <= ENERGY_TOL, f"{what}: energy error gpu {de_g:.3e} vs oracle {de_r:.3e}"
    assert dL <= 1e-12
    assert rep["ratio_with_backward_term"] <= 1.0, rep


def test_config4_full_semi_active_100_steps():
    """BASELINE.json:configs[3]: N = 131072 with 1024 active embryos, dt = 6 d, 100 steps."""
    _trajectory_vs_oracle(3, "config4 x100", 1e-9)


@pytest.mark.slow
def test_config2_full_1000_steps():
    """BASELINE.json:configs[1]: N = 16384 + 2 giants, dt = 6 d, 1000 steps -- "after 1000 steps, relative energy error
    must stay within 1e-9 of the oracle run"."""
    _trajectory_vs_oracle(1, "config2 x1000", 1e-7)


def _trajectory_vs_golden(k, x_tol_all, x_tol_most):
    path = os.path.join(_GOLDEN, f"config{k + 1}_trajectory.txt")
    assert os.path.exists(path), f"{path} is missing: run python -m oracle.make_golden --config {k}"
    g = make_golden.load(path)
    d = nb_inputs.make_config(k)
    assert make_golden.input_sha(d) == g["input_sha256"], "the generator no longer produces the input the golden run started from"
    nsteps = int(g["nsteps"])
    assert nsteps == d.nsteps and float(g["n1"]) == 3.0 and float(g["n2"]) == 0.0 and int(g["kepler_fail"]) == 0
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.0, pair_capacity=1 << 22)
    legs = int(g.get("legs", 1))      # a golden run written in legs is `legs` consecutive calls (oracle/make_golden.py)
    for _ in range(legs):
        st.step(d.dt, nsteps // legs)
    xg, vg, accg, rcg = st.host()
    status = st.nb.nb_status()
    assert status["kepler_fail"] == 0 and status["pairs_dropped"] == 0
    E0 = oracle.diagnostics(d.x, d.v, d.m, d.M_star, G_GAUSS)
    Eg = oracle.diagnostics(xg, vg, d.m, d.M_star, G_GAUSS)
    assert E0["E"] == float(g["E0"])                     # same diagnostic, same input: bit for bit
    de_g = (Eg["E"] - E0["E"]) / E0["E"]
    de_r = float(g["dE_over_E"])
    dL = np.linalg.norm(Eg["L"] - np.array(g["L1"])) / np.linalg.norm(np.array(g["L1"]))
    rows = g["row_index"]
    scale_x = np.linalg.norm(g["x"], axis=1, keepdims=True)
    scale_v = np.linalg.norm(g["v"], axis=1, keepdims=True)
    scale_a = np.linalg.norm(g["acc"], axis=1, keepdims=True)
    ex = np.max(np.abs(xg[rows] - g["x"]) / scale_x, axis=1)
    ev = np.max(np.abs(vg[rows] - g["v"]) / scale_v, axis=1)
    ea = np.max(np.abs(accg[rows] - g["acc"]) / scale_a, axis=1)
    gp, n = st.get_pairs()
    cg = canon_pairs(gp)
    sha = hashlib.sha256(np.ascontiguousarray(cg, dtype=np.int32).tobytes()).hexdigest()
    record(check="trajectory_vs_golden", config=k + 1, name=d.name, N=d.N, nsteps=nsteps, dE_gpu=de_g, dE_oracle=de_r,
           dE_diff=abs(de_g - de_r), dL_vs_oracle=dL, rows=int(rows.size), rel_dx_max=float(ex.max()), rel_dx_median=float(np.median(ex)),
           rel_dv_max=float(ev.max()), rel_dacc_max=float(ea.max()), rel_dacc_median=float(np.median(ea)),
           pairs_gpu=int(n), pairs_oracle=int(g["pairs_sure"]), pairs_borderline=int(g["pairs_borderline"]),
           pair_list_identical=(sha == g["pairs_sha256"]), geometry=str(st.nb.force_geometry(d.N)))
    assert abs(de_g - de_r) <= ENERGY_TOL, f"energy error gpu {de_g:.3e} vs oracle {de_r:.3e}"
    assert dL <= 1e-12
    # states: every sampled row within x_tol_all, 99 % of them within x_tol_most (bodies inside an encounter amplify
    # the last-bit differences of the two runs; the rest follows them to ~1e-12)
    assert ex.max() <= x_tol_all and ev.max() <= x_tol_all
    assert np.quantile(ex, 0.99) <= x_tol_most and np.quantile(ev, 0.99) <= x_tol_most
    assert np.quantile(ea, 0.99) <= 100 * x_tol_most
    # pair list of the final evaluation: same pairs unless a pair sits within the trajectories' difference of its radius
    assert abs(int(n) - int(g["pairs_sure"])) <= 2 + int(g["pairs_borderline"])
    # and it is exactly the list of the GPU's own final state (complete, no duplicates)
    if d.N <= 65536:
        sure, border = oracle.pairs(xg, rcg)
        assert_pairs_match(gp, n, sure, border, f"config{k + 1} final pairs")


def test_config3_full_200_steps_against_golden():
    """BASELINE.json:configs[2]: N = 65536 ring, dt = 3 d, 200 steps (the bench workload)."""
    _trajectory_vs_golden(2, 1e-6, 1e-9)


@pytest.mark.slow
def test_config5_full_10_steps_against_golden():
    """BASELINE.json:configs[4]: N = 524288, dt = 3 d, 10 steps."""
    _trajectory_vs_golden(4, 1e-9, 1e-11)


# ------------------------------------------------------------------------------------------ complete pair lists
@pytest.mark.parametrize("n2", [0.0, 0.4])
def test_complete_pair_list_and_all_rows_config3(n2):
    """N = 65536 in the bench configuration (Newton-III kernel, S = 512, I = 4, sorted staging with test-free far tiles):
    EVERY row's acceleration and the COMPLETE pair list against the oracle -- a wrong arcs_are_far decision would lose
    pairs here."""
    d = nb_inputs.make_config(2)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, n2)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=n2, pair_capacity=1 << 23)
    geo = st.nb.force_geometry(d.N)
    assert geo.tile_j == -512 and geo.i_per_thread == 4          # the configuration bench.py times
    st.set_rcrit(rc)
    st.kick(0.0)
    acc = st.acc.cpu().numpy()
    gp, n = st.get_pairs()
    sure, border = oracle.pairs(d.x, rc, cap=1 << 23)
    info = assert_pairs_match(gp, n, sure, border, f"config3 n2={n2} complete pair list")
    acc_ref, ab, _ = oracle.accel(d.x, d.m, rc, G_GAUSS, want_abs=True)
    rep = _acc_report(acc, acc_ref, ab)
    record(check="all_rows_complete_pairs", config=3, N=d.N, n2=n2, pairs=info, acc=rep, geometry=str(geo))
    assert rep["ratio_with_backward_term"] <= 1.0, rep
    assert info["n_sure"] > (1000 if n2 == 0.0 else 1000000)


@pytest.mark.slow
@pytest.mark.parametrize("cfg", [4, 3])
def test_complete_pair_list_large_configs_by_kdtree(cfg):
    """N = 524288 (config 5) and N = 131072 semi-active (config 4): the COMPLETE pair list against an independent route --
    scipy's cKDTree.query_pairs(max rc) followed by the max-radius rule r_ij < max(rc_i, rc_j) (strict, same fp64
    expression for r^2 as the definition) -- which none of the oracle's O(N^2) loops could afford on every row."""
    d = nb_inputs.make_config(cfg)
    na = d.n_active if d.n_active < d.N else 0
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, 0.0)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n_active=na, n1=3.0, n2=0.0, pair_capacity=1 << 22)
    st.set_rcrit(rc)
    st.kick(0.0)
    gp, n = st.get_pairs()
    cand = cKDTree(d.x).query_pairs(float(rc.max()) * (1 + 1e-9), output_type="ndarray")
    i, j = cand[:, 0], cand[:, 1]
    dx = d.x[j] - d.x[i]
    r2 = (dx[:, 0] * dx[:, 0] + dx[:, 1] * dx[:, 1]) + dx[:, 2] * dx[:, 2]
    rc2 = np.maximum(rc[i], rc[j]) ** 2
    keep = (r2 < rc2 * (1 - 2e-12))
    edge = ~keep & (np.abs(r2 / np.where(rc2 > 0, rc2, 1.0) - 1.0) <= 2e-12) & (rc2 > 0)
    if na:
        act = np.minimum(i, j) < na
        keep &= act
        edge &= act
    sure = canon_pairs(np.stack([np.minimum(i, j), np.maximum(i, j)], axis=1)[keep])
    border = canon_pairs(np.stack([np.minimum(i, j), np.maximum(i, j)], axis=1)[edge])
    info = assert_pairs_match(gp, n, sure, border, f"{d.name} complete pair list (cKDTree)")
    record(check="complete_pairs_kdtree", config=cfg + 1, N=d.N, pairs=info, geometry=str(st.nb.force_geometry(d.N)))
    assert info["n_sure"] > 100


# ------------------------------------------------------------------------------------------ host-buffer entry points
def test_step_host_and_kick_host_match_the_oracle():
    """nb_step_host / nb_kick_host (HOST pointers; the e2e leg of bench.py): 3 steps as 1 + 2 with reuse_acc chaining,
    rcrit == NULL, a pair buffer that overflows, against oracle.step / oracle.accel / oracle.pairs."""
    import paper_2604_09184_b200 as nb
    d = nb_inputs.make_config(1, n_override=3000)           # config-2 shape with both giants; ragged tile tail
    N = d.N
    cap = 1 << 16
    ref = oracle.step(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3, n1=3.0, n2=0.4)
    x, v, m = d.x.copy(), d.v.copy(), d.m.copy()
    rc = np.zeros(N); acc = np.zeros((N, 3)); pairs = np.full((cap, 2), -1, dtype=np.int32); npairs = np.zeros(1, dtype=np.int64)
    nb.nb_release()                                         # a fresh private arena: its status words start at zero
    nb.configure(None, pair_capacity=cap, G=G_GAUSS, n1=3.0, n2=0.4)
    nb.nb_step_host(x, v, m, d.M_star, d.dt, rc, acc, pairs, npairs, 1)
    nb.configure(None, pair_capacity=cap, G=G_GAUSS, n1=3.0, n2=0.4, reuse_acc=True)     # acc, rc, pairs of the last call are reused
    nb.nb_step_host(x, v, m, d.M_star, d.dt, rc, acc, pairs, npairs, 2)
    ex = np.max(np.abs(x - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(v - ref["v"])) / np.max(np.abs(ref["v"]))
    assert ex <= 1e-13 and ev <= 1e-13, (ex, ev)
    assert np.max(np.abs(rc - ref["rcrit"]) / ref["rcrit"]) <= 1e-12
    acc_ref, ab, _ = oracle.accel(x, m, rc, G_GAUSS, want_abs=True)
    assert_acc_close(acc, acc_ref, "nb_step_host final acc", ab)
    sure, border = oracle.pairs(x, rc)
    n = int(npairs[0])
    assert n > 50
    assert_pairs_match(pairs[:n], n, sure, border, "nb_step_host final pairs")
    status = nb.nb_status()
    assert status["kepler_fail"] == 0 and status["pairs_dropped"] == 0

    # rcrit == NULL in nb_step_host: neither read nor returned; same trajectory
    x2, v2 = d.x.copy(), d.v.copy()
    acc2 = np.zeros((N, 3))
    nb.configure(None, pair_capacity=cap, G=G_GAUSS, n1=3.0, n2=0.4)
    nb.nb_step_host(x2, v2, m, d.M_star, d.dt, None, acc2, pairs, npairs, 3)
    assert np.max(np.abs(x2 - ref["x"])) <= 1e-13 * np.max(np.abs(ref["x"])) and np.max(np.abs(v2 - ref["v"])) <= 1e-13 * np.max(np.abs(ref["v"]))

    # nb_kick_host: caller's rcrit, dt != 0, then rcrit == NULL (a0 inside), then an overflowing pair buffer
    rc_in = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, 0.4)
    vk = d.v.copy(); acck = np.zeros((N, 3))
    nb.nb_kick_host(d.x, vk, m, d.M_star, 0.5 * d.dt, rc_in, acck, pairs, npairs)
    v_ref, acc_ref = oracle.kick(d.x, d.v, m, 0.5 * d.dt, rc_in, G_GAUSS)
    _, ab, _ = oracle.accel(d.x, m, rc_in, G_GAUSS, want_abs=True)
    assert_acc_close(acck, acc_ref, "nb_kick_host acc", ab)
    assert np.max(np.abs(vk - v_ref)) <= 1e-12 * np.max(np.abs(v_ref))
    sure, border = oracle.pairs(d.x, rc_in)
    n_full = int(npairs[0])
    assert_pairs_match(pairs[:n_full], n_full, sure, border, "nb_kick_host pairs")
    vk2 = d.v.copy(); acck2 = np.zeros((N, 3))
    nb.nb_kick_host(d.x, vk2, m, d.M_star, 0.5 * d.dt, None, acck2, pairs, npairs)     # rcrit by a0 with dt = 0.5 d.dt
    rc_half = oracle.rcrit(d.x, d.v, d.m, d.M_star, 0.5 * d.dt, G_GAUSS, 3.0, 0.4)
    acc_ref2, ab2, _ = oracle.accel(d.x, m, rc_half, G_GAUSS, want_abs=True)
    assert_acc_close(acck2, acc_ref2, "nb_kick_host acc (rcrit NULL)", ab2)
    small = 16
    nb.configure(None, pair_capacity=small, G=G_GAUSS, n1=3.0, n2=0.4)
    nb.nb_status_reset()
    ps = np.full((small, 2), -1, dtype=np.int32)
    vk3 = d.v.copy()
    nb.nb_kick_host(d.x, vk3, m, d.M_star, 0.0, rc_in, acck, ps, npairs)
    assert int(npairs[0]) == n_full and nb.nb_status()["pairs_dropped"] == n_full - small
    keys = set(map(tuple, sure.tolist())) | set(map(tuple, border.tolist()))
    assert all(tuple(p) in keys for p in ps.tolist()) and len({tuple(p) for p in ps.tolist()}) == small
    assert np.array_equal(vk3, d.v)
    nb.nb_release()


def test_step_host_through_the_newton3_kernel_banded_and_not():
    """nb_step_host with the Newton-III kernel forced (sorted staging, tail splitting) and with the banded evaluation on top
    (nb_config.slot_bytes_max forced down): the private arena is sized by nb_workspace_bytes for either geometry; same
    trajectory as oracle.step, same final pair list."""
    import paper_2604_09184_b200 as nb
    d = nb_inputs.make_config(1, n_override=3000)
    N, cap = d.N, 1 << 16
    ref = oracle.step(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3, n1=3.0, n2=0.4)
    sure, border = oracle.pairs(ref["x"], ref["rcrit"])
    npad = -(-N // 128) * 128
    for slot_cap in (0, 24 * (N + npad) * 4 + 8):
        x, v = d.x.copy(), d.v.copy()
        rc = np.zeros(N); acc = np.zeros((N, 3)); pairs = np.full((cap, 2), -1, dtype=np.int32); npairs = np.zeros(1, dtype=np.int64)
        nb.nb_release()
        nb.configure(None, pair_capacity=cap, G=G_GAUSS, n1=3.0, n2=0.4, force_kernel=2, sym_block=128, sort_staging=1,
                     slot_bytes_max=slot_cap)
        nb.nb_step_host(x, v, d.m, d.M_star, d.dt, rc, acc, pairs, npairs, 3)
        ex = np.max(np.abs(x - ref["x"])) / np.max(np.abs(ref["x"]))
        ev = np.max(np.abs(v - ref["v"])) / np.max(np.abs(ref["v"]))
        assert ex <= 1e-13 and ev <= 1e-13, (slot_cap, ex, ev)
        n = int(npairs[0])
        assert_pairs_match(pairs[:n], n, sure, border, f"nb_step_host Newton-III, slot cap {slot_cap}")
        acc_ref, ab, _ = oracle.accel(x, d.m, rc, G_GAUSS, want_abs=True)
        assert_acc_close(acc, acc_ref, f"nb_step_host Newton-III acc, slot cap {slot_cap}", ab)
        assert nb.nb_status()["kepler_fail"] == 0 and nb.nb_status()["pairs_dropped"] == 0
    nb.nb_release()
