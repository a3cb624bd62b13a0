"""-m gpu: nb_kick_static (include/nbkick.h) -- the kick with its scratch in the library's static device array, for
callers that cannot allocate -- against the existing path (nb_kick with the caller-owned workspace), on two calls in a
row that share the array.  Collected last on purpose (pytest -x): a failure here hides nothing.
Passes alone in a fresh process and after the other tests (it configures the library itself)."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import GpuState, assert_acc_close, assert_pairs_match, canon_pairs, torch_mod

pytestmark = pytest.mark.gpu


def _both_paths(d, n1, n2, dt, what):
    """nb_kick (workspace of nb_configure) and nb_kick_static (static array) on the same input; returns the static
    call's accelerations.  Tolerance: the acceleration allowance of tests/gpu_util.py with the existing path as the
    reference (the two run the same kernels in the same geometry, so they agree bit for bit: asserted as well)."""
    torch = torch_mod()
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, n1, n2)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=n1, n2=n2, pair_capacity=1 << 18)
    st.set_rcrit(rc)
    st.kick(dt)
    _, v_ref, acc_ref, _ = st.host()
    p_ref, n_ref = st.get_pairs()
    # the new entry point: fresh outputs, same inputs; the configured workspace is poisoned first to show it is not used
    nb = st.nb
    x = torch.from_numpy(d.x).cuda(); v = torch.from_numpy(d.v).cuda(); m = torch.from_numpy(d.m).cuda()
    rcd = torch.from_numpy(rc).cuda()
    acc = torch.full((d.N, 3), float("nan"), dtype=torch.float64, device="cuda")
    pairs = torch.full((1 << 18, 2), -1, dtype=torch.int32, device="cuda")
    npairs = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    status8 = torch.full((8,), -1, dtype=torch.int64, device="cuda")
    before = torch.cuda.memory_allocated()
    nb.nb_kick_static(x, v, m, d.M_star, dt, rcd, acc, pairs, npairs, status8)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    acc_s, v_s = acc.cpu().numpy(), v.cpu().numpy()
    assert_acc_close(acc_s, acc_ref, what + ": static scratch vs workspace path")
    assert np.array_equal(acc_s, acc_ref) and np.array_equal(v_s, v_ref), what + ": same kernels, same geometry"
    n = int(npairs.item())
    assert n == n_ref
    assert np.array_equal(canon_pairs(pairs[:n].cpu().numpy()), canon_pairs(p_ref))
    assert status8.cpu().tolist() == [0] * 8
    # and against the oracle, like every other kick test
    a_or, ab, _ = oracle.accel(d.x, d.m, rc, G_GAUSS, want_abs=True)
    assert_acc_close(acc_s, a_or, what + ": static scratch vs oracle", ab)
    sure, border = oracle.pairs(d.x, rc)
    assert_pairs_match(pairs[:n].cpu().numpy(), n, sure, border, what)
    return n


def test_static_scratch_kick_two_calls_in_a_row():
    import paper_2604_09184_b200 as nb
    nb.nb_kick_static_setup()
    # first call: N = 4096 (Newton-III kernel, 6.0 MB of the 8 MiB array), dense pairs;
    # second call: config 1 in full (N = 2048, one-sided kernel, another carving of the same bytes), few pairs --
    # the array still holds the first call's slots, staged bodies and counters
    d1 = nb_inputs.make_config(2, n_override=4096)
    n_first = _both_paths(d1, 3.0, 0.4, 0.5 * d1.dt, "N=4096 ring, Eq. 7 radius")
    d2 = nb_inputs.make_config(0)
    n_second = _both_paths(d2, 3.0, 0.0, 0.5 * d2.dt, "config 1, 3 R_Hill")
    assert n_first > 100 and n_second < n_first
    # and the first input once more: identical to its first run (nothing of call two leaks into call three)
    assert _both_paths(d1, 3.0, 0.4, 0.5 * d1.dt, "N=4096 ring again") == n_first


def test_static_scratch_counters_belong_to_the_call():
    """Device-side conditions are counted in the static array and handed out per call: a pair list that overflows in
    one call leaves nothing behind for the next."""
    torch = torch_mod()
    d = nb_inputs.make_config(2, n_override=3000)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 30.0, 0.0)
    sure, border = oracle.pairs(d.x, rc)
    cap = 64
    assert sure.shape[0] > cap
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, pair_capacity=cap)
    acc = torch.zeros((d.N, 3), dtype=torch.float64, device="cuda")
    npairs = torch.zeros(1, dtype=torch.int64, device="cuda")
    status8 = torch.zeros(8, dtype=torch.int64, device="cuda")
    rcd = torch.from_numpy(rc).cuda()
    st.nb.nb_kick_static(st.x, st.v, st.m, d.M_star, 0.0, rcd, acc, st.pairs, npairs, status8)
    torch.cuda.synchronize()
    n = int(npairs.item())
    assert sure.shape[0] <= n <= sure.shape[0] + border.shape[0]
    assert int(status8[0].item()) == n - cap                      # pairs dropped, this call
    st.nb.nb_kick_static(st.x, st.v, st.m, d.M_star, 0.0, rcd, acc, None, None, status8)
    torch.cuda.synchronize()
    assert status8.cpu().tolist() == [0] * 8                      # no detection, nothing dropped, nothing left over
    assert st.nb.nb_status()["pairs_dropped"] == 0                # the configured workspace never saw either call


def test_static_scratch_rejects_sizes_beyond_the_array():
    import paper_2604_09184_b200 as nb
    torch = torch_mod()
    N = 16384
    assert nb.workspace_bytes(N) > (8 << 20)
    d = nb_inputs.make_config(0, n_override=N)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS)
    acc = torch.full((N, 3), 5.0, dtype=torch.float64, device="cuda")
    with pytest.raises(nb.NbError) as e:
        nb.nb_kick_static(st.x, st.v, st.m, d.M_star, 0.0, st.rcrit, acc)
    assert e.value.code == nb.binding.NB_E_WORKSPACE
    assert "NB_STATIC_SCRATCH_BYTES" in str(e.value) and "8388608" in str(e.value)
    torch.cuda.synchronize()
    assert float(acc.min().item()) == 5.0 and float(acc.max().item()) == 5.0     # nothing was launched
