"""-m gpu parity of the Newton-III force kernel (force_sym.cuh; nb_config.force_kernel =
NB_FORCE_SYMMETRIC) against the CPU oracle: same bar as the one-sided kernel (test_gpu_kick.py) --
accelerations within the north_star tolerance, pair lists bit-exact after the canonical sort.
Sizes straddle the super-block size S, the 128*I chunk and the 32-body rotation block; the
diagonal ("mixed") blocks, the padding bodies and the deferred exact pass are all exercised."""
import numpy as np
import pytest

import nb_inputs
import oracle
from nb_inputs import G_GAUSS

from gpu_util import GpuState, assert_acc_close, assert_pairs_match
from test_gpu_kick import _kick_case

pytestmark = pytest.mark.gpu

SYM = 2  # NB_FORCE_SYMMETRIC


def _geometry_is_symmetric(N):
    import paper_2604_09184_b200 as nb
    return nb.force_geometry(N).tile_j < 0


@pytest.mark.parametrize("ipt,S", [(1, 256), (2, 256), (2, 512), (4, 512), (4, 1024), (4, 128), (4, 256), (2, 128), (1, 128)])
@pytest.mark.parametrize("N", [1, 2, 31, 32, 33, 255, 256, 257, 700, 1100])
def test_sym_random_cluster_newtonian(N, ipt, S):
    x, v, m = nb_inputs.random_cluster(N, seed=100 + N)
    info = _kick_case(x, v, m, np.zeros(N), force_kernel=SYM, i_per_thread=ipt, sym_block=S,
                      what=f"sym cluster N={N} I={ipt} S={S}")
    assert _geometry_is_symmetric(N)
    assert info["n_gpu"] == 0


@pytest.mark.parametrize("kind", [0, 1])
@pytest.mark.parametrize("ipt,S", [(1, 256), (2, 256), (4, 512), (4, 128), (4, 256), (2, 128)])
def test_sym_cluster_with_changeover_and_pairs(kind, ipt, S):
    N = 1000
    x, v, m = nb_inputs.random_cluster(N, seed=5, scale=0.2)
    rng = np.random.default_rng(9)
    rc = rng.uniform(0.0, 0.06, N)
    rc[::7] = 0.0
    info = _kick_case(x, v, m, rc, kind=kind, dt=0.37, force_kernel=SYM, i_per_thread=ipt, sym_block=S,
                      what=f"sym changeover kind={kind} I={ipt} S={S}")
    assert info["n_sure"] > 300


@pytest.mark.parametrize("ipt,S", [(2, 256), (4, 512), (4, 128), (4, 256)])
def test_sym_chain_lattice_and_all_pairs(ipt, S):
    tune = dict(force_kernel=SYM, i_per_thread=ipt, sym_block=S)
    N = 300
    x, v, m = nb_inputs.chain_1d(N)
    for rcv, expect in ((1.5, N - 1), (2.5, 2 * N - 3)):
        info = _kick_case(x, v, m, np.full(N, rcv), G=1.0, what=f"sym chain rc={rcv}", **tune)
        assert info["n_gpu"] == expect
    n = 7
    x, v, m = nb_inputs.cubic_lattice(n)
    info = _kick_case(x, v, m, np.full(n ** 3, 1.2), G=1.0, what="sym lattice", **tune)
    assert info["n_gpu"] == 3 * n * n * (n - 1)
    # every pair inside every critical radius: the deferred exact pass does all the work
    N = 333
    x, v, m = nb_inputs.random_cluster(N, seed=17, scale=0.05)
    info = _kick_case(x, v, m, np.full(N, 10.0), what="sym all pairs", pair_capacity=1 << 17, **tune)
    assert info["n_gpu"] == N * (N - 1) // 2


@pytest.mark.parametrize("ipt,S", [(1, 256), (4, 512), (4, 128), (4, 256)])
def test_sym_coincident_bodies(ipt, S):
    tune = dict(force_kernel=SYM, i_per_thread=ipt, sym_block=S)
    x, v, m = nb_inputs.random_cluster(300, seed=3)
    x[7] = x[21]      # same 32-block (mixed visit)
    x[40] = x[290]    # different blocks (symmetric visit)
    rc = np.full(300, 0.01)
    info = _kick_case(x, v, m, rc, what="sym coincident rc>0", **tune)
    assert info["n_gpu"] >= 2
    _kick_case(x, v, m, np.zeros(300), what="sym coincident rc=0", **tune)  # checks the singular count


@pytest.mark.parametrize("cfg,n_override", [(0, 2048), (1, 3000), (2, 4096), (4, 5000)])
@pytest.mark.parametrize("n1,n2", [(3.0, 0.0), (3.0, 0.4), (30.0, 0.0)])
def test_sym_disk_configs_reduced(cfg, n_override, n1, n2):
    d = nb_inputs.make_config(cfg, n_override=n_override)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, n1, n2)
    info = _kick_case(d.x, d.v, d.m, rc, dt=0.5 * d.dt, force_kernel=SYM, what=f"sym {d.name} n1={n1} n2={n2}")
    assert _geometry_is_symmetric(d.N)
    if n1 == 30.0 or n2 > 0:
        assert info["n_sure"] > 0


def test_sym_semi_active_falls_back_to_tiles():
    import paper_2604_09184_b200 as nb
    d = nb_inputs.make_config(3, n_override=4096)
    assert d.n_active < d.N
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, 0.4)
    _kick_case(d.x, d.v, d.m, rc, n_active=d.n_active, force_kernel=SYM, what="sym requested, semi-active")
    assert nb.force_geometry(d.N).tile_j > 0  # a passive body has no second side to serve


def test_sym_bitwise_reproducible_and_close_to_tiles():
    d = nb_inputs.make_config(2, n_override=6000)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, 0.4)
    out = []
    for fk in (SYM, SYM, 1):
        st = GpuState(d.x, d.v, d.m, G=G_GAUSS, force_kernel=fk)
        st.set_rcrit(rc)
        st.kick(0.0)
        gp, n = st.get_pairs()
        out.append((st.acc.cpu().numpy().copy(), {tuple(p) for p in gp.tolist()}))
    assert np.array_equal(out[0][0], out[1][0]), "the symmetric kernel is not run-to-run reproducible"
    assert out[0][1] == out[1][1] == out[2][1]
    scale = np.linalg.norm(out[2][0], axis=1, keepdims=True)
    assert np.max(np.abs(out[0][0] - out[2][0]) / scale) < 1e-12


@pytest.mark.parametrize("nsteps", [1, 3, 100])
def test_sym_step_matches_oracle(nsteps):
    d = nb_inputs.make_config(1, n_override=1498)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, force_kernel=SYM, sym_block=256)
    st.step(d.dt, nsteps)
    xg, vg, ag, rcg = st.host()
    ref = oracle.step(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, nsteps, n1=3.0, n2=0.4)
    tol = 1e-13 if nsteps <= 3 else 1e-9
    assert np.max(np.abs(xg - ref["x"])) <= tol * np.max(np.abs(ref["x"]))
    assert np.max(np.abs(vg - ref["v"])) <= tol * np.max(np.abs(ref["v"]))
    acc_ref, ab, _ = oracle.accel(xg, d.m, rcg, G_GAUSS, want_abs=True)
    assert_acc_close(ag, acc_ref, f"sym step x{nsteps}: final acc", ab)
    sure, border = oracle.pairs(xg, rcg)
    gp, n = st.get_pairs()
    assert_pairs_match(gp, n, sure, border, f"sym step x{nsteps}")
    D0 = oracle.diagnostics(d.x, d.v, d.m, d.M_star, G_GAUSS)
    Dg = oracle.diagnostics(xg, vg, d.m, d.M_star, G_GAUSS)
    Dr = oracle.diagnostics(ref["x"], ref["v"], d.m, d.M_star, G_GAUSS)
    assert abs((Dg["E"] - D0["E"]) / D0["E"] - (Dr["E"] - D0["E"]) / D0["E"]) <= 1e-9


def test_sym_pair_overflow_counts_and_null_pairs():
    N = 900
    x, v, m = nb_inputs.random_cluster(N, seed=11, scale=0.1)
    rc = np.full(N, 0.05)
    sure, border = oracle.pairs(x, rc)
    acc_ref, ab, _ = oracle.accel(x, m, rc, G_GAUSS, want_abs=True)
    st = GpuState(x, v, m, G=G_GAUSS, pair_capacity=100, force_kernel=SYM, sym_block=256, i_per_thread=2)
    st.set_rcrit(rc)
    st.kick(0.0, with_pairs=False)                       # pairs = NULL: detection skipped, weights still applied
    assert_acc_close(st.acc.cpu().numpy(), acc_ref, "sym pairs=NULL", ab)
    st.kick(0.0, with_pairs=True)
    gp, n = st.get_pairs()
    assert sure.shape[0] <= n <= sure.shape[0] + border.shape[0] and n > 100
    assert gp.shape[0] == 100 and st.nb.nb_status()["pairs_dropped"] == n - 100
    assert_acc_close(st.acc.cpu().numpy(), acc_ref, "sym overflow", ab)
    allowed = {tuple(p) for p in np.concatenate([sure, border]).tolist()}
    assert all(tuple(p) in allowed for p in gp.tolist())


def test_sym_everything_in_the_exact_path_at_larger_n():
    """rc larger than the cluster: every one of the N(N-1)/2 pairs goes through the deferred exact pass."""
    N = 1500
    x, v, m = nb_inputs.random_cluster(N, seed=23, scale=0.05)
    info = _kick_case(x, v, m, np.full(N, 10.0), force_kernel=SYM, sym_block=512, i_per_thread=4,
                      pair_capacity=1 << 21, what="sym all pairs N=1500")
    assert info["n_gpu"] == N * (N - 1) // 2


def test_auto_selection_threshold():
    import paper_2604_09184_b200 as nb
    for N, want_sym in ((4095, False), (4096, True)):
        nb.configure(N, G=G_GAUSS)
        assert (nb.force_geometry(N).tile_j < 0) == want_sym
    d = nb_inputs.make_config(1, n_override=4100)        # just above the threshold, ragged: N = 4102
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 3.0, 0.4)
    rows = np.unique(np.concatenate([np.arange(0, d.N, 97), [d.N - 1, d.N - 2]]))
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, pair_capacity=1 << 20)
    assert _geometry_is_symmetric(d.N)
    st.set_rcrit(rc)
    st.kick(0.0)
    acc_ref, ab, _ = oracle.accel(d.x, d.m, rc, G_GAUSS, rows=rows, want_abs=True)
    assert_acc_close(st.acc.cpu().numpy()[rows], acc_ref, "auto sym N=4102 sampled rows", ab)
    sure, border = oracle.pairs(d.x, rc)
    gp, n = st.get_pairs()
    assert_pairs_match(gp, n, sure, border, "auto sym N=4102")


@pytest.mark.parametrize("seed", range(16))
def test_sym_randomized_shapes_against_oracle(seed):
    """Random N, mass spectrum, clustering and critical radii (including zero radii, a few huge ones and test
    particles): both force kernels against the oracle, same pair list from both."""
    rng = np.random.default_rng(1000 + seed)
    N = int(rng.integers(2, 1400))
    scale = float(rng.choice([0.02, 0.2, 2.0]))
    x, v, m = nb_inputs.random_cluster(N, seed=seed, scale=scale)
    m = m * rng.choice([0.0, 1.0, 1.0, 30.0], size=N)            # test particles and a few heavy bodies
    rc = rng.uniform(0.0, 0.08 * scale, N) * rng.choice([0.0, 1.0, 1.0, 1.0], size=N)
    big = rng.choice(N, size=max(1, N // 200), replace=False)
    rc[big] = 0.5 * scale                                         # a "giant": large radius next to small ones
    ipt = int(rng.choice([1, 2, 4])); S = int(rng.choice([256, 512, 1024]))
    kind = int(rng.integers(0, 2))
    info_s = _kick_case(x, v, m, rc, kind=kind, force_kernel=SYM, i_per_thread=ipt, sym_block=S,
                        what=f"random seed={seed} N={N} I={ipt} S={S} (Newton III)")
    info_t = _kick_case(x, v, m, rc, kind=kind, force_kernel=1, what=f"random seed={seed} N={N} (one-sided)")
    assert info_s["n_gpu"] == info_t["n_gpu"]


# ---- sorted staging (sort_staging.cuh): the staged bodies are permuted into azimuthal order; everything the caller
# sees (accelerations, pair indices, velocities) must be unchanged up to the summation order ----------------------
SORT = dict(force_kernel=SYM, sort_staging=1)


@pytest.mark.parametrize("ipt,S", [(1, 256), (2, 256), (4, 512), (4, 128), (4, 256)])
@pytest.mark.parametrize("N", [1, 2, 33, 257, 700, 1100])
def test_sorted_staging_cluster_with_changeover_and_pairs(N, ipt, S):
    x, v, m = nb_inputs.random_cluster(N, seed=300 + N, scale=0.2)
    rng = np.random.default_rng(N)
    rc = rng.uniform(0.0, 0.06, N)
    rc[::7] = 0.0
    _kick_case(x, v, m, rc, dt=0.37, i_per_thread=ipt, sym_block=S, what=f"sorted N={N} I={ipt} S={S}", **SORT)


def test_sorted_staging_counts_coincident_and_all_pairs():
    N = 300
    x, v, m = nb_inputs.chain_1d(N)
    for rcv, expect in ((1.5, N - 1), (2.5, 2 * N - 3)):
        assert _kick_case(x, v, m, np.full(N, rcv), G=1.0, what=f"sorted chain rc={rcv}", **SORT)["n_gpu"] == expect
    x, v, m = nb_inputs.cubic_lattice(7)
    assert _kick_case(x, v, m, np.full(343, 1.2), G=1.0, what="sorted lattice", **SORT)["n_gpu"] == 3 * 49 * 6
    x, v, m = nb_inputs.random_cluster(300, seed=3)
    x[7] = x[21]; x[40] = x[290]
    assert _kick_case(x, v, m, np.full(300, 0.01), what="sorted coincident rc>0", **SORT)["n_gpu"] >= 2
    _kick_case(x, v, m, np.zeros(300), what="sorted coincident rc=0", **SORT)
    N = 700
    x, v, m = nb_inputs.random_cluster(N, seed=23, scale=0.05)
    assert _kick_case(x, v, m, np.full(N, 10.0), what="sorted all pairs", pair_capacity=1 << 19, **SORT)["n_gpu"] == N * (N - 1) // 2


@pytest.mark.parametrize("cfg,n_override,n1,n2", [(0, 2048, 3.0, 0.4), (1, 3000, 3.0, 0.4), (2, 4096, 30.0, 0.0), (4, 5000, 3.0, 0.0)])
def test_sorted_staging_disk_configs_reduced(cfg, n_override, n1, n2):
    """Disks are where the order matters: most super-tiles skip the test, the near-diagonal ones and the ones that hold a
    giant planet (critical radius ~1 AU) do not."""
    d = nb_inputs.make_config(cfg, n_override=n_override)
    rc = oracle.rcrit(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, n1, n2)
    for S in (256, 512):
        info = _kick_case(d.x, d.v, d.m, rc, dt=0.5 * d.dt, sym_block=S, what=f"sorted {d.name} S={S}", **SORT)
        assert info["n_sure"] > 0


@pytest.mark.parametrize("nsteps", [3, 100])
def test_sorted_staging_step_matches_oracle_and_is_reproducible(nsteps):
    d = nb_inputs.make_config(1, n_override=1498)
    out = []
    for _ in range(2):
        st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, sym_block=256, **SORT)
        st.step(d.dt, nsteps)
        out.append(st.host())
    assert all(np.array_equal(a, b) for a, b in zip(out[0], out[1])), "sorted staging is not run-to-run reproducible"
    xg, vg, ag, rcg = out[0]
    ref = oracle.step(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, nsteps, n1=3.0, n2=0.4)
    tol = 1e-13 if nsteps <= 3 else 1e-9
    assert np.max(np.abs(xg - ref["x"])) <= tol * np.max(np.abs(ref["x"]))
    assert np.max(np.abs(vg - ref["v"])) <= tol * np.max(np.abs(ref["v"]))
    acc_ref, ab, _ = oracle.accel(xg, d.m, rcg, G_GAUSS, want_abs=True)
    assert_acc_close(ag, acc_ref, f"sorted step x{nsteps}: final acc", ab)
    sure, border = oracle.pairs(xg, rcg)
    gp, n = st.get_pairs()
    assert_pairs_match(gp, n, sure, border, f"sorted step x{nsteps}")


def test_sorted_staging_with_encounters_resolved():
    d = nb_inputs.make_config(1, n_override=900)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, resolve_encounters=True, pair_capacity=1 << 16,
                  sym_block=256, **SORT)
    st.step(d.dt, 10)
    xg, vg, _, _ = st.host()
    ref = oracle.step_enc(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 10, n1=3.0, n2=0.4)
    assert ref["stats"]["integrated"] > 0
    assert np.max(np.abs(xg - ref["x"])) <= 1e-9 * np.max(np.abs(ref["x"]))
    assert np.max(np.abs(vg - ref["v"])) <= 1e-9 * np.max(np.abs(ref["v"]))


# ---- banded evaluation (nb_config.slot_bytes_max): the tile columns in several launches, folded into acc band by band

def _band_cap(N, S, band):
    """slot_bytes_max that yields `band` tile columns per launch (24 (N + Npad) bytes per column)"""
    npad = -(-N // S) * S
    return 24 * (N + npad) * band + 8


@pytest.mark.parametrize("N,ipt,S,band,sort", [(3000, 4, 128, 5, 0), (3000, 4, 128, 1, 0), (3333, 4, 256, 3, 1), (2500, 2, 256, 4, 0),
                                               (5000, 4, 512, 2, 1), (3000, 4, 128, 23, 1)])
def test_banded_evaluation_against_oracle(N, ipt, S, band, sort):
    import paper_2604_09184_b200 as nb
    x, v, m = nb_inputs.random_cluster(N, seed=700 + N + band, scale=0.2)
    rng = np.random.default_rng(band)
    rc = rng.uniform(0.0, 0.05, N)
    rc[::5] = 0.0
    tune = dict(force_kernel=SYM, i_per_thread=ipt, sym_block=S, sort_staging=1 if sort else 2, slot_bytes_max=_band_cap(N, S, band))
    info = _kick_case(x, v, m, rc, dt=0.37, what=f"banded N={N} I={ipt} S={S} band={band} sorted={sort}", **tune)
    assert info["n_sure"] > 100
    # the banded workspace is the small one (two sets of `band` column slots against T slots)
    T = -(-N // S)
    if 3 * band <= T:
        ws_band = nb.workspace_bytes(N)
        nb.set_flags(slot_bytes_max=0)
        assert ws_band < nb.workspace_bytes(N)
    # same pair list and (to rounding order) the same accelerations as the one-launch evaluation; bit-reproducible
    out = []
    for cap in (_band_cap(N, S, band), _band_cap(N, S, band), 0):
        st = GpuState(x, v, m, G=G_GAUSS, **dict(tune, slot_bytes_max=cap))
        st.set_rcrit(rc)
        st.kick(0.0)
        gp, n = st.get_pairs()
        out.append((st.acc.cpu().numpy().copy(), {tuple(p) for p in gp[:n].tolist()}))
    assert np.array_equal(out[0][0], out[1][0]), "the banded evaluation is not run-to-run reproducible"
    assert out[0][1] == out[1][1] == out[2][1]
    scale = np.linalg.norm(out[2][0], axis=1, keepdims=True)
    assert np.max(np.abs(out[0][0] - out[2][0]) / scale) < 1e-12


@pytest.mark.parametrize("use_graph", [True, False])
def test_banded_step_matches_oracle(use_graph):
    d = nb_inputs.make_config(1, n_override=1498)
    st = GpuState(d.x, d.v, d.m, d.M_star, G=G_GAUSS, n1=3.0, n2=0.4, force_kernel=SYM, sym_block=128, use_graph=use_graph,
                  slot_bytes_max=_band_cap(d.N, 128, 5))
    st.step(d.dt, 20)
    xg, vg, ag, rcg = st.host()
    ref = oracle.step(d.x, d.v, d.m, d.M_star, d.dt, G_GAUSS, 20, n1=3.0, n2=0.4)
    ex = np.max(np.abs(xg - ref["x"])) / np.max(np.abs(ref["x"]))
    ev = np.max(np.abs(vg - ref["v"])) / np.max(np.abs(ref["v"]))
    print(f"banded step x20 graph={use_graph}: rel dx {ex:.2e} dv {ev:.2e}")
    assert ex <= 1e-11 and ev <= 1e-11
    sure, border = oracle.pairs(ref["x"], ref["rcrit"])
    gp, n = st.get_pairs()
    assert_pairs_match(gp, n, sure, border, "banded step")
