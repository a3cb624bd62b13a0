"""-m "not gpu": the C-ABI library builds for sm_100a, loads, and exports every symbol include/nbkick.h
declares; host-side argument validation and launch geometry (no compute calls without a GPU)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def nb():
    import paper_2604_09184_b200 as nb
    nb.build.build()
    nb.load()
    return nb


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "nbkick.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nb_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported(nb):
    decl = _declared_symbols()
    assert len(decl) >= 15
    lib = nb.load()
    for name in decl:
        assert hasattr(lib, name), f"libnbkick.so does not export {name}"
    assert sorted(nb.SYMBOLS) == decl, "binding.SYMBOLS is out of date with include/nbkick.h"
    assert "sm_100a" in nb.nb_version()


def test_no_torch_types_in_abi():
    src = open(os.path.join(ROOT, "include", "nbkick.h")).read()
    assert "torch" not in src.lower().replace("pytorch", "") and "at::" not in src and "c10" not in src


def test_config_struct_matches_header(nb):
    cfg = nb.default_config()
    assert cfg.n1 == 3.0 and cfg.n2 == 0.4 and cfg.use_graph == 1 and cfg.changeover_kind == 0
    assert abs(cfg.G - 0.01720209895 ** 2) < 1e-20
    fields = [f[0] for f in nb.NbConfig._fields_]
    src = open(os.path.join(ROOT, "include", "nbkick.h")).read()
    body = src[src.index("typedef struct nb_config"):src.index("} nb_config;")]
    order = [re.findall(r"(\w+);", line)[0] for line in body.splitlines() if re.search(r"\w+;\s*(/\*|$)", line)]
    assert order == fields


def test_configure_validation(nb):
    lib = nb.load()
    cfg = nb.default_config()
    assert lib.nb_configure(C.byref(cfg)) == 0
    for field, bad in (("G", -1.0), ("n1", -3.0), ("n2", float("nan")), ("pair_capacity", -1), ("n_active", -5),
                       ("changeover_kind", 7), ("i_per_thread", 3), ("j_splits", -2), ("sym_block", 300), ("slot_bytes_max", -1)):
        c = nb.default_config()
        setattr(c, field, bad)
        assert lib.nb_configure(C.byref(c)) == nb.binding.NB_E_BADARG, field
        assert lib.nb_last_error()
    assert lib.nb_configure(None) == nb.binding.NB_E_NULL
    assert lib.nb_configure(C.byref(nb.default_config())) == 0


def test_host_side_argument_checks_need_no_gpu(nb):
    lib = nb.load()
    assert lib.nb_configure(C.byref(nb.default_config())) == 0
    one = C.c_void_p(4096)  # never dereferenced: validation fails first
    assert lib.nb_kick(one, one, one, 1.0, 0, 1.0, one, one, None, None) == nb.binding.NB_E_BADN
    assert lib.nb_kick(one, one, one, 1.0, 1 << 31, 1.0, one, one, None, None) == nb.binding.NB_E_BADN
    assert lib.nb_kick(one, one, one, 0.0, 10, 1.0, one, one, None, None) == nb.binding.NB_E_BADARG
    assert lib.nb_kick(one, one, one, 1.0, 10, float("inf"), one, one, None, None) == nb.binding.NB_E_BADARG
    assert lib.nb_kick(None, one, one, 1.0, 10, 1.0, one, one, None, None) == nb.binding.NB_E_NULL
    assert lib.nb_kick(one, one, one, 1.0, 10, 1.0, one, one, one, None) == nb.binding.NB_E_NULL  # pairs without npairs
    assert lib.nb_kick(one, one, one, 1.0, 10, 1.0, one, one, None, None) == nb.binding.NB_E_WORKSPACE
    assert lib.nb_drift_kepler(one, None, 1.0, 10, 1.0) == nb.binding.NB_E_NULL
    assert lib.nb_step(one, one, one, 1.0, 10, 1.0, one, one, None, None, -1) == nb.binding.NB_E_BADARG
    c = nb.default_config()
    c.n_active = 11
    assert lib.nb_configure(C.byref(c)) == 0
    assert lib.nb_kick(one, one, one, 1.0, 10, 1.0, one, one, None, None) == nb.binding.NB_E_BADARG
    assert lib.nb_configure(C.byref(nb.default_config())) == 0


def test_geometry_and_workspace(nb):
    """Launch geometry for BASELINE.json's five sizes: every body covered, every j-tile owned by exactly
    one split, enough CTAs to fill 148 SMs where the problem allows, workspace grows with N."""
    lib = nb.load()
    prev = 0
    for N, n_active in ((2048, 0), (16386, 0), (65536, 0), (131072, 1024), (524288, 0)):
        c = nb.default_config()
        c.n_active = n_active
        assert lib.nb_configure(C.byref(c)) == 0
        g = nb.force_geometry(N)
        assert g.threads in (32, 64, 128) and g.i_per_thread in (1, 2, 4)
        nj = n_active or N
        ws = nb.workspace_bytes(N)
        if g.tile_j < 0:
            # Newton-III kernel: fully active and large enough; super-blocks of S bodies cover N, one CTA
            # per unordered pair of super-blocks, one partial slot per super-block
            S = -g.tile_j
            assert not n_active and N >= 4096
            # CTAs of W warps whose chunks of 32 W I bodies tile the super-block; always 12 warps per SM at I = 4
            assert S in (128, 256, 512, 1024, 2048) and S % (g.threads * g.i_per_thread) == 0
            assert g.threads == min(128, S // g.i_per_thread) or g.i_per_thread != 4
            assert g.i_blocks == g.j_splits == -(-N // S)
            # enough waves of CTAs (16 at S = 512, 5 at S = 256), else the smallest block
            slots = 148 * (1536 // min(S, 512))
            assert g.i_blocks * (g.i_blocks + 1) // 2 >= (16 if S >= 512 else 5) * slots or S == 128
            full = 24 * N * g.j_splits
            if full <= 4 << 30:
                assert ws >= 36 * N + full
            else:
                # banded evaluation (nb_config.slot_bytes_max, default 4 GiB): the slots of one band of tile columns only
                assert (2 << 30) < ws - 100 * N <= (4 << 30) + (1 << 26)
        else:
            assert g.tile_j == 128 and g.threads == 128
            assert g.i_blocks * g.threads * g.i_per_thread >= N > (g.i_blocks - 1) * g.threads * g.i_per_thread
            tiles = -(-nj // g.tile_j)
            per = -(-tiles // g.j_splits)
            assert (g.j_splits - 1) * per < tiles <= g.j_splits * per
            assert g.i_blocks * g.j_splits >= 148
            assert ws >= 64 * nj + 24 * N * g.j_splits
        if not n_active:
            assert ws > prev
            prev = ws
    assert nb.workspace_bytes(0) == 0
    # the kernel choice can be forced either way; semi-active requests fall back to the one-sided kernel
    c = nb.default_config()
    c.force_kernel = 1
    assert lib.nb_configure(C.byref(c)) == 0 and nb.force_geometry(65536).tile_j == 128
    c.force_kernel, c.sym_block, c.i_per_thread = 2, 256, 1
    assert lib.nb_configure(C.byref(c)) == 0 and nb.force_geometry(700).tile_j == -256
    c.n_active = 100
    assert lib.nb_configure(C.byref(c)) == 0 and nb.force_geometry(700).tile_j == 128
    c = nb.default_config()
    c.sym_block = 300
    assert lib.nb_configure(C.byref(c)) == nb.binding.NB_E_BADARG
    assert lib.nb_configure(C.byref(nb.default_config())) == 0


def test_product_path_does_not_touch_the_oracle():
    """The CUDA package must not import, link or read anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2604_09184_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "nb_oracle" not in txt and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2604_09184_b200\b", txt, flags=re.M), f
            assert "nbkick" not in txt, f


def test_geometry_of_the_mixed_precision_kernels(nb):
    """NB_PRECISION_MIXED (host logic, no GPU): fully active N >= 4096 takes the Newton-III kernel on double-single positions
    (same super-block rule as the fp64 kernel, 32 more bytes per staged body), bands when the slots would pass the cap;
    semi-active mode takes the one-sided double-single kernel (32 bytes more per active body); with one i-body per thread
    (small N) the fp64 kernel runs and the workspace is the fp64 one."""
    lib = nb.load()

    def geo(N, n_active=0, precision=1, **kw):
        c = nb.default_config()
        c.n_active, c.precision = n_active, precision
        for k, v in kw.items():
            setattr(c, k, v)
        assert lib.nb_configure(C.byref(c)) == 0
        return nb.force_geometry(N), nb.workspace_bytes(N)

    for N in (4096, 16386, 65536):
        g64, w64 = geo(N, precision=0)
        g32, w32 = geo(N)
        assert g32.tile_j == g64.tile_j < 0 and g32.i_per_thread == 4 and g32.threads == g64.threads
        npad = -(-N // -g32.tile_j) * -g32.tile_j
        T = npad // -g32.tile_j
        # the fp64 staged arrays (72 B per body, doubled blocks; the exact pass reads them), two float4 arrays in the same
        # layout (64 B per body), one slot per super-block
        assert w32 >= 72 * npad + 64 * npad + 24 * N * T
        assert w32 <= w64 + 64 * npad + 4096                                          # nothing else grows
    g, w = geo(524288)
    assert g.tile_j == -512 and w <= (4 << 30) + 200 * 524288                      # banded: slots within the 4 GiB cap
    g, w = geo(131072, n_active=1024)
    g0, w0 = geo(131072, n_active=1024, precision=0)
    assert g.tile_j == 128 and g.i_per_thread == 2 and w - w0 == 1024 * 32         # one-sided double-single records
    g, w = geo(2048)
    g0, w0 = geo(2048, precision=0)
    assert g.tile_j == 128 and g.i_per_thread == 1 and w == w0                     # small N: the fp64 kernel
