"""Helpers of the -m gpu parity tests: run the CUDA path through the C ABI (via the thin binding) and
compare with the CPU oracle.  Tolerances are the north_star's, written out here:

* accelerations: |da_c| <= max(1e-12 * max(|a_c|, 1e-3 * ||a_i||_2), 32 eps * sum_j |t_jc|) for every body
  and component (reading S9: "relative error 1e-12 per component"; the second term is the
  backward-error allowance of ANY fp64 evaluation of the sum for components whose terms t_jc cancel --
  condition number sum|t| / |sum t| >~ 1e3 inside dense encounters, or exactly symmetric lattices --
  where plain numpy fp64 misses the literal bound by the same factor; sum|t| comes from the oracle);
* pairs: bit-exact after canonical sort, except pairs within 1e-12 relative of the threshold
  (2e-12 in r^2), which the oracle lists separately: sure <= gpu <= sure + borderline;
* energy: |(dE/E)_gpu - (dE/E)_oracle| <= 1e-9.
"""
from __future__ import annotations

import numpy as np

ACC_RTOL = 1e-12
ACC_FLOOR = 1e-3
ACC_BACKWARD = 32 * 2.220446049250313e-16  # x sum_j |term|: fp64 rounding of the terms + two-level summation
ENERGY_TOL = 1e-9


def torch_mod():
    import torch
    return torch


def to_dev(a, dtype=None):
    torch = torch_mod()
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.to(dtype)


def acc_error(acc_gpu: np.ndarray, acc_ref: np.ndarray, abs_sum=None):
    """Returns (worst ratio of |da_c| to its allowance, literal max relative error per component)."""
    d = np.abs(acc_gpu - acc_ref)
    norm = np.linalg.norm(acc_ref, axis=1, keepdims=True)
    allow = ACC_RTOL * np.maximum(np.abs(acc_ref), ACC_FLOOR * norm)
    if abs_sum is not None:
        allow = np.maximum(allow, ACC_BACKWARD * abs_sum)
    allow = np.where(allow > 0.0, allow, np.finfo(float).tiny)
    ratio = float(np.max(d / allow)) if d.size else 0.0
    with np.errstate(divide="ignore", invalid="ignore"):
        lit = np.where(acc_ref != 0.0, d / np.abs(acc_ref), 0.0)
    return ratio, float(np.max(lit)) if lit.size else 0.0


def assert_acc_close(acc_gpu, acc_ref, what="", abs_sum=None):
    assert np.all(np.isfinite(acc_gpu)), f"{what}: non-finite acceleration from the CUDA path"
    ratio, lit = acc_error(acc_gpu, acc_ref, abs_sum)
    assert ratio <= 1.0, f"{what}: acceleration error {ratio:.3g} x the allowance (literal max rel {lit:.3g})"
    return ratio, lit


def canon_pairs(p: np.ndarray) -> np.ndarray:
    p = np.asarray(p, dtype=np.int32).reshape(-1, 2)
    if p.shape[0] == 0:
        return p
    return np.unique(p, axis=0)


def _keys(p):
    p = np.asarray(p, dtype=np.int64).reshape(-1, 2)
    return p[:, 0] * (1 << 32) + p[:, 1]


def assert_pairs_match(gpu_pairs, n_gpu, sure, border, what=""):
    """gpu list has no duplicates, is ordered (min,max), contains every sure pair and nothing outside
    sure + borderline."""
    gpu_pairs = np.asarray(gpu_pairs).reshape(-1, 2)
    assert n_gpu == gpu_pairs.shape[0], f"{what}: npairs {n_gpu} but {gpu_pairs.shape[0]} rows read"
    if gpu_pairs.shape[0]:
        assert np.all(gpu_pairs[:, 0] < gpu_pairs[:, 1]), f"{what}: a pair is not (min,max)"
    cg = canon_pairs(gpu_pairs)
    assert cg.shape[0] == gpu_pairs.shape[0], f"{what}: duplicate pairs in the CUDA list"
    kg, ks, kb = _keys(cg), _keys(sure), _keys(border)
    missing = np.setdiff1d(ks, kg)
    extra = np.setdiff1d(kg, np.union1d(ks, kb))
    assert missing.size == 0, f"{what}: {missing.size} sure pairs missing from the CUDA list"
    assert extra.size == 0, f"{what}: {extra.size} CUDA pairs are neither sure nor borderline"
    return dict(n_gpu=int(cg.shape[0]), n_sure=int(ks.size), n_border=int(kb.size))


class GpuState:
    """Device copies of one workload + output buffers, configured library."""

    def __init__(self, x, v, m, M_star=1.0, *, G, n_active=0, n1=3.0, n2=0.0, kind=0, pair_capacity=1 << 20,
                 i_per_thread=0, j_splits=0, use_graph=True, **tune):
        import paper_2604_09184_b200 as nb
        torch = torch_mod()
        self.nb = nb
        self.N = int(np.asarray(m).shape[0])
        self.M_star = float(M_star)
        self.x, self.v, self.m = to_dev(x), to_dev(v), to_dev(m)
        self.acc = torch.zeros((self.N, 3), dtype=torch.float64, device="cuda")
        self.rcrit = torch.zeros(self.N, dtype=torch.float64, device="cuda")
        self.cap = int(pair_capacity)
        self.pairs = torch.full((max(self.cap, 1), 2), -1, dtype=torch.int32, device="cuda")
        self.npairs = torch.zeros(1, dtype=torch.int64, device="cuda")
        nb.configure(self.N, pair_capacity=self.cap, n_active=n_active, G=G, n1=n1, n2=n2, changeover_kind=kind,
                     i_per_thread=i_per_thread, j_splits=j_splits, use_graph=use_graph, **tune)
        nb.nb_status_reset()

    def set_rcrit(self, rc):
        self.rcrit.copy_(to_dev(rc))

    def kick(self, dt, with_pairs=True, rcrit_given=True):
        self.nb.nb_kick(self.x, self.v, self.m, self.M_star, dt, self.rcrit if rcrit_given else None, self.acc,
                        self.pairs if with_pairs else None, self.npairs if with_pairs else None)
        torch_mod().cuda.synchronize()

    def step(self, dt, nsteps, with_pairs=True):
        self.nb.nb_step(self.x, self.v, self.m, self.M_star, dt, self.rcrit, self.acc,
                        self.pairs if with_pairs else None, self.npairs if with_pairs else None, nsteps)
        torch_mod().cuda.synchronize()

    def get_pairs(self):
        n = int(self.npairs.item())
        keep = min(n, self.cap)
        return self.pairs[:keep].cpu().numpy(), n

    def host(self):
        return self.x.cpu().numpy(), self.v.cpu().numpy(), self.acc.cpu().numpy(), self.rcrit.cpu().numpy()
