"""Synthetic disk generator (BASELINE.json:configs).

Units (reading S14): AU, day, solar mass; G = k^2 with the Gaussian
constant k = 0.01720209895.  The paper's initial conditions are statistical
recipes ("nearly circular and coplanar", "disk between
0.5 AU and 4 AU ... 5 M_earth ... MMSN", PAPER.md:204 N grid, PAPER.md:231 giants);
no dataset exists, these seeded draws stand in for them.

Only input construction lives here: orbital elements -> heliocentric position,
barycentric velocity.  None of the integrator's arithmetic.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

K_GAUSS = 0.01720209895
G_GAUSS = K_GAUSS * K_GAUSS
M_EARTH = 1.0 / 332946.0487
M_JUP = 1.0 / 1047.348644
RHO_2GCC = 3.367443e6  # 2 g/cm^3 in M_sun / AU^3 (radii only; unused by the hot path)


@dataclass
class DiskState:
    """One synthetic workload.  x: heliocentric [N,3]; v: barycentric [N,3]; m: [N]."""

    name: str
    x: np.ndarray
    v: np.ndarray
    m: np.ndarray
    M_star: float
    dt: float
    nsteps: int
    n_active: int  # == N unless semi-active (BASELINE.json:configs[3])
    radius: np.ndarray
    seed: int
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.m.shape[0])

    @property
    def interactions_per_eval(self) -> int:
        return self.N * self.n_active


def _solve_kepler(M: np.ndarray, e: np.ndarray) -> np.ndarray:
    """Eccentric anomaly for the INPUT orbits only (not the integrator's drift)."""
    E = M + e * np.sin(M)
    for _ in range(60):
        dE = (E - e * np.sin(E) - M) / (1.0 - e * np.cos(E))
        E = E - dE
        if np.max(np.abs(dE)) < 1e-15:
            break
    return E


def elements_to_cartesian(a, e, inc, w, O, M, mu):
    """Keplerian elements -> heliocentric position and velocity, gravitational parameter mu."""
    a, e, inc, w, O, M = (np.asarray(t, dtype=np.float64) for t in (a, e, inc, w, O, M))
    mu = np.asarray(mu, dtype=np.float64)
    E = _solve_kepler(M, e)
    cE, sE = np.cos(E), np.sin(E)
    b = np.sqrt(1.0 - e * e)
    xp = a * (cE - e)
    yp = a * b * sE
    n = np.sqrt(mu / (a * a * a))
    rr = 1.0 - e * cE
    vxp = -a * n * sE / rr
    vyp = a * n * b * cE / rr
    cw, sw = np.cos(w), np.sin(w)
    cO, sO = np.cos(O), np.sin(O)
    ci, si = np.cos(inc), np.sin(inc)
    r11 = cO * cw - sO * sw * ci
    r12 = -cO * sw - sO * cw * ci
    r21 = sO * cw + cO * sw * ci
    r22 = -sO * sw + cO * cw * ci
    r31 = sw * si
    r32 = cw * si
    x = np.stack([r11 * xp + r12 * yp, r21 * xp + r22 * yp, r31 * xp + r32 * yp], axis=-1)
    v = np.stack([r11 * vxp + r12 * vyp, r21 * vxp + r22 * vyp, r31 * vxp + r32 * vyp], axis=-1)
    return np.ascontiguousarray(x), np.ascontiguousarray(v)


def _draw_disk(rng, N, a_in, a_out, sig_e, sig_i, profile):
    """Draw order per body array: u_a, e, i, omega, Omega, M."""
    u = rng.random(N)
    if profile == "sigma_r-1.5":  # Sigma ~ r^-1.5, equal masses => dN/da ~ a^-1/2
        a = (math.sqrt(a_in) + u * (math.sqrt(a_out) - math.sqrt(a_in))) ** 2
    elif profile == "uniform_a":
        a = a_in + u * (a_out - a_in)
    else:
        raise ValueError(profile)
    e = rng.rayleigh(sig_e, N)
    inc = rng.rayleigh(sig_i, N)
    w = rng.random(N) * 2.0 * math.pi
    O = rng.random(N) * 2.0 * math.pi
    M = rng.random(N) * 2.0 * math.pi
    return a, e, inc, w, O, M


# name, N, a_in, a_out, sig_e, sig_i, profile, dt, nsteps, seed
CONFIGS = [
    dict(name="c1_N2048_equal", N=2048, a_in=0.5, a_out=4.0, sig_e=0.01, sig_i=0.005,
         profile="sigma_r-1.5", dt=6.0, nsteps=100, seed=1001, total_mearth=2.0),
    dict(name="c2_N16384_giants", N=16384, a_in=0.5, a_out=4.0, sig_e=0.01, sig_i=0.005,
         profile="sigma_r-1.5", dt=6.0, nsteps=1000, seed=1002, total_mearth=5.0,
         giants=[(1.0, 5.2, 0.05), (0.3, 9.5, 0.05)]),
    dict(name="c3_N65536_ring", N=65536, a_in=0.7, a_out=1.0, sig_e=0.002, sig_i=0.001,
         profile="uniform_a", dt=3.0, nsteps=200, seed=1003, powerlaw=(1e-4, 1e-2, 2.5)),
    dict(name="c4_N131072_semiactive", N=131072, a_in=0.5, a_out=3.0, sig_e=0.01, sig_i=0.005,
         profile="sigma_r-1.5", dt=6.0, nsteps=100, seed=1004, n_active=1024,
         embryo_mearth=0.02),
    dict(name="c5_N524288_equal", N=524288, a_in=0.3, a_out=4.0, sig_e=0.005, sig_i=0.0025,
         profile="sigma_r-1.5", dt=3.0, nsteps=10, seed=1005, total_mearth=5.0),
]


def make_config(k: int, n_override: int | None = None, seed: int | None = None) -> DiskState:
    """Workload k (0-based index into BASELINE.json:configs).

    `n_override` shrinks the planetesimal count for tests (total disk mass, giants and
    the active fraction are kept); the full-size call is the benchmark workload.
    """
    c = CONFIGS[k]
    N = int(n_override) if n_override is not None else c["N"]
    sd = c["seed"] if seed is None else seed
    rng = np.random.default_rng(sd)
    M_star = 1.0
    a, e, inc, w, O, M = _draw_disk(rng, N, c["a_in"], c["a_out"], c["sig_e"], c["sig_i"], c["profile"])
    n_active = N
    if "powerlaw" in c:
        m_lo, m_hi, q = c["powerlaw"]
        p = q - 1.0
        u = rng.random(N)
        m = (m_lo ** (-p) - u * (m_lo ** (-p) - m_hi ** (-p))) ** (-1.0 / p) * M_EARTH
    elif "n_active" in c:
        n_active = max(1, (c["n_active"] * N) // c["N"])
        m = np.zeros(N)
        m[:n_active] = c["embryo_mearth"] * M_EARTH
    else:
        m = np.full(N, c["total_mearth"] * M_EARTH / max(N, 1))
    if "giants" in c:
        ng = len(c["giants"])
        ga = np.array([g[1] for g in c["giants"]])
        ge = np.array([g[2] for g in c["giants"]])
        gm = np.array([g[0] * M_JUP for g in c["giants"]])
        gw = rng.random(ng) * 2.0 * math.pi
        gO = rng.random(ng) * 2.0 * math.pi
        gM = rng.random(ng) * 2.0 * math.pi
        a = np.concatenate([a, ga]); e = np.concatenate([e, ge]); inc = np.concatenate([inc, np.zeros(ng)])
        w = np.concatenate([w, gw]); O = np.concatenate([O, gO]); M = np.concatenate([M, gM])
        m = np.concatenate([m, gm])
        n_active = m.shape[0]
    xh, vh = elements_to_cartesian(a, e, inc, w, O, M, G_GAUSS * (M_star + m))
    # democratic coordinates: heliocentric r, barycentric v
    v_star = -(m[:, None] * vh).sum(axis=0) / (M_star + m.sum())
    vb = vh + v_star
    radius = np.cbrt(3.0 * m / (4.0 * math.pi * RHO_2GCC))
    return DiskState(name=c["name"] if n_override is None else f'{c["name"]}@N{N}',
                     x=np.ascontiguousarray(xh), v=np.ascontiguousarray(vb), m=np.ascontiguousarray(m),
                     M_star=M_star, dt=c["dt"], nsteps=c["nsteps"], n_active=int(n_active),
                     radius=radius, seed=sd, meta=dict(config_index=k, a=a, e=e, inc=inc))


# ---- tiny hand-made cases for pins and edge tests (positions/masses only; no method arithmetic) ----

def two_body(m1=1e-3, m2=2e-3, sep=0.01, center=(1.0, 0.0, 0.0), direction=(0.6, 0.0, 0.8)):
    d = np.asarray(direction, dtype=np.float64)
    d = d / np.linalg.norm(d)
    c = np.asarray(center, dtype=np.float64)
    x = np.stack([c - 0.5 * sep * d, c + 0.5 * sep * d])
    v = np.zeros((2, 3))
    m = np.array([m1, m2])
    return x, v, m


def chain_1d(N, spacing=1.0, origin=(10.0, 0.0, 0.0)):
    x = np.zeros((N, 3))
    x[:, 0] = origin[0] + spacing * np.arange(N)
    x[:, 1] = origin[1]
    x[:, 2] = origin[2]
    return x, np.zeros((N, 3)), np.full(N, 1e-9)


def cubic_lattice(n, spacing=1.0, origin=(5.0, 5.0, 5.0)):
    g = np.arange(n) * spacing
    X, Y, Z = np.meshgrid(g, g, g, indexing="ij")
    x = np.stack([X.ravel() + origin[0], Y.ravel() + origin[1], Z.ravel() + origin[2]], axis=1)
    N = x.shape[0]
    return np.ascontiguousarray(x), np.zeros((N, 3)), np.full(N, 1e-9)


def random_cluster(N, seed=7, scale=1.0, mass_lo=1e-9, mass_hi=1e-6, center=(1.0, 0.0, 0.0)):
    rng = np.random.default_rng(seed)
    x = rng.normal(size=(N, 3)) * scale + np.asarray(center)
    v = rng.normal(size=(N, 3)) * 0.01
    m = np.exp(rng.uniform(math.log(mass_lo), math.log(mass_hi), N))
    return np.ascontiguousarray(x), np.ascontiguousarray(v), m
