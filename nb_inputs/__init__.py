"""Seeded synthetic planetesimal-disk inputs shared by the oracle and the CUDA path.

This module holds NONE of the method's arithmetic (no kick, no pair test, no
drift, no r_crit): it only turns random orbital elements into the state the
paper's integrator takes -- heliocentric positions, barycentric velocities,
masses ("democratic coordinates") -- with the shapes that
BASELINE.json:configs fixes and SURVEY.md section 8(d) spells out.  It imports
neither `oracle/` nor `paper_2604_09184_b200/`.
"""
from .disks import (  # noqa: F401
    G_GAUSS,
    K_GAUSS,
    M_EARTH,
    M_JUP,
    CONFIGS,
    DiskState,
    make_config,
    elements_to_cartesian,
    two_body,
    chain_1d,
    cubic_lattice,
    random_cluster,
)
