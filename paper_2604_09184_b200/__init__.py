"""paper_2604_09184_b200 -- B200-native (sm_100a) direct-summation kick, close-encounter pair list and
Kepler drift of the hybrid symplectic planet-formation integrator (arxiv 2604.09184).

The product is the C-ABI library libnbkick.so (include/nbkick.h; sources in csrc/); this package is
its thin Python binding.  No CPU fallback exists: the calls raise if the library is not built.
"""
from . import build  # noqa: F401
from .binding import *  # noqa: F401,F403
from .binding import (NbConfig, NbError, SYMBOLS, configure, default_config, force_geometry, lib_path, load,  # noqa: F401
                      nb_drift_kepler, nb_encounter, nb_fp64_peak, nb_groups, nb_kick, nb_merge, nb_kick_host, nb_force_time, nb_force_time_reset, nb_last_force_ms, nb_rcrit, set_flags, nb_release,
                      nb_shift, nb_status, nb_status_reset, nb_step, nb_step_host, nb_version, workspace_bytes)
