"""B200-native two-site DMRG hot path of arxiv 2503.20700 (H_eff psi, renormalisation, sweep, 1-/2-RDM).

Everything is computed by the CUDA library csrc/ -> libdmrg_b200.so behind the C ABI of include/dmrg_b200.h;
`binding` only marshals arguments.  Importing this package without the built library raises (no CPU fallback).
"""
from .binding import *  # noqa: F401,F403
from . import binding  # noqa: F401
