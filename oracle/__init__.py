"""fp64 CPU oracle (test infrastructure only; see mvd_oracle.py header)."""
from .mvd_oracle import *  # noqa: F401,F403
from .mvd_oracle import Oracle, back_projector, deconvolve, deconvolve_blocked  # noqa: F401
