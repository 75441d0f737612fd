"""B200-native hydrodynamic timestep of the FARGO3D method (arXiv 1602.02359).

`Fargo` wraps the C-ABI library (include/fargo.h, csrc/*.cu); `workloads` builds the seeded synthetic
inputs of the five BASELINE.json configs.  The CPU oracle under oracle/ is test infrastructure and is
never imported from here.
"""
from . import workloads  # noqa: F401
from .binding import Fargo, load, library_path, STAGES  # noqa: F401
