"""B200-native CLVisc hydro step (arXiv:1802.04449): C-ABI CUDA library + thin ctypes binding.

The package holds the CUDA sources (csrc/), their build step (build.py), the binding (hydro.py) and the
seeded synthetic input generators (inputs.py).  It never imports oracle/.
"""
from .hydro import Hydro, HydroError, from_config, load_library  # noqa: F401
