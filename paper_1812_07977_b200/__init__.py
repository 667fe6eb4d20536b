"""B200-native RK2 step of the 3D compressible-Euler finite-volume update (arXiv 1812.07977).

`Hydro` (binding.py) wraps the C-ABI library `libhydro_b200.so` declared in include/hydro.h;
`inputs` holds the seeded synthetic workloads.  There is no CPU fallback: using `Hydro`
without the built CUDA library raises.
"""
from . import inputs  # noqa: F401


def __getattr__(name):
    if name in ("Hydro", "HydroError", "load_library", "build"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
