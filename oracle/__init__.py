"""CPU fp64 oracle for the RK2 Euler step (test infrastructure, not the product).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the CUDA package.
"""
from .hydro_oracle import (  # noqa: F401
    OracleHydro, OracleError, build, lib, sum3, minmod, primitive, hll_flux,
    set_threads, get_threads, BC_OUTFLOW, BC_REFLECT, BC_PERIODIC,
)
