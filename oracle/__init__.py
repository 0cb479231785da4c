"""ORACLE — test infrastructure, not product code.

ctypes loader for ``oracle/*.cpp``: ``spin_oracle.cpp`` (the plain CPU restatement of the paper's checkerboard
Metropolis sweep) and its extensions ``dmc_oracle.cpp`` (Algorithm 2), ``general_oracle.cpp`` (per-bond couplings and
fields), ``stencil_oracle.cpp`` (other geometries), ``cpm_oracle.cpp`` (cellular Potts); each file's header names the
passages it follows and its pins.
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from the CUDA package.
"""
from .oracle import *  # noqa: F401,F403
