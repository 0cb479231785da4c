"""ORACLE — test infrastructure, not product code.

ctypes loader for ``oracle/spin_oracle.cpp`` (the plain CPU restatement of the paper's
checkerboard Metropolis sweep; see that file's header for the passages it follows and its pins).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from the CUDA package.
"""
from .oracle import *  # noqa: F401,F403
