"""paper_2304_01772_b200 — B200-native checkerboard Metropolis sweeps (Ising / Potts) behind libspin.so.

``binding`` mirrors include/spin.h one to one (argument marshalling only); ``workloads`` holds the seeded
synthetic input recipes of the five BASELINE.json configurations; ``build`` compiles csrc/ for sm_100a.
"""
from . import workloads  # noqa: F401
from .binding import *  # noqa: F401,F403
