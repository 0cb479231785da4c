"""Physics at sizes the oracle cannot reach in test time: the GPU path against Onsager's exact 2D Ising energy and
Yang's spontaneous magnetisation, standard errors across independent replicas.  The GPU
lattices are bit-identical to the oracle's wherever both were run, so this checks nothing new about the rule; it
checks that long runs on large lattices through the public API (both layouts, streaming kernels, traces through
spin_sweep_measure) land where the physics says."""
import numpy as np
import pytest

import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu

U_030 = -0.704499070832      # Onsager, beta = 0.30 (J = 1, h = 0), energy per spin
U_060 = -1.909086177684      # beta = 0.60
M_060 = 0.973608667440       # Yang


@pytest.mark.parametrize("layout", [sp.SPIN_LAYOUT_INT8, sp.SPIN_LAYOUT_BITPACKED])
def test_onsager_energy_high_temperature(layout):
    B, L, n_therm, n_meas = 64, 512, 200, 300
    with sp.spin_create_ex(B, L, sp.SPIN_MODEL_ISING, seed=2024, layout=layout) as sim:
        sim.spin_sweep(0.30, 1.0, 0.0, n_therm, 0)
        E, M = sim.spin_sweep_measure(0.30, 1.0, 0.0, n_meas, n_therm)
    u = E.mean(axis=0) / (L * L)                      # per-replica time average of J * E_int / N
    mean, se = u.mean(), u.std(ddof=1) / np.sqrt(B)
    assert abs(mean - U_030) < 4 * se + 1e-3, (mean, se)


def test_onsager_energy_and_yang_magnetisation_cold_start():
    B, L, n_therm, n_meas = 64, 512, 300, 300
    with sp.spin_create_ex(B, L, sp.SPIN_MODEL_ISING, seed=7) as sim:
        sim.spin_set_spins(np.ones((B, L, L), dtype=np.int8))      # cold start: no stripe states
        sim.spin_sweep(0.60, 1.0, 0.0, n_therm, 0)
        E, M = sim.spin_sweep_measure(0.60, 1.0, 0.0, n_meas, n_therm)
    u = E.mean(axis=0) / (L * L)
    m = np.abs(M).mean(axis=0) / (L * L)
    assert abs(u.mean() - U_060) < 4 * u.std(ddof=1) / np.sqrt(B) + 1e-3
    assert abs(m.mean() - M_060) < 4 * m.std(ddof=1) / np.sqrt(B) + 1e-3
