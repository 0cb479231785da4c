"""GPU parity for +-J couplings (spin_set_bonds; bit-packed Ising layout) against the oracle, bit for bit."""
import numpy as np
import pytest

import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu


def _rand_bonds(seed, B, L):
    rng = np.random.default_rng(seed)
    return ((2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8),
            (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8))


def _mk(batch, L, seed, layout=sp.SPIN_LAYOUT_BITPACKED):
    return sp.spin_create_ex(batch, L, sp.SPIN_MODEL_ISING, seed=seed, layout=layout)


@pytest.mark.parametrize("L,batch,J,h,betas", [
    (64, 3, 1.0, 0.0, [0.3, 0.8, 20.0]),
    (128, 2, 1.0, 0.05, [0.5, 1.2]),
    (192, 2, -1.0, 0.2, [0.4, 0.0]),
])
def test_sweeps_with_random_bonds_match_oracle_every_sweep(oracle_mod, L, batch, J, h, betas):
    seed, n = 300 + L, 10
    Jh, Jv = _rand_bonds(L, batch, L)
    ref = oracle_mod.init(batch, L, seed=seed)
    with _mk(batch, L, seed) as sim:
        sim.spin_set_bonds(Jh, Jv)
        for t in range(n):
            sim.spin_sweep(betas, J, h, 1, t)
            oracle_mod.sweep_bonds(ref, Jh, Jv, betas, J, h, seed=seed, n_sweeps=1, sweep_offset=t)
            assert np.array_equal(sim.spin_get_spins(), ref), "lattice differs after sweep %d" % t
            E, M = sim.spin_observables()
            Eo, Mo = oracle_mod.ising_bonds_observables(ref, Jh, Jv)
            assert np.array_equal(E, Eo) and np.array_equal(M, Mo)


def test_long_rows_trace_and_removal(oracle_mod):
    """A launch big enough for the 8-rows-per-thread variant (L = 1024), traces through spin_sweep_measure, a bond
    sample broadcast over the batch, and spin_set_bonds(None, None) restoring the uniform model."""
    L, batch, seed, n = 1024, 8, 31, 4
    Jh, Jv = _rand_bonds(1, 1, L)
    beta = np.linspace(0.4, 1.0, batch)
    ref = oracle_mod.init(batch, L, seed=seed)
    Eo, Mo = oracle_mod.sweep_bonds(ref, Jh, Jv, beta, 1.0, 0.0, seed=seed, n_sweeps=n, trace=True)
    with _mk(batch, L, seed) as sim:
        sim.spin_set_bonds(Jh[0], Jv[0])
        E, M = sim.spin_sweep_measure(beta, 1.0, 0.0, n, 0)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
        assert np.array_equal(sim.spin_get_spins(), ref)
        sim.spin_set_bonds(None, None)
        sim.spin_sweep(beta, 1.0, 0.0, 2, n)
        oracle_mod.sweep(ref, beta, 1.0, 0.0, seed=seed, n_sweeps=2, sweep_offset=n)
        assert np.array_equal(sim.spin_get_spins(), ref)
        assert np.array_equal(sim.spin_observables()[0], oracle_mod.ising_observables(ref)[0])


def test_mattis_gauge_on_the_gpu(oracle_mod):
    """J_ij = xi_i xi_j, s' = xi s: the GPU trajectory with bonds is the gauge image of its own uniform trajectory."""
    L, batch, seed = 64, 4, 17
    rng = np.random.default_rng(3)
    xi = (2 * rng.integers(0, 2, size=(batch, L, L)) - 1).astype(np.int8)
    Jh, Jv = xi * np.roll(xi, -1, axis=2), xi * np.roll(xi, -1, axis=1)
    beta = [0.2, 0.44, 0.7, 1.5]
    with _mk(batch, L, seed) as f, _mk(batch, L, seed) as g:
        g.spin_set_spins((f.spin_get_spins() * xi).astype(np.int8))
        g.spin_set_bonds(Jh, Jv)
        f.spin_sweep(beta, 1.0, 0.0, 20, 0)
        g.spin_sweep(beta, 1.0, 0.0, 20, 0)
        assert np.array_equal(g.spin_get_spins(), (f.spin_get_spins() * xi).astype(np.int8))
        assert np.array_equal(g.spin_observables()[0], f.spin_observables()[0])


def test_set_bonds_argument_checks():
    Jh, Jv = _rand_bonds(0, 2, 64)
    with _mk(2, 64, 1) as sim:
        before = sim.spin_get_spins()
        bad = Jh.copy()
        bad[1, 3, 5] = 0
        with pytest.raises(sp.SpinError):
            sim.spin_set_bonds(bad, Jv)
        sim.spin_sweep([0.5, 0.5], 1.0, 0.0, 1, 0)          # still the uniform model
        assert not np.array_equal(sim.spin_get_spins(), before)
    with _mk(2, 64, 1, layout=sp.SPIN_LAYOUT_INT8) as sim:       # int8 layout: accepted (general kernels), still validated
        with pytest.raises(sp.SpinError):
            sim.spin_set_bonds(bad, Jv)
        sim.spin_set_bonds(Jh, Jv)
        with pytest.raises(sp.SpinError):                          # bond signs and real couplings exclude each other
            sim.spin_set_couplings(Jh.astype(float), Jv.astype(float), np.zeros((2, 64, 64)))
