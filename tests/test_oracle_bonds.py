"""Pins for the oracle's +-J couplings (Eq. 1 with per-bond J_ij; the
+-J spin glass of Fig. 9).  None of them re-uses the oracle's own formula: uniform bonds must reproduce
the uniform model bit for bit, a Mattis gauge transformation must map trajectories exactly, the zero-temperature
half-sweep is recomputed with numpy rolls, the observables with an independent definition, and the long-run energy is
compared with a brute-force Boltzmann average over all 2^16 states of a 4x4 torus."""
import numpy as np
import pytest


def _rand_bonds(rng, B, L):
    return ((2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8),
            (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8))


def _local_field(s, Jh, Jv):
    """nn_eff with numpy rolls: right, left, down, up neighbours weighted by the bond that joins them."""
    return (Jh * np.roll(s, -1, axis=2) + np.roll(Jh, 1, axis=2) * np.roll(s, 1, axis=2) +
            Jv * np.roll(s, -1, axis=1) + np.roll(Jv, 1, axis=1) * np.roll(s, 1, axis=1))


@pytest.mark.parametrize("L", [2, 4, 6, 16])
def test_uniform_bonds_equal_the_uniform_model(oracle_mod, L):
    B, beta = 3, [0.2, 0.44, 0.9]
    a = oracle_mod.init(B, L, seed=7)
    b = a.copy()
    ones = np.ones((B, L, L), dtype=np.int8)
    Ea, Ma = oracle_mod.sweep(a, beta, 1.0, 0.05, seed=7, n_sweeps=9, trace=True)
    Eb, Mb = oracle_mod.sweep_bonds(b, ones, ones, beta, 1.0, 0.05, seed=7, n_sweeps=9, trace=True)
    assert np.array_equal(a, b) and np.array_equal(Ea, Eb) and np.array_equal(Ma, Mb)
    # all bonds -1 with J = -1 is the same Hamiltonian again
    c = oracle_mod.init(B, L, seed=7)
    oracle_mod.sweep_bonds(c, -ones, -ones, beta, -1.0, 0.05, seed=7, n_sweeps=9)
    assert np.array_equal(a, c)


@pytest.mark.parametrize("L", [2, 4, 10])
def test_mattis_gauge_maps_trajectories_exactly(oracle_mod, L):
    """J_ij = xi_i xi_j and s' = xi s: same energy changes, same random words, so s'(t) = xi s(t) for all t."""
    B, beta = 4, [0.1, 0.44, 0.7, 20.0]
    rng = np.random.default_rng(L)
    xi = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    Jh, Jv = xi * np.roll(xi, -1, axis=2), xi * np.roll(xi, -1, axis=1)
    f = oracle_mod.init(B, L, seed=11)
    g = (f * xi).astype(np.int8)
    for t in range(8):
        oracle_mod.sweep(f, beta, 1.0, 0.0, seed=11, n_sweeps=1, sweep_offset=t)
        oracle_mod.sweep_bonds(g, Jh, Jv, beta, 1.0, 0.0, seed=11, n_sweeps=1, sweep_offset=t)
        assert np.array_equal(g, (f * xi).astype(np.int8)), "gauge image differs after sweep %d" % t
        assert np.array_equal(oracle_mod.ising_observables(f)[0], oracle_mod.ising_bonds_observables(g, Jh, Jv)[0])


def test_zero_temperature_half_sweep_recomputed_with_rolls(oracle_mod):
    """beta = 20, h = 0: every threshold of a dE > 0 class is 0, so a site flips iff s * nn_eff <= 0."""
    B, L = 3, 8
    rng = np.random.default_rng(5)
    Jh, Jv = _rand_bonds(rng, B, L)
    s = oracle_mod.init(B, L, seed=2)
    ii, jj = np.meshgrid(np.arange(L), np.arange(L), indexing="ij")
    for t in range(4):
        for colour in (0, 1):
            nn = _local_field(s.astype(np.int64), Jh.astype(np.int64), Jv.astype(np.int64))
            flip = (((ii + jj) & 1) == colour)[None] & (s * nn <= 0)
            expect = np.where(flip, -s, s).astype(np.int8)
            got = s.copy()
            oracle_mod.ising_bonds_half_sweep(got, Jh, Jv, 20.0, 1.0, 0.0, seed=9, t=t, colour=colour)
            assert np.array_equal(got, expect), "sweep %d colour %d" % (t, colour)
            s = got


def test_observables_against_an_independent_definition(oracle_mod):
    B, L = 4, 6
    rng = np.random.default_rng(9)
    Jh, Jv = _rand_bonds(rng, B, L)
    s = oracle_mod.init(B, L, seed=3).astype(np.int64)
    E, M = oracle_mod.ising_bonds_observables(s.astype(np.int8), Jh, Jv)
    # every bond once, from an explicit list of (site, site, sign) triples
    Eo = np.zeros(B, dtype=np.int64)
    for b in range(B):
        for i in range(L):
            for j in range(L):
                Eo[b] -= Jh[b, i, j] * s[b, i, j] * s[b, i, (j + 1) % L]
                Eo[b] -= Jv[b, i, j] * s[b, i, j] * s[b, (i + 1) % L, j]
    assert np.array_equal(E, Eo) and np.array_equal(M, s.sum(axis=(1, 2)))
    # and half the bond-weighted local-field sum
    assert np.array_equal(E, -(s * _local_field(s, Jh.astype(np.int64), Jv.astype(np.int64))).sum(axis=(1, 2)) // 2)


def test_long_run_energy_matches_brute_force_boltzmann_average(oracle_mod):
    """4x4 torus, one random +-J sample, beta = 0.5, h = 0.1: <E> over all 2^16 states vs 512 replicas x 400 sweeps."""
    L, beta, h, R = 4, 0.5, 0.1, 512
    rng = np.random.default_rng(123)
    Jh1, Jv1 = _rand_bonds(rng, 1, L)
    states = ((np.arange(1 << 16)[:, None] >> np.arange(16)[None]) & 1).astype(np.int64) * 2 - 1
    S = states.reshape(-1, L, L)
    bond = (Jh1[0] * S * np.roll(S, -1, axis=2) + Jv1[0] * S * np.roll(S, -1, axis=1)).sum(axis=(1, 2))
    H = -bond - h * S.sum(axis=(1, 2))
    w = np.exp(-beta * (H - H.min()))
    exact = float((w * H).sum() / w.sum()) / 16.0
    lat = oracle_mod.init(R, L, seed=77)
    Jh, Jv = np.broadcast_to(Jh1, (R, L, L)), np.broadcast_to(Jv1, (R, L, L))
    oracle_mod.sweep_bonds(lat, Jh, Jv, beta, 1.0, h, seed=77, n_sweeps=200)
    Et, Mt = oracle_mod.sweep_bonds(lat, Jh, Jv, beta, 1.0, h, seed=77, n_sweeps=400, sweep_offset=200, trace=True)
    per_replica = (Et - h * Mt).mean(axis=0) / 16.0
    mean, se = per_replica.mean(), per_replica.std(ddof=1) / np.sqrt(R)
    assert abs(mean - exact) < 4 * se + 1e-3, (mean, exact, se)
