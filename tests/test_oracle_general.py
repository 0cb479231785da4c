"""Pins of the general-coupling oracle (oracle/general_oracle.cpp; Eq. 1 with J_ij and B_i, Eq. 5 with the field term,
PAPER.md:99-103, 166): special cases that reduce to the already pinned uniform / +-J oracle bit for bit, an exact gauge
symmetry, brute-force Boltzmann sums on tiny lattices, limits, and observables against explicit numpy definitions."""
import itertools

import numpy as np
import pytest

import oracle


def test_uniform_couplings_reduce_to_the_uniform_oracle():
    B, L, seed = 3, 12, 5
    beta = [0.3, 0.44, 0.6]
    for J, h in ((1.0, 0.0), (0.5, 0.25), (2.0, -0.5), (-1.0, 0.125)):     # exactly representable: both dE orders agree
        a = oracle.init(B, L, seed=seed)
        b = a.copy()
        oracle.sweep(a, beta, J, h, seed=seed, n_sweeps=6)
        oracle.sweep_general(b, np.full((L, L), J), np.full((L, L), J), np.full((L, L), h), beta, seed, 6)
        assert np.array_equal(a, b), (J, h)


def test_pm1_couplings_reduce_to_the_bond_sign_oracle():
    B, L, seed = 2, 10, 8
    rng = np.random.default_rng(1)
    Jh = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    Jv = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    a = oracle.init(B, L, seed=seed)
    b = a.copy()
    oracle.sweep_bonds(a, Jh, Jv, [0.5, 0.9], 1.0, 0.25, seed, 5, sweep_offset=3)
    oracle.sweep_general(b, Jh.astype(float), Jv.astype(float), np.full((B, L, L), 0.25), [0.5, 0.9], seed, 5, sweep_offset=3)
    assert np.array_equal(a, b)
    E, M = oracle.ising_general_observables(b, Jh.astype(float), Jv.astype(float), np.zeros((B, L, L)))
    Eo, Mo = oracle.ising_bonds_observables(b, Jh, Jv)
    assert np.array_equal(E, Eo.astype(float)) and np.array_equal(M, Mo)


def test_gauge_transformation_maps_trajectories_exactly():
    """s' = x s, J'_ij = x_i J_ij x_j, B'_i = x_i B_i with x = +-1: dE is bitwise the same (sign changes are exact), so the
    trajectories map onto each other at every sweep.  Breaks if any of the four bonds is mis-indexed."""
    B, L, seed = 2, 8, 13
    rng = np.random.default_rng(2)
    Jh, Jv, Bf = rng.normal(size=(B, L, L)), rng.normal(size=(B, L, L)), 0.3 * rng.normal(size=(B, L, L))
    x = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    Jh2 = x * Jh * np.roll(x, -1, axis=2)
    Jv2 = x * Jv * np.roll(x, -1, axis=1)
    a = oracle.init(B, L, seed=seed)
    b = (a * x).astype(np.int8)
    for t in range(6):
        oracle.sweep_general(a, Jh, Jv, Bf, [0.4, 1.1], seed, 1, sweep_offset=t)
        oracle.sweep_general(b, Jh2, Jv2, x * Bf, [0.4, 1.1], seed, 1, sweep_offset=t)
        assert np.array_equal(b, a * x), t
    Ea, _ = oracle.ising_general_observables(a, Jh, Jv, Bf)
    Eb, _ = oracle.ising_general_observables(b, Jh2, Jv2, x * Bf)
    assert np.allclose(Ea, Eb, rtol=0, atol=1e-12)


def _all_states(n):
    return np.array(list(itertools.product((-1, 1), repeat=n)), dtype=np.int8)


def test_long_run_energy_matches_the_boltzmann_sum_on_4x4_with_random_real_couplings():
    L, seed, beta, R = 4, 3, 0.7, 512
    rng = np.random.default_rng(7)
    Jh, Jv, Bf = rng.normal(size=(L, L)), rng.normal(size=(L, L)), 0.5 * rng.normal(size=(L, L))
    states = _all_states(L * L).reshape(-1, L, L)
    E = -(Jh * states * np.roll(states, -1, axis=2)).sum((1, 2)) - (Jv * states * np.roll(states, -1, axis=1)).sum((1, 2)) \
        - (Bf * states).sum((1, 2))
    w = np.exp(-beta * (E - E.min()))
    exact_E = float((w * E).sum() / w.sum())
    exact_M = float((w * states.sum((1, 2))).sum() / w.sum())
    lat = oracle.init(R, L, seed=seed)
    oracle.sweep_general(lat, Jh, Jv, Bf, beta, seed, 200)
    accE, accM, n = np.zeros(R), np.zeros(R), 0
    for t in range(200, 600):
        oracle.sweep_general(lat, Jh, Jv, Bf, beta, seed, 1, sweep_offset=t)
        e, m = oracle.ising_general_observables(lat, Jh, Jv, Bf)
        accE += e; accM += m; n += 1
    for acc, exact in ((accE / n, exact_E), (accM / n, exact_M)):
        se = acc.std(ddof=1) / np.sqrt(R)
        assert abs(acc.mean() - exact) <= 4 * se + 1e-9, (acc.mean(), exact, se)


def test_observables_against_an_explicit_bond_list():
    B, L = 2, 6
    rng = np.random.default_rng(4)
    s = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    Jh, Jv, Bf = rng.normal(size=(B, L, L)), rng.normal(size=(B, L, L)), rng.normal(size=(B, L, L))
    E, M = oracle.ising_general_observables(s, Jh, Jv, Bf)
    for b in range(B):
        e = 0.0
        for i in range(L):
            for j in range(L):
                e -= Jh[b, i, j] * s[b, i, j] * s[b, i, (j + 1) % L] + Jv[b, i, j] * s[b, i, j] * s[b, (i + 1) % L, j]
                e -= Bf[b, i, j] * s[b, i, j]
        assert abs(E[b] - e) < 1e-10 and M[b] == s[b].sum()


def test_large_field_and_low_temperature_limits():
    L, seed = 8, 2
    lat = oracle.init(2, L, seed=seed)
    field = np.where(np.indices((L, L)).sum(0) % 3 == 0, -50.0, 50.0)          # |B| beats any neighbour sum
    oracle.sweep_general(lat, np.ones((L, L)), np.ones((L, L)), field, [5.0, 5.0], seed, 2)
    assert np.array_equal(lat[0], np.sign(field).astype(np.int8)) and np.array_equal(lat[1], lat[0])


# ---- Potts with a field on the state label and +-1 bond signs ---------------------------------------------------------
def test_potts_general_reduces_to_the_potts_oracle():
    B, L, seed, q = 3, 10, 4, [3, 5, 8]
    beta = [0.8, 1.0, 1.4]
    a = oracle.init(B, L, seed=seed, q=q)
    b, c = a.copy(), a.copy()
    oracle.sweep(a, beta, 1.0, 0.0, seed=seed, n_sweeps=5, q=q)
    oracle.sweep_potts_general(b, q, beta, 1.0, 0.0, seed, 5)
    oracle.sweep_potts_general(c, q, beta, 1.0, 0.0, seed, 5, Jh=np.ones((L, L), np.int8), Jv=np.ones((L, L), np.int8))
    assert np.array_equal(a, b) and np.array_equal(a, c)
    E, S, M = oracle.potts_general_observables(a, q)
    Eo, Mo = oracle.potts_observables(a, q)
    assert np.array_equal(E, Eo) and np.array_equal(M, Mo) and np.array_equal(S, a.astype(np.int64).sum((1, 2)))


@pytest.mark.parametrize("q,h,bonds", [(3, 0.4, False), (3, -0.3, True), (4, 0.25, True)])
def test_potts_field_long_run_matches_the_boltzmann_sum_on_2x2(q, h, bonds):
    L, seed, beta, J, R = 2, 6, 0.9, 1.0, 768
    rng = np.random.default_rng(q)
    Jh = (2 * rng.integers(0, 2, size=(L, L)) - 1).astype(np.int8) if bonds else None
    Jv = (2 * rng.integers(0, 2, size=(L, L)) - 1).astype(np.int8) if bonds else None
    states = np.array(list(itertools.product(range(q), repeat=4)), dtype=np.int8).reshape(-1, L, L)
    Eint, S, _ = oracle.potts_general_observables(np.ascontiguousarray(states), q, Jh, Jv)   # explicit check of these below
    H = J * Eint - h * S
    w = np.exp(-beta * (H - H.min()))
    exact = float((w * H).sum() / w.sum())
    lat = oracle.init(R, L, seed=seed, q=q)
    oracle.sweep_potts_general(lat, q, beta, J, h, seed, 100, Jh, Jv)
    acc, n = np.zeros(R), 0
    for t in range(100, 500):
        oracle.sweep_potts_general(lat, q, beta, J, h, seed, 1, Jh, Jv, sweep_offset=t)
        e, s, _ = oracle.potts_general_observables(lat, q, Jh, Jv)
        acc += J * e - h * s; n += 1
    se = (acc / n).std(ddof=1) / np.sqrt(R)
    assert abs((acc / n).mean() - exact) <= 4 * se + 1e-9, ((acc / n).mean(), exact, se)


def test_potts_general_observables_against_explicit_loops():
    B, L, q = 2, 4, 5
    rng = np.random.default_rng(11)
    s = rng.integers(0, q, size=(B, L, L)).astype(np.int8)
    Jh = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    Jv = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    E, S, M = oracle.potts_general_observables(s, q, Jh, Jv)
    for b in range(B):
        e = 0
        for i in range(L):
            for j in range(L):
                e -= Jh[b, i, j] * int(s[b, i, j] == s[b, i, (j + 1) % L]) + Jv[b, i, j] * int(s[b, i, j] == s[b, (i + 1) % L, j])
        assert E[b] == e and S[b] == s[b].sum() and M[b] == np.bincount(s[b].ravel()).max()


def test_potts_strong_field_at_low_temperature_selects_the_top_label():
    L, seed, q = 6, 9, 4
    lat = oracle.init(2, L, seed=seed, q=q)
    oracle.sweep_potts_general(lat, q, [8.0, 8.0], 1.0, 30.0, seed, 40)
    assert np.all(lat == q - 1)
    lat = oracle.init(2, L, seed=seed, q=q)
    oracle.sweep_potts_general(lat, q, [8.0, 8.0], 1.0, -30.0, seed, 40)
    assert np.all(lat == 0)


def test_schedule_equals_the_same_sweeps_called_one_by_one():
    B, L, seed = 2, 8, 12
    steps = np.array([[0.2, 0.3], [0.5, 0.6], [1.0, 1.2]])
    a = oracle.init(B, L, seed=seed)
    b = a.copy()
    oracle.sweep_schedule(a, steps, 1.0, 0.0, seed, 4, sweep_offset=2)
    for k in range(3):
        oracle.sweep(b, steps[k], 1.0, 0.0, seed=seed, n_sweeps=4, sweep_offset=2 + 4 * k)
    assert np.array_equal(a, b)
