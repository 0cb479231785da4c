"""Pins of the other-geometry oracle (oracle/stencil_oracle.cpp): triangular lattice,
3D cubic lattice, square lattice with second neighbours.  Brute-force Boltzmann sums over every state of tiny lattices
(energies from an explicit bond list written here), the exact 4x4 square-lattice values of SURVEY Q7 for J2 = 0,
RNG-free limits, the colouring property the checkerboard needs, and one site recomputed by hand."""
import itertools

import numpy as np
import pytest

import oracle
from oracle import STENCIL_CUBIC as CUB, STENCIL_SQUARE_NNN as NNN, STENCIL_TRIANGULAR as TRI

OFFS = {TRI: ([(-1, 0), (1, 0), (0, -1), (0, 1), (1, 1), (-1, -1)], []),
        CUB: ([(-1, 0, 0), (1, 0, 0), (0, -1, 0), (0, 1, 0), (0, 0, -1), (0, 0, 1)], []),
        NNN: ([(-1, 0), (1, 0), (0, -1), (0, 1)], [(-1, -1), (-1, 1), (1, -1), (1, 1)])}


def _bond_sums(stencil, s):
    """(sum over first-neighbour bonds of s s', same for second neighbours), each bond once, for [..., *lattice] arrays:
    half of the sum over all ordered neighbour pairs (with multiplicity)."""
    nd = 3 if stencil == CUB else 2
    axes = tuple(range(s.ndim - nd, s.ndim))
    out = []
    for offs in OFFS[stencil]:
        tot = np.zeros(s.shape[:-nd], dtype=np.int64)
        for o in offs:
            tot += (s.astype(np.int64) * np.roll(s, tuple(-x for x in o), axis=axes)).sum(axes)
        out.append(tot // 2)
    return out


def _colour(stencil, idx):
    if stencil == TRI:
        return (idx[0] + idx[1]) % 3
    if stencil == CUB:
        return (idx[0] + idx[1] + idx[2]) & 1
    return 2 * (idx[0] & 1) + (idx[1] & 1)


@pytest.mark.parametrize("stencil,L", [(TRI, 3), (TRI, 6), (TRI, 9), (CUB, 2), (CUB, 4), (NNN, 2), (NNN, 4), (NNN, 6)])
def test_colour_classes_are_independent_sets_and_observables_match_bond_lists(stencil, L):
    shape = oracle.stencil_shape(stencil, 1, L)[1:]
    idx = np.indices(shape)
    col = _colour(stencil, idx)
    for offs in OFFS[stencil]:
        for o in offs:
            nb = np.roll(col, tuple(-x for x in o), axis=tuple(range(len(shape))))
            if L > 2:
                assert not np.any(nb == col), (stencil, L, o)          # no neighbour shares a site's colour
    s = oracle.stencil_init(stencil, 3, L, seed=5)
    E1, E2, M = oracle.stencil_observables(stencil, s)
    b1, b2 = _bond_sums(stencil, s)
    assert np.array_equal(E1, -b1) and np.array_equal(E2, -b2) and np.array_equal(M, s.reshape(3, -1).sum(1))


@pytest.mark.parametrize("stencil,L", [(TRI, 6), (CUB, 4), (NNN, 6)])
def test_beta_zero_flips_everything_and_a_pass_touches_one_colour(stencil, L):
    s = oracle.stencil_init(stencil, 2, L, seed=3)
    a = s.copy()
    oracle.stencil_sweep(stencil, a, 0.0, 1.0, 0.5, 0.1, 3, 1)
    assert np.array_equal(a, -s)
    b = s.copy()
    oracle.stencil_colour_pass(stencil, b, 0.0, 1.0, 0.5, 0.1, 3, 0, 1)
    col = _colour(stencil, np.indices(s.shape[1:]))
    assert np.array_equal(b[:, col == 1], -s[:, col == 1]) and np.array_equal(b[:, col != 1], s[:, col != 1])


@pytest.mark.parametrize("stencil,L", [(TRI, 6), (CUB, 4), (NNN, 4)])
def test_low_temperature_energy_never_increases_and_ground_state_is_fixed(stencil, L):
    J1, J2, h = 1.0, 0.5, 0.0
    s = oracle.stencil_init(stencil, 2, L, seed=8)
    ncol = {TRI: 3, CUB: 2, NNN: 4}[stencil]
    E1, E2, _ = oracle.stencil_observables(stencil, s)
    prev = J1 * E1 + J2 * E2
    for t in range(4):
        for c in range(ncol):
            oracle.stencil_colour_pass(stencil, s, 30.0, J1, J2, h, 8, t, c)
            E1, E2, _ = oracle.stencil_observables(stencil, s)
            cur = J1 * E1 + J2 * E2
            assert np.all(cur <= prev)
            prev = cur
    up = np.ones_like(s)
    oracle.stencil_sweep(stencil, up, 30.0, J1, J2, h, 8, 3)
    assert np.all(up == 1)


def _exact(stencil, shape, beta, J1, J2, h):
    n = int(np.prod(shape))
    states = np.array(list(itertools.product((-1, 1), repeat=n)), dtype=np.int8).reshape((-1,) + shape)
    b1, b2 = _bond_sums(stencil, states)
    M = states.reshape(len(states), -1).sum(1).astype(np.int64)
    H = -J1 * b1 - J2 * b2 - h * M
    w = np.exp(-beta * (H - H.min()))
    return float((w * H).sum() / w.sum()), float((w * np.abs(M)).sum() / w.sum())


@pytest.mark.parametrize("stencil,L,beta,J1,J2,h", [
    # (3x3 triangular at h = 0 has closed deterministic cycles under "dE <= 0 always accepts", like the 2x2 square
    # lattice of SURVEY W1: a property of the rule, so the brute-force comparisons use a small field there)
    (TRI, 3, 0.25, 1.0, 0.0, 0.15), (TRI, 3, 0.5, -1.0, 0.0, 0.1),       # ferromagnet; frustrated antiferromagnet
    (TRI, 3, 0.3, 1.0, 0.0, -0.2),
    (CUB, 2, 0.15, 1.0, 0.0, 0.0), (CUB, 2, 0.1, 1.0, 0.0, 0.3),          # 2x2x2: every neighbour counted twice
    (NNN, 4, 0.3, 1.0, 0.5, 0.0), (NNN, 4, 0.4, 1.0, -0.4, 0.1), (NNN, 2, 0.2, 1.0, 0.3, 0.0)])
def test_long_run_averages_match_brute_force_boltzmann_sums(stencil, L, beta, J1, J2, h):
    shape = oracle.stencil_shape(stencil, 1, L)[1:]
    exact_H, exact_absM = _exact(stencil, shape, beta, J1, J2, h)
    R, seed = 512, 17
    s = oracle.stencil_init(stencil, R, L, seed=seed)
    oracle.stencil_sweep(stencil, s, beta, J1, J2, h, seed, 200)
    accH, accM, n = np.zeros(R), np.zeros(R), 0
    for t in range(200, 600):
        oracle.stencil_sweep(stencil, s, beta, J1, J2, h, seed, 1, sweep_offset=t)
        E1, E2, M = oracle.stencil_observables(stencil, s)
        accH += J1 * E1 + J2 * E2 - h * M
        accM += np.abs(M)
        n += 1
    for acc, exact in ((accH / n, exact_H), (accM / n, exact_absM)):
        se = acc.std(ddof=1) / np.sqrt(R)
        assert abs(acc.mean() - exact) <= 4 * se + 1e-9, (acc.mean(), exact, se)


def test_square_nnn_with_J2_zero_samples_the_square_lattice_ising_model():
    """4x4, J2 = 0, beta = 0.44: <E>/N = -1.562847028104, <|M|>/N = 0.842715640981 (exact enumeration)."""
    R, seed, L, beta = 1024, 23, 4, 0.44
    s = oracle.stencil_init(NNN, R, L, seed=seed)
    oracle.stencil_sweep(NNN, s, beta, 1.0, 0.0, 0.0, seed, 200)
    accE, accM, n = np.zeros(R), np.zeros(R), 0
    for t in range(200, 500):
        oracle.stencil_sweep(NNN, s, beta, 1.0, 0.0, 0.0, seed, 1, sweep_offset=t)
        E1, _, M = oracle.stencil_observables(NNN, s)
        accE += E1 / 16.0; accM += np.abs(M) / 16.0; n += 1
    for acc, exact in ((accE / n, -1.562847028104), (accM / n, 0.842715640981)):
        assert abs(acc.mean() - exact) <= 4 * acc.std(ddof=1) / np.sqrt(R)


@pytest.mark.parametrize("stencil,L,site", [(TRI, 6, (4, 3)), (CUB, 4, (1, 2, 2)), (NNN, 6, (3, 4))])
def test_one_site_by_hand(stencil, L, site):
    seed, t, beta, J1, J2, h, b, roff = 0xABCDEF0123456789, (1 << 32) + 9, 0.35, 1.0, 0.6, 0.1, 1, 4
    s = oracle.stencil_init(stencil, 2, L, seed=seed)
    col = _colour(stencil, np.indices(s.shape[1:]))
    c = int(col[site])
    flat_same = np.flatnonzero(col.ravel() == c)
    n = int(np.searchsorted(flat_same, np.ravel_multi_index(site, s.shape[1:])))     # index among the colour's sites
    ctr = [n >> 2, b + roff, t & 0xFFFFFFFF, ((t >> 32) & 0xFFFFFF) | (c << 24) | (3 << 28)]
    r = int(oracle.philox4x32_10(ctr, [seed & 0xFFFFFFFF, seed >> 32])[n & 3])
    lat = s[b]
    nn = [sum(int(lat[tuple((np.array(site) + np.array(o)) % L)]) for o in offs) for offs in OFFS[stencil]]
    dE = 2.0 * float(lat[site]) * (J1 * nn[0] + J2 * nn[1] + h)
    accept = dE <= 0 or r < int(np.floor(np.exp(-beta * dE) * 2.0 ** 32))
    x = s.copy()
    oracle.stencil_colour_pass(stencil, x, beta, J1, J2, h, seed, t, c, replica_offset=roff)
    assert x[b][site] == (-lat[site] if accept else lat[site])
    # initial value of that site: natural index p, group p >> 2, word p & 3, domain INIT
    p = int(np.ravel_multi_index(site, s.shape[1:]))
    w = int(oracle.philox4x32_10([p >> 2, b, 0, 0], [seed & 0xFFFFFFFF, seed >> 32])[p & 3])
    assert lat[site] == (1 if w & 0x80000000 else -1)


def test_chunking_and_replica_independence():
    for stencil, L in ((TRI, 6), (CUB, 4), (NNN, 6)):
        s = oracle.stencil_init(stencil, 3, L, seed=2)
        a, c = s.copy(), s.copy()
        beta = [0.2, 0.3, 0.4]
        oracle.stencil_sweep(stencil, a, beta, 1.0, 0.2, 0.0, 2, 7)
        oracle.stencil_sweep(stencil, c, beta, 1.0, 0.2, 0.0, 2, 3)
        oracle.stencil_sweep(stencil, c, beta, 1.0, 0.2, 0.0, 2, 4, sweep_offset=3)
        assert np.array_equal(a, c)
        one = oracle.stencil_init(stencil, 1, L, seed=2, replica_offset=2)
        assert np.array_equal(one[0], s[2])
        oracle.stencil_sweep(stencil, one, beta[2:], 1.0, 0.2, 0.0, 2, 7, replica_offset=2)
        assert np.array_equal(one[0], a[2])
