"""Pins of the Cellular-Potts oracle (oracle/cpm_oracle.cpp; Eq. 7, Table II).  The energy change of
a proposal is checked against the difference of an explicit Eq.-7 Hamiltonian written here (exact integers), the
proposal direction / random words / acceptance by a by-hand site through the exported Philox, the beta = 0 pass by a
numpy gather, and the invariants of a copy dynamics."""
import numpy as np
import pytest

import oracle
from paper_2304_01772_b200 import workloads

MOORE = [(-1, -1), (-1, 0), (-1, 1), (0, -1), (0, 1), (1, -1), (1, 0), (1, 1)]
JT = workloads.CPM_TABLE_II


def hamiltonian(lat, tau, Jtab, lam, A):
    """Eq. 7 as written: 1/2 sum_x sum_{y in Moore(x)} J (1 - delta) + lambda sum_{cells} (a - A)^2."""
    L = lat.shape[0]
    tot = 0
    for i in range(L):
        for j in range(L):
            for di, dj in MOORE:
                sy = lat[(i + di) % L, (j + dj) % L]
                if sy != lat[i, j]:
                    tot += int(Jtab[tau[lat[i, j]], tau[sy]])
    assert tot % 2 == 0
    area = np.bincount(lat.ravel(), minlength=len(tau))
    return tot // 2 + lam * int(((area[1:] - A[1:]) ** 2).sum())


def _random_setup(L, q, seed):
    rng = np.random.default_rng(seed)
    lat = rng.integers(0, q, size=(L, L)).astype(np.int8)
    tau = np.concatenate([[0], rng.integers(1, 3, size=q - 1)]).astype(np.int32)
    A = np.concatenate([[0], rng.integers(1, 9, size=q - 1)]).astype(np.int32)
    return lat, tau, A


@pytest.mark.parametrize("L,q,lam", [(4, 3, 1), (6, 5, 2), (8, 9, 0), (2, 3, 1)])
def test_delta_equals_difference_of_the_explicit_hamiltonian(L, q, lam):
    lat, tau, A = _random_setup(L, q, 10 * L + q)
    rng = np.random.default_rng(1)
    H0 = hamiltonian(lat, tau, JT, lam, A)
    for _ in range(40):
        i, j, new = int(rng.integers(0, L)), int(rng.integers(0, L)), int(rng.integers(0, q))
        after = lat.copy()
        after[i, j] = new
        assert oracle.cpm_delta(lat, tau, JT, lam, A, i, j, new) == hamiltonian(after, tau, JT, lam, A) - H0, (i, j, new)


def test_observables_match_the_explicit_hamiltonian_and_counts():
    lat, tau, A = _random_setup(8, 7, 3)
    spins = np.ascontiguousarray(np.stack([lat, np.roll(lat, 3, axis=1)]))
    Ha, Hr, areas, bl = oracle.cpm_observables(spins, tau, JT, 2, A)
    for b in range(2):
        assert Ha[b] + Hr[b] == hamiltonian(spins[b], tau, JT, 2, A)
        assert np.array_equal(areas[b], np.bincount(spins[b].ravel(), minlength=7)) and areas[b].sum() == 64
        cnt = np.zeros((3, 3), dtype=np.int64)
        for i in range(8):
            for j in range(8):
                for di, dj in MOORE:
                    s, sy = spins[b, i, j], spins[b, (i + di) % 8, (j + dj) % 8]
                    if s != sy:
                        lo, hi = sorted((tau[s], tau[sy]))
                        cnt[lo, hi] += 1
        assert np.array_equal(bl[b], cnt // 2)


def test_one_site_by_hand():
    L, q, seed, t, b, roff, lam, beta = 8, 6, 0x0123456789ABCDEF, (1 << 32) + 2, 1, 3, 1, 0.125
    lat, tau, A = _random_setup(L, q, 5)
    spins = np.ascontiguousarray(np.stack([lat, lat.T.copy()]))
    i, j = 5, 2                                                   # colour 2 (5 & 1) + (2 & 1) = 2
    c = 2
    n = (i >> 1) * (L // 2) + (j >> 1)
    w = oracle.philox4x32_10([n >> 1, b + roff, t & 0xFFFFFFFF, ((t >> 32) & 0xFFFFFF) | (c << 24) | (4 << 28)],
                             [seed & 0xFFFFFFFF, seed >> 32])
    r_prop, r_acc = int(w[2 * (n & 1)]), int(w[2 * (n & 1) + 1])
    di, dj = MOORE[r_prop >> 29]
    cur = spins[b]
    new = int(cur[(i + di) % L, (j + dj) % L])
    after = cur.copy(); after[i, j] = new
    dH = hamiltonian(after, tau, JT, lam, A) - hamiltonian(cur, tau, JT, lam, A)
    accept = dH <= 0 or r_acc < int(np.floor(np.exp(-beta * dH) * 2.0 ** 32))
    x = spins.copy()
    oracle.cpm_colour_pass(x, tau, JT, lam, A, beta, seed, t, c, replica_offset=roff)
    assert x[b, i, j] == (new if accept else cur[i, j])


def test_beta_zero_pass_is_a_gather_from_the_chosen_neighbour():
    L, q, seed, t = 10, 8, 77, 4
    lat, tau, A = _random_setup(L, q, 9)
    spins = np.ascontiguousarray(lat[None])
    for c in range(4):
        expect = spins[0].copy()
        for i in range(c >> 1, L, 2):
            for j in range(c & 1, L, 2):
                n = (i >> 1) * (L // 2) + (j >> 1)
                w = oracle.philox4x32_10([n >> 1, 0, t, (c << 24) | (4 << 28)], [seed, 0])
                di, dj = MOORE[int(w[2 * (n & 1)]) >> 29]
                expect[i, j] = spins[0, (i + di) % L, (j + dj) % L]
        oracle.cpm_colour_pass(spins, tau, JT, 1, A, 0.0, seed, t, c)
        assert np.array_equal(spins[0], expect), c


def test_invariants_of_the_copy_dynamics():
    B, L = 3, 40
    spins, tau, A = workloads.cpm_initial(B, L, cells_per_side=6, cell_size=5, seed=2)
    spins = spins.copy()
    ids0 = set(np.unique(spins))
    H0 = sum(oracle.cpm_observables(spins, tau, JT, 1, A)[k] for k in (0, 1))
    oracle.cpm_sweep(spins, tau, JT, 1, A, [0.125, 0.125, 0.5], 4, 30)
    Ha, Hr, areas, bl = oracle.cpm_observables(spins, tau, JT, 1, A)
    assert set(np.unique(spins)) <= ids0 and np.all(areas.sum(1) == L * L)
    assert not np.array_equal(spins[0], spins[1])                  # replicas draw different words
    # an all-medium lattice never changes; a lattice filled by one cell with lambda = 0 neither
    z = np.zeros((1, 8, 8), dtype=np.int8)
    oracle.cpm_sweep(z, tau, JT, 1, A, 0.125, 1, 5)
    assert not z.any()
    one = np.full((1, 8, 8), 3, dtype=np.int8)
    oracle.cpm_sweep(one, tau, JT, 0, A, 0.125, 1, 5)
    assert np.all(one == 3)
    # cold dynamics lower the energy of the square aggregate (cell sorting / rounding)
    cold = workloads.cpm_initial(1, L, seed=2)[0].copy()
    oracle.cpm_sweep(cold, tau, JT, 1, A, 2.0, 4, 30)
    assert sum(oracle.cpm_observables(cold, tau, JT, 1, A)[k][0] for k in (0, 1)) < H0[0]


def test_chunking_and_replica_offset():
    spins, tau, A = workloads.cpm_initial(2, 36, seed=1)
    a, c = spins.copy(), spins.copy()
    oracle.cpm_sweep(a, tau, JT, 1, A, 0.125, 9, 6)
    oracle.cpm_sweep(c, tau, JT, 1, A, 0.125, 9, 2)
    oracle.cpm_sweep(c, tau, JT, 1, A, 0.125, 9, 4, sweep_offset=2)
    assert np.array_equal(a, c)
    one = spins[1:2].copy()
    oracle.cpm_sweep(one, tau, JT, 1, A, 0.125, 9, 6, replica_offset=1)
    assert np.array_equal(one[0], a[1])


def test_table_ii_and_parameters_are_the_papers():
    """workloads.CPM_TABLE_II / cpm_initial against the values the paper prints (tests/golden/cpm_table_ii.txt)."""
    import os
    idx = {"medium": 0, "light": 1, "dark": 2}
    want = np.full((3, 3), -1, dtype=np.int64)
    params = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "cpm_table_ii.txt")):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] in idx:
            want[idx[f[0]], idx[f[1]]] = want[idx[f[1]], idx[f[0]]] = int(f[2])      # symmetric
        else:
            params[f[0]] = int(f[1])
    assert np.array_equal(workloads.CPM_TABLE_II, want)
    spins, tau, A = workloads.cpm_initial(1, 40)
    assert len(tau) == params["identifiers"] and tau[0] == 0 and set(tau[1:]) <= {1, 2}
    assert np.all(A[1:] == params["A"]) and np.all(np.bincount(spins.ravel(), minlength=37)[1:] == params["A"])
