"""Deterministic pins of the oracle (CPU only).  Each test names the SURVEY.md section 8(c) pin
(Q1..Q14) and the PAPER.md passage the pinned function follows."""
import math

import numpy as np
import pytest

from conftest import read_golden


# ---------------------------------------------------------------- Q1: Philox known answers
def test_philox_known_answer_vectors(oracle_mod):
    for name, words in read_golden("philox_kat.txt").items():
        w = [int(x, 16) for x in words]
        out = oracle_mod.philox4x32_10(w[0:4], w[4:6])
        assert [int(x) for x in out] == w[6:10], name


def test_philox_bijection_and_avalanche(oracle_mod):
    # A counter-based generator must give distinct outputs for distinct counters, and one flipped
    # counter bit must change about half of the 128 output bits.
    outs = set()
    base = oracle_mod.philox4x32_10([5, 6, 7, 8], [1, 2])
    flips = []
    for word in range(4):
        for bit in range(0, 32, 5):
            c = [5, 6, 7, 8]
            c[word] ^= 1 << bit
            o = oracle_mod.philox4x32_10(c, [1, 2])
            outs.add(tuple(int(x) for x in o))
            flips.append(sum(bin(int(a) ^ int(b)).count("1") for a, b in zip(o, base)))
    assert len(outs) == 28
    assert 50 < np.mean(flips) < 78


# ---------------------------------------------------------------- Q2: threshold tables
def _closed_form_T(x):
    if x <= 0.0:
        return None
    return min(int(math.floor(math.exp(-x) * 4294967296.0)), 0xFFFFFFFF)


def test_ising_table_closed_form(oracle_mod):
    # dE = H(-s) - H(s) with H = -J s nn - h s  (Eq. 1; reading P1)
    for beta, J, h in [(0.44, 1.0, 0.0), (0.4407, 1.0, 0.01), (0.3, -1.0, 0.2), (1.7, 0.5, -0.3), (0.0, 1.0, 0.0)]:
        T, always = oracle_mod.ising_table(beta, J, h)
        for si, s in enumerate((-1, 1)):
            for ni, nn in enumerate((-4, -2, 0, 2, 4)):
                H_old = -J * s * nn - h * s
                H_new = -J * (-s) * nn - h * (-s)
                want = _closed_form_T(beta * (H_new - H_old))
                idx = 5 * si + ni
                if want is None:
                    assert always[idx]
                else:
                    assert not always[idx]
                    assert abs(int(T[idx]) - want) <= 1  # 1 ulp of exp() may move the floor by one


def test_potts_table_closed_form(oracle_mod):
    for beta, J in [(1.005052538742, 1.0), (0.5, 2.0), (0.9, -1.0), (0.0, 1.0)]:
        T, always = oracle_mod.potts_table(beta, J)
        for di, dn in enumerate(range(-4, 5)):
            want = _closed_form_T(beta * (-J * dn))  # H = -J * (number of equal neighbours)
            if want is None:
                assert always[di]
            else:
                assert not always[di] and abs(int(T[di]) - want) <= 1


def test_tables_survey_values(oracle_mod):
    g = read_golden("threshold_tables.txt")
    bc3 = math.log(1.0 + math.sqrt(3.0))
    cases = {
        "ising beta=0.44 J=1 h=0": oracle_mod.ising_table(0.44, 1.0, 0.0),
        "ising beta=0.4407 J=1 h=0.01": oracle_mod.ising_table(0.4407, 1.0, 0.01),
        "potts3 beta=bc J=1": oracle_mod.potts_table(bc3, 1.0),
    }
    for key, (T, always) in cases.items():
        for idx, tok in enumerate(g[key]):
            if tok == "A":
                assert always[idx], (key, idx)
            else:
                assert not always[idx] and int(T[idx]) == int(tok, 16), (key, idx)


def test_table_extremes(oracle_mod):
    T, always = oracle_mod.ising_table(20.0, 1.0, 0.0)  # exp(-80) 2^32 < 1 -> never accept
    assert [int(t) for t, a in zip(T, always) if not a] == [0, 0, 0, 0]
    T, always = oracle_mod.ising_table(1e-12, 1.0, 0.0)  # p -> 1 clips to 2^32-1, not to "always"
    assert int(T[0]) == 0xFFFFFFFF and not always[0]


# ---------------------------------------------------------------- O3: init
def test_init_keying_and_balance(oracle_mod):
    s = oracle_mod.init(3, 16, seed=7)
    assert set(np.unique(s)) == {-1, 1}
    # site p uses word p&3 of group p>>2, domain INIT: recompute site (b=2, p=37) from the generator
    p, b = 37, 2
    out = oracle_mod.philox4x32_10([p >> 2, b, 0, 0], [7, 0])
    assert s[b].reshape(-1)[p] == (1 if int(out[p & 3]) >> 31 else -1)
    big = oracle_mod.init(1, 256, seed=11)
    assert abs(int(big.sum())) < 4 * 256  # 4 sigma of a fair coin over 65536 sites
    pq = oracle_mod.init(2, 64, seed=3, q=[3, 8])
    assert set(np.unique(pq[0])) == {0, 1, 2} and set(np.unique(pq[1])) == set(range(8))
    out = oracle_mod.philox4x32_10([100 >> 2, 1, 0, 0], [3, 0])
    assert pq[1].reshape(-1)[100] == (int(out[100 & 3]) * 8) >> 32
    counts = np.bincount(pq[1].reshape(-1), minlength=8)
    assert np.all(np.abs(counts - 512) < 4 * math.sqrt(512 * 7 / 8))
    # replica_offset shifts the replica key: replica 1 of a batch == replica 0 of an offset-1 handle
    assert np.array_equal(oracle_mod.init(1, 16, seed=7, replica_offset=1)[0], s[1])


# ---------------------------------------------------------------- Q3: beta = 0
@pytest.mark.parametrize("L", [2, 4, 6, 16])
def test_beta_zero_flips_everything(oracle_mod, L):
    s0 = oracle_mod.init(3, L, seed=21)
    s = s0.copy()
    E0, M0 = oracle_mod.ising_observables(s0)
    oracle_mod.sweep(s, 0.0, 1.0, 0.3, seed=21, n_sweeps=1)
    assert np.array_equal(s, -s0)
    E1, M1 = oracle_mod.ising_observables(s)
    assert np.array_equal(E1, E0) and np.array_equal(M1, -M0)


def test_half_sweep_touches_one_colour(oracle_mod):
    L = 8
    s0 = oracle_mod.init(2, L, seed=5)
    ii, jj = np.meshgrid(np.arange(L), np.arange(L), indexing="ij")
    for colour in (0, 1):
        s = s0.copy()
        oracle_mod.ising_half_sweep(s, 0.0, 1.0, 0.0, seed=5, t=0, colour=colour)
        mask = ((ii + jj) & 1) == colour
        assert np.array_equal(s[:, mask], -s0[:, mask]) and np.array_equal(s[:, ~mask], s0[:, ~mask])


# ---------------------------------------------------------------- Q4: Z2 mirror at h = 0
def test_z2_mirror_trajectory(oracle_mod):
    a = oracle_mod.init(2, 12, seed=9)
    b = -a
    Ea, Ma = oracle_mod.sweep(a, [0.3, 0.5], 1.0, 0.0, seed=9, n_sweeps=20, trace=True)
    Eb, Mb = oracle_mod.sweep(b, [0.3, 0.5], 1.0, 0.0, seed=9, n_sweeps=20, trace=True)
    assert np.array_equal(a, -b) and np.array_equal(Ea, Eb) and np.array_equal(Ma, -Mb)


# ---------------------------------------------------------------- Q5: chunking, replica independence
def test_chunking_and_replica_independence(oracle_mod):
    beta = np.array([0.3, 0.44, 0.6])
    a = oracle_mod.init(3, 10, seed=13)
    b = a.copy()
    oracle_mod.sweep(a, beta, 1.0, 0.05, seed=13, n_sweeps=10)
    oracle_mod.sweep(b, beta, 1.0, 0.05, seed=13, n_sweeps=4, sweep_offset=0)
    oracle_mod.sweep(b, beta, 1.0, 0.05, seed=13, n_sweeps=6, sweep_offset=4)
    assert np.array_equal(a, b)
    solo = oracle_mod.init(1, 10, seed=13, replica_offset=2)
    oracle_mod.sweep(solo, beta[2:], 1.0, 0.05, seed=13, n_sweeps=10, replica_offset=2)
    assert np.array_equal(solo[0], a[2])
    # Potts, mixed q
    q = [3, 8]
    pa = oracle_mod.init(2, 8, seed=4, q=q)
    pb = pa.copy()
    oracle_mod.sweep(pa, [1.0, 1.3], 1.0, 0.0, seed=4, n_sweeps=7, q=q)
    oracle_mod.sweep(pb, [1.0, 1.3], 1.0, 0.0, seed=4, n_sweeps=3, q=q)
    oracle_mod.sweep(pb, [1.0, 1.3], 1.0, 0.0, seed=4, n_sweeps=4, sweep_offset=3, q=q)
    assert np.array_equal(pa, pb)
    solo = oracle_mod.init(1, 8, seed=4, q=8, replica_offset=1)
    oracle_mod.sweep(solo, 1.3, 1.0, 0.0, seed=4, n_sweeps=7, q=8, replica_offset=1)
    assert np.array_equal(solo[0], pa[1])


def test_sweep_uses_time_colour_and_seed(oracle_mod):
    base = oracle_mod.init(1, 16, seed=2)
    outs = []
    for seed, off in [(2, 0), (2, 1), (3, 0), (2, 1 << 32)]:
        s = base.copy()
        oracle_mod.sweep(s, 0.44, 1.0, 0.0, seed=seed, n_sweeps=1, sweep_offset=off)
        outs.append(s)
    for a in range(4):
        for b in range(a + 1, 4):
            assert not np.array_equal(outs[a], outs[b])


def test_high_sweep_index_field_by_hand(oracle_mod):
    """Pins the placement of bits 32..55 of t in counter word 3 (O2): at t = 2^32 + 5 and t = (0xABCDEF << 32) + 7 every
    site of a half-sweep is recomputed here from the exported Philox with c3 = (t >> 32) & 0xFFFFFF | colour << 24 |
    1 << 28 written out; a wrong shift or mask in the oracle's counter assembly fails it."""
    L, seed, beta, J, h = 8, 0x5DEECE66D1234567, 0.37, 1.0, 0.05
    T, always = oracle_mod.ising_table(beta, J, h)
    for t in ((1 << 32) + 5, (0xABCDEF << 32) + 7):
        for colour in (0, 1):
            lat = oracle_mod.init(1, L, seed=3)
            expect = lat[0].copy()
            for i in range(L):
                for j in range(L):
                    if (i + j) & 1 != colour:
                        continue
                    n = i * (L // 2) + (j >> 1)
                    ctr = [n >> 2, 0, t & 0xFFFFFFFF, ((t >> 32) & 0xFFFFFF) | (colour << 24) | (1 << 28)]
                    r = int(oracle_mod.philox4x32_10(ctr, [seed & 0xFFFFFFFF, seed >> 32])[n & 3])
                    s0 = int(lat[0, i, j])
                    nn = int(lat[0, (i - 1) % L, j]) + int(lat[0, (i + 1) % L, j]) + int(lat[0, i, (j - 1) % L]) + int(lat[0, i, (j + 1) % L])
                    cls = 5 * ((s0 + 1) // 2) + (nn + 4) // 2
                    if always[cls] or r < int(T[cls]):
                        expect[i, j] = -s0
            oracle_mod.ising_half_sweep(lat, beta, J, h, seed, t, colour)
            assert np.array_equal(lat[0], expect), (t, colour)


# ---------------------------------------------------------------- Q6: observables
def _numpy_ising_obs(s):
    s = s.astype(np.int64)
    bonds = (s * np.roll(s, 1, axis=1)).sum(axis=(1, 2)) + (s * np.roll(s, 1, axis=2)).sum(axis=(1, 2))
    return -bonds, s.sum(axis=(1, 2))


def _numpy_potts_obs(s, q):
    bonds = (s == np.roll(s, 1, axis=1)).sum(axis=(1, 2)) + (s == np.roll(s, 1, axis=2)).sum(axis=(1, 2))
    M = np.array([np.bincount(s[b].reshape(-1), minlength=q[b]).max() for b in range(s.shape[0])])
    return -bonds, M


@pytest.mark.parametrize("L", [2, 4, 10, 32])
def test_ising_observables_definition_and_invariants(oracle_mod, L):
    # E_int = -(sum over bonds, each once) = -sum_sites s*(right + down) (Eq. 1; reading P2)
    s = oracle_mod.init(4, L, seed=17)
    oracle_mod.sweep(s, [0.2, 0.4, 0.5, 0.7], 1.0, 0.0, seed=17, n_sweeps=5)
    E, M = oracle_mod.ising_observables(s)
    En, Mn = _numpy_ising_obs(s)
    assert np.array_equal(E, En) and np.array_equal(M, Mn)
    N = L * L
    assert np.all((E - 2 * N) % 4 == 0) and np.all(np.abs(E) <= 2 * N)
    assert np.all((M - N) % 2 == 0) and np.all(np.abs(M) <= N)
    ones = np.ones((1, L, L), dtype=np.int8)
    assert oracle_mod.ising_observables(ones) == (np.array([-2 * N]), np.array([N]))
    assert oracle_mod.ising_observables(-ones) == (np.array([-2 * N]), np.array([-N]))


def test_potts_observables_definition_and_invariants(oracle_mod):
    q = [3, 8, 2, 5]
    for L in (2, 4, 12):
        s = oracle_mod.init(4, L, seed=19, q=q)
        oracle_mod.sweep(s, [0.8, 1.2, 0.9, 1.0], 1.0, 0.0, seed=19, n_sweeps=4, q=q)
        E, M = oracle_mod.potts_observables(s, q)
        En, Mn = _numpy_potts_obs(s, q)
        assert np.array_equal(E, En) and np.array_equal(M, Mn)
        N = L * L
        assert np.all(E <= 0) and np.all(E >= -2 * N)
        assert all(-(-N // qq) <= m <= N for qq, m in zip(q, M))
        for b in range(4):
            assert s[b].min() >= 0 and s[b].max() < q[b]
    same = np.full((1, 6, 6), 2, dtype=np.int8)
    assert oracle_mod.potts_observables(same, 3) == (np.array([-72]), np.array([36]))


def test_trace_and_moments(oracle_mod):
    s = oracle_mod.init(2, 8, seed=23)
    ref = s.copy()
    mom = np.zeros((2, 8), dtype=np.int64)
    Et, Mt = oracle_mod.sweep(s, [0.3, 0.6], 1.0, 0.1, seed=23, n_sweeps=6, trace=True, moments=mom)
    for t in range(6):
        oracle_mod.sweep(ref, [0.3, 0.6], 1.0, 0.1, seed=23, n_sweeps=1, sweep_offset=t)
        E, M = _numpy_ising_obs(ref)
        assert np.array_equal(E, Et[t]) and np.array_equal(M, Mt[t])
    for b in range(2):
        E = [int(x) for x in Et[:, b]]
        M = [int(x) for x in Mt[:, b]]
        e2 = sum(e * e for e in E)
        want = [6, sum(E), e2 & (2 ** 64 - 1), e2 >> 64, sum(M), sum(abs(m) for m in M),
                sum(m * m for m in M), sum(e * m for e, m in zip(E, M))]
        got = [int(x) for x in mom[b]]
        got[2] &= 2 ** 64 - 1
        assert got == want


def test_moments_128bit_carry(oracle_mod):
    mom = np.zeros((1, 8), dtype=np.int64)
    E = np.array([-(2 ** 33)], dtype=np.int64)  # E^2 = 2^66 overflows 64 bits
    M = np.array([3], dtype=np.int64)
    for _ in range(3):
        oracle_mod.accumulate_moments(mom, E, M)
    total = 3 * 2 ** 66
    assert (int(mom[0, 2]) & (2 ** 64 - 1)) == total & (2 ** 64 - 1) and int(mom[0, 3]) == total >> 64
    assert int(mom[0, 0]) == 3 and int(mom[0, 1]) == -3 * 2 ** 33 and int(mom[0, 6]) == 27


# ---------------------------------------------------------------- O5/O6: one site by hand
def test_single_site_rule_ising(oracle_mod):
    # Recompute one colour-1 site of one half-sweep from the generator, table and neighbours.
    L, seed, t, b = 8, 31, 5, 1
    s0 = oracle_mod.init(2, L, seed=seed)
    beta = [0.44, 0.35]
    s = s0.copy()
    oracle_mod.ising_half_sweep(s, beta, 1.0, 0.2, seed=seed, t=t, colour=1)
    T, always = oracle_mod.ising_table(beta[b], 1.0, 0.2)
    for (i, j) in [(0, 1), (3, 0), (7, 6), (4, 7)]:
        assert (i + j) & 1 == 1
        lat = s0[b].astype(int)
        nn = lat[(i - 1) % L, j] + lat[(i + 1) % L, j] + lat[i, (j - 1) % L] + lat[i, (j + 1) % L]
        n = i * (L // 2) + (j >> 1)
        out = oracle_mod.philox4x32_10([n >> 2, b, t, (1 << 24) | (1 << 28)], [seed, 0])
        r = int(out[n & 3])
        idx = 5 * ((lat[i, j] + 1) // 2) + (nn + 4) // 2
        acc = bool(always[idx]) or r < int(T[idx])
        assert s[b, i, j] == (-lat[i, j] if acc else lat[i, j])


def test_single_site_rule_potts(oracle_mod):
    L, seed, t, q = 8, 33, 2, [3, 8]
    s0 = oracle_mod.init(2, L, seed=seed, q=q)
    beta = [1.0, 1.3]
    s = s0.copy()
    oracle_mod.potts_half_sweep(s, q, beta, 1.0, seed=seed, t=t, colour=0)
    changed = 0
    for b in range(2):
        T, always = oracle_mod.potts_table(beta[b], 1.0)
        lat = s0[b].astype(int)
        for i in range(L):
            for j in range(L):
                if (i + j) & 1:
                    assert s[b, i, j] == lat[i, j]
                    continue
                n = i * (L // 2) + (j >> 1)
                out = oracle_mod.philox4x32_10([n >> 1, b, t, (0 << 24) | (2 << 28)], [seed, 0])
                rp, ra = int(out[2 * (n & 1)]), int(out[2 * (n & 1) + 1])
                new = (lat[i, j] + 1 + ((rp * (q[b] - 1)) >> 32)) % q[b]
                assert new != lat[i, j]  # one of the q-1 *other* states
                nb = [lat[(i - 1) % L, j], lat[(i + 1) % L, j], lat[i, (j - 1) % L], lat[i, (j + 1) % L]]
                dn = sum(x == new for x in nb) - sum(x == lat[i, j] for x in nb)
                acc = bool(always[dn + 4]) or ra < int(T[dn + 4])
                assert s[b, i, j] == (new if acc else lat[i, j])
                changed += acc
    assert changed > 10


def test_potts_proposal_uniform_over_other_states(oracle_mod):
    # beta = 0 accepts every proposal: the new state is never the old one and is uniform over the rest
    q = 5
    s0 = oracle_mod.init(1, 64, seed=41, q=q)
    s = s0.copy()
    oracle_mod.sweep(s, 0.0, 1.0, 0.0, seed=41, n_sweeps=1, q=q)
    assert np.all(s != s0)
    shift = (s.astype(int) - s0.astype(int)) % q
    counts = np.bincount(shift.reshape(-1), minlength=q)[1:]
    assert np.all(np.abs(counts - 1024) < 4 * math.sqrt(1024 * 0.75))


# ---------------------------------------------------------------- Q12: T -> 0
def test_zero_temperature(oracle_mod):
    L = 16
    s = oracle_mod.init(4, L, seed=51)
    E_prev, _ = oracle_mod.ising_observables(s)
    for t in range(30):
        for colour in (0, 1):
            oracle_mod.ising_half_sweep(s, 20.0, 1.0, 0.0, seed=51, t=t, colour=colour)
            E, _ = oracle_mod.ising_observables(s)
            assert np.all(E <= E_prev)
            E_prev = E
    assert np.all(E_prev < -1.5 * L * L)  # ground state (-2N) or a stripe state
    for sign in (1, -1):
        g = np.full((1, L, L), sign, dtype=np.int8)
        oracle_mod.sweep(g, 20.0, 1.0, 0.0, seed=51, n_sweeps=3)
        assert np.all(g == sign)
        g = np.full((1, L, L), sign, dtype=np.int8)
        oracle_mod.sweep(g, 20.0, 1.0, 0.5, seed=51, n_sweeps=3)  # all -1 is metastable: dE = 8J-2h > 0
        assert np.all(g == sign)
    p = np.full((1, L, L), 4, dtype=np.int8)
    oracle_mod.sweep(p, 20.0, 1.0, 0.0, seed=51, n_sweeps=3, q=6)
    assert np.all(p == 4)


# ---------------------------------------------------------------- Q14: second opinion
def test_second_opinion_trajectories(oracle_mod):
    g = read_golden("second_opinion_q14.txt")
    s = oracle_mod.init(4, 32, seed=1)
    E0, M0 = oracle_mod.ising_observables(s)
    Et, Mt = oracle_mod.sweep(s, 0.44, 1.0, 0.0, seed=1, n_sweeps=1000, trace=True)
    for b in range(4):
        want = [int(x) for x in g["ising L=32 seed=1 beta=0.44 replica%d" % b]]
        got = [int(E0[b]), int(M0[b])]
        for t in range(5):
            got += [int(Et[t, b]), int(Mt[t, b])]
        assert got == want
    assert [int(Et[999, 0]), int(Mt[999, 0])] == [int(x) for x in g["ising L=32 seed=1 beta=0.44 replica0 after1000"]]

    s = oracle_mod.init(1, 8, seed=1)
    assert "".join("+" if x > 0 else "-" for x in s[0, 0]) == g["ising L=8 seed=1 beta=0.44 row0"][0]
    E0, M0 = oracle_mod.ising_observables(s)
    Et, Mt = oracle_mod.sweep(s, 0.44, 1.0, 0.0, seed=1, n_sweeps=3, trace=True)
    got = [int(E0[0]), int(M0[0])] + [int(v) for t in range(3) for v in (Et[t, 0], Mt[t, 0])]
    assert got == [int(x) for x in g["ising L=8 seed=1 beta=0.44 replica0"]]

    for q, off, key in [(3, 0, "potts L=8 seed=4 q=3 beta=bc replica0"), (8, 64, "potts L=8 seed=4 q=8 beta=bc replica64")]:
        bc = math.log(1.0 + math.sqrt(q))
        s = oracle_mod.init(1, 8, seed=4, q=q, replica_offset=off)
        assert "".join(str(int(x)) for x in s[0, 0]) == g[key + " row0"][0]
        E0, M0 = oracle_mod.potts_observables(s, q)
        Et, Mt = oracle_mod.sweep(s, bc, 1.0, 0.0, seed=4, n_sweeps=3, q=q, replica_offset=off, trace=True)
        got = [int(E0[0]), int(M0[0])] + [int(v) for t in range(3) for v in (Et[t, 0], Mt[t, 0])]
        assert got == [int(x) for x in g[key]]
