"""Statistical / exact-physics pins of the oracle (CPU only; fixed seeds, so deterministic).

Q7  exact enumeration of the 2^16 states of the 4x4 Ising torus vs long-run averages (4 SE)
Q8  Onsager's exact energy per spin at beta = 0.30 and 0.60 on L = 128 (4 SE + 1e-3)
Q9  half-sweep detailed balance + sweep stationarity on 2x2 from the transition matrix, and the
    oracle's empirical one-sweep transition frequencies against that matrix
Q10 exact enumeration of small Potts tori (brute force 2x2; transfer-matrix density of states 4x4)
Q11 Potts self-dual point beta_c = ln(1+sqrt(q)): energy bracket around -(1+1/sqrt(q))
The exact values are recomputed here by brute force (independently of the oracle) and cross-checked
against tests/golden/exact_small_lattices.txt.
"""
import itertools
import math

import numpy as np
import pytest
from scipy import integrate

from conftest import read_golden

GOLD = read_golden("exact_small_lattices.txt")


def _gold(key):
    return [float(x) for x in GOLD[key]]


# ------------------------------------------------------------------ brute-force helpers (test side)
def _all_ising_states(L):
    n = L * L
    idx = np.arange(1 << n, dtype=np.int64)
    bits = ((idx[:, None] >> np.arange(n)) & 1).astype(np.int64)
    return (2 * bits - 1).reshape(-1, L, L)


def _ising_bond_sum(s):
    return (s * np.roll(s, 1, axis=1)).sum(axis=(1, 2)) + (s * np.roll(s, 1, axis=2)).sum(axis=(1, 2))


def _exact_ising(L, beta, h):
    s = _all_ising_states(L)
    S = _ising_bond_sum(s)
    M = s.sum(axis=(1, 2))
    H = -1.0 * S - h * M
    w = np.exp(-beta * (H - H.min()))
    Z = w.sum()
    N = L * L
    e = (w * H).sum() / Z
    e2 = (w * H * H).sum() / Z
    return e / N, (w * np.abs(M)).sum() / Z / N, beta * beta * (e2 - e * e) / N, S


def _replica_average(oracle_mod, L, B, beta, h, seed, therm, meas, start=None):
    s = oracle_mod.init(B, L, seed=seed) if start is None else start
    oracle_mod.sweep(s, beta, 1.0, h, seed=seed, n_sweeps=therm)
    Et, Mt = oracle_mod.sweep(s, beta, 1.0, h, seed=seed, n_sweeps=meas, sweep_offset=therm, trace=True)
    return Et, Mt


def _check(mean_per_replica, exact, extra=0.0):
    B = len(mean_per_replica)
    se = mean_per_replica.std(ddof=1) / math.sqrt(B)
    assert abs(mean_per_replica.mean() - exact) <= 4 * se + extra, (mean_per_replica.mean(), exact, se)
    return se


# ------------------------------------------------------------------ Q7
def test_4x4_enumeration_matches_survey_values():
    for key in ("ising4x4 0.20 0", "ising4x4 0.30 0", "ising4x4 0.44 0", "ising4x4 0.60 0"):
        beta = float(key.split()[1])
        e, m, c, S = _exact_ising(4, beta, 0.0)
        ge, gm, gc = _gold(key)
        assert abs(e - ge) < 1e-11 and abs(m - gm) < 1e-11 and abs(c - gc) < 1e-10
    e, m, _, S = _exact_ising(4, 0.44, 0.01)
    ge, gm = _gold("ising4x4 0.44 0.01")
    assert abs(e - ge) < 1e-11 and abs(m - gm) < 1e-11
    dos = [int(x) for x in GOLD["ising4x4 dos"]]
    for S_abs, count in zip(dos[0::2], dos[1::2]):
        assert int((np.abs(S) == S_abs).sum()) == (count if S_abs == 0 else 2 * count) or \
               int((S == S_abs).sum()) == count


@pytest.mark.parametrize("beta,h", [(0.30, 0.0), (0.44, 0.0), (0.60, 0.0), (0.44, 0.01)])
def test_4x4_ising_long_run_averages(oracle_mod, beta, h):
    e_exact, m_exact, c_exact, _ = _exact_ising(4, beta, h)
    B, N = 512, 16
    Et, Mt = _replica_average(oracle_mod, 4, B, beta, h, seed=1234, therm=300, meas=3000)
    H = 1.0 * Et - h * Mt  # energy = J E_int - h M  (O8)
    _check(H.mean(axis=0) / N, e_exact)
    _check(np.abs(Mt).mean(axis=0) / N, m_exact)
    # specific heat from the pooled variance; loose (it is a fluctuation quantity)
    c = beta * beta * H.var() / N
    assert abs(c - c_exact) < 0.05 * c_exact + 0.01


# ------------------------------------------------------------------ Q8
def _onsager_u(beta):
    # u = -coth(2b) [1 + (2/pi)(2 tanh^2(2b) - 1) K(k)], k = 2 sinh(2b)/cosh^2(2b), J = 1
    k = 2.0 * math.sinh(2 * beta) / math.cosh(2 * beta) ** 2
    K, _ = integrate.quad(lambda th: 1.0 / math.sqrt(1.0 - (k * math.sin(th)) ** 2), 0.0, math.pi / 2)
    return -(1.0 / math.tanh(2 * beta)) * (1.0 + (2.0 / math.pi) * (2.0 * math.tanh(2 * beta) ** 2 - 1.0) * K)


def test_onsager_formula_matches_survey_values():
    assert abs(_onsager_u(0.30) - _gold("onsager 0.30")[0]) < 1e-10
    assert abs(_onsager_u(0.60) - _gold("onsager 0.60")[0]) < 1e-10


@pytest.mark.parametrize("beta,cold", [(0.30, False), (0.60, True)])
def test_onsager_energy_L128(oracle_mod, beta, cold):
    L, B = 128, 8
    start = np.ones((B, L, L), dtype=np.int8) if cold else None  # W2: beta=0.60 must start cold
    Et, Mt = _replica_average(oracle_mod, L, B, beta, 0.0, seed=77, therm=300, meas=700, start=start)
    u = Et.mean(axis=0) / (L * L)
    _check(u, _onsager_u(beta), extra=1e-3)
    if cold:
        m_exact = (1.0 - math.sinh(2 * beta) ** -4) ** 0.125  # Yang's spontaneous magnetisation
        assert abs(np.abs(Mt).mean() / (L * L) - m_exact) < 2e-3


# ------------------------------------------------------------------ Q9
def _half_sweep_matrix_2x2(p_of_class, colour):
    """16x16 transition matrix of one colour's half-sweep on the 2x2 torus, from class probabilities.
    On L=2 up==down and left==right (multiplicity 2, O1), so nn = 2*(vertical + horizontal)."""
    states = _all_ising_states(2)
    P = np.zeros((16, 16))
    sites = [(i, j) for i in range(2) for j in range(2) if (i + j) & 1 == colour]
    for a, s in enumerate(states):
        for flips in itertools.product((0, 1), repeat=len(sites)):
            prob = 1.0
            t = s.copy()
            for (i, j), f in zip(sites, flips):
                nn = 2 * s[1 - i, j] + 2 * s[i, 1 - j]
                p = p_of_class[5 * ((s[i, j] + 1) // 2) + (nn + 4) // 2]
                prob *= p if f else 1.0 - p
                if f:
                    t[i, j] = -s[i, j]
            b = int((((t.reshape(-1) + 1) // 2) << np.arange(4)).sum())
            P[a, b] += prob
    return P


@pytest.mark.parametrize("beta,h", [(0.44, 0.0), (0.44, 0.5), (0.2, -0.3)])
def test_detailed_balance_2x2_from_table(oracle_mod, beta, h):
    T, always = oracle_mod.ising_table(beta, 1.0, h)
    p = np.where(always, 1.0, T.astype(np.float64) / 4294967296.0)
    states = _all_ising_states(2)
    H = -1.0 * _ising_bond_sum(states) - h * states.sum(axis=(1, 2))
    pi = np.exp(-beta * H)
    pi /= pi.sum()
    P0, P1 = _half_sweep_matrix_2x2(p, 0), _half_sweep_matrix_2x2(p, 1)
    for P in (P0, P1):
        assert np.allclose(P.sum(axis=1), 1.0)
        flow = pi[:, None] * P
        assert np.abs(flow - flow.T).max() < 1e-9  # reversible up to the 2^-32 quantisation
    assert np.abs(pi @ (P0 @ P1) - pi).max() < 1e-9  # the sweep is stationary (it is not reversible)


def test_one_sweep_transition_frequencies_2x2(oracle_mod):
    beta, h, reps = 0.44, 0.3, 4000
    T, always = oracle_mod.ising_table(beta, 1.0, h)
    p = np.where(always, 1.0, T.astype(np.float64) / 4294967296.0)
    P = _half_sweep_matrix_2x2(p, 0) @ _half_sweep_matrix_2x2(p, 1)  # colour 0 first (reading P3)
    states = _all_ising_states(2).astype(np.int8)
    for a in range(16):
        s = np.repeat(states[a:a + 1], reps, axis=0).copy()
        oracle_mod.sweep(s, beta, 1.0, h, seed=99, n_sweeps=1, sweep_offset=a)
        code = (((s.reshape(reps, 4).astype(np.int64) + 1) // 2) << np.arange(4)).sum(axis=1)
        freq = np.bincount(code, minlength=16) / reps
        se = np.sqrt(np.maximum(P[a] * (1 - P[a]), 1e-12) / reps)
        assert np.all(np.abs(freq - P[a]) <= 4 * se + 1e-9), a
        assert np.all(freq[P[a] == 0] == 0)


def test_2x2_h0_closed_cycle_warning_W1(oracle_mod):
    # W1: at h=0 the states with both colour pairs unequal flip deterministically for ever.
    s = np.array([[[1, 1], [-1, -1]]], dtype=np.int8)
    seen = []
    for t in range(4):
        oracle_mod.sweep(s, 0.44, 1.0, 0.0, seed=3, n_sweeps=1, sweep_offset=t)
        seen.append(s.copy())
    assert np.array_equal(seen[0], -np.array([[[1, 1], [-1, -1]]])) and np.array_equal(seen[1], -seen[0])


# ------------------------------------------------------------------ Q10
def _exact_potts_bruteforce(L, q, beta):
    n = L * L
    states = np.array(list(itertools.product(range(q), repeat=n)), dtype=np.int64).reshape(-1, L, L)
    D = (states == np.roll(states, 1, axis=1)).sum(axis=(1, 2)) + (states == np.roll(states, 1, axis=2)).sum(axis=(1, 2))
    nmax = np.array([np.bincount(s.reshape(-1), minlength=q).max() for s in states])
    w = np.exp(beta * (D - D.max()))
    return -(w * D).sum() / w.sum() / n, (w * nmax).sum() / w.sum() / n


def _exact_potts_energy_transfer(L, q, beta):
    """<E>/N of the LxL Potts torus from an integer density of states built with a polynomial-valued
    row transfer matrix: entry = x^(bonds inside the new row + bonds between rows)."""
    rows = np.array(list(itertools.product(range(q), repeat=L)))
    R = len(rows)
    horiz = (rows == np.roll(rows, 1, axis=1)).sum(axis=1)
    vert = (rows[:, None, :] == rows[None, :, :]).sum(axis=2)
    deg = 2 * L * L + 1
    expo = vert + horiz[None, :]
    Tm = np.zeros((R, R, deg), dtype=object)
    for a in range(R):
        for b in range(R):
            Tm[a, b, expo[a, b]] = 1
    def mul(A, B):
        out = np.zeros((R, R, deg), dtype=object)
        for d1 in range(deg):
            if not A[:, :, d1].any():
                continue
            for d2 in range(deg - d1):
                if not B[:, :, d2].any():
                    continue
                out[:, :, d1 + d2] += A[:, :, d1].dot(B[:, :, d2])
        return out
    P = Tm
    for _ in range(L - 1):
        P = mul(P, Tm)
    g = np.array([sum(P[a, a, d] for a in range(R)) for d in range(deg)], dtype=object)
    assert sum(g) == q ** (L * L)
    d = np.arange(deg, dtype=np.float64)
    gf = np.array([float(x) for x in g])
    w = gf * np.exp(beta * (d - d.max()))
    return -(w * d).sum() / w.sum() / (L * L)


def test_potts_exact_values_match_survey():
    for q in (3, 8):
        bc = math.log(1.0 + math.sqrt(q))
        for f in (0.5, 1.0, 1.5):
            e, m = _exact_potts_bruteforce(2, q, f * bc)
            ge, gm = _gold("potts %d 2 %.1f" % (q, f))
            assert abs(e - ge) < 1e-10 and abs(m - gm) < 1e-10
    bc = math.log(1.0 + math.sqrt(3))
    for f in (0.5, 1.0, 1.5):
        assert abs(_exact_potts_energy_transfer(4, 3, f * bc) - _gold("potts 3 4 %.1f" % f)[0]) < 1e-10


def _potts_run(oracle_mod, L, q, beta, B, seed, therm, meas):
    s = oracle_mod.init(B, L, seed=seed, q=q)
    oracle_mod.sweep(s, beta, 1.0, 0.0, seed=seed, n_sweeps=therm, q=q)
    return oracle_mod.sweep(s, beta, 1.0, 0.0, seed=seed, n_sweeps=meas, sweep_offset=therm, q=q, trace=True)


@pytest.mark.parametrize("q,L,f", [(3, 4, 0.5), (3, 4, 1.0), (3, 4, 1.5), (3, 2, 1.0), (8, 2, 1.0), (8, 4, 0.5), (8, 4, 1.0)])
def test_potts_long_run_averages(oracle_mod, q, L, f):
    beta = f * math.log(1.0 + math.sqrt(q))
    gold = _gold("potts %d %d %.1f" % (q, L, f))
    Et, Mt = _potts_run(oracle_mod, L, q, beta, B=384, seed=4321, therm=400, meas=2500)
    N = L * L
    _check(Et.mean(axis=0) / N, gold[0])
    if len(gold) > 1:
        _check(Mt.mean(axis=0) / N, gold[1])


def test_potts_q2_is_ising(oracle_mod):
    # q=2 Potts at beta_P = 2 beta_I has the Ising Boltzmann weights: E_P/N = -(2 + |e_I|)/2 ... (Q10)
    e_ising, _, c_ising, _ = _exact_ising(4, 0.44, 0.0)
    Et, Mt = _potts_run(oracle_mod, 4, 2, 0.88, B=384, seed=555, therm=300, meas=2500)
    _check(Et.mean(axis=0) / 16, -(2.0 - e_ising) / 2.0)


# ------------------------------------------------------------------ Q11
@pytest.mark.parametrize("q", [3, 8])
def test_potts_self_dual_point_bracket(oracle_mod, q):
    bc = math.log(1.0 + math.sqrt(q))
    u_c = -(1.0 + 1.0 / math.sqrt(q))
    L, B = 32, 6
    beta = np.array([0.5 * bc, 0.5 * bc, 0.9 * bc, 1.1 * bc, 1.5 * bc, 1.5 * bc])
    s = np.zeros((B, L, L), dtype=np.int8)  # cold start so the ordered side needs no nucleation
    oracle_mod.sweep(s, beta, 1.0, 0.0, seed=8, n_sweeps=400, q=q)
    Et, _ = oracle_mod.sweep(s, beta, 1.0, 0.0, seed=8, n_sweeps=300, sweep_offset=400, q=q, trace=True)
    u = Et.mean(axis=0) / (L * L)
    assert u[0] > u_c + 0.3 and u[1] > u_c + 0.3      # disordered side well above
    assert u[4] < u_c - 0.3 and u[5] < u_c - 0.3      # ordered side well below
    assert u[2] > u[3]                                 # crossing near beta_c
    assert u[2] > u_c - 0.05 and u[3] < u_c + 0.05
