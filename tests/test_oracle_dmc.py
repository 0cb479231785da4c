"""Pins of the Differentiable-Monte-Carlo oracle (oracle/dmc_oracle.cpp; Algorithm 2 and Eq. 4).

None of these re-types the oracle's formula and compares it with itself: the gradients are pinned by central finite
differences of the forward pass, the forward pass by its alpha -> infinity limit (the discrete Algorithm-1 oracle,
pinned on its own in test_oracle_*.py), by a by-hand site through the exported Philox, and by the invariants the paper
states (0 < q < 1, spins stay in [-1, 1], Eq. 4 returns +-1)."""
import numpy as np
import pytest

import oracle


def _setup(B, L, seed, glass=True):
    rng = np.random.default_rng(seed)
    s = rng.uniform(-1.0, 1.0, size=(B, L, L))
    if glass:
        Jh = rng.normal(0.0, 1.0, size=(B, L, L))
        Jv = rng.normal(0.0, 1.0, size=(B, L, L))
    else:
        Jh = np.ones((B, L, L))
        Jv = np.ones((B, L, L))
    beta = rng.uniform(0.3, 0.9, size=B)
    return s, Jh, Jv, beta


def _loss(s, Jh, Jv, h, beta, alpha, seed, n_sweeps, target):
    x = s.copy()
    oracle.dmc_forward(x, Jh, Jv, h, beta, alpha, seed, n_sweeps)
    return float(np.sum((target - x) ** 2))          # Eq. 8


@pytest.mark.parametrize("L,n_sweeps,alpha", [(4, 1, 3.0), (4, 3, 8.0), (6, 2, 5.0), (2, 2, 4.0)])
def test_gradients_match_central_finite_differences(L, n_sweeps, alpha):
    B, seed, h = 2, 11, 0.15
    s, Jh, Jv, beta = _setup(B, L, seed + L)
    target = np.sign(np.random.default_rng(5).normal(size=(B, L, L)))
    x = s.copy()
    traj = oracle.dmc_forward(x, Jh, Jv, h, beta, alpha, seed, n_sweeps, want_traj=True)
    assert np.array_equal(traj[-1], x) and np.array_equal(traj[0], s)
    gs, gjh, gjv, gb, gh = oracle.dmc_backward(traj, Jh, Jv, h, beta, alpha, seed, 2.0 * (x - target))
    eps = 1e-6
    rng = np.random.default_rng(3)

    def fd(arr, idx):
        a = arr.copy(); a[idx] += eps
        b = arr.copy(); b[idx] -= eps
        return a, b

    args = dict(s=s, Jh=Jh, Jv=Jv, h=h, beta=beta)

    def loss_with(**kw):
        a = dict(args); a.update(kw)
        return _loss(a["s"], a["Jh"], a["Jv"], a["h"], a["beta"], alpha, seed, n_sweeps, target)

    for name, grad in (("s", gs), ("Jh", gjh), ("Jv", gjv)):
        for _ in range(12):
            idx = tuple(int(rng.integers(0, n)) for n in grad.shape)
            up, dn = fd(args[name], idx)
            num = (loss_with(**{name: up}) - loss_with(**{name: dn})) / (2 * eps)
            assert abs(num - grad[idx]) <= 1e-6 * max(1.0, abs(num)), (name, idx, num, grad[idx])
    for b in range(B):
        up, dn = fd(beta, b)
        num = (loss_with(beta=up) - loss_with(beta=dn)) / (2 * eps)
        assert abs(num - gb[b]) <= 1e-6 * max(1.0, abs(num)), ("beta", b, num, gb[b])
    num = (loss_with(h=h + eps) - loss_with(h=h - eps)) / (2 * eps)
    assert abs(num - gh.sum()) <= 1e-6 * max(1.0, abs(num)), ("h", num, gh.sum())


@pytest.mark.parametrize("L,glass", [(8, False), (16, True), (2, True)])
def test_alpha_to_infinity_then_eq4_is_algorithm_1(L, glass):
    """Alg. 2 with alpha -> infinity 'becomes the standard Metropolis algorithm': on a +-1 lattice with
    +-1 bond signs the discretised DMC trajectory equals the discrete oracle's (same Philox words; the two acceptance
    tests r24 < p and r32 < floor(p 2^32) differ with probability 2^-24 per site, never on these seeds)."""
    B, seed, h, n_sweeps = 3, 21, 0.0 if not glass else 0.05, 6
    rng = np.random.default_rng(L)
    spins = oracle.init(B, L, seed=seed)
    if glass:
        Jh = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
        Jv = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    else:
        Jh = np.ones((B, L, L), dtype=np.int8)
        Jv = np.ones((B, L, L), dtype=np.int8)
    beta = np.array([0.3, 0.44, 0.7])
    s = spins.astype(np.float64)
    ref = spins.copy()
    for t in range(n_sweeps):
        oracle.dmc_forward(s, Jh, Jv, h, beta, 1e13, seed, 1, sweep_offset=t)
        oracle.dmc_discretise(s)
        oracle.sweep_bonds(ref, Jh, Jv, beta, 1.0, h, seed, 1, sweep_offset=t)
        assert np.array_equal(s.astype(np.int8), ref), t
    if not glass:      # and the bond-free discrete oracle
        ref2 = spins.copy()
        oracle.sweep(ref2, beta, 1.0, h, seed=seed, n_sweeps=n_sweeps)
        assert np.array_equal(ref2, ref)


def test_q_in_unit_interval_and_spins_stay_bounded():
    B, L, seed = 4, 12, 9
    s, Jh, Jv, beta = _setup(B, L, 2)
    for t in range(5):
        for c in (0, 1):
            before = s.copy()
            q = oracle.dmc_half_sweep(s, Jh, Jv, 0.1, beta, 6.0, seed, t, c, want_q=True)
            ii, jj = np.indices((L, L))
            own = ((ii + jj) & 1) == c
            assert np.all(np.isnan(q[:, ~own])) and np.all((q[:, own] > 0.0) & (q[:, own] <= 1.0))   # < 1 up to rounding (p can be e^8)
            assert np.array_equal(s[:, ~own], before[:, ~own])                   # the other colour is untouched
            assert np.allclose(s[:, own], before[:, own] * (1.0 - 2.0 * q[:, own]), rtol=0, atol=1e-15)
            assert np.all(np.abs(s) <= 1.0)
    d = oracle.dmc_discretise(s.copy())
    assert set(np.unique(d)) <= {-1.0, 1.0} and np.array_equal(d, np.where(s < 0, -1.0, 1.0))
    assert oracle.dmc_discretise(np.array([0.0, -0.0, -1e-300]))[0] == 1.0       # Eq. 4: s >= 0 -> +1


def test_alpha_zero_halves_every_updated_spin_to_zero():
    s, Jh, Jv, beta = _setup(2, 6, 4)
    oracle.dmc_forward(s, Jh, Jv, 0.0, beta, 0.0, 1, 1)
    assert np.all(s == 0.0)                                                      # q = 1/2: s (1 - 2q) = 0


def test_one_site_by_hand_from_the_philox_word():
    """Site (3, 2) of replica 1, L = 6, colour (3+2)&1 = 1, sweep t = 2^32 + 5: counter words, word index, r, F, p, q."""
    B, L, seed, t, alpha, h = 2, 6, 0x1234567887654321, (1 << 32) + 5, 4.0, -0.2
    s, Jh, Jv, beta = _setup(B, L, 8)
    i, j, b = 3, 2, 1
    n = i * (L // 2) + (j >> 1)
    ctr = [n >> 2, b + 7, t & 0xFFFFFFFF, ((t >> 32) & 0xFFFFFF) | (1 << 24) | (1 << 28)]
    w = int(oracle.philox4x32_10(ctr, [seed & 0xFFFFFFFF, seed >> 32])[n & 3])
    r = (w >> 8) / 2.0 ** 24
    F = (Jv[b, i - 1, j] * s[b, i - 1, j] + Jv[b, i, j] * s[b, (i + 1) % L, j] + Jh[b, i, j - 1] * s[b, i, j - 1]
         + Jh[b, i, j] * s[b, i, (j + 1) % L] + h)
    p = np.exp(-beta[b] * 2.0 * s[b, i, j] * F)
    q = 1.0 / (1.0 + np.exp(-alpha * (p - r)))
    expect = q * (-s[b, i, j]) + (1.0 - q) * s[b, i, j]
    x = s.copy()
    oracle.dmc_half_sweep(x, Jh, Jv, h, beta, alpha, seed, t, 1, replica_offset=7)
    assert abs(x[b, i, j] - expect) < 1e-15
    # the t-high field matters (2^32 + 5 is not 5) and so does the replica offset
    y = s.copy(); oracle.dmc_half_sweep(y, Jh, Jv, h, beta, alpha, seed, 5, 1, replica_offset=7)
    z = s.copy(); oracle.dmc_half_sweep(z, Jh, Jv, h, beta, alpha, seed, t, 1, replica_offset=0)
    assert x[b, i, j] != y[b, i, j] and x[b, i, j] != z[b, i, j]


def test_chunked_forward_equals_one_call_and_replicas_are_independent():
    s, Jh, Jv, beta = _setup(3, 8, 6)
    a = s.copy(); oracle.dmc_forward(a, Jh, Jv, 0.1, beta, 5.0, 3, 5)
    c = s.copy()
    oracle.dmc_forward(c, Jh, Jv, 0.1, beta, 5.0, 3, 2)
    oracle.dmc_forward(c, Jh, Jv, 0.1, beta, 5.0, 3, 3, sweep_offset=2)
    assert np.array_equal(a, c)
    one = s[2:3].copy()
    oracle.dmc_forward(one, Jh[2:3], Jv[2:3], 0.1, beta[2:3], 5.0, 3, 5, replica_offset=2)
    assert np.array_equal(one[0], a[2])
