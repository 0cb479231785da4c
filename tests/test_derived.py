"""Host logic: float-derived quantities from the exact integer moments (energy per spin, |m|, specific heat,
susceptibility).  Computed from exact integers in rational arithmetic, so equal moments give bit-equal doubles; checked
here against plain numpy statistics of the oracle's traces (relative 1e-12, the north star's bar)."""
import numpy as np

from paper_2304_01772_b200 import derived


def test_thermodynamics_from_moments_match_trace_statistics(oracle_mod):
    B, L, n = 4, 8, 300
    beta = np.array([0.2, 0.4, 0.44, 0.6])
    J, h = 1.0, 0.05
    lat = oracle_mod.init(B, L, seed=4)
    mom = np.zeros((B, 8), dtype=np.int64)
    E, M = oracle_mod.sweep(lat, beta, J, h, seed=4, n_sweeps=n, trace=True, moments=mom)
    d = derived.thermodynamics(mom, beta, J, h, L)
    N = L * L
    # exact rational reference from the traces (python ints), then the same single rounding
    from fractions import Fraction
    for b in range(B):
        Hs = [Fraction(J) * int(e) - Fraction(h) * int(m) for e, m in zip(E[:, b], M[:, b])]
        meanH = sum(Hs) / n
        varH = sum(x * x for x in Hs) / n - meanH * meanH
        absM = Fraction(sum(abs(int(m)) for m in M[:, b]), n)
        M2 = Fraction(sum(int(m) ** 2 for m in M[:, b]), n)
        bb = Fraction(float(beta[b]))
        ref = (float(meanH / N), float(absM / N), float(bb * bb * varH / N), float(bb * (M2 - absM ** 2) / N))
        got = (d["u"][b], d["abs_m"][b], d["c"][b], d["chi"][b])
        for g, r in zip(got, ref):
            assert g == r or abs(g - r) <= 1e-12 * abs(r), (got, ref)
        # and against straightforward float64 numpy statistics (loose: those cancel in floating point)
        Hf = J * E[:, b].astype(np.float64) - h * M[:, b].astype(np.float64)
        assert abs(d["u"][b] - Hf.mean() / N) < 1e-12
        assert abs(d["c"][b] - beta[b] ** 2 * Hf.var() / N) < 1e-9
    assert np.all(d["n"] == n)


def test_128_bit_energy_square_limbs_and_empty_replicas():
    mom = np.zeros((2, 8), dtype=np.int64)
    E = 2 ** 35 + 12345                                   # E^2 needs more than 64 bits after a few samples
    tot = 5 * E * E
    mom[0] = [5, 5 * E, np.int64(np.uint64(tot & (2 ** 64 - 1)).astype(np.int64)), tot >> 64, 0, 0, 0, 0]
    d = derived.thermodynamics(mom, 1.0, 1.0, 0.0, 4)
    assert d["c"][0] == 0.0 and d["u"][0] == float(E) / 16.0   # all samples equal: zero variance, exactly
    assert np.isnan(d["u"][1]) and d["n"][1] == 0
