"""Float-derived quantities from the exact integer moments (energy = J E_int - h M, per-spin
averages, specific heat, susceptibility are computed on the host in double FROM THE EXACT INTEGERS, so two paths whose
integers agree give the same doubles).  The moments are those of spin_sweep_measure:
[n, sum E, sum E^2 (low 64 bits), sum E^2 (high 64 bits), sum M, sum |M|, sum M^2, sum E*M] per replica.

All differences of large numbers (variances) are taken in exact rational arithmetic (python integers / Fraction) and
rounded to double once, at the end."""
from fractions import Fraction

import numpy as np


def _exact(mom_row):
    m = [int(x) for x in mom_row]
    n = m[0]
    sumE2 = (m[3] << 64) + (m[2] & ((1 << 64) - 1))          # two 64-bit limbs, low limb stored as a signed int64
    return n, m[1], sumE2, m[4], m[5], m[6], m[7]


def thermodynamics(moments, beta, J, h, L, model="ising"):
    """Per replica: energy per spin u = <H>/N, |m| = <|M|>/N, specific heat c = beta^2 (<H^2> - <H>^2)/N,
    susceptibility chi = beta (<M^2> - <|M|>^2)/N, with H = J E_int - h M (Ising) or J E_int (Potts, h = 0).
    Returns a dict of float64 arrays; replicas without samples give NaN."""
    moments = np.asarray(moments, dtype=np.int64)
    B = moments.shape[0]
    beta = np.broadcast_to(np.asarray(beta, dtype=np.float64), (B,))
    Jf, hf = Fraction(float(J)), Fraction(float(h) if model == "ising" else 0.0)
    N = L * L
    out = {k: np.full(B, np.nan) for k in ("u", "abs_m", "c", "chi", "n")}
    for b in range(B):
        n, sE, sE2, sM, sA, sM2, sEM = _exact(moments[b])
        out["n"][b] = n
        if n == 0:
            continue
        meanH = (Jf * sE - hf * sM) / n
        meanH2 = (Jf * Jf * sE2 - 2 * Jf * hf * sEM + hf * hf * sM2) / n
        bb = Fraction(float(beta[b]))
        out["u"][b] = float(meanH / N)
        out["abs_m"][b] = float(Fraction(sA, n) / N)
        out["c"][b] = float(bb * bb * (meanH2 - meanH * meanH) / N)
        out["chi"][b] = float(bb * (Fraction(sM2, n) - Fraction(sA, n) ** 2) / N)
    return out
