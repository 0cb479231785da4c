"""Seeded synthetic inputs of the five BASELINE.json configurations (DESIGN.md
section 4).  Input recipes only: shapes, seeds, per-replica beta / q arrays, sweep counts.  This module
holds none of the method's arithmetic and is the only module both the CUDA path's callers and the
oracle's callers (tests, bench) share."""
import math

import numpy as np


class Workload:
    def __init__(self, name, model, batch, L, seed, beta, J, h, n_sweeps, q=None, layout="int8", therm=0,
                 measure=False, note=""):
        self.name, self.model, self.batch, self.L, self.seed = name, model, batch, L, seed
        self.beta = np.ascontiguousarray(beta, dtype=np.float64)
        self.J, self.h, self.n_sweeps, self.q, self.layout = J, h, n_sweeps, q, layout
        self.therm, self.measure, self.note = therm, measure, note
        assert self.beta.shape == (batch,)

    @property
    def sites(self):
        return self.batch * self.L * self.L

    @property
    def updates(self):
        return self.sites * self.n_sweeps


def potts_beta_c(q):
    return math.log(1.0 + math.sqrt(float(q)))


def config(index, layout=None):
    """index 1..5 = BASELINE.json configs[0..4]."""
    if index == 1:
        return Workload("C1", "ising", 4, 32, 1, np.full(4, 0.44), 1.0, 0.0, 1000, measure=True,
                        note="E, M recorded each sweep")
    if index == 2:
        beta = np.array([0.30 + 0.30 * b / 63.0 for b in range(64)])
        return Workload("C2", "ising", 64, 1024, 2, beta, 1.0, 0.0, 2000)
    if index == 3:
        return Workload("C3", "ising", 4, 8192, 3, np.full(4, 0.4407), 1.0, 0.01, 500, layout=layout or "bits",
                        note="bit-packed and int8 layouts both exercised")
    if index == 4:
        q = np.array([3] * 64 + [8] * 64, dtype=np.int32)
        beta = np.array([0.5 * potts_beta_c(q[b]) + potts_beta_c(q[b]) * (b % 64) / 63.0 for b in range(128)])
        return Workload("C4", "potts", 128, 512, 4, beta, 1.0, 0.0, 1000, q=q)
    if index == 5:
        beta = np.array([0.2 + 0.5 * b / 1023.0 for b in range(1024)])
        return Workload("C5", "ising", 1024, 256, 5, beta, 1.0, 0.0, 10000, therm=2000, measure=True,
                        note="moments accumulated after 2000 thermalisation sweeps")
    raise ValueError("config index must be 1..5")


def paper_table3_shapes():
    """The corners of the paper's Table III: (batch, L) at beta = 0.44, seed 6, 200 sweeps."""
    out = []
    for batch, L in [(1, 640), (16, 640), (1, 2560), (16, 2560)]:
        out.append(Workload("P_%dx%d" % (batch, L), "ising", batch, L, 6, np.full(batch, 0.44), 1.0, 0.0, 200))
    return out


def random_ising_lattice(batch, L, seed):
    """A seeded +-1 lattice for set_spins tests (numpy generator; not the method's Philox init)."""
    rng = np.random.default_rng(seed)
    return (2 * rng.integers(0, 2, size=(batch, L, L), dtype=np.int8) - 1).astype(np.int8)


def random_potts_lattice(batch, L, q, seed):
    rng = np.random.default_rng(seed)
    q = np.broadcast_to(np.asarray(q), (batch,))
    out = np.empty((batch, L, L), dtype=np.int8)
    for b in range(batch):
        out[b] = rng.integers(0, int(q[b]), size=(L, L), dtype=np.int8)
    return out
