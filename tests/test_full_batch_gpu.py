"""Whole-batch parity at the BASELINE.json shapes: EVERY replica of C2, C3 (both layouts), C4 and C5 after a multi-sweep call, the
oracle running one replica per host thread (ctypes releases the GIL; the oracle itself stays single-threaded).
Sized for about a minute on a 16-core host."""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu


def _threads():
    try:
        return max(1, min(32, len(os.sched_getaffinity(0))))
    except AttributeError:
        return max(1, min(32, os.cpu_count() or 1))


def _check_all_replicas(oracle_mod, cfg, n_sweeps, layout="int8"):
    w = sp.workloads.config(cfg, layout=layout)
    potts = w.model == "potts"
    sim = sp.spin_create_ex(w.batch, w.L, sp.SPIN_MODEL_POTTS if potts else sp.SPIN_MODEL_ISING, q_per_replica=w.q,
                            seed=w.seed, layout=sp.SPIN_LAYOUT_BITPACKED if layout == "bits" else sp.SPIN_LAYOUT_INT8)
    with sim:
        sim.spin_sweep(w.beta, w.J, w.h, n_sweeps, 0)
        got = sim.spin_get_spins()
        E, M = sim.spin_observables()

    def one(b):
        qb = int(w.q[b]) if potts else None
        ref = oracle_mod.init(1, w.L, seed=w.seed, q=qb, replica_offset=b)
        oracle_mod.sweep(ref, w.beta[b:b + 1], w.J, w.h, seed=w.seed, n_sweeps=n_sweeps, q=qb, replica_offset=b)
        Eo, Mo = oracle_mod.potts_observables(ref, qb) if potts else oracle_mod.ising_observables(ref)
        return bool(np.array_equal(got[b], ref[0])) and int(E[b]) == int(Eo[0]) and int(M[b]) == int(Mo[0])

    with ThreadPoolExecutor(_threads()) as ex:
        ok = list(ex.map(one, range(w.batch)))
    bad = [b for b, v in enumerate(ok) if not v]
    assert not bad, "replicas differing from the oracle after %d sweeps: %s" % (n_sweeps, bad[:10])


def test_config2_every_replica(oracle_mod):
    _check_all_replicas(oracle_mod, 2, n_sweeps=60)     # 64 x 1024^2 x 60 = 4.0e9 updates on the host


@pytest.mark.parametrize("layout", ["int8", "bits"])
def test_config3_every_replica(oracle_mod, layout):
    _check_all_replicas(oracle_mod, 3, n_sweeps=5, layout=layout)   # 4 x 8192^2 x 5 = 1.3e9 updates per layout


def test_config4_every_replica(oracle_mod):
    _check_all_replicas(oracle_mod, 4, n_sweeps=80)     # 128 x 512^2 x 80 = 2.7e9 updates (two words per site)


def test_config5_every_replica(oracle_mod):
    _check_all_replicas(oracle_mod, 5, n_sweeps=60)     # 1024 x 256^2 x 60 = 4.0e9 updates


@pytest.mark.skipif(os.environ.get("SPIN_FULL_CONFIGS") != "1",
                    reason="full-length configurations: 2e10-7e11 host updates, minutes to an hour; set SPIN_FULL_CONFIGS=1")
@pytest.mark.parametrize("cfg,layout", [(2, "int8"), (3, "int8"), (3, "bits"), (4, "int8"), (5, "int8")])
def test_full_length_configuration_every_replica(oracle_mod, cfg, layout):
    """The complete BASELINE.json configuration (all sweeps, all replicas) against the oracle: final lattice, E, M."""
    _check_all_replicas(oracle_mod, cfg, n_sweeps=sp.workloads.config(cfg).n_sweeps, layout=layout)
