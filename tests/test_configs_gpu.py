"""GPU parity at the BASELINE.json shapes, in the launch configuration bench.py times.

The full configurations are 1e11-7e11 updates; the oracle does about 2e7 per second.  So (SURVEY 8(d) parity
schedule): C1 is compared completely (all 1000 sweeps, E/M trace and final lattice); for C2-C5 the GPU runs the
full batch at full size and single replicas are compared against the oracle run alone with replica_offset,
lattice and E/M after every one of the first sweeps."""
import numpy as np
import pytest

import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu


def _create(w, layout=None):
    layout = layout or w.layout
    lay = sp.SPIN_LAYOUT_BITPACKED if layout == "bits" else sp.SPIN_LAYOUT_INT8
    if w.model == "potts":
        return sp.spin_create_ex(w.batch, w.L, sp.SPIN_MODEL_POTTS, q_per_replica=w.q, seed=w.seed)
    return sp.spin_create_ex(w.batch, w.L, sp.SPIN_MODEL_ISING, seed=w.seed, layout=lay)


@pytest.mark.parametrize("policy", [sp.SPIN_POLICY_AUTO, sp.SPIN_POLICY_STREAMING])
def test_config1_complete(oracle_mod, policy):
    """All 1000 sweeps, every (E, M), final lattice: once as bench.py runs it (AUTO: one resident launch) and once
    through the two-launches-per-sweep kernels."""
    w = sp.workloads.config(1)
    ref = oracle_mod.init(w.batch, w.L, seed=w.seed)
    Eo, Mo = oracle_mod.sweep(ref, w.beta, w.J, w.h, seed=w.seed, n_sweeps=w.n_sweeps, trace=True)
    with _create(w) as sim:
        sim.spin_set_policy(policy)
        assert (sim.spin_kernel_variant() == "ising_int8_resident") == (policy == sp.SPIN_POLICY_AUTO)
        E, M = sim.spin_sweep_measure(w.beta, w.J, w.h, w.n_sweeps, 0)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
        assert np.array_equal(sim.spin_get_spins(), ref)


def _compare_after_one_call(oracle_mod, w, replicas, n_sweeps, policy=sp.SPIN_POLICY_AUTO):
    """The whole batch runs n_sweeps in ONE spin_sweep call (the way bench.py drives it); sampled replicas are then
    compared with the oracle run alone: lattice, E_int, M."""
    q = None if w.q is None else w.q
    with _create(w) as sim:
        sim.spin_set_policy(policy)
        sim.spin_sweep(w.beta, w.J, w.h, n_sweeps, 0)
        got = sim.spin_get_spins()
        E, M = sim.spin_observables()
    for b in replicas:
        qb = None if q is None else int(q[b])
        ref = oracle_mod.init(1, w.L, seed=w.seed, q=qb, replica_offset=b)
        oracle_mod.sweep(ref, w.beta[b:b + 1], w.J, w.h, seed=w.seed, n_sweeps=n_sweeps, q=qb, replica_offset=b)
        assert np.array_equal(got[b], ref[0]), "replica %d differs after %d sweeps" % (b, n_sweeps)
        Eo, Mo = oracle_mod.ising_observables(ref) if qb is None else oracle_mod.potts_observables(ref, qb)
        assert int(E[b]) == int(Eo[0]) and int(M[b]) == int(Mo[0])


def _compare_sampled_replicas(oracle_mod, w, replicas, n_sweeps, layout=None):
    q = None if w.q is None else w.q
    with _create(w, layout) as sim:
        refs = {}
        for b in replicas:
            refs[b] = oracle_mod.init(1, w.L, seed=w.seed, q=None if q is None else int(q[b]), replica_offset=b)
        got = sim.spin_get_spins()
        for b in replicas:
            assert np.array_equal(got[b], refs[b][0]), "init differs, replica %d" % b
        for t in range(n_sweeps):
            sim.spin_sweep(w.beta, w.J, w.h, 1, t)
            got = sim.spin_get_spins()
            E, M = sim.spin_observables()
            for b in replicas:
                qb = None if q is None else int(q[b])
                oracle_mod.sweep(refs[b], w.beta[b:b + 1], w.J, w.h, seed=w.seed, n_sweeps=1, sweep_offset=t, q=qb,
                                 replica_offset=b)
                assert np.array_equal(got[b], refs[b][0]), "replica %d differs after sweep %d" % (b, t)
                if qb is None:
                    Eo, Mo = oracle_mod.ising_observables(refs[b])
                else:
                    Eo, Mo = oracle_mod.potts_observables(refs[b], qb)
                assert int(E[b]) == int(Eo[0]) and int(M[b]) == int(Mo[0])


def test_config2_sampled_replicas(oracle_mod):
    _compare_sampled_replicas(oracle_mod, sp.workloads.config(2), [0, 31, 63], n_sweeps=3)
    _compare_after_one_call(oracle_mod, sp.workloads.config(2), [0, 63], n_sweeps=100)


@pytest.mark.parametrize("layout", ["int8", "bits"])
def test_config3_all_replicas(oracle_mod, layout):
    # 8192^2 = 6.7e7 sites per replica: all four replicas, 3 sweeps, lattice and (E, M) after every sweep
    # (8e8 oracle updates per layout)
    _compare_sampled_replicas(oracle_mod, sp.workloads.config(3), [0, 1, 2, 3], n_sweeps=3, layout=layout)


def test_config4_sampled_replicas(oracle_mod):
    _compare_sampled_replicas(oracle_mod, sp.workloads.config(4), [0, 63, 64, 127], n_sweeps=5)
    _compare_after_one_call(oracle_mod, sp.workloads.config(4), [5, 100], n_sweeps=200)


def test_config5_sampled_replicas_and_moments(oracle_mod):
    w = sp.workloads.config(5)
    _compare_sampled_replicas(oracle_mod, w, [0, 512, 1023], n_sweeps=5)
    _compare_after_one_call(oracle_mod, w, [1, 511, 1022], n_sweeps=1000)
    _compare_after_one_call(oracle_mod, w, [2, 1000], n_sweeps=50, policy=sp.SPIN_POLICY_RESIDENT)
    # thermalise, then moments over a window: all 1024 replicas on the GPU (AUTO: the resident kernel with fused
    # reductions; STREAMING: half-sweep kernels + reduction kernels), three replicas checked against the oracle
    n_therm, n_meas = 20, 60
    expect = {}
    for b in (0, 700, 1023):
        ref = oracle_mod.init(1, w.L, seed=w.seed, replica_offset=b)
        oracle_mod.sweep(ref, w.beta[b:b + 1], w.J, w.h, seed=w.seed, n_sweeps=n_therm, replica_offset=b)
        mo = np.zeros((1, 8), dtype=np.int64)
        oracle_mod.sweep(ref, w.beta[b:b + 1], w.J, w.h, seed=w.seed, n_sweeps=n_meas, sweep_offset=n_therm,
                         replica_offset=b, moments=mo)
        expect[b] = (mo[0], ref[0])
    for policy in (sp.SPIN_POLICY_AUTO, sp.SPIN_POLICY_STREAMING):
        with _create(w) as sim:
            sim.spin_set_policy(policy)
            sim.spin_sweep(w.beta, w.J, w.h, n_therm, 0)
            mom = np.zeros((w.batch, 8), dtype=np.int64)
            sim.spin_sweep_measure(w.beta, w.J, w.h, n_meas, n_therm, trace=False, moments=mom)
            got = sim.spin_get_spins()
        for b, (mo, lat) in expect.items():
            assert np.array_equal(mom[b], mo), "moments differ, replica %d, policy %d" % (b, policy)
            assert np.array_equal(got[b], lat)
