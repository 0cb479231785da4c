"""GPU parity over the launch plans of the row-marching kernels (csrc/spin_internal.cuh, plan_rows): 2, 4 or 8 rows per
thread and the point where a half-sweep releases the next launch (at block exit, at the first instruction, at a thread's
last rows) are chosen from the size of the launch.  The result may not depend on any of it: one shape per branch of each
kernel's planner, streaming policy, lattice and observables against the oracle after every compared sweep.

w8 = threads of the 8-row grid / (128 x 148 x resident blocks per SM: int8 Ising 5, bit-packed 8, Potts 4).  From
0.3 / 0.15 / 0.2 waves upwards (and batch >= 2) the batch runs as two replica groups on two streams with their own
thresholds; `_plan` below restates the rules of csrc/ (ising_int8.cu, ising_bits.cu, potts_int8.cu, spin_api.cu)."""
import numpy as np
import pytest

import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu


def _w8(batch, L, layout, slots_per_sm):
    per = (L // 8) * (L >> (6 if layout == "bits" else 5))
    return per * batch / (128.0 * 148 * slots_per_sm)


def _plan(kind, batch, L):
    """(rows per thread, replica groups) the library picks for a streaming half-sweep of this shape."""
    layout = "bits" if kind == "bits" else "int8"
    w8 = _w8(batch, L, layout, {"int8": 5, "bits": 8, "potts": 4}[kind])
    groups = 2 if batch >= 2 and w8 >= {"int8": 0.3, "bits": 0.15, "potts": 0.2}[kind] else 1
    lo, hi = {"int8": ((0.25, 1.2), (0.6, 1.2)), "bits": ((0.3, 0.75), (0.3, 0.75)), "potts": ((0.3, 1.5), (0.55, 1.2))}[kind][groups - 1]
    per8 = (L // 8) * (L >> (6 if layout == "bits" else 5))
    return (2 if per8 < 64 or w8 < lo else 4 if w8 < hi else 8), groups


ISING_PLANS = [
    # batch, L, layout, expected (rows, groups), J, h
    (2, 1024, "int8", (2, 1), 1.0, 0.0),        # w8 0.09
    (100, 256, "int8", (4, 1), -1.0, 0.2),      # w8 0.27, many replicas per wave
    (1, 4096, "int8", (4, 1), 1.0, 0.01),       # w8 0.69, one replica: no groups
    (8, 1024, "int8", (2, 2), 1.0, 0.01),       # w8 0.35
    (16, 1024, "int8", (4, 2), 1.0, 0.0),       # w8 0.69
    (30, 1024, "int8", (8, 2), 1.0, 0.0),       # w8 1.30, released at the first instruction
    (3, 64, "int8", (2, 1), 1.0, 0.0),          # fewer than 64 eight-row threads per replica
    (4, 1024, "bits", (2, 1), 1.0, 0.01),       # w8 0.05, released at the last rows
    (12, 1024, "bits", (2, 2), 1.0, 0.0),       # w8 0.16, released at exit
    (32, 1024, "bits", (4, 2), -1.0, 0.2),      # w8 0.43
    (60, 1024, "bits", (8, 2), 1.0, 0.0),       # w8 0.81
    (1, 8192, "bits", (8, 1), 1.0, 0.0),        # w8 0.86, one replica
]


@pytest.mark.parametrize("batch,L,layout,rows,J,h", ISING_PLANS)
def test_ising_every_plan_equals_oracle(oracle_mod, batch, L, layout, rows, J, h):
    assert rows == _plan(layout, batch, L), "the case no longer hits the branch it names"
    seed = 300 + batch
    beta = np.linspace(0.3, 0.6, batch)
    if batch > 1:
        beta[-1] = 20.0                                       # one replica with never-accepted classes
    lay = sp.SPIN_LAYOUT_BITPACKED if layout == "bits" else sp.SPIN_LAYOUT_INT8
    ref = oracle_mod.init(batch, L, seed=seed)
    with sp.spin_create_ex(batch, L, sp.SPIN_MODEL_ISING, seed=seed, layout=lay) as sim:
        sim.spin_set_policy(sp.SPIN_POLICY_STREAMING)
        for t0, n in ((0, 1), (1, 3)):
            l0 = sim.spin_kernel_launches()
            sim.spin_sweep(beta, J, h, n, t0)
            assert sim.spin_kernel_launches() - l0 == 2 * n * rows[1]        # colours x sweeps x replica groups
            oracle_mod.sweep(ref, beta, J, h, seed=seed, n_sweeps=n, sweep_offset=t0)
            assert np.array_equal(sim.spin_get_spins(), ref), "lattice differs after sweep %d" % (t0 + n - 1)
        E, M = sim.spin_observables()
        Eo, Mo = oracle_mod.ising_observables(ref)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)


@pytest.mark.parametrize("batch,L,rows", [(2, 512, (2, 1)), (1, 4096, (4, 1)), (32, 512, (2, 2)), (64, 512, (4, 2)),
                                          (120, 512, (8, 2))])
def test_potts_every_plan_equals_oracle(oracle_mod, batch, L, rows):
    assert rows == _plan("potts", batch, L), "the case no longer hits the branch it names"
    seed = 400 + batch
    q = np.array([3, 8, 5, 127][: min(batch, 4)] + [3 + (b % 6) for b in range(max(0, batch - 4))], dtype=np.int32)
    beta = np.linspace(0.5, 1.6, batch)
    if batch > 1:
        beta[0] = 25.0                                        # never-accepted classes
    ref = oracle_mod.init(batch, L, seed=seed, q=q)
    with sp.spin_create_ex(batch, L, sp.SPIN_MODEL_POTTS, q_per_replica=q, seed=seed) as sim:
        for t0, n in ((0, 1), (1, 2)):
            l0 = sim.spin_kernel_launches()
            sim.spin_sweep(beta, 1.0, 0.0, n, t0)
            assert sim.spin_kernel_launches() - l0 == 2 * n * rows[1]        # colours x sweeps x replica groups
            oracle_mod.sweep(ref, beta, 1.0, 0.0, seed=seed, n_sweeps=n, sweep_offset=t0, q=q)
            assert np.array_equal(sim.spin_get_spins(), ref), "lattice differs after sweep %d" % (t0 + n - 1)
        E, M = sim.spin_observables()
        Eo, Mo = oracle_mod.potts_observables(ref, q)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)


@pytest.mark.parametrize("batch,L", [(4, 1024), (32, 1024), (60, 1024)])
def test_bit_packed_bonds_every_plan_equals_oracle(oracle_mod, batch, L):
    """The +-J variant of the bit-packed kernel has its own instantiations per rows-per-thread."""
    seed = 500 + batch
    rng = np.random.default_rng(seed)
    Jh = (2 * rng.integers(0, 2, size=(1, L, L)) - 1).astype(np.int8)
    Jv = (2 * rng.integers(0, 2, size=(1, L, L)) - 1).astype(np.int8)
    beta = np.linspace(0.4, 1.2, batch)
    ref = oracle_mod.init(batch, L, seed=seed)
    with sp.spin_create_ex(batch, L, sp.SPIN_MODEL_ISING, seed=seed, layout=sp.SPIN_LAYOUT_BITPACKED) as sim:
        sim.spin_set_bonds(Jh[0], Jv[0])
        sim.spin_sweep(beta, 1.0, 0.05, 3, 7)
        oracle_mod.sweep_bonds(ref, Jh, Jv, beta, 1.0, 0.05, seed=seed, n_sweeps=3, sweep_offset=7)
        assert np.array_equal(sim.spin_get_spins(), ref)
        E, M = sim.spin_observables()
        Eo, Mo = oracle_mod.ising_bonds_observables(ref, Jh, Jv)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)


# ----------------------------------------------------------------- replica groups on two streams (csrc/spin_api.cu)
@pytest.mark.parametrize("model,batch,L,layout", [("ising", 31, 1024, "bits"), ("ising", 13, 1024, "int8"),
                                                  ("potts", 27, 512, "int8")])
def test_two_replica_groups_sweep_schedule_and_later_calls(oracle_mod, model, batch, L, layout):
    """From 0.3 waves of 8-row blocks upwards a streaming sweep runs as two replica groups on two streams (odd batches
    split unevenly); later operations of the handle (observables, a schedule, a measured sweep, get_spins) must see both
    groups finished, and spin_sweep_schedule runs every step on both."""
    seed = 600 + batch
    assert _plan("potts" if model == "potts" else layout, batch, L)[1] == 2, "the case no longer runs as two groups"
    q = None if model == "ising" else np.array([3 + (b % 6) for b in range(batch)], dtype=np.int32)
    h = 0.02 if model == "ising" else 0.0
    beta = np.linspace(0.4, 1.1, batch)
    ref = oracle_mod.init(batch, L, seed=seed, q=q)
    lay = sp.SPIN_LAYOUT_BITPACKED if layout == "bits" else sp.SPIN_LAYOUT_INT8
    mdl = sp.SPIN_MODEL_ISING if model == "ising" else sp.SPIN_MODEL_POTTS
    obs = oracle_mod.ising_observables if model == "ising" else (lambda s: oracle_mod.potts_observables(s, q))
    with sp.spin_create_ex(batch, L, mdl, q_per_replica=q, seed=seed, layout=lay) as sim:
        l0 = sim.spin_kernel_launches()
        sim.spin_sweep(beta, 1.0, h, 2, 0)
        assert sim.spin_kernel_launches() - l0 == 2 * 2 * 2          # sweeps x colours x groups
        oracle_mod.sweep(ref, beta, 1.0, h, seed=seed, n_sweeps=2, q=q)
        E, M = sim.spin_observables()                                 # on the handle's stream, right after the join
        Eo, Mo = obs(ref)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
        steps = np.stack([beta, beta[::-1], 0.5 * beta])
        sim.spin_sweep_schedule(steps, 1.0, h, 2, sweep_offset=2)
        oracle_mod.sweep_schedule(ref, steps, 1.0, h, seed, 2, sweep_offset=2, q=q)
        assert np.array_equal(sim.spin_get_spins(), ref)
        Et, Mt = sim.spin_sweep_measure(beta, 1.0, h, 2, 8)
        Eo, Mo = oracle_mod.sweep(ref, beta, 1.0, h, seed=seed, n_sweeps=2, sweep_offset=8, q=q, trace=True)
        assert np.array_equal(Et, Eo) and np.array_equal(Mt, Mo)
        assert np.array_equal(sim.spin_get_spins(), ref)


# ----------------------------------------------------------------- SPIN_POLICY_GRAPH: sweeps replayed from a CUDA graph
def _oracle_sweep_threads(oracle_mod, ref, beta, h, seed, n, t0, q):
    """oracle.sweep replica by replica on host threads (replica_offset = b): same lattices, a fraction of the wall time."""
    from concurrent.futures import ThreadPoolExecutor

    def one(b):
        oracle_mod.sweep(ref[b:b + 1], beta[b:b + 1], 1.0, h, seed=seed, n_sweeps=n, sweep_offset=t0,
                         q=None if q is None else q[b:b + 1], replica_offset=b)
    with ThreadPoolExecutor(16) as ex:
        list(ex.map(one, range(ref.shape[0])))


@pytest.mark.parametrize("model,batch,L,layout,calls", [
    ("ising", 3, 96, "int8", (64 * 2 + 5, 64, 7)), ("ising", 2, 128, "bits", (64 * 2 + 5, 64, 7)),
    ("potts", 2, 64, "int8", (64 * 2 + 5, 64, 7)),
    ("ising", 13, 1024, "int8", (67, 64)), ("ising", 12, 1024, "bits", (67, 64)), ("potts", 27, 512, "int8", (67, 64))])
def test_graph_policy_equals_oracle(oracle_mod, model, batch, L, layout, calls):
    """The kernels of a graph read the sweep index from device memory: replays of 64 sweeps, the ragged rest as plain
    launches, a later call that replays the same graph, a sweep index that crosses 2^32 inside a replay, one and two
    replica groups, never-accepted classes; short calls stream."""
    import torch
    seed = 700 + batch + L
    q = None if model == "ising" else np.array([3 + (b % 6) for b in range(batch)], dtype=np.int32)
    h = 0.02 if model == "ising" else 0.0
    beta = np.linspace(0.4, 1.1, batch)
    beta[-1] = 22.0
    ref = oracle_mod.init(batch, L, seed=seed, q=q)
    lay = sp.SPIN_LAYOUT_BITPACKED if layout == "bits" else sp.SPIN_LAYOUT_INT8
    mdl = sp.SPIN_MODEL_ISING if model == "ising" else sp.SPIN_MODEL_POTTS
    groups = _plan("potts" if model == "potts" else layout, batch, L)[1]
    assert groups == (2 if L >= 512 else 1)
    stream = torch.cuda.Stream()                              # the legacy default stream cannot be captured
    with sp.spin_create_ex(batch, L, mdl, q_per_replica=q, seed=seed, layout=lay, cuda_stream=stream.cuda_stream) as sim:
        sim.spin_set_policy(sp.SPIN_POLICY_GRAPH)
        t0 = (1 << 32) - 70
        for n in calls:
            l0 = sim.spin_kernel_launches()
            sim.spin_sweep(beta, 1.0, h, n, t0)
            replays = n // 64
            # per replay: 64 sweeps x 2 colours x groups + the node that advances the index; + 1 kernel that sets it per call
            want = replays * (64 * 2 * groups + 1) + (1 if replays else 0) + (n % 64) * 2 * groups
            assert sim.spin_kernel_launches() - l0 == want
            _oracle_sweep_threads(oracle_mod, ref, beta, h, seed, n, t0, q)
            assert np.array_equal(sim.spin_get_spins(), ref), n
            t0 += n
        E, M = sim.spin_observables()
        Eo, Mo = oracle_mod.ising_observables(ref) if model == "ising" else oracle_mod.potts_observables(ref, q)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
    # on the legacy default stream the policy falls back to plain launches
    with sp.spin_create_ex(batch, L, mdl, q_per_replica=q, seed=seed, layout=lay) as sim:
        sim.spin_set_policy(sp.SPIN_POLICY_GRAPH)
        l0 = sim.spin_kernel_launches()
        sim.spin_sweep(beta, 1.0, h, 64, 0)
        assert sim.spin_kernel_launches() - l0 == 64 * 2 * groups


def test_graph_policy_with_bonds_rebuilds_the_graph(oracle_mod):
    """+-J couplings on the bit-packed layout: the graph holds the pointer to the sign planes and is captured again after
    spin_set_bonds replaced or removed them."""
    import torch
    batch, L, seed = 2, 256, 77
    rng = np.random.default_rng(seed)
    mk = lambda: (2 * rng.integers(0, 2, size=(batch, L, L)) - 1).astype(np.int8)
    beta = np.linspace(0.5, 1.5, batch)
    ref = oracle_mod.init(batch, L, seed=seed)
    stream = torch.cuda.Stream()
    with sp.spin_create_ex(batch, L, sp.SPIN_MODEL_ISING, seed=seed, layout=sp.SPIN_LAYOUT_BITPACKED,
                           cuda_stream=stream.cuda_stream) as sim:
        sim.spin_set_policy(sp.SPIN_POLICY_GRAPH)
        t = 0
        for bonds in (None, (mk(), mk()), (mk(), mk()), None):
            l0 = sim.spin_kernel_launches()
            if bonds is None:
                sim.spin_set_bonds(None, None)
                sim.spin_sweep(beta, 1.0, 0.0, 66, t)
                oracle_mod.sweep(ref, beta, 1.0, 0.0, seed=seed, n_sweeps=66, sweep_offset=t)
            else:
                sim.spin_set_bonds(bonds[0], bonds[1])
                sim.spin_sweep(beta, 1.0, 0.0, 66, t)
                oracle_mod.sweep_bonds(ref, bonds[0], bonds[1], beta, 1.0, 0.0, seed=seed, n_sweeps=66, sweep_offset=t)
            assert np.array_equal(sim.spin_get_spins(), ref)
            t += 66


# ----------------------------------------------------------------- spin_sweep_measure on the streaming path (fused E / M)
@pytest.mark.parametrize("batch,L", [(13, 1024), (40, 256), (3, 96)])
def test_fused_measure_two_groups_traces_and_moments(oracle_mod, batch, L):
    """The colour-1 launch adds the E / M sums, the next sweep's colour-0 launch (or the finalisation kernel after the last
    sweep) turns them into the sample: traces and moments against the oracle, two replica groups, a replica with
    never-accepted classes, a second call that continues, launch counts (no reduction launches any more)."""
    seed, n = 800 + batch, 5
    groups = _plan("int8", batch, L)[1]
    beta = np.linspace(0.3, 0.6, batch)
    beta[-1] = 20.0
    ref = oracle_mod.init(batch, L, seed=seed)
    mom_o = np.zeros((batch, 8), dtype=np.int64)
    Eo, Mo = oracle_mod.sweep(ref, beta, 1.0, 0.03, seed=seed, n_sweeps=n, sweep_offset=4, trace=True, moments=mom_o)
    with sp.spin_create_ex(batch, L, sp.SPIN_MODEL_ISING, seed=seed) as sim:
        sim.spin_set_policy(sp.SPIN_POLICY_STREAMING)
        mom = np.zeros((batch, 8), dtype=np.int64)
        l0 = sim.spin_kernel_launches()
        E1, M1 = sim.spin_sweep_measure(beta, 1.0, 0.03, 2, 4, moments=mom)
        assert sim.spin_kernel_launches() - l0 == (2 * 2 + 1) * groups      # sweeps x colours + one finalisation, per group
        E2, M2 = sim.spin_sweep_measure(beta, 1.0, 0.03, n - 2, 6, moments=mom)
        assert np.array_equal(np.vstack([E1, E2]), Eo) and np.array_equal(np.vstack([M1, M2]), Mo)
        assert np.array_equal(mom, mom_o)
        assert np.array_equal(sim.spin_get_spins(), ref)
        # moments only (no trace), then a plain sweep and the stand-alone reduction agree with the oracle
        sim.spin_sweep_measure(beta, 1.0, 0.03, 2, 4 + n, trace=False, moments=mom)
        oracle_mod.sweep(ref, beta, 1.0, 0.03, seed=seed, n_sweeps=2, sweep_offset=4 + n, moments=mom_o)
        assert np.array_equal(mom, mom_o)
        E, M = sim.spin_observables()
        Eo2, Mo2 = oracle_mod.ising_observables(ref)
        assert np.array_equal(E, Eo2) and np.array_equal(M, Mo2)
