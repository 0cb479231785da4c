"""GPU parity tests (-m gpu): the CUDA path through the C ABI vs the CPU oracle, bit for bit.

Bar (BASELINE.json north star): lattices identical after every compared sweep, E_int and M identical as exact
integers, threshold tables identical.  Small cases compare everything; the full-size cases compare all
replicas for a few sweeps and single replicas (via replica_offset on the oracle side) for longer."""
import math

import numpy as np
import pytest

import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu


def _layout(name):
    return sp.SPIN_LAYOUT_BITPACKED if name == "bits" else sp.SPIN_LAYOUT_INT8


def _mk_ising(batch, L, seed, layout="int8", replica_offset=0, policy=None):
    sim = sp.spin_create_ex(batch, L, sp.SPIN_MODEL_ISING, seed=seed, layout=_layout(layout),
                            replica_offset=replica_offset)
    if policy is not None:
        sim.spin_set_policy(policy)
    return sim


# every int8 Ising case runs through the three kernel families: the two-launches-per-sweep HBM kernels, the
# shared-memory-resident multi-sweep kernel and the persistent cooperative kernel (each used when the shape allows it,
# else the call falls back to streaming)
POLICIES = [sp.SPIN_POLICY_STREAMING, sp.SPIN_POLICY_RESIDENT, sp.SPIN_POLICY_PERSISTENT, sp.SPIN_POLICY_TILED]


def _mk_potts(batch, L, q, seed, replica_offset=0):
    q = np.broadcast_to(np.asarray(q, dtype=np.int32), (batch,))
    return sp.spin_create_ex(batch, L, sp.SPIN_MODEL_POTTS, q_per_replica=q, seed=seed, replica_offset=replica_offset)


# ----------------------------------------------------------------------------------------- init (row a0)
@pytest.mark.parametrize("L,layout", [(2, "int8"), (4, "int8"), (6, "int8"), (10, "int8"), (32, "int8"),
                                      (96, "int8"), (64, "bits"), (192, "bits")])
def test_init_matches_oracle_ising(oracle_mod, L, layout):
    with _mk_ising(3, L, seed=11, layout=layout, replica_offset=5) as sim:
        got = sim.spin_get_spins()
    assert np.array_equal(got, oracle_mod.init(3, L, seed=11, replica_offset=5))


def test_init_matches_oracle_potts(oracle_mod):
    q = [3, 8, 2, 127, 5]
    for L in (2, 6, 32, 64):
        with _mk_potts(5, L, q, seed=4) as sim:
            got = sim.spin_get_spins()
        assert np.array_equal(got, oracle_mod.init(5, L, seed=4, q=q))


def test_set_get_roundtrip_and_validation():
    for L, layout in [(2, "int8"), (6, "int8"), (32, "int8"), (64, "bits"), (128, "bits")]:
        with _mk_ising(3, L, seed=1, layout=layout) as sim:
            lat = sp.workloads.random_ising_lattice(3, L, seed=L)
            sim.spin_set_spins(lat)
            assert np.array_equal(sim.spin_get_spins(), lat)
            bad = lat.copy()
            bad[1, 0, 1] = 0
            with pytest.raises(sp.SpinError):
                sim.spin_set_spins(bad)
            assert np.array_equal(sim.spin_get_spins(), lat)  # unchanged after a rejected set
    with _mk_potts(2, 8, [3, 8], seed=1) as sim:
        lat = sp.workloads.random_potts_lattice(2, 8, [3, 8], seed=2)
        sim.spin_set_spins(lat)
        assert np.array_equal(sim.spin_get_spins(), lat)
        bad = lat.copy()
        bad[0, 0, 0] = 3
        with pytest.raises(sp.SpinError):
            sim.spin_set_spins(bad)


# ----------------------------------------------------------------------------------------- Ising sweeps
ISING_CASES = [
    # L, batch, layout, J, h, betas
    (2, 3, "int8", 1.0, 0.0, [0.2, 0.44, 0.9]),
    (4, 4, "int8", 1.0, 0.01, [0.1, 0.44, 0.6, 20.0]),
    (6, 2, "int8", 1.0, 0.0, [0.3, 0.5]),
    (10, 3, "int8", -1.0, 0.2, [0.3, 0.44, 0.0]),
    (32, 4, "int8", 1.0, 0.0, [0.44] * 4),
    (64, 3, "int8", 1.0, 0.01, [0.3, 0.4407, 20.0]),
    (96, 2, "int8", 0.7, -0.3, [0.5, 1.0]),
    (160, 2, "int8", 1.0, 0.0, [0.44, 0.6]),
    (64, 3, "bits", 1.0, 0.01, [0.3, 0.4407, 20.0]),
    (128, 2, "bits", 1.0, 0.0, [0.44, 0.0]),
    (192, 2, "bits", -1.0, 0.2, [0.4, 0.8]),
]


@pytest.mark.parametrize("policy", POLICIES)
@pytest.mark.parametrize("L,batch,layout,J,h,betas", ISING_CASES)
def test_ising_sweeps_match_oracle_every_sweep(oracle_mod, L, batch, layout, J, h, betas, policy):
    seed, n = 100 + L, 12
    ref = oracle_mod.init(batch, L, seed=seed)
    with _mk_ising(batch, L, seed=seed, layout=layout, policy=policy) as sim:
        if policy == sp.SPIN_POLICY_RESIDENT and layout == "bits":
            assert sim.spin_kernel_variant() == "ising_bits_resident"
        elif policy == sp.SPIN_POLICY_RESIDENT and L % 32 == 0:
            assert sim.spin_kernel_variant() == "ising_int8_resident"
        for t in range(n):
            sim.spin_sweep(betas, J, h, 1, t)
            oracle_mod.sweep(ref, betas, J, h, seed=seed, n_sweeps=1, sweep_offset=t)
            got = sim.spin_get_spins()
            assert np.array_equal(got, ref), "lattice differs after sweep %d" % t
            E, M = sim.spin_observables()
            Eo, Mo = oracle_mod.ising_observables(ref)
            assert np.array_equal(E, Eo) and np.array_equal(M, Mo)


def test_ising_chunking_offsets_and_replica_offset(oracle_mod):
    L, seed = 64, 9
    beta = [0.3, 0.44, 0.6]
    with _mk_ising(3, L, seed=seed) as a, _mk_ising(3, L, seed=seed) as b, \
            _mk_ising(1, L, seed=seed, replica_offset=2) as solo:
        a.spin_sweep(beta, 1.0, 0.0, 10, 0)
        b.spin_sweep(beta, 1.0, 0.0, 4, 0)
        b.spin_sweep(beta, 1.0, 0.0, 6, 4)
        solo.spin_sweep(beta[2:], 1.0, 0.0, 10, 0)
        la = a.spin_get_spins()
        assert np.array_equal(la, b.spin_get_spins())
        assert np.array_equal(la[2], solo.spin_get_spins()[0])
    big = (1 << 32) + 3  # sweep index beyond 32 bits goes into counter word 3
    ref = oracle_mod.init(1, 32, seed=seed)
    oracle_mod.sweep(ref, 0.44, 1.0, 0.0, seed=seed, n_sweeps=2, sweep_offset=big)
    with _mk_ising(1, 32, seed=seed) as sim:
        sim.spin_sweep(0.44, 1.0, 0.0, 2, big)
        assert np.array_equal(sim.spin_get_spins(), ref)
    seed64 = (0xDEADBEEF << 32) | 0x12345678  # both key words
    ref = oracle_mod.init(2, 32, seed=seed64)
    oracle_mod.sweep(ref, 0.44, 1.0, 0.0, seed=seed64, n_sweeps=3)
    with _mk_ising(2, 32, seed=seed64) as sim:
        sim.spin_sweep(0.44, 1.0, 0.0, 3, 0)
        assert np.array_equal(sim.spin_get_spins(), ref)


def test_bitpacked_equals_int8(oracle_mod):
    L, seed = 256, 3
    with _mk_ising(2, L, seed=seed, layout="int8") as a, _mk_ising(2, L, seed=seed, layout="bits") as b:
        assert np.array_equal(a.spin_get_spins(), b.spin_get_spins())
        a.spin_sweep(0.4407, 1.0, 0.01, 25, 0)
        b.spin_sweep(0.4407, 1.0, 0.01, 25, 0)
        assert np.array_equal(a.spin_get_spins(), b.spin_get_spins())
        Ea, Ma = a.spin_observables()
        Eb, Mb = b.spin_observables()
        assert np.array_equal(Ea, Eb) and np.array_equal(Ma, Mb)


def test_set_spins_then_sweep(oracle_mod):
    L = 32
    lat = sp.workloads.random_ising_lattice(2, L, seed=77)
    ref = lat.copy()
    oracle_mod.sweep(ref, [0.4, 0.5], 1.0, 0.0, seed=5, n_sweeps=3, sweep_offset=7)
    with _mk_ising(2, L, seed=5) as sim:
        sim.spin_set_spins(lat)
        sim.spin_sweep([0.4, 0.5], 1.0, 0.0, 3, 7)
        assert np.array_equal(sim.spin_get_spins(), ref)


# ----------------------------------------------------------------------------------------- Potts sweeps
POTTS_CASES = [
    (2, [3, 8], [1.0, 1.3]),
    (4, [3, 8, 2], [0.5, 1.34, 0.88]),
    (6, [3, 5], [1.0, 20.0]),
    (10, [8, 127], [1.2, 2.0]),
    (32, [3, 8, 2, 127], [1.005, 1.342, 0.0, 3.0]),
    (64, [3, 8], [20.0, 0.7]),
    (96, [4, 7], [1.1, 1.3]),
    (64, [16, 17, 15, 33], [1.6, 1.6, 20.0, 1.9]),   # both sides of the q <= 16 (shift-free indicators) boundary
]


@pytest.mark.parametrize("L,q,betas", POTTS_CASES)
def test_potts_sweeps_match_oracle_every_sweep(oracle_mod, L, q, betas):
    seed, n, batch = 200 + L, 10, len(q)
    ref = oracle_mod.init(batch, L, seed=seed, q=q)
    with _mk_potts(batch, L, q, seed=seed) as sim:
        for t in range(n):
            sim.spin_sweep(betas, 1.0, 0.0, 1, t)
            oracle_mod.sweep(ref, betas, 1.0, 0.0, seed=seed, n_sweeps=1, sweep_offset=t, q=q)
            assert np.array_equal(sim.spin_get_spins(), ref), "lattice differs after sweep %d" % t
            E, M = sim.spin_observables()
            Eo, Mo = oracle_mod.potts_observables(ref, q)
            assert np.array_equal(E, Eo) and np.array_equal(M, Mo)


def test_potts_negative_J(oracle_mod):
    q, L, seed = [3, 6], 32, 8
    ref = oracle_mod.init(2, L, seed=seed, q=q)
    oracle_mod.sweep(ref, [0.8, 1.1], -1.0, 0.0, seed=seed, n_sweeps=4, q=q)
    with _mk_potts(2, L, q, seed=seed) as sim:
        sim.spin_sweep([0.8, 1.1], -1.0, 0.0, 4, 0)
        assert np.array_equal(sim.spin_get_spins(), ref)


# ----------------------------------------------------------------------------------------- measurements
@pytest.mark.parametrize("policy", POLICIES)
@pytest.mark.parametrize("L", [32, 96, 256])
def test_sweep_measure_trace_and_moments(oracle_mod, policy, L):
    seed, n = 1, 40
    beta = [0.3, 0.44, 0.5, 0.6]
    ref = oracle_mod.init(4, L, seed=seed)
    mom_o = np.zeros((4, 8), dtype=np.int64)
    Eo, Mo = oracle_mod.sweep(ref, beta, 1.0, 0.05, seed=seed, n_sweeps=n, trace=True, moments=mom_o)
    with _mk_ising(4, L, seed=seed, policy=policy) as sim:
        mom = np.zeros((4, 8), dtype=np.int64)
        E1, M1 = sim.spin_sweep_measure(beta, 1.0, 0.05, 15, 0, moments=mom)
        E2, M2 = sim.spin_sweep_measure(beta, 1.0, 0.05, n - 15, 15, moments=mom)   # moments are in/out
        assert np.array_equal(np.vstack([E1, E2]), Eo) and np.array_equal(np.vstack([M1, M2]), Mo)
        assert np.array_equal(mom, mom_o)
        assert np.array_equal(sim.spin_get_spins(), ref)
        # float-derived quantities (north star: relative 1e-12 in double): the product's host post-processing of the
        # GPU moments against an independent exact evaluation of the oracle's traces (python rationals)
        from fractions import Fraction
        from paper_2304_01772_b200 import derived
        dg = derived.thermodynamics(mom, beta, 1.0, 0.05, L)
        for b in range(4):
            Hs = [Fraction(1.0) * int(e) - Fraction(0.05) * int(m) for e, m in zip(Eo[:, b], Mo[:, b])]
            meanH = sum(Hs) / n
            c_ref = float(Fraction(float(beta[b])) ** 2 * (sum(x * x for x in Hs) / n - meanH * meanH) / (L * L))
            u_ref = float(meanH / (L * L))
            assert abs(dg["u"][b] - u_ref) <= 1e-12 * abs(u_ref) and abs(dg["c"][b] - c_ref) <= 1e-12 * abs(c_ref)


def test_resident_multi_sweep_call_equals_streaming(oracle_mod):
    """One resident launch for 25 sweeps (t crossing 2^32, beta = 20 never-classes, odd batch) == streaming == oracle."""
    L, seed, off = 64, 77, (1 << 32) - 10
    beta = [0.2, 0.4407, 20.0, 0.6, 0.0]
    ref = oracle_mod.init(5, L, seed=seed, replica_offset=3)
    oracle_mod.sweep(ref, beta, 1.0, 0.01, seed=seed, n_sweeps=25, sweep_offset=off, replica_offset=3)
    for policy in POLICIES:
        with _mk_ising(5, L, seed=seed, replica_offset=3, policy=policy) as sim:
            sim.spin_sweep(beta, 1.0, 0.01, 25, off)
            assert np.array_equal(sim.spin_get_spins(), ref)
            with pytest.raises(sp.SpinError):
                sim.spin_set_policy(7)


def test_sweep_measure_potts(oracle_mod):
    seed = 1
    q = [3, 8]
    ref = oracle_mod.init(2, 16, seed=seed, q=q)
    mom_o = np.zeros((2, 8), dtype=np.int64)
    Eo, Mo = oracle_mod.sweep(ref, [1.0, 1.3], 1.0, 0.0, seed=seed, n_sweeps=20, q=q, trace=True, moments=mom_o)
    with _mk_potts(2, 16, q, seed=seed) as sim:
        mom = np.zeros((2, 8), dtype=np.int64)
        E, M = sim.spin_sweep_measure([1.0, 1.3], 1.0, 0.0, 20, 0, moments=mom)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo) and np.array_equal(mom, mom_o)


def test_invalid_sweep_arguments_leave_lattice_untouched():
    with _mk_ising(2, 32, seed=1) as sim:
        before = sim.spin_get_spins()
        for beta, n, off in [([0.4, float("nan")], 1, 0), ([0.4, -1.0], 1, 0), ([0.4, 0.4], -1, 0),
                             ([0.4, 0.4], 1, -1), ([0.4, 0.4], 1, 1 << 56)]:
            with pytest.raises(sp.SpinError):
                sim.spin_sweep(beta, 1.0, 0.0, n, off)
        sim.spin_sweep([0.4, 0.4], 1.0, 0.0, 0, 0)  # zero sweeps is a no-op
        assert np.array_equal(sim.spin_get_spins(), before)


def test_caller_owned_buffer_and_stream(oracle_mod):
    import torch
    L, batch, seed = 64, 2, 6
    buf = torch.empty(sp.spin_buffer_bytes(batch, L, 0, 0), dtype=torch.int8, device="cuda")
    stream = torch.cuda.Stream()
    sim = sp.spin_create_ex(batch, L, sp.SPIN_MODEL_ISING, seed=seed, device_buffer=buf.data_ptr(),
                            buffer_bytes=buf.numel(), cuda_stream=stream.cuda_stream, keepalive=buf)
    ref = oracle_mod.init(batch, L, seed=seed)
    oracle_mod.sweep(ref, 0.44, 1.0, 0.0, seed=seed, n_sweeps=5)
    sim.spin_sweep(0.44, 1.0, 0.0, 5, 0)
    sim.spin_synchronize()
    # the caller's tensor holds the split layout [B][2][L][L/2]
    split = buf.view(batch, 2, L, L // 2).cpu().numpy()
    nat = np.empty((batch, L, L), dtype=np.int8)
    for i in range(L):
        for c in range(2):
            nat[:, i, ((i + c) & 1)::2] = split[:, c, i, :]
    assert np.array_equal(nat, ref) and np.array_equal(sim.spin_get_spins(), ref)
    Ed = torch.zeros(batch, dtype=torch.int64, device="cuda")
    Md = torch.zeros(batch, dtype=torch.int64, device="cuda")
    sim.spin_observables_dev(Ed.data_ptr(), Md.data_ptr())
    sim.spin_synchronize()
    Eo, Mo = oracle_mod.ising_observables(ref)
    assert np.array_equal(Ed.cpu().numpy(), Eo) and np.array_equal(Md.cpu().numpy(), Mo)
    sim.spin_destroy()


# ------------------------------------------------------------- persistent cooperative kernel (launch-bound shapes)
@pytest.mark.parametrize("batch,L,n", [(1, 640, 12), (3, 128, 20), (2, 1024, 6), (5, 96, 15), (1, 2560, 3)])
def test_persistent_kernel_many_sweeps_in_one_launch(oracle_mod, batch, L, n):
    """All sweeps of a call in one cooperative launch, grid barrier between half-sweeps (the paper's Table III shapes,
    PAPER.md:252-276): lattice, E and M equal the oracle's; chunked calls continue the same trajectory."""
    seed, beta = 60 + L, np.linspace(0.3, 0.6, batch)
    ref = oracle_mod.init(batch, L, seed=seed)
    with _mk_ising(batch, L, seed, policy=sp.SPIN_POLICY_PERSISTENT) as sim:
        assert sim.spin_kernel_variant() == "ising_int8_persistent"
        l0 = sim.spin_kernel_launches()
        sim.spin_sweep(beta, 1.0, 0.02, n, 3)
        assert sim.spin_kernel_launches() - l0 == 1
        oracle_mod.sweep(ref, beta, 1.0, 0.02, seed=seed, n_sweeps=n, sweep_offset=3)
        assert np.array_equal(sim.spin_get_spins(), ref)
        sim.spin_sweep(beta, 1.0, 0.02, 2, 3 + n)
        oracle_mod.sweep(ref, beta, 1.0, 0.02, seed=seed, n_sweeps=2, sweep_offset=3 + n)
        assert np.array_equal(sim.spin_get_spins(), ref)
        E, M = sim.spin_observables()
        Eo, Mo = oracle_mod.ising_observables(ref)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
        # a never-accepted class (beta = 20) cannot use the kernel: the call streams, results unchanged
        sim.spin_sweep(np.full(batch, 20.0), 1.0, 0.0, 2, 100)
        oracle_mod.sweep(ref, np.full(batch, 20.0), 1.0, 0.0, seed=seed, n_sweeps=2, sweep_offset=100)
        assert np.array_equal(sim.spin_get_spins(), ref)


# ------------------------------------------------------------- temporally blocked tile kernel (launch-bound shapes)
@pytest.mark.parametrize("batch,L,n", [(1, 640, 13), (3, 128, 9), (2, 1024, 6), (5, 96, 7), (1, 2560, 5), (1, 16, 11),
                                       (2, 40, 6), (7, 200, 5), (150, 64, 5)])
def test_tiled_kernel_equals_oracle(oracle_mod, batch, L, n):
    """Tiles with halos advance several sweeps per launch in shared memory: sweep counts that are not multiples of the
    sweeps per launch, tile grids that do not divide the lattice, regions that wrap around small lattices, never-classes."""
    seed = 80 + L
    beta = np.linspace(0.25, 0.65, batch)
    ref = oracle_mod.init(batch, L, seed=seed)
    with _mk_ising(batch, L, seed, policy=sp.SPIN_POLICY_TILED) as sim:
        assert sim.spin_kernel_variant() == "ising_int8_tiled"
        sim.spin_sweep(beta, 1.0, 0.03, n, 2)
        oracle_mod.sweep(ref, beta, 1.0, 0.03, seed=seed, n_sweeps=n, sweep_offset=2)
        assert np.array_equal(sim.spin_get_spins(), ref)
        sim.spin_sweep(beta, 1.0, 0.03, 1, 2 + n)
        oracle_mod.sweep(ref, beta, 1.0, 0.03, seed=seed, n_sweeps=1, sweep_offset=2 + n)
        assert np.array_equal(sim.spin_get_spins(), ref)
        E, M = sim.spin_observables()
        Eo, Mo = oracle_mod.ising_observables(ref)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
        cold = np.full(batch, 20.0)
        sim.spin_sweep(cold, 1.0, 0.0, 3, (1 << 32) - 1)
        oracle_mod.sweep(ref, cold, 1.0, 0.0, seed=seed, n_sweeps=3, sweep_offset=(1 << 32) - 1)
        assert np.array_equal(sim.spin_get_spins(), ref)


@pytest.mark.parametrize("batch,L,variant", [(2, 256, "ising_int8_tiled"), (16, 128, "ising_int8_tiled"),
                                             (1, 1024, "ising_int8_tiled"), (16, 64, "ising_int8_tiled"),
                                             (17, 128, "ising_int8_resident"), (4, 32, "ising_int8_resident"),
                                             (4, 640, "ising_int8_tiled"), (2, 1056, "ising_int8_rows128"),
                                             (150, 224, "ising_int8_rows128")])
def test_auto_policy_small_launches(oracle_mod, batch, L, variant):
    """What SPIN_POLICY_AUTO picks around the tile kernel's corner (<= 16 replicas, <= 2^21 sites, L >= 64), each pick
    against the oracle; spin_sweep_measure on the same handle (never tiled) continues the same trajectory."""
    seed, n = 90 + L, 6
    beta = np.linspace(0.3, 0.6, batch)
    ref = oracle_mod.init(batch, L, seed=seed)
    with _mk_ising(batch, L, seed) as sim:
        assert sim.spin_kernel_variant() == variant
        sim.spin_sweep(beta, 1.0, 0.01, n, 0)
        oracle_mod.sweep(ref, beta, 1.0, 0.01, seed=seed, n_sweeps=n)
        assert np.array_equal(sim.spin_get_spins(), ref)
        E, M = sim.spin_sweep_measure(beta, 1.0, 0.01, 2, n)
        Eo, Mo = oracle_mod.sweep(ref, beta, 1.0, 0.01, seed=seed, n_sweeps=2, sweep_offset=n, trace=True)
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
        assert np.array_equal(sim.spin_get_spins(), ref)


def test_bits_resident_kernel_many_sweeps_in_one_launch(oracle_mod):
    """Bit-packed replica resident in one CTA: 1024^2 = 128 KiB of shared memory, all sweeps of a call in one
    launch; equals the oracle, the streaming bit-packed kernel and continues across calls and a schedule."""
    for batch, L, n in ((2, 1024, 5), (3, 256, 17), (1, 1280, 3)):
        seed, beta = 70 + L, np.linspace(0.3, 0.6, batch)
        ref = oracle_mod.init(batch, L, seed=seed)
        with _mk_ising(batch, L, seed, layout="bits", policy=sp.SPIN_POLICY_RESIDENT) as sim:
            assert sim.spin_kernel_variant() == "ising_bits_resident"
            l0 = sim.spin_kernel_launches()
            sim.spin_sweep(beta, 1.0, 0.02, n, 4)
            assert sim.spin_kernel_launches() - l0 == 1
            oracle_mod.sweep(ref, beta, 1.0, 0.02, seed=seed, n_sweeps=n, sweep_offset=4)
            assert np.array_equal(sim.spin_get_spins(), ref)
            steps = np.stack([beta * 0.5, beta * 2.0])
            sim.spin_sweep_schedule(steps, 1.0, 0.0, 2, sweep_offset=4 + n)
            oracle_mod.sweep_schedule(ref, steps, 1.0, 0.0, seed, 2, sweep_offset=4 + n)
            assert np.array_equal(sim.spin_get_spins(), ref)
            E, M = sim.spin_observables()
            Eo, Mo = oracle_mod.ising_observables(ref)
            assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
