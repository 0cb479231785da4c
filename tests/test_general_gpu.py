"""GPU bit-parity of SURVEY.md 8(f) #2 through the C ABI against oracle/general_oracle.cpp: +-J bond signs on the int8
Ising layout and on Potts, real-valued J_ij with per-site fields B_i (host-built per-site thresholds), the Potts field
term of Eq. 5, and the annealing schedule call (the Monte Carlo arm of Fig. 9)."""
import numpy as np
import pytest

import oracle
import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu


def _signs(seed, B, L):
    rng = np.random.default_rng(seed)
    return ((2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8),
            (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8))


@pytest.mark.parametrize("L", [2, 6, 10, 32, 64, 96])
def test_int8_ising_bond_signs_equal_oracle(L):
    B, seed = 3, 40 + L
    Jh, Jv = _signs(L, B, L)
    beta = [0.3, 0.7, 20.0]
    ref = oracle.init(B, L, seed=seed)
    with sp.spin_create_ex(B, L, sp.SPIN_MODEL_ISING, seed=seed) as sim:
        sim.spin_set_bonds(Jh, Jv)
        for t in range(6):
            sim.spin_sweep(beta, 0.8, 0.05, 1, t)
            oracle.sweep_bonds(ref, Jh, Jv, beta, 0.8, 0.05, seed, 1, sweep_offset=t)
            assert np.array_equal(sim.spin_get_spins(), ref), t
            E, M = sim.spin_observables()
            Eo, Mo = oracle.ising_bonds_observables(ref, Jh, Jv)
            assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
        Et, Mt = sim.spin_sweep_measure(beta, 0.8, 0.05, 3, 6)
        Eo, Mo = oracle.sweep_bonds(ref, Jh, Jv, beta, 0.8, 0.05, seed, 3, sweep_offset=6, trace=True)
        assert np.array_equal(Et, Eo) and np.array_equal(Mt, Mo)
        sim.spin_set_bonds(None, None)                                  # back to the uniform model
        sim.spin_sweep(beta, 0.8, 0.05, 2, 9)
        oracle.sweep(ref, beta, 0.8, 0.05, seed=seed, n_sweeps=2, sweep_offset=9)
        assert np.array_equal(sim.spin_get_spins(), ref)


def test_int8_and_bitpacked_bond_paths_agree():
    B, L, seed = 2, 128, 3
    Jh, Jv = _signs(1, B, L)
    out = []
    for layout in (sp.SPIN_LAYOUT_INT8, sp.SPIN_LAYOUT_BITPACKED):
        with sp.spin_create_ex(B, L, sp.SPIN_MODEL_ISING, seed=seed, layout=layout) as sim:
            sim.spin_set_bonds(Jh, Jv)
            sim.spin_sweep([0.5, 1.0], 1.0, 0.0, 10, 0)
            out.append((sim.spin_get_spins(), sim.spin_observables()))
    assert np.array_equal(out[0][0], out[1][0])
    assert np.array_equal(out[0][1][0], out[1][1][0]) and np.array_equal(out[0][1][1], out[1][1][1])


@pytest.mark.parametrize("L", [2, 4, 10, 32, 64])
def test_real_couplings_and_site_fields_equal_oracle(L):
    B, seed = 3, 70 + L
    rng = np.random.default_rng(L)
    Jh, Jv, Bf = rng.normal(size=(B, L, L)), rng.normal(size=(B, L, L)), 0.4 * rng.normal(size=(B, L, L))
    beta = np.array([0.2, 0.9, 15.0])
    ref = oracle.init(B, L, seed=seed)
    with sp.spin_create_ex(B, L, sp.SPIN_MODEL_ISING, seed=seed) as sim:
        sim.spin_set_couplings(Jh, Jv, Bf)
        for t in range(5):
            sim.spin_sweep(beta, 1.0, 0.0, 1, t)                       # J, h arguments are ignored with real couplings
            oracle.sweep_general(ref, Jh, Jv, Bf, beta, seed, 1, sweep_offset=t)
            assert np.array_equal(sim.spin_get_spins(), ref), t
        Eo, Mo = oracle.ising_general_observables(ref, Jh, Jv, Bf)
        E = sim.spin_energy_general()
        assert np.all(np.abs(E - Eo) <= 1e-12 * np.maximum(1.0, np.abs(Eo)))
        assert np.array_equal(sim.spin_observables()[1], Mo)
        beta2 = beta * 0.5                                              # a new beta rebuilds the thresholds
        sim.spin_sweep(beta2, 1.0, 0.0, 3, 5)
        oracle.sweep_general(ref, Jh, Jv, Bf, beta2, seed, 3, sweep_offset=5)
        assert np.array_equal(sim.spin_get_spins(), ref)
        sim.spin_set_couplings(None, None, None)
        sim.spin_sweep(beta, 1.0, 0.1, 2, 8)
        oracle.sweep(ref, beta, 1.0, 0.1, seed=seed, n_sweeps=2, sweep_offset=8)
        assert np.array_equal(sim.spin_get_spins(), ref)


def test_real_couplings_argument_checks():
    with sp.spin_create_ex(1, 8, sp.SPIN_MODEL_ISING, seed=1) as sim:
        z = np.zeros((1, 8, 8))
        bad = z.copy(); bad[0, 1, 1] = np.inf
        with pytest.raises(sp.SpinError):
            sim.spin_set_couplings(bad, z, z)
        with pytest.raises(sp.SpinError):
            sim.spin_energy_general()
    with sp.spin_create_ex(1, 64, sp.SPIN_MODEL_ISING, seed=1, layout=sp.SPIN_LAYOUT_BITPACKED) as sim:
        with pytest.raises(sp.SpinError) as e:
            sim.spin_set_couplings(np.zeros((1, 64, 64)), np.zeros((1, 64, 64)), np.zeros((1, 64, 64)))
        assert e.value.code == sp.SPIN_ERR_UNSUPPORTED


@pytest.mark.parametrize("L,q,h,bonds", [(2, [3, 8], 0.3, False), (6, [3, 5], -0.2, True), (32, [4, 8], 0.15, True),
                                         (64, [3, 127], 0.05, False), (32, [3, 8], 0.0, True)])
def test_potts_field_and_bond_signs_equal_oracle(L, q, h, bonds):
    B, seed = 2, 90 + L
    Jh, Jv = _signs(L + 1, B, L) if bonds else (None, None)
    beta = [0.7, 1.2]
    ref = oracle.init(B, L, seed=seed, q=q)
    with sp.spin_create_ex(B, L, sp.SPIN_MODEL_POTTS, q_per_replica=np.array(q, dtype=np.int32), seed=seed) as sim:
        if bonds:
            sim.spin_set_bonds(Jh, Jv)
        for t in range(5):
            sim.spin_sweep(beta, 1.0, h, 1, t)
            oracle.sweep_potts_general(ref, q, beta, 1.0, h, seed, 1, Jh, Jv, sweep_offset=t)
            assert np.array_equal(sim.spin_get_spins(), ref), t
            Eo, So, Mo = oracle.potts_general_observables(ref, q, Jh, Jv)
            E, M = sim.spin_observables()
            assert np.array_equal(E, Eo) and np.array_equal(M, Mo) and np.array_equal(sim.spin_potts_label_sum(), So)
        sim.spin_sweep(beta, -1.0, 0.0, 2, 5)                          # h = 0 without... (bond signs keep the general kernel)
        oracle.sweep_potts_general(ref, q, beta, -1.0, 0.0, seed, 2, Jh, Jv, sweep_offset=5)
        assert np.array_equal(sim.spin_get_spins(), ref)


@pytest.mark.parametrize("layout,L,policy", [("int8", 32, sp.SPIN_POLICY_RESIDENT), ("int8", 64, sp.SPIN_POLICY_STREAMING),
                                             ("bits", 128, sp.SPIN_POLICY_AUTO), ("int8", 10, sp.SPIN_POLICY_AUTO)])
def test_schedule_equals_step_by_step_oracle(layout, L, policy):
    B, seed, n_steps, per = 3, 15, 6, 4
    steps = np.array([[0.1 + 0.2 * k + 0.01 * b for b in range(B)] for k in range(n_steps)])
    ref = oracle.init(B, L, seed=seed)
    lay = sp.SPIN_LAYOUT_BITPACKED if layout == "bits" else sp.SPIN_LAYOUT_INT8
    with sp.spin_create_ex(B, L, sp.SPIN_MODEL_ISING, seed=seed, layout=lay) as sim:
        sim.spin_set_policy(policy)
        sim.spin_sweep_schedule(steps, 1.0, 0.02, per, sweep_offset=7)
        oracle.sweep_schedule(ref, steps, 1.0, 0.02, seed, per, sweep_offset=7)
        assert np.array_equal(sim.spin_get_spins(), ref)
        sim.spin_sweep_schedule(steps[::-1], 1.0, 0.0, 2, sweep_offset=100)     # a second schedule reuses the buffers
        oracle.sweep_schedule(ref, steps[::-1], 1.0, 0.0, seed, 2, sweep_offset=100)
        assert np.array_equal(sim.spin_get_spins(), ref)


def test_annealing_of_the_pmJ_glass_in_one_call_equals_oracle_and_lowers_the_energy():
    """Fig. 9's Monte Carlo arm: random J in {-1, +1}, temperature annealed towards zero."""
    B, L, seed, n_steps, per = 2, 64, 77, 40, 5
    Jh, Jv = _signs(9, B, L)
    steps = np.array([[0.1 + 2.9 * k / (n_steps - 1)] * B for k in range(n_steps)])
    ref = oracle.init(B, L, seed=seed)
    with sp.spin_create_ex(B, L, sp.SPIN_MODEL_ISING, seed=seed, layout=sp.SPIN_LAYOUT_BITPACKED) as sim:
        sim.spin_set_bonds(Jh, Jv)
        E0 = sim.spin_observables()[0]
        sim.spin_sweep_schedule(steps, 1.0, 0.0, per)
        oracle.sweep_schedule(ref, steps, 1.0, 0.0, seed, per, Jh=Jh, Jv=Jv)
        assert np.array_equal(sim.spin_get_spins(), ref)
        E1 = sim.spin_observables()[0]
        assert np.array_equal(E1, oracle.ising_bonds_observables(ref, Jh, Jv)[0])
        assert np.all(E1 < E0) and np.all(E1 / (L * L) < -1.3)         # the 2D +-J ground state is near -1.40 per spin


def test_schedule_argument_checks():
    with sp.spin_create_ex(2, 8, sp.SPIN_MODEL_ISING, seed=1) as sim:
        before = sim.spin_get_spins()
        with pytest.raises(sp.SpinError):
            sim.spin_sweep_schedule(np.array([[0.1, -0.2]]), 1.0, 0.0, 3)
        assert np.array_equal(sim.spin_get_spins(), before)
        sim.spin_set_couplings(np.ones((8, 8)), np.ones((8, 8)), np.zeros((8, 8)))
        with pytest.raises(sp.SpinError) as e:
            sim.spin_sweep_schedule(np.array([[0.1, 0.2]]), 1.0, 0.0, 3)
        assert e.value.code == sp.SPIN_ERR_UNSUPPORTED


def test_schedule_with_int8_bond_signs_and_for_potts():
    """The schedule call on the remaining class-table models: +-J signs on the int8 layout, and the uniform Potts model."""
    B, L, seed = 2, 32, 55
    steps = np.array([[0.2, 0.3], [0.6, 0.7], [1.5, 2.0]])
    Jh, Jv = _signs(3, B, L)
    ref = oracle.init(B, L, seed=seed)
    with sp.spin_create_ex(B, L, sp.SPIN_MODEL_ISING, seed=seed) as sim:
        sim.spin_set_bonds(Jh, Jv)
        sim.spin_sweep_schedule(steps, 1.0, 0.0, 3, sweep_offset=1)
        oracle.sweep_schedule(ref, steps, 1.0, 0.0, seed, 3, sweep_offset=1, Jh=Jh, Jv=Jv)
        assert np.array_equal(sim.spin_get_spins(), ref)
    q = [3, 8]
    ref = oracle.init(B, L, seed=seed, q=q)
    with sp.spin_create_ex(B, L, sp.SPIN_MODEL_POTTS, q_per_replica=np.array(q, dtype=np.int32), seed=seed) as sim:
        sim.spin_sweep_schedule(steps, 1.0, 0.0, 3, sweep_offset=1)
        oracle.sweep_schedule(ref, steps, 1.0, 0.0, seed, 3, sweep_offset=1, q=q)
        assert np.array_equal(sim.spin_get_spins(), ref)
        with pytest.raises(sp.SpinError) as e:                       # a Potts field needs the general kernel: per-call only
            sim.spin_sweep_schedule(steps, 1.0, 0.1, 3)
        assert e.value.code == sp.SPIN_ERR_UNSUPPORTED


@pytest.mark.parametrize("L,B,h", [(32, 3, 0.25), (96, 5, -0.2), (256, 64, 0.1)])
def test_potts_field_on_the_row_marching_kernel(L, B, h):
    """A field on the state label with uniform couplings and L % 32 == 0 runs the row-marching Potts kernel's field variant
    (threshold by class and by new - old): ragged blocks, two replica groups (64 x 256^2), q from 2 to 127, thresholds of 0
    (beta = 30) and always-accept entries, chunked calls; E, M and the label sum against the oracle."""
    seed = 300 + L
    q = np.array([2, 3, 8, 127, 5, 16, 9][:min(B, 7)] + [3 + (b % 6) for b in range(max(0, B - 7))], dtype=np.int32)
    beta = np.linspace(0.4, 1.6, B)
    beta[-1] = 30.0
    ref = oracle.init(B, L, seed=seed, q=q)
    with sp.spin_create_ex(B, L, sp.SPIN_MODEL_POTTS, q_per_replica=q, seed=seed) as sim:
        l0 = sim.spin_kernel_launches()
        sim.spin_sweep(beta, 1.0, h, 3, 0)
        assert sim.spin_kernel_launches() - l0 == 3 * 2 * (2 if B >= 60 else 1)
        oracle.sweep_potts_general(ref, q, beta, 1.0, h, seed, 3, None, None, sweep_offset=0)
        assert np.array_equal(sim.spin_get_spins(), ref)
        sim.spin_sweep(beta, -0.5, -h, 2, (1 << 32) - 1)
        oracle.sweep_potts_general(ref, q, beta, -0.5, -h, seed, 2, None, None, sweep_offset=(1 << 32) - 1)
        assert np.array_equal(sim.spin_get_spins(), ref)
        Eo, So, Mo = oracle.potts_general_observables(ref, q, None, None)
        E, M = sim.spin_observables()
        assert np.array_equal(E, Eo) and np.array_equal(M, Mo) and np.array_equal(sim.spin_potts_label_sum(), So)
        sim.spin_sweep(beta, 1.0, 0.0, 2, 9)                            # back to the plain model on the same handle
        oracle.sweep(ref, beta, 1.0, 0.0, seed=seed, n_sweeps=2, sweep_offset=9, q=q)
        assert np.array_equal(sim.spin_get_spins(), ref)
