"""A size-independent physics check of the other-geometry kernels through the public API (no oracle involved): a chain
that samples the Boltzmann distribution of the stated Hamiltonian at inverse temperature beta obeys the
fluctuation-dissipation relation  d<H>/d(beta) = -(<H^2> - <H>^2).  The left side comes from runs at beta -+ delta, the
right side from the energy fluctuations at beta; both from the exact integer observables of `spin_stencil_observables`.
A wrong class table, a wrong neighbour list or a colouring that lets neighbours update together breaks the equality."""
import numpy as np
import pytest

import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _run(stencil, B, L, beta, J1, J2, h, seed, n_therm, n_meas):
    n = sp.spin_stencil_sites(stencil, L)
    d = torch.empty(B * n, dtype=torch.int8, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    sp.spin_stencil_init(stencil, B, L, d.data_ptr(), seed, cuda_stream=st)
    b = np.full(B, beta)
    sp.spin_stencil_sweep(stencil, B, L, d.data_ptr(), b, J1, J2, h, seed, n_therm, cuda_stream=st)
    H = np.zeros((n_meas, B))
    for t in range(n_meas):
        sp.spin_stencil_sweep(stencil, B, L, d.data_ptr(), b, J1, J2, h, seed, 2, sweep_offset=n_therm + 2 * t, cuda_stream=st)
        E1, E2, M = sp.spin_stencil_observables(stencil, B, L, d.data_ptr(), cuda_stream=st)
        H[t] = J1 * E1 + J2 * E2 - h * M
    return H


@pytest.mark.parametrize("stencil,L,beta,J1,J2,h", [
    (sp.SPIN_STENCIL_TRIANGULAR, 24, 0.18, 1.0, 0.0, 0.05),     # L % 12 == 0: byte-SIMD
    (sp.SPIN_STENCIL_TRIANGULAR, 21, 0.18, 1.0, 0.0, 0.05),     # the general kernel
    (sp.SPIN_STENCIL_CUBIC, 16, 0.15, 1.0, 0.0, 0.0),           # L % 16 == 0: the byte-SIMD kernel
    (sp.SPIN_STENCIL_CUBIC, 10, 0.15, 1.0, 0.0, 0.1),           # the general kernel
    (sp.SPIN_STENCIL_SQUARE_NNN, 32, 0.22, 1.0, 0.4, 0.0),      # byte-SIMD
    (sp.SPIN_STENCIL_SQUARE_NNN, 20, 0.3, 1.0, -0.3, 0.05)])    # general, frustrating second neighbours
def test_fluctuation_dissipation(stencil, L, beta, J1, J2, h):
    B, delta, n_therm, n_meas = 256, 0.01, 300, 400
    Hm = _run(stencil, B, L, beta - delta, J1, J2, h, 11, n_therm, n_meas)
    H0 = _run(stencil, B, L, beta, J1, J2, h, 12, n_therm, n_meas)
    Hp = _run(stencil, B, L, beta + delta, J1, J2, h, 13, n_therm, n_meas)
    # per-replica time averages are independent samples: standard errors across replicas
    dU = (Hp.mean(0).mean() - Hm.mean(0).mean()) / (2 * delta)
    dU_se = np.sqrt(Hp.mean(0).var(ddof=1) / B + Hm.mean(0).var(ddof=1) / B) / (2 * delta)
    # variance of H in the ensemble: pooled over replicas and measurement times (replicas are exchangeable)
    var_rep = np.array([np.mean((H0[:, b] - H0.mean()) ** 2) for b in range(B)])
    varH, varH_se = var_rep.mean(), var_rep.std(ddof=1) / np.sqrt(B)
    # central difference is exact up to O(delta^2 d^3U/dbeta^3): allow 2 % on top of 4 standard errors
    assert abs(dU + varH) <= 4 * np.hypot(dU_se, varH_se) + 0.02 * abs(varH), (dU, varH, dU_se, varH_se)


def _fdt(run, beta, delta, B):
    Hm, H0, Hp = run(beta - delta, 21), run(beta, 22), run(beta + delta, 23)
    dU = (Hp.mean(0).mean() - Hm.mean(0).mean()) / (2 * delta)
    dU_se = np.sqrt(Hp.mean(0).var(ddof=1) / B + Hm.mean(0).var(ddof=1) / B) / (2 * delta)
    var_rep = np.array([np.mean((H0[:, b] - H0.mean()) ** 2) for b in range(B)])
    varH, varH_se = var_rep.mean(), var_rep.std(ddof=1) / np.sqrt(B)
    assert abs(dU + varH) <= 4 * np.hypot(dU_se, varH_se) + 0.02 * abs(varH), (dU, varH, dU_se, varH_se)


def test_fluctuation_dissipation_real_couplings_and_site_fields():
    """H = -sum J_ij s s - sum B_i s with one random real sample shared by all replicas."""
    B, L, n_therm, n_meas = 256, 16, 300, 400
    rng = np.random.default_rng(5)
    Jh, Jv, Bf = rng.normal(size=(L, L)), rng.normal(size=(L, L)), 0.3 * rng.normal(size=(L, L))

    def run(beta, seed):
        with sp.spin_create_ex(B, L, sp.SPIN_MODEL_ISING, seed=seed) as sim:
            sim.spin_set_couplings(Jh, Jv, Bf)
            b = np.full(B, beta)
            sim.spin_sweep(b, 1.0, 0.0, n_therm, 0)
            H = np.zeros((n_meas, B))
            for t in range(n_meas):
                sim.spin_sweep(b, 1.0, 0.0, 2, n_therm + 2 * t)
                H[t] = sim.spin_energy_general()
            return H
    _fdt(run, 0.35, 0.01, B)


def test_fluctuation_dissipation_potts_with_field():
    """Eq. 5 with its field term on the state label: H = J E_int - h S."""
    B, L, q, J, h, n_therm, n_meas = 256, 16, 4, 1.0, 0.2, 300, 400

    def run(beta, seed):
        with sp.spin_create_ex(B, L, sp.SPIN_MODEL_POTTS, q_uniform=q, seed=seed) as sim:
            b = np.full(B, beta)
            sim.spin_sweep(b, J, h, n_therm, 0)
            H = np.zeros((n_meas, B))
            for t in range(n_meas):
                sim.spin_sweep(b, J, h, 2, n_therm + 2 * t)
                H[t] = J * sim.spin_observables()[0] - h * sim.spin_potts_label_sum()
            return H
    _fdt(run, 0.6, 0.01, B)
