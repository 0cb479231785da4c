"""GPU bit-parity of the Cellular Potts kernels (csrc/cpm.cu through the C ABI) against oracle/cpm_oracle.cpp: the lattice
after every sweep, adhesion / area energies, areas and boundary lengths as exact integers, on the paper's set-up (Table
II, 37 identifiers, k_B T = 8, A = 25, lambda = 1) and on random lattices with ragged Philox groups."""
import numpy as np
import pytest

import oracle
import paper_2304_01772_b200 as sp
from paper_2304_01772_b200 import workloads

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
JT = workloads.CPM_TABLE_II


def _check_obs(d, ref, B, L, tau, A, lam, st):
    Ha, Hr, ar, bl = sp.spin_cpm_observables(B, L, d.data_ptr(), tau, JT, lam, A, cuda_stream=st)
    oa, orr, oar, obl = oracle.cpm_observables(ref, tau, JT, lam, A)
    assert np.array_equal(Ha, oa) and np.array_equal(Hr, orr) and np.array_equal(ar, oar) and np.array_equal(bl, obl)


@pytest.mark.parametrize("L,cells,size", [(40, 6, 5), (64, 6, 5), (16, 3, 4)])
def test_paper_setup_equals_oracle(L, cells, size):
    B, seed, lam = 3, 12, 1
    spins, tau, A = workloads.cpm_initial(B, L, cells, size, seed=3)
    beta = np.array([1.0 / 8.0, 0.05, 1.0])
    ref = spins.copy()
    d = torch.from_numpy(spins.copy()).cuda()
    st = torch.cuda.current_stream().cuda_stream
    _check_obs(d, ref, B, L, tau, A, lam, st)
    for t in range(6):
        sp.spin_cpm_sweep(B, L, d.data_ptr(), tau, JT, lam, A, beta, seed, 1, sweep_offset=t, replica_offset=2, cuda_stream=st)
        oracle.cpm_sweep(ref, tau, JT, lam, A, beta, seed, 1, sweep_offset=t, replica_offset=2)
        assert np.array_equal(d.cpu().numpy(), ref), t
        _check_obs(d, ref, B, L, tau, A, lam, st)
    sp.spin_cpm_sweep(B, L, d.data_ptr(), tau, JT, lam, A, beta, seed, 20, sweep_offset=6, replica_offset=2, cuda_stream=st)
    oracle.cpm_sweep(ref, tau, JT, lam, A, beta, seed, 20, sweep_offset=6, replica_offset=2)
    assert np.array_equal(d.cpu().numpy(), ref)


@pytest.mark.parametrize("L,q,lam", [(2, 3, 1), (6, 5, 0), (10, 9, 3), (34, 127, 1)])
def test_random_lattices_equal_oracle(L, q, lam):
    B, seed = 2, 40 + L
    rng = np.random.default_rng(L)
    spins = rng.integers(0, q, size=(B, L, L)).astype(np.int8)
    tau = np.concatenate([[0], rng.integers(1, 3, size=q - 1)]).astype(np.int32)
    A = np.concatenate([[0], rng.integers(1, 12, size=q - 1)]).astype(np.int32)
    beta = np.array([0.0, 0.2])
    ref = spins.copy()
    d = torch.from_numpy(spins.copy()).cuda()
    st = torch.cuda.current_stream().cuda_stream
    for t in range(5):
        sp.spin_cpm_sweep(B, L, d.data_ptr(), tau, JT, lam, A, beta, seed, 1, sweep_offset=(1 << 32) + t, cuda_stream=st)
        oracle.cpm_sweep(ref, tau, JT, lam, A, beta, seed, 1, sweep_offset=(1 << 32) + t)
        assert np.array_equal(d.cpu().numpy(), ref), t
    _check_obs(d, ref, B, L, tau, A, lam, st)


@pytest.mark.parametrize("L,cells,size,B", [(192, 8, 6, 3), (260, 11, 8, 2)])
def test_large_lattices_take_the_three_launch_path(L, cells, size, B):
    """Lattices beyond one CTA's shared memory, or few large replicas (L > 128 with fewer than 148 replicas), run
    cpm_area_kernel + cpm_pass_kernel per colour pass instead of the resident kernel: same oracle, same bar."""
    seed, lam = 21, 2
    spins, tau, A = workloads.cpm_initial(B, L, cells, size, seed=4)
    beta = np.linspace(0.05, 0.5, B)
    ref = spins.copy()
    d = torch.from_numpy(spins.copy()).cuda()
    st = torch.cuda.current_stream().cuda_stream
    for t0, n in ((0, 1), (1, 1), (2, 3)):
        sp.spin_cpm_sweep(B, L, d.data_ptr(), tau, JT, lam, A, beta, seed, n, sweep_offset=t0, replica_offset=1, cuda_stream=st)
        oracle.cpm_sweep(ref, tau, JT, lam, A, beta, seed, n, sweep_offset=t0, replica_offset=1)
        assert np.array_equal(d.cpu().numpy(), ref), t0
    _check_obs(d, ref, B, L, tau, A, lam, st)


def test_argument_checks():
    spins, tau, A = workloads.cpm_initial(1, 16, 3, 4, seed=1)
    d = torch.from_numpy(spins.copy()).cuda()
    bad_J = JT.copy(); bad_J[0, 1] = 5
    for kw in (dict(L=15), dict(Jtab=bad_J), dict(beta=[1e-6]), dict(lam=-1)):
        a = dict(L=16, Jtab=JT, beta=[0.125], lam=1); a.update(kw)
        with pytest.raises(sp.SpinError):
            sp.spin_cpm_sweep(1, a["L"], d.data_ptr(), tau, a["Jtab"], a["lam"], A, a["beta"], 1, 1)
    assert np.array_equal(d.cpu().numpy(), spins)


def test_cell_sorting_as_in_the_papers_figure_6():
    """PAPER.md:288-294 (Fig. 5, 6): from the aggregate of square cells 'the interface between the blue cells and the medium
    vanish[es], while the boundary length between red cells with medium and red cells with blue cells approaches a minimum':
    with Table II one cell type ends up inside, wrapped by the other.  64 replicas, 2000 sweeps, through the public API."""
    B, L = 64, 64
    spins, tau, A = workloads.cpm_initial(B, L, 6, 5, seed=5)
    d = torch.from_numpy(spins.copy()).cuda()
    st = torch.cuda.current_stream().cuda_stream
    Ha0, _, ar0, bl0 = sp.spin_cpm_observables(B, L, d.data_ptr(), tau, JT, 1, A, cuda_stream=st)
    sp.spin_cpm_sweep(B, L, d.data_ptr(), tau, JT, 1, A, np.full(B, 1.0 / 8.0), 5, 2000, cuda_stream=st)
    Ha, Hr, ar, bl = sp.spin_cpm_observables(B, L, d.data_ptr(), tau, JT, 1, A, cuda_stream=st)
    ml0, ml = bl0[:, 0, 1].mean(), bl[:, 0, 1].mean()          # medium-light boundary
    assert ml < 0.4 * ml0, (ml0, ml)                           # 164 -> ~34: the light cells leave the surface
    assert bl[:, 0, 2].mean() > bl0[:, 0, 2].mean()            # the dark cells take it over
    assert bl[:, 1, 2].mean() < 0.7 * bl0[:, 1, 2].mean()      # light-dark contacts fall to a minimum (476 -> ~237)
    assert Ha.mean() < Ha0.mean()                              # adhesion energy decreases
    assert np.all((ar[:, 1:] > 0).sum(1) == 36)                # no cell disappears at lambda = 1, A = 25
    assert np.all(np.abs(ar[:, 1:] - 25).mean(1) < 6)          # areas stay near the target
