"""GPU bit-parity of the other lattice geometries (csrc/stencil.cu through the C ABI) against oracle/stencil_oracle.cpp:
initial lattice, the lattice after every sweep, E1 / E2 / M as exact integers; ragged Philox groups, tiny lattices with
neighbour multiplicity, beta = 0 and beta = 20, t >= 2^32, replica offsets, chunking."""
import numpy as np
import pytest

import oracle
import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

# cubic and second-neighbour lattices with L % 16 == 0 and triangular ones with L % 12 == 0 run the byte-SIMD kernels,
# every other shape the general one
CASES = ([(sp.SPIN_STENCIL_TRIANGULAR, L) for L in (3, 6, 9, 12, 30, 36, 96)]
         + [(sp.SPIN_STENCIL_CUBIC, L) for L in (2, 4, 6, 10, 16, 32, 48)]
         + [(sp.SPIN_STENCIL_SQUARE_NNN, L) for L in (2, 4, 6, 10, 16, 48, 64, 100)])


@pytest.mark.parametrize("stencil,L", CASES)
def test_sweeps_equal_oracle(stencil, L):
    B, seed, roff, t0 = 3, 1000 + L, 6, (1 << 32) - 2
    beta = np.array([0.0, 0.25, 20.0])
    J1, J2, h = 1.0, -0.35, 0.05
    n = sp.spin_stencil_sites(stencil, L)
    assert n == oracle.stencil_init(stencil, 1, L, seed=0)[0].size
    d = torch.empty(B * n, dtype=torch.int8, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    sp.spin_stencil_init(stencil, B, L, d.data_ptr(), seed, replica_offset=roff, cuda_stream=st)
    ref = oracle.stencil_init(stencil, B, L, seed=seed, replica_offset=roff)
    assert np.array_equal(d.cpu().numpy().reshape(ref.shape), ref)
    for k in range(5):
        sp.spin_stencil_sweep(stencil, B, L, d.data_ptr(), beta, J1, J2, h, seed, 1, sweep_offset=t0 + k, replica_offset=roff,
                              cuda_stream=st)
        oracle.stencil_sweep(stencil, ref, beta, J1, J2, h, seed, 1, sweep_offset=t0 + k, replica_offset=roff)
        assert np.array_equal(d.cpu().numpy().reshape(ref.shape), ref), k
        E1, E2, M = sp.spin_stencil_observables(stencil, B, L, d.data_ptr(), cuda_stream=st)
        o1, o2, om = oracle.stencil_observables(stencil, ref)
        assert np.array_equal(E1, o1) and np.array_equal(E2, o2) and np.array_equal(M, om)
    # one call of 4 sweeps = 4 calls of one
    sp.spin_stencil_sweep(stencil, B, L, d.data_ptr(), beta, J1, J2, h, seed, 4, sweep_offset=t0 + 5, replica_offset=roff, cuda_stream=st)
    oracle.stencil_sweep(stencil, ref, beta, J1, J2, h, seed, 4, sweep_offset=t0 + 5, replica_offset=roff)
    assert np.array_equal(d.cpu().numpy().reshape(ref.shape), ref)


def test_invalid_shapes_and_arguments():
    assert sp.spin_stencil_sites(sp.SPIN_STENCIL_TRIANGULAR, 4) == 0 and sp.spin_stencil_sites(sp.SPIN_STENCIL_CUBIC, 3) == 0
    assert sp.spin_stencil_sites(7, 4) == 0 and sp.spin_stencil_sites(sp.SPIN_STENCIL_SQUARE_NNN, 6) == 36
    d = torch.ones(64, dtype=torch.int8, device="cuda")
    for kw in (dict(L=5), dict(beta=[-0.1]), dict(J1=float("nan")), dict(n_sweeps=-1)):
        a = dict(L=4, beta=[0.3], J1=1.0, n_sweeps=1); a.update(kw)
        with pytest.raises(sp.SpinError):
            sp.spin_stencil_sweep(sp.SPIN_STENCIL_CUBIC, 1, a["L"], d.data_ptr(), a["beta"], a["J1"], 0.0, 0.0, 1, a["n_sweeps"])
    assert torch.all(d == 1).item()


@pytest.mark.parametrize("L,B", [(24, 5), (96, 2400)])
def test_triangular_row_marching_kernel(L, B):
    """The triangular byte-SIMD kernel marches 6 rows per thread, 12 when the launch is large (2400 x 96^2): every replica
    against the oracle after each of 2 sweeps and after a 3-sweep call, ragged blocks that straddle replicas (5 x 24^2)."""
    st = sp.SPIN_STENCIL_TRIANGULAR
    seed = 40 + L
    beta = np.linspace(0.05, 0.6, B)
    beta[-1] = 20.0
    n = sp.spin_stencil_sites(st, L)
    d = torch.empty(B * n, dtype=torch.int8, device="cuda")
    cs = torch.cuda.current_stream().cuda_stream
    sp.spin_stencil_init(st, B, L, d.data_ptr(), seed, cuda_stream=cs)
    ref = oracle.stencil_init(st, B, L, seed=seed)
    t = 0
    for k in (1, 1, 3):
        sp.spin_stencil_sweep(st, B, L, d.data_ptr(), beta, 1.0, 0.0, 0.07, seed, k, sweep_offset=t, cuda_stream=cs)
        oracle.stencil_sweep(st, ref, beta, 1.0, 0.0, 0.07, seed, k, sweep_offset=t)
        assert np.array_equal(d.cpu().numpy().reshape(ref.shape), ref), t
        t += k
    E1, E2, M = sp.spin_stencil_observables(st, B, L, d.data_ptr(), cuda_stream=cs)
    o1, o2, om = oracle.stencil_observables(st, ref)
    assert np.array_equal(E1, o1) and np.array_equal(M, om)
