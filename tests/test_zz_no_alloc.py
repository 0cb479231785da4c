"""spin_stencil_observables_noalloc (include/spin.h): the reductions of spin_stencil_observables with the accumulators in a
fixed device array inside the library instead of a per-call allocation.  Checked against the existing entry point as exact
integers (the bar of every reduction test here), on two calls in a row: the second call has a smaller batch and other
lattices, so sums left in the shared array by the first call would show.  Collected last on purpose (file name)."""
import numpy as np
import pytest

import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

NO_ALLOC_MAX_BATCH = 4096


def _both(stencil, batch, L, lattice, stream):
    out = torch.full((3, batch), -7, dtype=torch.int64, device="cuda")       # poisoned: every entry must be written
    with torch.cuda.stream(stream):
        sp.spin_stencil_observables_noalloc(stencil, batch, L, lattice.data_ptr(), out[0].data_ptr(), out[1].data_ptr(),
                                            out[2].data_ptr(), cuda_stream=stream.cuda_stream)
    stream.synchronize()
    want = sp.spin_stencil_observables(stencil, batch, L, lattice.data_ptr(), cuda_stream=stream.cuda_stream)
    return out.cpu().numpy(), want


@pytest.mark.parametrize("stencil,L", [(sp.SPIN_STENCIL_TRIANGULAR, 36), (sp.SPIN_STENCIL_CUBIC, 16),
                                       (sp.SPIN_STENCIL_SQUARE_NNN, 50)])
def test_two_calls_in_a_row_equal_the_allocating_path(stencil, L):
    stream = torch.cuda.Stream()
    n = sp.spin_stencil_sites(stencil, L)
    for batch, seed in ((37, 11), (5, 12)):
        lat = torch.empty(batch * n, dtype=torch.int8, device="cuda")
        sp.spin_stencil_init(stencil, batch, L, lat.data_ptr(), seed, cuda_stream=stream.cuda_stream)
        beta = np.linspace(0.1, 0.6, batch)
        sp.spin_stencil_sweep(stencil, batch, L, lat.data_ptr(), beta, 1.0, 0.3, 0.05, seed, 2, cuda_stream=stream.cuda_stream)
        got, (E1, E2, M) = _both(stencil, batch, L, lat, stream)
        assert np.array_equal(got[0], E1) and np.array_equal(got[1], E2) and np.array_equal(got[2], M), (batch, seed)
        assert np.any(E1 != 0) and np.any(M != 0)
    # NULL outputs are skipped, the others still written
    only_m = torch.full((batch,), -7, dtype=torch.int64, device="cuda")
    sp.spin_stencil_observables_noalloc(stencil, batch, L, lat.data_ptr(), None, None, only_m.data_ptr(),
                                        cuda_stream=stream.cuda_stream)
    stream.synchronize()
    assert np.array_equal(only_m.cpu().numpy(), M)


def test_maximum_batch_and_rejection_beyond_it():
    stencil, L = sp.SPIN_STENCIL_SQUARE_NNN, 4
    stream = torch.cuda.Stream()
    n = sp.spin_stencil_sites(stencil, L)
    batch = NO_ALLOC_MAX_BATCH
    lat = torch.empty((batch + 1) * n, dtype=torch.int8, device="cuda")
    sp.spin_stencil_init(stencil, batch + 1, L, lat.data_ptr(), 3, cuda_stream=stream.cuda_stream)
    got, (E1, E2, M) = _both(stencil, batch, L, lat, stream)
    assert np.array_equal(got[0], E1) and np.array_equal(got[1], E2) and np.array_equal(got[2], M)
    out = torch.full((3, batch + 1), -7, dtype=torch.int64, device="cuda")
    with pytest.raises(sp.SpinError) as err:
        sp.spin_stencil_observables_noalloc(stencil, batch + 1, L, lat.data_ptr(), out[0].data_ptr(), out[1].data_ptr(),
                                            out[2].data_ptr(), cuda_stream=stream.cuda_stream)
    assert "4096" in str(err.value)
    torch.cuda.synchronize()
    assert torch.all(out == -7).item()                                          # a rejected call touches nothing


def test_no_allocation_during_the_call():
    """The driver's free-memory figure does not move across calls (the allocating path draws from the stream-ordered pool)."""
    stencil, L, batch = sp.SPIN_STENCIL_CUBIC, 16, 64
    stream = torch.cuda.Stream()
    lat = torch.empty(batch * sp.spin_stencil_sites(stencil, L), dtype=torch.int8, device="cuda")
    out = torch.zeros((3, batch), dtype=torch.int64, device="cuda")
    sp.spin_stencil_init(stencil, batch, L, lat.data_ptr(), 9, cuda_stream=stream.cuda_stream)
    args = (stencil, batch, L, lat.data_ptr(), out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr())
    sp.spin_stencil_observables_noalloc(*args, cuda_stream=stream.cuda_stream)    # first call: symbol address looked up
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(20):
        sp.spin_stencil_observables_noalloc(*args, cuda_stream=stream.cuda_stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
