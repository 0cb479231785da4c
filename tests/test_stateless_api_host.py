"""Host logic of the stateless C-ABI calls (DMC, other geometries, cellular Potts): argument validation happens before any
CUDA call, so it is testable without a GPU (`-m "not gpu"`); a rejected call reports SPIN_ERR_INVALID with a reason."""
import ctypes

import numpy as np
import pytest

import paper_2304_01772_b200 as sp

DUMMY = 0x1000     # never dereferenced: every call below is rejected during validation


def _code(fn, *a, **kw):
    with pytest.raises(sp.SpinError) as e:
        fn(*a, **kw)
    assert sp.spin_last_error() != ""
    return e.value.code


def test_stencil_shapes():
    T, C, N = sp.SPIN_STENCIL_TRIANGULAR, sp.SPIN_STENCIL_CUBIC, sp.SPIN_STENCIL_SQUARE_NNN
    assert sp.spin_stencil_sites(T, 6) == 36 and sp.spin_stencil_sites(C, 4) == 64 and sp.spin_stencil_sites(N, 8) == 64
    for stencil, L in ((T, 4), (T, 0), (C, 3), (C, 1), (N, 7), (9, 4), (-1, 4)):
        assert sp.spin_stencil_sites(stencil, L) == 0
    assert _code(sp.spin_stencil_sweep, C, 1, 5, DUMMY, [0.3], 1.0, 0.0, 0.0, 1, 1) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_stencil_sweep, C, 1, 4, DUMMY, [-0.3], 1.0, 0.0, 0.0, 1, 1) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_stencil_sweep, C, 1, 4, DUMMY, [0.3], float("inf"), 0.0, 0.0, 1, 1) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_stencil_sweep, C, 1, 4, DUMMY, [0.3], 1.0, 0.0, 0.0, 1, -2) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_stencil_sweep, C, 1, 4, None, [0.3], 1.0, 0.0, 0.0, 1, 1) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_stencil_init, T, 0, 6, DUMMY, 1) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_stencil_sweep, T, 1, 6, DUMMY, [0.3], 1.0, 0.0, 0.0, 1, 1, replica_offset=1 << 32) == sp.SPIN_ERR_INVALID


def test_dmc_arguments():
    F32 = sp.SPIN_DTYPE_F32
    ok = dict(s_out_ptr=DUMMY)
    assert _code(sp.spin_dmc_forward, 1, 3, F32, DUMMY, DUMMY, DUMMY, 0.0, [0.5], 1.0, 1, 1, **ok) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_dmc_forward, 0, 4, F32, DUMMY, DUMMY, DUMMY, 0.0, [], 1.0, 1, 1, **ok) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_dmc_forward, 1, 4, 5, DUMMY, DUMMY, DUMMY, 0.0, [0.5], 1.0, 1, 1, **ok) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_dmc_forward, 1, 4, F32, DUMMY, DUMMY, DUMMY, 0.0, [float("nan")], 1.0, 1, 1, **ok) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_dmc_forward, 1, 4, F32, DUMMY, DUMMY, DUMMY, 0.0, [0.5], -1.0, 1, 1, **ok) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_dmc_forward, 1, 4, F32, DUMMY, DUMMY, DUMMY, 0.0, [0.5], 1.0, 1, 1 << 57, **ok) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_dmc_forward, 1, 4, F32, None, DUMMY, DUMMY, 0.0, [0.5], 1.0, 1, 1, **ok) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_dmc_backward, 1, 4, F32, DUMMY, DUMMY, DUMMY, 0.0, [0.5], 1.0, 1, 1, None, DUMMY, DUMMY, DUMMY) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_dmc_discretise, 9, DUMMY, 4) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_dmc_discretise, F32, None, 4) == sp.SPIN_ERR_INVALID


def test_cpm_arguments():
    tau, A = np.array([0, 1, 2], dtype=np.int32), np.array([0, 5, 5], dtype=np.int32)
    J = sp.workloads.CPM_TABLE_II
    assert _code(sp.spin_cpm_sweep, 1, 7, DUMMY, tau, J, 1, A, [0.125], 1, 1) == sp.SPIN_ERR_INVALID            # odd L
    bad = J.copy(); bad[1, 2] += 1
    assert _code(sp.spin_cpm_sweep, 1, 8, DUMMY, tau, bad, 1, A, [0.125], 1, 1) == sp.SPIN_ERR_INVALID          # asymmetric J
    assert _code(sp.spin_cpm_sweep, 1, 8, DUMMY, np.array([0, 1, 3], dtype=np.int32), J, 1, A, [0.125], 1, 1) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_cpm_sweep, 1, 8, DUMMY, tau, J, -1, A, [0.125], 1, 1) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_cpm_sweep, 1, 8, DUMMY, tau, J, 1, A, [-1.0], 1, 1) == sp.SPIN_ERR_INVALID
    assert _code(sp.spin_cpm_sweep, 1, 8, DUMMY, tau, J, 1, A, [1e-7], 1, 1) == sp.SPIN_ERR_UNSUPPORTED         # table would exceed 65536 entries
    assert _code(sp.spin_cpm_sweep, 1, 8, None, tau, J, 1, A, [0.125], 1, 1) == sp.SPIN_ERR_INVALID


def test_measurement_aid_rejects_null():
    assert sp.load_library().spin_measure_philox_compare_rate(None) == sp.SPIN_ERR_INVALID
