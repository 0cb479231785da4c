"""ctypes binding of include/spin.h.  Same names, argument marshalling only: every step of the path runs in
the CUDA kernels of libspin.so.  There is no fallback: if the library is missing it is built with nvcc, and if
that fails, or no CUDA device is present at spin_create time, an exception is raised."""
import ctypes
import os

import numpy as np

from . import build as _build

SPIN_OK, SPIN_ERR_INVALID, SPIN_ERR_NOMEM, SPIN_ERR_CUDA, SPIN_ERR_UNSUPPORTED = 0, -1, -2, -3, -4
SPIN_MODEL_ISING, SPIN_MODEL_POTTS = 0, 1
SPIN_LAYOUT_INT8, SPIN_LAYOUT_BITPACKED = 0, 1
SPIN_POLICY_AUTO, SPIN_POLICY_STREAMING, SPIN_POLICY_RESIDENT, SPIN_POLICY_PERSISTENT, SPIN_POLICY_TILED = 0, 1, 2, 3, 4
SPIN_POLICY_GRAPH = 5
SPIN_DTYPE_F32, SPIN_DTYPE_F64 = 0, 1
SPIN_STENCIL_TRIANGULAR, SPIN_STENCIL_CUBIC, SPIN_STENCIL_SQUARE_NNN = 0, 1, 2

__all__ = [
    "SPIN_OK", "SPIN_ERR_INVALID", "SPIN_ERR_NOMEM", "SPIN_ERR_CUDA", "SPIN_ERR_UNSUPPORTED",
    "SPIN_MODEL_ISING", "SPIN_MODEL_POTTS", "SPIN_LAYOUT_INT8", "SPIN_LAYOUT_BITPACKED",
    "SPIN_POLICY_AUTO", "SPIN_POLICY_STREAMING", "SPIN_POLICY_RESIDENT", "SPIN_POLICY_PERSISTENT", "SPIN_POLICY_TILED", "SPIN_POLICY_GRAPH",
    "SpinError", "load_library", "spin_last_error", "spin_buffer_bytes", "spin_threshold_table", "SpinSim", "spin_measure_philox_compare_rate",
    "SPIN_DTYPE_F32", "SPIN_DTYPE_F64", "SPIN_STENCIL_TRIANGULAR", "SPIN_STENCIL_CUBIC", "SPIN_STENCIL_SQUARE_NNN",
    "spin_stencil_sites", "spin_stencil_init", "spin_stencil_sweep", "spin_stencil_observables",
    "spin_stencil_observables_noalloc",
    "spin_cpm_sweep", "spin_cpm_observables", "spin_dmc_forward", "spin_dmc_backward", "spin_dmc_discretise",
    "spin_create", "spin_create_ex",
]

_lib = None


class SpinError(RuntimeError):
    def __init__(self, code, message):
        super().__init__("libspin error %d: %s" % (code, message))
        self.code = code


def load_library():
    """Load (building if needed) libspin.so and declare the prototypes of include/spin.h."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    if not os.path.exists(path):
        raise RuntimeError("libspin.so is missing and could not be built; there is no fallback path")
    lib = ctypes.CDLL(path)
    c = ctypes
    vp, i32, i64, u64, dbl, sz = c.c_void_p, c.c_int32, c.c_int64, c.c_uint64, c.c_double, c.c_size_t
    protos = {
        "spin_create": (vp, [i32, i32, i32, u64]),
        "spin_sweep": (c.c_int, [vp, vp, dbl, dbl, i64, i64]),
        "spin_observables": (c.c_int, [vp, vp, vp]),
        "spin_destroy": (None, [vp]),
        "spin_last_error": (c.c_char_p, []),
        "spin_buffer_bytes": (sz, [i32, i32, i32, i32]),
        "spin_create_ex": (vp, [i32, i32, i32, vp, i32, u64, i32, i64, vp, sz, vp]),
        "spin_set_stream": (c.c_int, [vp, vp]),
        "spin_get_spins": (c.c_int, [vp, vp]),
        "spin_set_spins": (c.c_int, [vp, vp]),
        "spin_sweep_measure": (c.c_int, [vp, vp, dbl, dbl, i64, i64, vp, vp, vp]),
        "spin_observables_dev": (c.c_int, [vp, vp, vp]),
        "spin_synchronize": (c.c_int, [vp]),
        "spin_threshold_table": (c.c_int, [i32, dbl, dbl, dbl, vp, vp]),
        "spin_kernel_launches": (i64, [vp]),
        "spin_kernel_variant": (c.c_char_p, [vp]),
        "spin_set_policy": (c.c_int, [vp, i32]),
        "spin_set_bonds": (c.c_int, [vp, vp, vp]),
        "spin_measure_philox_compare_rate": (c.c_int, [vp]),
        "spin_set_couplings": (c.c_int, [vp, vp, vp, vp]),
        "spin_energy_general": (c.c_int, [vp, vp]),
        "spin_potts_label_sum": (c.c_int, [vp, vp]),
        "spin_sweep_schedule": (c.c_int, [vp, vp, i64, dbl, dbl, i64, i64]),
        "spin_stencil_sites": (sz, [i32, i32]),
        "spin_stencil_init": (c.c_int, [i32, i32, i32, vp, u64, i64, vp]),
        "spin_stencil_sweep": (c.c_int, [i32, i32, i32, vp, vp, dbl, dbl, dbl, u64, i64, i64, i64, vp]),
        "spin_stencil_observables": (c.c_int, [i32, i32, i32, vp, vp, vp, vp, vp]),
        "spin_stencil_observables_noalloc": (c.c_int, [i32, i32, i32, vp, vp, vp, vp, vp]),
        "spin_cpm_sweep": (c.c_int, [i32, i32, i32, vp, vp, vp, i32, i64, vp, vp, u64, i64, i64, i64, vp]),
        "spin_cpm_observables": (c.c_int, [i32, i32, i32, vp, vp, vp, i32, i64, vp, vp, vp, vp, vp, vp]),
        "spin_dmc_forward": (c.c_int, [i32, i32, i32, vp, vp, vp, dbl, vp, dbl, u64, i64, i64, i64, vp, vp, vp]),
        "spin_dmc_backward": (c.c_int, [i32, i32, i32, vp, vp, vp, dbl, vp, dbl, u64, i64, i64, i64, vp, vp, vp, vp, vp, vp, vp]),
        "spin_dmc_discretise": (c.c_int, [i32, vp, i64, vp]),
    }
    for name, (res, args) in protos.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


EXPORTED_SYMBOLS = (
    "spin_create", "spin_sweep", "spin_observables", "spin_destroy", "spin_last_error", "spin_buffer_bytes",
    "spin_create_ex", "spin_set_stream", "spin_get_spins", "spin_set_spins", "spin_sweep_measure",
    "spin_observables_dev", "spin_synchronize", "spin_threshold_table", "spin_kernel_launches",
    "spin_kernel_variant", "spin_set_policy", "spin_set_bonds", "spin_measure_philox_compare_rate",
    "spin_dmc_forward", "spin_dmc_backward", "spin_dmc_discretise",
    "spin_set_couplings", "spin_energy_general", "spin_potts_label_sum", "spin_sweep_schedule",
    "spin_stencil_sites", "spin_stencil_init", "spin_stencil_sweep", "spin_stencil_observables",
    "spin_stencil_observables_noalloc",
    "spin_cpm_sweep", "spin_cpm_observables",
)


def spin_last_error():
    return load_library().spin_last_error().decode()


def _check(rc):
    if rc != SPIN_OK:
        raise SpinError(rc, spin_last_error())


def _np_ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def spin_buffer_bytes(batch, L, model, layout):
    return int(load_library().spin_buffer_bytes(batch, L, model, layout))


def spin_threshold_table(model, beta, J, h=0.0):
    """-> (T uint32[n], always bool[n]); n = 10 (Ising) or 9 (Potts).  Host only, needs no GPU."""
    T = np.zeros(10, dtype=np.uint32)
    a = np.zeros(10, dtype=np.uint8)
    n = load_library().spin_threshold_table(model, float(beta), float(J), float(h), _np_ptr(T), _np_ptr(a))
    if n < 0:
        raise SpinError(n, spin_last_error())
    return T[:n].copy(), a[:n].astype(bool)


def spin_measure_philox_compare_rate():
    """Stand-alone Philox-4x32-10 + compare rate of the current device, random words per ns (measurement aid)."""
    v = ctypes.c_double(0.0)
    _check(load_library().spin_measure_philox_compare_rate(ctypes.byref(v)))
    return float(v.value)


def _beta64(beta, batch):
    return np.ascontiguousarray(np.broadcast_to(np.asarray(beta, dtype=np.float64), (batch,)))


def spin_dmc_forward(batch, L, dtype, s0_ptr, Jh_ptr, Jv_ptr, h, beta, alpha, seed, n_sweeps, sweep_offset=0,
                     replica_offset=0, s_out_ptr=None, traj_ptr=None, cuda_stream=None):
    """Device pointers (ints) in, device results out; see include/spin.h."""
    b = _beta64(beta, batch)
    _check(load_library().spin_dmc_forward(batch, L, dtype, s0_ptr, Jh_ptr, Jv_ptr, float(h), _np_ptr(b), float(alpha),
                                           int(seed), int(replica_offset), int(n_sweeps), int(sweep_offset), s_out_ptr,
                                           traj_ptr, cuda_stream))


def spin_dmc_backward(batch, L, dtype, traj_ptr, Jh_ptr, Jv_ptr, h, beta, alpha, seed, n_sweeps, grad_out_ptr, grad_s0_ptr,
                      grad_Jh_ptr, grad_Jv_ptr, sweep_offset=0, replica_offset=0, cuda_stream=None, want_host=True):
    """-> (grad_beta, grad_h) float64[batch] on the host (None, None if not want_host: fully asynchronous)."""
    b = _beta64(beta, batch)
    gb = np.zeros(batch) if want_host else None
    gh = np.zeros(batch) if want_host else None
    _check(load_library().spin_dmc_backward(batch, L, dtype, traj_ptr, Jh_ptr, Jv_ptr, float(h), _np_ptr(b), float(alpha),
                                            int(seed), int(replica_offset), int(n_sweeps), int(sweep_offset), grad_out_ptr,
                                            grad_s0_ptr, grad_Jh_ptr, grad_Jv_ptr, _np_ptr(gb), _np_ptr(gh), cuda_stream))
    return gb, gh


def spin_stencil_sites(stencil, L):
    return int(load_library().spin_stencil_sites(stencil, L))


def spin_stencil_init(stencil, batch, L, lattice_ptr, seed, replica_offset=0, cuda_stream=None):
    _check(load_library().spin_stencil_init(stencil, batch, L, lattice_ptr, int(seed), int(replica_offset), cuda_stream))


def spin_stencil_sweep(stencil, batch, L, lattice_ptr, beta, J1, J2, h, seed, n_sweeps, sweep_offset=0, replica_offset=0,
                       cuda_stream=None):
    b = _beta64(beta, batch)
    _check(load_library().spin_stencil_sweep(stencil, batch, L, lattice_ptr, _np_ptr(b), float(J1), float(J2), float(h),
                                             int(seed), int(replica_offset), int(n_sweeps), int(sweep_offset), cuda_stream))


def spin_stencil_observables(stencil, batch, L, lattice_ptr, cuda_stream=None):
    E1, E2, M = (np.zeros(batch, dtype=np.int64) for _ in range(3))
    _check(load_library().spin_stencil_observables(stencil, batch, L, lattice_ptr, _np_ptr(E1), _np_ptr(E2), _np_ptr(M),
                                                   cuda_stream))
    return E1, E2, M


def spin_stencil_observables_noalloc(stencil, batch, L, lattice_ptr, E1_ptr, E2_ptr, M_ptr, cuda_stream=None):
    """E1_ptr / E2_ptr / M_ptr: DEVICE int64 [batch] (or None); asynchronous, allocates nothing (batch <= 4096)."""
    _check(load_library().spin_stencil_observables_noalloc(stencil, batch, L, lattice_ptr, E1_ptr, E2_ptr, M_ptr, cuda_stream))


def _cpm_arrays(tau, Jtab, A):
    tau = np.ascontiguousarray(tau, dtype=np.int32)
    Jtab = np.ascontiguousarray(Jtab, dtype=np.int32)
    A = np.ascontiguousarray(A, dtype=np.int32)
    assert Jtab.ndim == 2 and Jtab.shape[0] == Jtab.shape[1] and A.shape == tau.shape
    return tau, Jtab, A


def spin_cpm_sweep(batch, L, lattice_ptr, tau, Jtab, lam, A, beta, seed, n_sweeps, sweep_offset=0, replica_offset=0,
                   cuda_stream=None):
    tau, Jtab, A = _cpm_arrays(tau, Jtab, A)
    b = _beta64(beta, batch)
    _check(load_library().spin_cpm_sweep(batch, L, tau.shape[0], lattice_ptr, _np_ptr(tau), _np_ptr(Jtab), Jtab.shape[0],
                                         int(lam), _np_ptr(A), _np_ptr(b), int(seed), int(replica_offset), int(n_sweeps),
                                         int(sweep_offset), cuda_stream))


def spin_cpm_observables(batch, L, lattice_ptr, tau, Jtab, lam, A, cuda_stream=None):
    """-> (H_adh [B], H_area [B], areas [B][q], boundary [B][ntypes][ntypes]) int64."""
    tau, Jtab, A = _cpm_arrays(tau, Jtab, A)
    q, nt = tau.shape[0], Jtab.shape[0]
    Ha, Hr = np.zeros(batch, dtype=np.int64), np.zeros(batch, dtype=np.int64)
    ar, bl = np.zeros((batch, q), dtype=np.int64), np.zeros((batch, nt, nt), dtype=np.int64)
    _check(load_library().spin_cpm_observables(batch, L, q, lattice_ptr, _np_ptr(tau), _np_ptr(Jtab), nt, int(lam), _np_ptr(A),
                                               _np_ptr(Ha), _np_ptr(Hr), _np_ptr(ar), _np_ptr(bl), cuda_stream))
    return Ha, Hr, ar, bl


def spin_dmc_discretise(dtype, s_ptr, n, cuda_stream=None):
    _check(load_library().spin_dmc_discretise(dtype, s_ptr, int(n), cuda_stream))


class SpinSim:
    """Owner of one spin_sim* handle.  Methods are the C calls with numpy / raw-pointer marshalling."""

    def __init__(self, handle, batch, L, model, layout, keepalive=None):
        self._h = handle
        self.batch, self.L, self.model, self.layout = batch, L, model, layout
        self._keepalive = keepalive  # e.g. the torch tensor backing device_buffer

    def _beta(self, beta):
        b = np.ascontiguousarray(np.broadcast_to(np.asarray(beta, dtype=np.float64), (self.batch,)))
        return b

    def spin_sweep(self, beta, J, h, n_sweeps, sweep_offset=0):
        b = self._beta(beta)
        _check(load_library().spin_sweep(self._h, _np_ptr(b), float(J), float(h), int(n_sweeps), int(sweep_offset)))

    def spin_observables(self):
        E = np.zeros(self.batch, dtype=np.int64)
        M = np.zeros(self.batch, dtype=np.int64)
        _check(load_library().spin_observables(self._h, _np_ptr(E), _np_ptr(M)))
        return E, M

    def spin_observables_dev(self, E_ptr, M_ptr):
        _check(load_library().spin_observables_dev(self._h, E_ptr, M_ptr))

    def spin_get_spins(self, out=None):
        if out is None:
            out = np.empty((self.batch, self.L, self.L), dtype=np.int8)
        assert out.dtype == np.int8 and out.size == self.batch * self.L * self.L and out.flags["C_CONTIGUOUS"]
        _check(load_library().spin_get_spins(self._h, _np_ptr(out)))
        return out

    def spin_set_spins(self, spins):
        s = np.ascontiguousarray(spins, dtype=np.int8)
        assert s.size == self.batch * self.L * self.L
        _check(load_library().spin_set_spins(self._h, _np_ptr(s)))

    def spin_set_spins_ptr(self, host_ptr):
        """spin_set_spins from a raw host pointer (e.g. a pinned torch tensor's data_ptr())."""
        _check(load_library().spin_set_spins(self._h, host_ptr))

    def spin_sweep_measure(self, beta, J, h, n_sweeps, sweep_offset=0, trace=True, moments=None):
        b = self._beta(beta)
        Et = Mt = None
        if trace:
            Et = np.zeros((n_sweeps, self.batch), dtype=np.int64)
            Mt = np.zeros((n_sweeps, self.batch), dtype=np.int64)
        if moments is not None:
            assert moments.dtype == np.int64 and moments.shape == (self.batch, 8) and moments.flags["C_CONTIGUOUS"]
        _check(load_library().spin_sweep_measure(self._h, _np_ptr(b), float(J), float(h), int(n_sweeps),
                                                 int(sweep_offset), _np_ptr(Et), _np_ptr(Mt), _np_ptr(moments)))
        return Et, Mt

    def spin_set_stream(self, cuda_stream):
        _check(load_library().spin_set_stream(self._h, cuda_stream))

    def spin_synchronize(self):
        _check(load_library().spin_synchronize(self._h))

    def spin_kernel_launches(self):
        return int(load_library().spin_kernel_launches(self._h))

    def spin_set_bonds(self, Jh, Jv):
        """+-1 bond signs, natural layout [batch][L][L] (broadcast from [L][L]); (None, None) removes them."""
        if Jh is None and Jv is None:
            _check(load_library().spin_set_bonds(self._h, None, None))
            return
        shape = (self.batch, self.L, self.L)
        jh = np.ascontiguousarray(np.broadcast_to(np.asarray(Jh, dtype=np.int8), shape))
        jv = np.ascontiguousarray(np.broadcast_to(np.asarray(Jv, dtype=np.int8), shape))
        _check(load_library().spin_set_bonds(self._h, _np_ptr(jh), _np_ptr(jv)))

    def spin_set_couplings(self, Jh, Jv, B):
        """Real couplings / per-site fields, natural [batch][L][L] (broadcastable); (None, None, None) removes them."""
        if Jh is None and Jv is None and B is None:
            _check(load_library().spin_set_couplings(self._h, None, None, None))
            return
        shape = (self.batch, self.L, self.L)
        a = [np.ascontiguousarray(np.broadcast_to(np.asarray(x, dtype=np.float64), shape)) for x in (Jh, Jv, B)]
        _check(load_library().spin_set_couplings(self._h, _np_ptr(a[0]), _np_ptr(a[1]), _np_ptr(a[2])))

    def spin_energy_general(self):
        E = np.zeros(self.batch, dtype=np.float64)
        _check(load_library().spin_energy_general(self._h, _np_ptr(E)))
        return E

    def spin_potts_label_sum(self):
        S = np.zeros(self.batch, dtype=np.int64)
        _check(load_library().spin_potts_label_sum(self._h, _np_ptr(S)))
        return S

    def spin_sweep_schedule(self, beta_steps, J, h, sweeps_per_step, sweep_offset=0):
        bs = np.ascontiguousarray(np.asarray(beta_steps, dtype=np.float64))
        assert bs.ndim == 2 and bs.shape[1] == self.batch
        _check(load_library().spin_sweep_schedule(self._h, _np_ptr(bs), bs.shape[0], float(J), float(h), int(sweeps_per_step),
                                                  int(sweep_offset)))

    def spin_set_policy(self, policy):
        _check(load_library().spin_set_policy(self._h, int(policy)))

    def spin_kernel_variant(self):
        return load_library().spin_kernel_variant(self._h).decode()

    def spin_destroy(self):
        if self._h:
            load_library().spin_destroy(self._h)
            self._h = None
            self._keepalive = None

    def __del__(self):
        try:
            self.spin_destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.spin_destroy()


def spin_create(batch, L, q, seed):
    h = load_library().spin_create(batch, L, q, seed)
    if not h:
        raise SpinError(SPIN_ERR_INVALID, spin_last_error())
    return SpinSim(h, batch, L, SPIN_MODEL_ISING if q == 2 else SPIN_MODEL_POTTS, SPIN_LAYOUT_INT8)


def spin_create_ex(batch, L, model, q_per_replica=None, q_uniform=2, seed=0, layout=SPIN_LAYOUT_INT8,
                   replica_offset=0, device_buffer=None, buffer_bytes=0, cuda_stream=None, keepalive=None):
    qa = None
    if q_per_replica is not None:
        qa = np.ascontiguousarray(q_per_replica, dtype=np.int32)
        assert qa.shape == (batch,)
    h = load_library().spin_create_ex(batch, L, model, _np_ptr(qa), int(q_uniform), int(seed), layout,
                                      int(replica_offset), device_buffer, int(buffer_bytes), cuda_stream)
    if not h:
        raise SpinError(SPIN_ERR_INVALID, spin_last_error())
    return SpinSim(h, batch, L, model, layout, keepalive=keepalive)
