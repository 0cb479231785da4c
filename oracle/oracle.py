"""ORACLE — test infrastructure.  Thin ctypes wrappers over ``liboracle.so``.

Argument marshalling only; every step of the method is in ``spin_oracle.cpp``.
Lattices are numpy int8 arrays in the natural layout ``[batch][L][L]``.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "spin_oracle.cpp")
_SRCS = [_SRC, os.path.join(_HERE, "dmc_oracle.cpp"), os.path.join(_HERE, "general_oracle.cpp"),
         os.path.join(_HERE, "stencil_oracle.cpp"), os.path.join(_HERE, "cpm_oracle.cpp")]
_LIB = os.path.join(_HERE, "liboracle.so")

__all__ = [
    "build", "philox4x32_10", "ising_table", "potts_table", "init", "ising_half_sweep",
    "potts_half_sweep", "ising_observables", "potts_observables", "accumulate_moments", "sweep",
    "sweep_bonds", "ising_bonds_observables", "ising_bonds_half_sweep",
    "dmc_half_sweep", "dmc_forward", "dmc_discretise", "dmc_backward",
    "ising_general_half_sweep", "sweep_general", "ising_general_observables", "potts_general_half_sweep",
    "sweep_potts_general", "potts_general_observables", "sweep_schedule",
    "STENCIL_TRIANGULAR", "STENCIL_CUBIC", "STENCIL_SQUARE_NNN", "stencil_shape", "stencil_init", "stencil_colour_pass",
    "stencil_sweep", "stencil_observables",
    "cpm_delta", "cpm_colour_pass", "cpm_sweep", "cpm_observables",
]


def build(force=False):
    """Compile the oracle with ``g++ -O2 -ffp-contract=off`` (no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(p) for p in _SRCS):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", tmp] + _SRCS)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _l():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        c = ctypes
        p = c.c_void_p
        lib.oracle_philox4x32_10.argtypes = [p, p, p]
        lib.oracle_ising_table.argtypes = [c.c_double, c.c_double, c.c_double, p, p]
        lib.oracle_potts_table.argtypes = [c.c_double, c.c_double, p, p]
        lib.oracle_init.argtypes = [p, c.c_int32, c.c_int32, c.c_int32, p, c.c_uint64, c.c_int64]
        lib.oracle_ising_half_sweep.argtypes = [p, c.c_int32, c.c_int32, p, c.c_double, c.c_double,
                                                c.c_uint64, c.c_int64, c.c_int64, c.c_int32]
        lib.oracle_potts_half_sweep.argtypes = [p, c.c_int32, c.c_int32, p, p, c.c_double, c.c_uint64,
                                                c.c_int64, c.c_int64, c.c_int32]
        lib.oracle_ising_observables.argtypes = [p, c.c_int32, c.c_int32, p, p]
        lib.oracle_potts_observables.argtypes = [p, c.c_int32, c.c_int32, p, p, p]
        lib.oracle_accumulate_moments.argtypes = [p, c.c_int32, p, p]
        lib.oracle_sweep.argtypes = [p, c.c_int32, c.c_int32, c.c_int32, p, p, c.c_double, c.c_double,
                                     c.c_uint64, c.c_int64, c.c_int64, c.c_int64, p, p, p]
        lib.oracle_ising_bonds_observables.argtypes = [p, p, p, c.c_int32, c.c_int32, p, p]
        lib.oracle_ising_bonds_half_sweep.argtypes = [p, p, p, c.c_int32, c.c_int32, p, c.c_double, c.c_double,
                                                      c.c_uint64, c.c_int64, c.c_int64, c.c_int32]
        lib.oracle_sweep_bonds.argtypes = [p, p, p, c.c_int32, c.c_int32, p, c.c_double, c.c_double, c.c_uint64,
                                           c.c_int64, c.c_int64, c.c_int64, p, p]
        d = c.c_double
        lib.oracle_ising_general_half_sweep.argtypes = [p, p, p, p, c.c_int32, c.c_int32, p, c.c_uint64, c.c_int64,
                                                        c.c_int64, c.c_int32]
        lib.oracle_ising_general_observables.argtypes = [p, p, p, p, c.c_int32, c.c_int32, p, p]
        lib.oracle_potts_general_half_sweep.argtypes = [p, p, p, c.c_int32, c.c_int32, p, p, d, d, c.c_uint64, c.c_int64,
                                                        c.c_int64, c.c_int32]
        lib.oracle_potts_general_observables.argtypes = [p, p, p, c.c_int32, c.c_int32, p, p, p, p]
        lib.oracle_stencil_sites.argtypes = [c.c_int32, c.c_int32]
        lib.oracle_stencil_sites.restype = c.c_int64
        lib.oracle_stencil_init.argtypes = [p, c.c_int32, c.c_int32, c.c_int32, c.c_uint64, c.c_int64]
        lib.oracle_stencil_colour_pass.argtypes = [p, c.c_int32, c.c_int32, c.c_int32, p, d, d, d, c.c_uint64, c.c_int64,
                                                   c.c_int64, c.c_int32]
        lib.oracle_stencil_sweep.argtypes = [p, c.c_int32, c.c_int32, c.c_int32, p, d, d, d, c.c_uint64, c.c_int64,
                                             c.c_int64, c.c_int64]
        lib.oracle_stencil_observables.argtypes = [p, c.c_int32, c.c_int32, c.c_int32, p, p, p]
        lib.oracle_cpm_delta.argtypes = [p, c.c_int32, c.c_int32, p, p, c.c_int32, c.c_int64, p, c.c_int32, c.c_int32, c.c_int32]
        lib.oracle_cpm_delta.restype = c.c_int64
        lib.oracle_cpm_colour_pass.argtypes = [p, c.c_int32, c.c_int32, c.c_int32, p, p, c.c_int32, c.c_int64, p, p,
                                               c.c_uint64, c.c_int64, c.c_int64, c.c_int32]
        lib.oracle_cpm_sweep.argtypes = [p, c.c_int32, c.c_int32, c.c_int32, p, p, c.c_int32, c.c_int64, p, p, c.c_uint64,
                                         c.c_int64, c.c_int64, c.c_int64]
        lib.oracle_cpm_observables.argtypes = [p, c.c_int32, c.c_int32, c.c_int32, p, p, c.c_int32, c.c_int64, p, p, p, p, p]
        lib.oracle_dmc_half_sweep.argtypes = [p, p, p, c.c_int32, c.c_int32, d, p, d, c.c_uint64, c.c_int64, c.c_int64,
                                              c.c_int32, p]
        lib.oracle_dmc_forward.argtypes = [p, p, p, c.c_int32, c.c_int32, d, p, d, c.c_uint64, c.c_int64, c.c_int64,
                                           c.c_int64, p]
        lib.oracle_dmc_discretise.argtypes = [p, c.c_int64]
        lib.oracle_dmc_backward.argtypes = [p, p, p, c.c_int32, c.c_int32, d, p, d, c.c_uint64, c.c_int64, c.c_int64,
                                            c.c_int64, p, p, p, p, p, p]
        _lib = lib
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _lattice(spins):
    assert spins.dtype == np.int8 and spins.ndim == 3 and spins.shape[1] == spins.shape[2]
    assert spins.flags["C_CONTIGUOUS"]
    return spins.shape[0], spins.shape[1]


def _q_array(q, batch):
    if q is None:
        return None
    qa = np.ascontiguousarray(np.broadcast_to(np.asarray(q, dtype=np.int32), (batch,)))
    return qa


def _beta_array(beta, batch):
    return np.ascontiguousarray(np.broadcast_to(np.asarray(beta, dtype=np.float64), (batch,)))


def philox4x32_10(ctr, key):
    ctr = np.asarray(ctr, dtype=np.uint32)
    key = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    _l().oracle_philox4x32_10(_ptr(ctr), _ptr(key), _ptr(out))
    return out


def ising_table(beta, J, h):
    """-> (T uint32[10], always bool[10]); class = 5*(s+1)/2 + (nn+4)/2."""
    T = np.zeros(10, dtype=np.uint32)
    a = np.zeros(10, dtype=np.uint8)
    _l().oracle_ising_table(float(beta), float(J), float(h), _ptr(T), _ptr(a))
    return T, a.astype(bool)


def potts_table(beta, J):
    """-> (T uint32[9], always bool[9]); class = dn+4."""
    T = np.zeros(9, dtype=np.uint32)
    a = np.zeros(9, dtype=np.uint8)
    _l().oracle_potts_table(float(beta), float(J), _ptr(T), _ptr(a))
    return T, a.astype(bool)


def init(batch, L, seed, q=None, replica_offset=0):
    """Initial lattices (O3).  q=None -> Ising; q int or int[batch] -> Potts."""
    spins = np.zeros((batch, L, L), dtype=np.int8)
    qa = _q_array(q, batch)
    _l().oracle_init(_ptr(spins), batch, L, 0 if q is None else 1, _ptr(qa), int(seed), int(replica_offset))
    return spins


def ising_half_sweep(spins, beta, J, h, seed, t, colour, replica_offset=0):
    B, L = _lattice(spins)
    ba = _beta_array(beta, B)
    _l().oracle_ising_half_sweep(_ptr(spins), B, L, _ptr(ba), float(J), float(h), int(seed),
                                 int(replica_offset), int(t), int(colour))


def potts_half_sweep(spins, q, beta, J, seed, t, colour, replica_offset=0):
    B, L = _lattice(spins)
    ba = _beta_array(beta, B)
    qa = _q_array(q, B)
    _l().oracle_potts_half_sweep(_ptr(spins), B, L, _ptr(qa), _ptr(ba), float(J), int(seed),
                                 int(replica_offset), int(t), int(colour))


def ising_observables(spins):
    B, L = _lattice(spins)
    E = np.zeros(B, dtype=np.int64)
    M = np.zeros(B, dtype=np.int64)
    _l().oracle_ising_observables(_ptr(spins), B, L, _ptr(E), _ptr(M))
    return E, M


def potts_observables(spins, q):
    B, L = _lattice(spins)
    qa = _q_array(q, B)
    E = np.zeros(B, dtype=np.int64)
    M = np.zeros(B, dtype=np.int64)
    _l().oracle_potts_observables(_ptr(spins), B, L, _ptr(qa), _ptr(E), _ptr(M))
    return E, M


def accumulate_moments(moments, E, M):
    B = moments.shape[0]
    assert moments.dtype == np.int64 and moments.shape == (B, 8) and moments.flags["C_CONTIGUOUS"]
    E = np.ascontiguousarray(E, dtype=np.int64)
    M = np.ascontiguousarray(M, dtype=np.int64)
    _l().oracle_accumulate_moments(_ptr(moments), B, _ptr(E), _ptr(M))


def sweep(spins, beta, J, h, seed, n_sweeps, sweep_offset=0, q=None, replica_offset=0,
          trace=False, moments=None):
    """Run sweeps in place.  Returns (E_trace, M_trace) int64[n_sweeps][batch] if trace else None."""
    B, L = _lattice(spins)
    ba = _beta_array(beta, B)
    qa = _q_array(q, B)
    Et = Mt = None
    if trace:
        Et = np.zeros((n_sweeps, B), dtype=np.int64)
        Mt = np.zeros((n_sweeps, B), dtype=np.int64)
    if moments is not None:
        assert moments.dtype == np.int64 and moments.shape == (B, 8) and moments.flags["C_CONTIGUOUS"]
    _l().oracle_sweep(_ptr(spins), B, L, 0 if q is None else 1, _ptr(qa), _ptr(ba), float(J), float(h),
                      int(seed), int(replica_offset), int(n_sweeps), int(sweep_offset),
                      _ptr(Et), _ptr(Mt), _ptr(moments))
    return (Et, Mt) if trace else None


def _bonds(J, B, L):
    a = np.ascontiguousarray(np.broadcast_to(np.asarray(J, dtype=np.int8), (B, L, L)))
    assert np.all(np.abs(a) == 1), "bond signs must be +-1"
    return a


def ising_bonds_observables(spins, Jh, Jv):
    """E_int = -sum_bonds J_ij s_i s_j, M = sum s for +-1 bond signs Jh (right bonds), Jv (down bonds)."""
    B, L = _lattice(spins)
    jh, jv = _bonds(Jh, B, L), _bonds(Jv, B, L)
    E = np.zeros(B, dtype=np.int64)
    M = np.zeros(B, dtype=np.int64)
    _l().oracle_ising_bonds_observables(_ptr(spins), _ptr(jh), _ptr(jv), B, L, _ptr(E), _ptr(M))
    return E, M


def sweep_bonds(spins, Jh, Jv, beta, J, h, seed, n_sweeps, sweep_offset=0, replica_offset=0, trace=False):
    """Ising sweeps with +-1 bond signs (Jh[b][i][j]: bond (i,j)-(i,j+1); Jv[b][i][j]: bond (i,j)-(i+1,j)), in place."""
    B, L = _lattice(spins)
    ba = _beta_array(beta, B)
    jh, jv = _bonds(Jh, B, L), _bonds(Jv, B, L)
    Et = Mt = None
    if trace:
        Et = np.zeros((n_sweeps, B), dtype=np.int64)
        Mt = np.zeros((n_sweeps, B), dtype=np.int64)
    _l().oracle_sweep_bonds(_ptr(spins), _ptr(jh), _ptr(jv), B, L, _ptr(ba), float(J), float(h), int(seed),
                            int(replica_offset), int(n_sweeps), int(sweep_offset), _ptr(Et), _ptr(Mt))
    return (Et, Mt) if trace else None


def ising_bonds_half_sweep(spins, Jh, Jv, beta, J, h, seed, t, colour, replica_offset=0):
    B, L = _lattice(spins)
    ba = _beta_array(beta, B)
    jh, jv = _bonds(Jh, B, L), _bonds(Jv, B, L)
    _l().oracle_ising_bonds_half_sweep(_ptr(spins), _ptr(jh), _ptr(jv), B, L, _ptr(ba), float(J), float(h),
                                       int(seed), int(replica_offset), int(t), int(colour))


# ---- Differentiable Monte Carlo (dmc_oracle.cpp; Algorithm 2, Eq. 4) ------------------------------------------
def _f64(a, shape):
    a = np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.float64), shape))
    return a


def _dmc_lattice(s):
    assert s.dtype == np.float64 and s.ndim == 3 and s.shape[1] == s.shape[2] and s.flags["C_CONTIGUOUS"]
    return s.shape[0], s.shape[1]


def dmc_half_sweep(s, Jh, Jv, h, beta, alpha, seed, t, colour, replica_offset=0, want_q=False):
    """One DMC half-sweep in place on the float64 lattice s [B][L][L]; returns q [B][L][L] (NaN elsewhere) if want_q."""
    B, L = _dmc_lattice(s)
    jh, jv, ba = _f64(Jh, (B, L, L)), _f64(Jv, (B, L, L)), _beta_array(beta, B)
    q = np.full((B, L, L), np.nan) if want_q else None
    _l().oracle_dmc_half_sweep(_ptr(s), _ptr(jh), _ptr(jv), B, L, float(h), _ptr(ba), float(alpha), int(seed),
                               int(replica_offset), int(t), int(colour), _ptr(q))
    return q


def dmc_forward(s, Jh, Jv, h, beta, alpha, seed, n_sweeps, sweep_offset=0, replica_offset=0, want_traj=False):
    """n_sweeps DMC sweeps in place; returns the trajectory [2 n_sweeps + 1][B][L][L] if want_traj."""
    B, L = _dmc_lattice(s)
    jh, jv, ba = _f64(Jh, (B, L, L)), _f64(Jv, (B, L, L)), _beta_array(beta, B)
    traj = np.zeros((2 * n_sweeps + 1, B, L, L)) if want_traj else None
    _l().oracle_dmc_forward(_ptr(s), _ptr(jh), _ptr(jv), B, L, float(h), _ptr(ba), float(alpha), int(seed),
                            int(replica_offset), int(n_sweeps), int(sweep_offset), _ptr(traj))
    return traj


def dmc_discretise(s):
    assert s.dtype == np.float64 and s.flags["C_CONTIGUOUS"]
    _l().oracle_dmc_discretise(_ptr(s), s.size)
    return s


def dmc_backward(traj, Jh, Jv, h, beta, alpha, seed, grad_out, sweep_offset=0, replica_offset=0):
    """-> (grad_s0, grad_Jh, grad_Jv [B][L][L], grad_beta [B], grad_h [B]) of a loss whose gradient with respect to the
    final lattice is grad_out; traj from dmc_forward(..., want_traj=True)."""
    assert traj.dtype == np.float64 and traj.ndim == 4 and traj.flags["C_CONTIGUOUS"]
    n_sweeps, B, L = (traj.shape[0] - 1) // 2, traj.shape[1], traj.shape[2]
    jh, jv, ba = _f64(Jh, (B, L, L)), _f64(Jv, (B, L, L)), _beta_array(beta, B)
    go = _f64(grad_out, (B, L, L))
    gs, gjh, gjv = np.zeros((B, L, L)), np.zeros((B, L, L)), np.zeros((B, L, L))
    gb, gh = np.zeros(B), np.zeros(B)
    _l().oracle_dmc_backward(_ptr(traj), _ptr(jh), _ptr(jv), B, L, float(h), _ptr(ba), float(alpha), int(seed),
                             int(replica_offset), int(n_sweeps), int(sweep_offset), _ptr(go), _ptr(gs), _ptr(gjh),
                             _ptr(gjv), _ptr(gb), _ptr(gh))
    return gs, gjh, gjv, gb, gh


# ---- general couplings and fields (general_oracle.cpp; Eq. 1 and Eq. 5 as the paper writes them) ---------------------
def ising_general_half_sweep(spins, Jh, Jv, B, beta, seed, t, colour, replica_offset=0):
    Bn, L = _lattice(spins)
    jh, jv, fb, ba = _f64(Jh, (Bn, L, L)), _f64(Jv, (Bn, L, L)), _f64(B, (Bn, L, L)), _beta_array(beta, Bn)
    _l().oracle_ising_general_half_sweep(_ptr(spins), _ptr(jh), _ptr(jv), _ptr(fb), Bn, L, _ptr(ba), int(seed),
                                         int(replica_offset), int(t), int(colour))


def sweep_general(spins, Jh, Jv, B, beta, seed, n_sweeps, sweep_offset=0, replica_offset=0):
    """Ising sweeps with real couplings Jh, Jv and per-site fields B (natural [batch][L][L], broadcastable), in place."""
    for t in range(sweep_offset, sweep_offset + n_sweeps):
        for colour in (0, 1):
            ising_general_half_sweep(spins, Jh, Jv, B, beta, seed, t, colour, replica_offset)


def ising_general_observables(spins, Jh, Jv, B):
    """-> (E float64[batch] = -sum J s s - sum B s, M int64[batch])."""
    Bn, L = _lattice(spins)
    jh, jv, fb = _f64(Jh, (Bn, L, L)), _f64(Jv, (Bn, L, L)), _f64(B, (Bn, L, L))
    E = np.zeros(Bn)
    M = np.zeros(Bn, dtype=np.int64)
    _l().oracle_ising_general_observables(_ptr(spins), _ptr(jh), _ptr(jv), _ptr(fb), Bn, L, _ptr(E), _ptr(M))
    return E, M


def _opt_bonds(J, Bn, L):
    return None if J is None else _bonds(J, Bn, L)


def potts_general_half_sweep(spins, q, beta, J, h, seed, t, colour, Jh=None, Jv=None, replica_offset=0):
    Bn, L = _lattice(spins)
    assert (Jh is None) == (Jv is None)
    jh, jv, ba, qa = _opt_bonds(Jh, Bn, L), _opt_bonds(Jv, Bn, L), _beta_array(beta, Bn), _q_array(q, Bn)
    _l().oracle_potts_general_half_sweep(_ptr(spins), _ptr(jh), _ptr(jv), Bn, L, _ptr(qa), _ptr(ba), float(J), float(h),
                                         int(seed), int(replica_offset), int(t), int(colour))


def sweep_potts_general(spins, q, beta, J, h, seed, n_sweeps, Jh=None, Jv=None, sweep_offset=0, replica_offset=0):
    """Potts sweeps with a field h on the state label and optional +-1 bond signs, in place."""
    for t in range(sweep_offset, sweep_offset + n_sweeps):
        for colour in (0, 1):
            potts_general_half_sweep(spins, q, beta, J, h, seed, t, colour, Jh, Jv, replica_offset)


def potts_general_observables(spins, q, Jh=None, Jv=None):
    """-> (E_int = -sum_bonds J_ij delta, S = sum of state labels, M = max_k N_k), int64[batch] each."""
    Bn, L = _lattice(spins)
    jh, jv, qa = _opt_bonds(Jh, Bn, L), _opt_bonds(Jv, Bn, L), _q_array(q, Bn)
    E, S, M = (np.zeros(Bn, dtype=np.int64) for _ in range(3))
    _l().oracle_potts_general_observables(_ptr(spins), _ptr(jh), _ptr(jv), Bn, L, _ptr(qa), _ptr(E), _ptr(S), _ptr(M))
    return E, S, M


def sweep_schedule(spins, beta_steps, J, h, seed, sweeps_per_step, sweep_offset=0, q=None, replica_offset=0, Jh=None,
                   Jv=None):
    """Annealing schedule (Fig. 9's Monte Carlo arm): step k runs sweeps_per_step sweeps at beta_steps[k]
    ([n_steps][batch]); the sweep index keeps counting across steps."""
    beta_steps = np.asarray(beta_steps, dtype=np.float64)
    t = sweep_offset
    for k in range(beta_steps.shape[0]):
        if Jh is not None and q is None:
            sweep_bonds(spins, Jh, Jv, beta_steps[k], J, h, seed, sweeps_per_step, sweep_offset=t, replica_offset=replica_offset)
        else:
            sweep(spins, beta_steps[k], J, h, seed, sweeps_per_step, sweep_offset=t, q=q, replica_offset=replica_offset)
        t += sweeps_per_step


# ---- other lattice geometries (stencil_oracle.cpp) -----------------------------------------
STENCIL_TRIANGULAR, STENCIL_CUBIC, STENCIL_SQUARE_NNN = 0, 1, 2


def stencil_shape(stencil, batch, L):
    return (batch, L, L, L) if stencil == STENCIL_CUBIC else (batch, L, L)


def stencil_init(stencil, batch, L, seed, replica_offset=0):
    spins = np.zeros(stencil_shape(stencil, batch, L), dtype=np.int8)
    _l().oracle_stencil_init(_ptr(spins), stencil, batch, L, int(seed), int(replica_offset))
    return spins


def _stencil_lattice(stencil, spins):
    assert spins.dtype == np.int8 and spins.flags["C_CONTIGUOUS"] and spins.ndim == (5 if False else (4 if stencil == STENCIL_CUBIC else 3))
    return spins.shape[0], spins.shape[1]


def stencil_colour_pass(stencil, spins, beta, J1, J2, h, seed, t, colour, replica_offset=0):
    B, L = _stencil_lattice(stencil, spins)
    ba = _beta_array(beta, B)
    _l().oracle_stencil_colour_pass(_ptr(spins), stencil, B, L, _ptr(ba), float(J1), float(J2), float(h), int(seed),
                                    int(replica_offset), int(t), int(colour))


def stencil_sweep(stencil, spins, beta, J1, J2, h, seed, n_sweeps, sweep_offset=0, replica_offset=0):
    B, L = _stencil_lattice(stencil, spins)
    ba = _beta_array(beta, B)
    _l().oracle_stencil_sweep(_ptr(spins), stencil, B, L, _ptr(ba), float(J1), float(J2), float(h), int(seed),
                              int(replica_offset), int(n_sweeps), int(sweep_offset))


def stencil_observables(stencil, spins):
    """-> (E1, E2, M) int64[batch]: minus the first- / second-neighbour bond sums, and sum s."""
    B, L = _stencil_lattice(stencil, spins)
    E1, E2, M = (np.zeros(B, dtype=np.int64) for _ in range(3))
    _l().oracle_stencil_observables(_ptr(spins), stencil, B, L, _ptr(E1), _ptr(E2), _ptr(M))
    return E1, E2, M


# ---- Cellular Potts model (cpm_oracle.cpp; Eq. 7, Table II) ----------------------------------------
def _cpm_params(tau, Jtab, A):
    tau = np.ascontiguousarray(tau, dtype=np.int32)
    Jtab = np.ascontiguousarray(Jtab, dtype=np.int32)
    A = np.ascontiguousarray(A, dtype=np.int32)
    q, nt = tau.shape[0], Jtab.shape[0]
    assert Jtab.shape == (nt, nt) and A.shape == (q,) and tau.min() >= 0 and tau.max() < nt
    return tau, Jtab, A, q, nt


def cpm_delta(lat, tau, Jtab, lam, A, i, j, new):
    """dH of the proposal lat[i][j] -> new on one lattice [L][L] (areas counted from lat)."""
    tau, Jtab, A, q, nt = _cpm_params(tau, Jtab, A)
    assert lat.dtype == np.int8 and lat.ndim == 2 and lat.flags["C_CONTIGUOUS"]
    return int(_l().oracle_cpm_delta(_ptr(lat), lat.shape[0], q, _ptr(tau), _ptr(Jtab), nt, int(lam), _ptr(A), int(i), int(j), int(new)))


def cpm_colour_pass(spins, tau, Jtab, lam, A, beta, seed, t, colour, replica_offset=0):
    B, L = _lattice(spins)
    tau, Jtab, A, q, nt = _cpm_params(tau, Jtab, A)
    ba = _beta_array(beta, B)
    _l().oracle_cpm_colour_pass(_ptr(spins), B, L, q, _ptr(tau), _ptr(Jtab), nt, int(lam), _ptr(A), _ptr(ba), int(seed),
                                int(replica_offset), int(t), int(colour))


def cpm_sweep(spins, tau, Jtab, lam, A, beta, seed, n_sweeps, sweep_offset=0, replica_offset=0):
    B, L = _lattice(spins)
    tau, Jtab, A, q, nt = _cpm_params(tau, Jtab, A)
    ba = _beta_array(beta, B)
    _l().oracle_cpm_sweep(_ptr(spins), B, L, q, _ptr(tau), _ptr(Jtab), nt, int(lam), _ptr(A), _ptr(ba), int(seed),
                          int(replica_offset), int(n_sweeps), int(sweep_offset))


def cpm_observables(spins, tau, Jtab, lam, A):
    """-> (H_adh [B], H_area [B], areas [B][q], boundary [B][ntypes][ntypes]) int64."""
    B, L = _lattice(spins)
    tau, Jtab, A, q, nt = _cpm_params(tau, Jtab, A)
    Ha, Hr = np.zeros(B, dtype=np.int64), np.zeros(B, dtype=np.int64)
    ar, bl = np.zeros((B, q), dtype=np.int64), np.zeros((B, nt, nt), dtype=np.int64)
    _l().oracle_cpm_observables(_ptr(spins), B, L, q, _ptr(tau), _ptr(Jtab), nt, int(lam), _ptr(A), _ptr(Ha), _ptr(Hr),
                                _ptr(ar), _ptr(bl))
    return Ha, Hr, ar, bl
