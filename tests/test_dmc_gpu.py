"""GPU parity of the Differentiable-Monte-Carlo kernels (csrc/dmc.cu, through the C ABI) against the fp64 oracle
(oracle/dmc_oracle.cpp): Algorithm 2 forward (every stored half-sweep state, elementwise), the hand-written backward
(dJ per bond, dbeta, dh, ds0), Eq. 4, the alpha -> infinity limit, and a finite-difference check run on the GPU.

Tolerances.  fp64 kernel vs fp64 oracle: same operation order, the only difference is CUDA's
exp vs glibc's (<= 2 ulp): 1e-12 absolute per half-sweep state, growing with the number of half-sweeps.  fp32 kernel
vs fp64 oracle on fp32-representable inputs: the error of one update is 2|s| (alpha/4) dp with dp ~ p (|beta dE| + 2) 6e-8
where q is not saturated (p <~ 1), i.e. ~1e-6 at alpha = 6, multiplied by the per-half-sweep Jacobian (up to ~alpha): the
bound used is 2e-5 absolute after 2 sweeps, and 2e-3 of the largest gradient entry for the backward pass."""
import numpy as np
import pytest

import oracle
import paper_2304_01772_b200 as sp

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _inputs(B, L, seed, dtype, glass=True):
    rng = np.random.default_rng(seed)
    f = np.float32 if dtype == sp.SPIN_DTYPE_F32 else np.float64
    s = rng.uniform(-1.0, 1.0, size=(B, L, L)).astype(f)
    if glass:
        Jh = rng.normal(0.0, 0.7, size=(B, L, L)).astype(f)
        Jv = rng.normal(0.0, 0.7, size=(B, L, L)).astype(f)
    else:
        Jh = np.ones((B, L, L), dtype=f)
        Jv = np.ones((B, L, L), dtype=f)
    beta = rng.uniform(0.3, 0.9, size=B)
    return s, Jh, Jv, beta


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _run_gpu(dtype, s, Jh, Jv, h, beta, alpha, seed, n_sweeps, grad_out_fn=None, replica_offset=0, sweep_offset=0):
    B, L = s.shape[0], s.shape[1]
    tdt = torch.float32 if dtype == sp.SPIN_DTYPE_F32 else torch.float64
    ds, dJh, dJv = _dev(s), _dev(Jh), _dev(Jv)
    traj = torch.empty((2 * n_sweeps + 1, B, L, L), dtype=tdt, device="cuda")
    out = torch.empty_like(ds)
    st = torch.cuda.current_stream().cuda_stream
    sp.spin_dmc_forward(B, L, dtype, ds.data_ptr(), dJh.data_ptr(), dJv.data_ptr(), h, beta, alpha, seed, n_sweeps,
                        sweep_offset=sweep_offset, replica_offset=replica_offset, s_out_ptr=out.data_ptr(),
                        traj_ptr=traj.data_ptr(), cuda_stream=st)
    res = {"traj": traj.cpu().numpy(), "out": out.cpu().numpy()}
    if grad_out_fn is not None:
        go = _dev(grad_out_fn(res["out"]).astype(s.dtype))
        gs, gjh, gjv = torch.empty_like(ds), torch.empty_like(ds), torch.empty_like(ds)
        gb, gh = sp.spin_dmc_backward(B, L, dtype, traj.data_ptr(), dJh.data_ptr(), dJv.data_ptr(), h, beta, alpha, seed,
                                      n_sweeps, go.data_ptr(), gs.data_ptr(), gjh.data_ptr(), gjv.data_ptr(),
                                      sweep_offset=sweep_offset, replica_offset=replica_offset, cuda_stream=st)
        res.update(gs=gs.cpu().numpy(), gjh=gjh.cpu().numpy(), gjv=gjv.cpu().numpy(), gb=gb, gh=gh)
    return res


def _run_oracle(s, Jh, Jv, h, beta, alpha, seed, n_sweeps, grad_out_fn=None, replica_offset=0, sweep_offset=0):
    x = s.astype(np.float64)
    traj = oracle.dmc_forward(x, Jh.astype(np.float64), Jv.astype(np.float64), h, beta, alpha, seed, n_sweeps,
                              sweep_offset=sweep_offset, replica_offset=replica_offset, want_traj=True)
    res = {"traj": traj, "out": x}
    if grad_out_fn is not None:
        gs, gjh, gjv, gb, gh = oracle.dmc_backward(traj, Jh.astype(np.float64), Jv.astype(np.float64), h, beta, alpha, seed,
                                                   grad_out_fn(x), sweep_offset=sweep_offset, replica_offset=replica_offset)
        res.update(gs=gs, gjh=gjh, gjv=gjv, gb=gb, gh=gh)
    return res


@pytest.mark.parametrize("L", [2, 4, 6, 32, 50, 256])
def test_fp64_kernel_equals_oracle(L):
    B, seed, h, alpha, n = 3, 17, 0.1, 6.0, 2
    s, Jh, Jv, beta = _inputs(B, L, L, sp.SPIN_DTYPE_F64)
    target = np.sign(np.random.default_rng(1).normal(size=s.shape))
    gfn = lambda x: 2.0 * (x - target)                                             # Eq. 8
    g = _run_gpu(sp.SPIN_DTYPE_F64, s, Jh, Jv, h, beta, alpha, seed, n, gfn, replica_offset=5, sweep_offset=(1 << 32) + 3)
    o = _run_oracle(s, Jh, Jv, h, beta, alpha, seed, n, gfn, replica_offset=5, sweep_offset=(1 << 32) + 3)
    assert np.array_equal(g["traj"][0], s) and np.array_equal(g["traj"][-1], g["out"])
    for k in range(1, 2 * n + 1):
        assert np.max(np.abs(g["traj"][k] - o["traj"][k])) <= 1e-12 * 4 ** k, k
    for key in ("gs", "gjh", "gjv", "gb", "gh"):
        scale = max(1.0, np.max(np.abs(o[key])))
        assert np.max(np.abs(g[key] - o[key])) <= 1e-10 * scale, key


@pytest.mark.parametrize("L,glass", [(4, True), (32, True), (50, True), (256, False), (1024, True)])
def test_fp32_kernel_within_tolerance_of_oracle(L, glass):
    B, seed, h, alpha, n = 2, 23, 0.05, 6.0, 2
    s, Jh, Jv, beta = _inputs(B, L, 100 + L, sp.SPIN_DTYPE_F32, glass)
    target = np.sign(np.random.default_rng(2).normal(size=s.shape))
    gfn = lambda x: 2.0 * (x - target)
    g = _run_gpu(sp.SPIN_DTYPE_F32, s, Jh, Jv, h, beta, alpha, seed, n, gfn)
    o = _run_oracle(s, Jh, Jv, h, beta, alpha, seed, n, gfn)
    err = [float(np.max(np.abs(g["traj"][k] - o["traj"][k]))) for k in range(2 * n + 1)]
    assert err[0] == 0.0 and max(err) <= 2e-5, err
    for key in ("gs", "gjh", "gjv", "gb", "gh"):
        scale = max(1.0, np.max(np.abs(o[key])))
        assert np.max(np.abs(g[key] - o[key])) <= 2e-3 * scale, (key, np.max(np.abs(g[key] - o[key])), scale)


def test_without_trajectory_and_in_place_give_the_same_final_lattice():
    B, L, seed = 2, 64, 3
    s, Jh, Jv, beta = _inputs(B, L, 7, sp.SPIN_DTYPE_F32)
    ref = _run_gpu(sp.SPIN_DTYPE_F32, s, Jh, Jv, 0.0, beta, 5.0, seed, 3)["out"]
    ds, dJh, dJv = _dev(s), _dev(Jh), _dev(Jv)
    sp.spin_dmc_forward(B, L, sp.SPIN_DTYPE_F32, ds.data_ptr(), dJh.data_ptr(), dJv.data_ptr(), 0.0, beta, 5.0, seed, 3,
                        s_out_ptr=ds.data_ptr(), cuda_stream=torch.cuda.current_stream().cuda_stream)      # in place
    assert np.array_equal(ds.cpu().numpy(), ref)
    # chunked = one call
    ds2 = _dev(s)
    for t in range(3):
        sp.spin_dmc_forward(B, L, sp.SPIN_DTYPE_F32, ds2.data_ptr(), dJh.data_ptr(), dJv.data_ptr(), 0.0, beta, 5.0, seed, 1,
                            sweep_offset=t, s_out_ptr=ds2.data_ptr(), cuda_stream=torch.cuda.current_stream().cuda_stream)
    assert np.array_equal(ds2.cpu().numpy(), ref)


@pytest.mark.parametrize("L", [8, 24, 64, 256, 1024, 2048])
def test_fused_sweep_kernel_matches_oracle_and_its_own_trajectory(L):
    """fp32 with L % 8 == 0 runs the fused two-colour sweep kernel (one launch per sweep, tiles of rows with a recomputed
    halo row): final state with and without a stored trajectory is bit-identical (odd and even sweep counts, in place),
    the stored intermediate states chain correctly, and everything stays within the fp32 tolerance of the oracle."""
    B, seed, h, alpha = 2, 41, 0.02, 6.0
    s, Jh, Jv, beta = _inputs(B, L, 300 + L, sp.SPIN_DTYPE_F32)
    st = torch.cuda.current_stream().cuda_stream
    for n in (1, 2, 3):
        g = _run_gpu(sp.SPIN_DTYPE_F32, s, Jh, Jv, h, beta, alpha, seed, n)
        ds, dJh, dJv = _dev(s), _dev(Jh), _dev(Jv)
        out = torch.empty_like(ds)
        sp.spin_dmc_forward(B, L, sp.SPIN_DTYPE_F32, ds.data_ptr(), dJh.data_ptr(), dJv.data_ptr(), h, beta, alpha, seed, n,
                            s_out_ptr=out.data_ptr(), cuda_stream=st)
        assert np.array_equal(out.cpu().numpy(), g["out"]), n
        sp.spin_dmc_forward(B, L, sp.SPIN_DTYPE_F32, ds.data_ptr(), dJh.data_ptr(), dJv.data_ptr(), h, beta, alpha, seed, n,
                            s_out_ptr=ds.data_ptr(), cuda_stream=st)
        assert np.array_equal(ds.cpu().numpy(), g["out"]), n
        if L <= 256 and n == 2:
            o = _run_oracle(s, Jh, Jv, h, beta, alpha, seed, n)
            err = [float(np.max(np.abs(g["traj"][k] - o["traj"][k]))) for k in range(2 * n + 1)]
            assert max(err) <= 2e-5, err
        # every stored state is one half-sweep of the previous one: colour c sites of state k+1 differ, the others not
        ii, jj = np.indices((L, L))
        for k in range(2 * n):
            other = ((ii + jj) & 1) != (k & 1)
            assert np.array_equal(g["traj"][k + 1][:, other], g["traj"][k][:, other]), k


def test_alpha_to_infinity_then_eq4_reproduces_the_discrete_sweep():
    """'at the limit alpha -> infinity becomes the standard Metropolis algorithm'.  fp32 kernel, +-J glass,
    against the discrete Algorithm-1 oracle (the two acceptance tests differ with probability ~2^-24 per site)."""
    B, L, seed, n = 3, 64, 31, 5
    rng = np.random.default_rng(4)
    spins = oracle.init(B, L, seed=seed)
    Jh = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    Jv = (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    beta = np.array([0.3, 0.5, 0.8])
    ds, dJh, dJv = _dev(spins.astype(np.float32)), _dev(Jh.astype(np.float32)), _dev(Jv.astype(np.float32))
    st = torch.cuda.current_stream().cuda_stream
    ref = spins.copy()
    for t in range(n):
        sp.spin_dmc_forward(B, L, sp.SPIN_DTYPE_F32, ds.data_ptr(), dJh.data_ptr(), dJv.data_ptr(), 0.05, beta, 1e12, seed, 1,
                            sweep_offset=t, s_out_ptr=ds.data_ptr(), cuda_stream=st)
        sp.spin_dmc_discretise(sp.SPIN_DTYPE_F32, ds.data_ptr(), ds.numel(), st)
        oracle.sweep_bonds(ref, Jh, Jv, beta, 1.0, 0.05, seed, 1, sweep_offset=t)
        assert np.array_equal(ds.cpu().numpy().astype(np.int8), ref), t


def test_gradients_by_finite_differences_on_the_gpu():
    """The backward kernels against central differences of the forward KERNEL (fp64), independent of the oracle."""
    B, L, seed, h, alpha, n = 2, 8, 5, 0.1, 5.0, 2
    s, Jh, Jv, beta = _inputs(B, L, 9, sp.SPIN_DTYPE_F64)
    target = np.sign(np.random.default_rng(3).normal(size=s.shape))
    gfn = lambda x: 2.0 * (x - target)
    g = _run_gpu(sp.SPIN_DTYPE_F64, s, Jh, Jv, h, beta, alpha, seed, n, gfn)

    def loss(**kw):
        a = dict(s=s, Jh=Jh, Jv=Jv, h=h, beta=beta); a.update(kw)
        out = _run_gpu(sp.SPIN_DTYPE_F64, a["s"], a["Jh"], a["Jv"], a["h"], a["beta"], alpha, seed, n)["out"]
        return float(np.sum((target - out) ** 2))

    eps, rng = 1e-6, np.random.default_rng(0)
    for name, key in (("s", "gs"), ("Jh", "gjh"), ("Jv", "gjv")):
        base = dict(s=s, Jh=Jh, Jv=Jv)[name]
        for _ in range(6):
            idx = tuple(int(rng.integers(0, m)) for m in base.shape)
            up, dn = base.copy(), base.copy()
            up[idx] += eps; dn[idx] -= eps
            num = (loss(**{name: up}) - loss(**{name: dn})) / (2 * eps)
            assert abs(num - g[key][idx]) <= 1e-6 * max(1.0, abs(num)), (name, idx)
    for b in range(B):
        up, dn = beta.copy(), beta.copy()
        up[b] += eps; dn[b] -= eps
        num = (loss(beta=up) - loss(beta=dn)) / (2 * eps)
        assert abs(num - g["gb"][b]) <= 1e-6 * max(1.0, abs(num))
    num = (loss(h=h + eps) - loss(h=h - eps)) / (2 * eps)
    assert abs(num - g["gh"].sum()) <= 1e-6 * max(1.0, abs(num))


def test_invalid_arguments_are_rejected():
    d = torch.zeros((1, 4, 4), dtype=torch.float32, device="cuda")
    p = d.data_ptr()
    for kw in (dict(L=3), dict(beta=[-1.0]), dict(alpha=-1.0), dict(dtype=7)):
        a = dict(L=4, beta=[0.5], alpha=1.0, dtype=sp.SPIN_DTYPE_F32); a.update(kw)
        with pytest.raises(sp.SpinError):
            sp.spin_dmc_forward(1, a["L"], a["dtype"], p, p, p, 0.0, a["beta"], a["alpha"], 1, 1, s_out_ptr=p)
    with pytest.raises(sp.SpinError):
        sp.spin_dmc_forward(1, 4, sp.SPIN_DTYPE_F32, p, p, p, 0.0, [0.5], 1.0, 1, 1, s_out_ptr=None)
    assert torch.count_nonzero(d).item() == 0
