#!/usr/bin/env python
"""bench.py — throughput of the checkerboard Metropolis hot path on B200 (contract in the task statement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]

A "step" is one pass of the whole hot path over one batch: the acceptance-table build for the batch's betas,
all sweeps of the configuration (colour 0 + colour 1 each) and the per-replica E / M reductions.  At N = 1 the
headline workload is BASELINE.json configs[1] (C2: Ising 64 x 1024^2, 2000 sweeps), and the same JSON line carries a
`per_config` block with every BASELINE.json configuration (C1, C2, C3 in both layouts, C4, C5 sweeps only and C5 with
moments), the paper's Table III shapes, and the differentiable-MC path, each timed the same way.  With N > 1
(torchrun) every rank runs the same number of replicas with replica_offset = rank * batch: replicas are
independent, there is no data-path collective ("weak" scaling).  Rank 0 prints ONE JSON line.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "spin flips/ns (attempted updates)"
UNIT = "flips/ns"
# Roofline denominators: algorithmic integer ops per attempted update
# ("Philox plus compare", BASELINE.json north star): 40 per Philox call shared by 4 Ising / 2 Potts sites + 1.
OPS_PER_UPDATE = {"ising": 11.0, "potts": 21.0}
# INT32 peak per the north star / BASELINE.md: 64 lanes/SM/clk x 148 SMs x max SM clock.
INT32_LANES_PER_SM = 64
N_SM = 148


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
               "samples": len(sm), "sm_mhz_min": float(min(sm))}
        try:
            pw = [float(line.split(",")[2]) for line in self.lines if len(line.split(",")) >= 7]
            out["power_w_max"] = max(pw)
        except ValueError:
            pass
        return out


def _ncu_traffic(kernel_variant, w):
    """DRAM bytes per launch of the dominant kernel from the committed `ncu --set full` capture summary
    (profiles/r2_traffic.csv: kernel variant, workload, dram read + write bytes per launch), or None."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    if not os.path.exists(p):
        return None
    for line in open(p):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 4 and f[0] == kernel_variant and f[1] == w.name:
            try:
                return float(f[2]) + float(f[3])
            except ValueError:
                return None
    return None


def _cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def oracle_throughput(w, target_seconds, max_threads=None):
    """Time the oracle, as it stands, on a bounded sample of workload w: whole replicas on separate host threads
    (the oracle itself is single-threaded; ctypes releases the GIL).  Returns (flips/ns, threads, sample text)."""
    import oracle
    oracle.build()
    threads = max(1, min(_cores(), w.batch, max_threads or 1 << 30))
    q = None if w.q is None else [int(x) for x in w.q[:threads]]

    def run(n_sweeps, lat):
        def one(b):
            qb = None if q is None else q[b]
            oracle.sweep(lat[b:b + 1], w.beta[b:b + 1], w.J, w.h, seed=w.seed, n_sweeps=n_sweeps, q=qb, replica_offset=b)
        ts = [threading.Thread(target=one, args=(b,)) for b in range(threads)]
        t0 = time.perf_counter()
        for t in ts:
            t.start()
        for t in ts:
            t.join()
        return time.perf_counter() - t0

    lat = np.concatenate([oracle.init(1, w.L, seed=w.seed, q=None if q is None else q[b], replica_offset=b)
                          for b in range(threads)])
    t1 = run(1, lat)  # calibration sweep (also warms caches)
    n = int(max(1, min(w.n_sweeps, target_seconds / max(t1, 1e-6))))
    dt = run(n, lat)
    flips = float(threads) * w.L * w.L * n
    sample = "%d replicas of %s (L=%d) x %d sweeps, one replica per host thread" % (threads, w.name, w.L, n)
    return flips / dt / 1e9, threads, sample, dt


def run_reference(args, w, rank, world):
    """--impl reference: the oracle (unmodified, host cores), same metric/config; rank 0 only."""
    if rank != 0:
        return
    vals, times = [], []
    per_step = max(2.0, min(20.0, 60.0 / max(1, args.steps + args.warmup)))
    info = None
    for i in range(args.warmup + args.steps):
        v, threads, sample, dt = oracle_throughput(w, per_step)
        info = (threads, sample)
        if i >= args.warmup:
            vals.append(v)
            times.append(dt)
    value = float(np.mean(vals))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int8", "data": "synthetic",
        "config": _config_dict(w, world, "oracle sample: " + info[1]),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": info[0], "kind": "oracle", "sample": info[1]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def _config_dict(w, world, extra=None):
    d = {"workload": "%s: %s %dx%d^2 periodic, batch %d per GPU, %d sweeps, J=%g h=%g, seed %d, layout %s" % (
        w.name, w.model, w.batch, w.L, w.batch, w.n_sweeps, w.J, w.h, w.seed, w.layout),
        "baseline_config_index": int(w.name[1:]) - 1 if w.name[1:].isdigit() else None,
        "global_batch": w.batch * world, "L": w.L, "sweeps_per_step": w.n_sweeps,
        "parallelism": "replicas sharded over %d GPU(s), no collective" % world,
        "l2": "L2 flushed (256 MiB write) between timed steps; the lattice (%.0f MiB) is re-swept %d times inside a step"
              % (w.sites * (0.125 if w.layout == "bits" else 1.0) / 2 ** 20, w.n_sweeps)}
    if extra:
        d["note"] = extra
    return d


class Runner:
    """Times one workload through the binding: device-resident steps with CUDA events on the handle's stream, then
    end-to-end steps (host lattice in, host observables out) with the host clock around synchronising calls."""

    def __init__(self, sp, torch, sharding, rank, world, local_rank):
        self.sp, self.torch, self.sharding = sp, torch, sharding
        self.rank, self.world, self.local_rank = rank, world, local_rank
        self.stream = torch.cuda.Stream()
        self.flush = torch.empty(256 << 20, dtype=torch.int8, device="cuda")

    def create(self, w, policy=None):
        sp, torch = self.sp, self.torch
        lay = sp.SPIN_LAYOUT_BITPACKED if w.layout == "bits" else sp.SPIN_LAYOUT_INT8
        model = sp.SPIN_MODEL_POTTS if w.model == "potts" else sp.SPIN_MODEL_ISING
        nbytes = sp.spin_buffer_bytes(w.batch, w.L, model, lay)
        buf = torch.empty(nbytes, dtype=torch.int8, device="cuda")
        sim = sp.spin_create_ex(w.batch, w.L, model, q_per_replica=w.q, seed=w.seed, layout=lay,
                                replica_offset=self.sharding.replica_offset(self.rank, w.batch),
                                device_buffer=buf.data_ptr(), buffer_bytes=nbytes,
                                cuda_stream=self.stream.cuda_stream, keepalive=buf)
        if policy is not None:
            sim.spin_set_policy(policy)
        return sim

    def run(self, w, mode, steps, warmup, policy=None, e2e_steps=None, barrier=lambda: None, prepare=None):
        """mode: 'sweep' (spin_sweep + spin_observables_dev), 'trace' (spin_sweep_measure with per-sweep E, M traces),
        'moments' (w.therm plain sweeps, then spin_sweep_measure with moments and no trace)."""
        torch, stream = self.torch, self.stream
        sim = self.create(w, policy)
        if prepare:
            prepare(sim)
        E_dev = torch.zeros(w.batch, dtype=torch.int64, device="cuda")
        M_dev = torch.zeros(w.batch, dtype=torch.int64, device="cuda")
        state = {"offset": 0, "per_call": None, "host_ms": []}

        def step(events=None):
            off = state["offset"]
            if events:
                events[0].record(stream)
            if mode == "sweep":
                l0 = sim.spin_kernel_launches()
                th = time.perf_counter()
                sim.spin_sweep(w.beta, w.J, w.h, w.n_sweeps, off)
                state["host_ms"].append((time.perf_counter() - th) * 1e3)     # host time to enqueue the call's launches
                state["per_call"] = sim.spin_kernel_launches() - l0
                if events:
                    events[1].record(stream)
                sim.spin_observables_dev(E_dev.data_ptr(), M_dev.data_ptr())
            elif mode == "schedule":
                l0 = sim.spin_kernel_launches()
                sim.spin_sweep_schedule(w.beta_steps, w.J, w.h, w.n_sweeps // len(w.beta_steps), off)
                state["per_call"] = sim.spin_kernel_launches() - l0
                if events:
                    events[1].record(stream)
                sim.spin_observables_dev(E_dev.data_ptr(), M_dev.data_ptr())
            elif mode == "trace":
                sim.spin_sweep_measure(w.beta, w.J, w.h, w.n_sweeps, off, trace=True)
                if events:
                    events[1].record(stream)
            else:
                mom = np.zeros((w.batch, 8), dtype=np.int64)
                if w.therm:
                    sim.spin_sweep(w.beta, w.J, w.h, w.therm, off)
                l0 = sim.spin_kernel_launches()
                sim.spin_sweep_measure(w.beta, w.J, w.h, w.n_sweeps - w.therm, off + w.therm, trace=False, moments=mom)
                state["measure_launches"] = sim.spin_kernel_launches() - l0
                if events:
                    events[1].record(stream)
            if events:
                events[2].record(stream)
            state["offset"] = off + w.n_sweeps

        for _ in range(warmup):
            step()
        sim.spin_synchronize()
        torch.cuda.synchronize()
        ev = [tuple(torch.cuda.Event(enable_timing=True) for _ in range(3)) for _ in range(steps)]
        launches0 = sim.spin_kernel_launches()
        barrier()
        torch.cuda.synchronize()
        state["host_ms"] = []
        for k in range(steps):
            with torch.cuda.stream(stream):
                self.flush.fill_(k)  # L2 flush, outside the timed interval of the step
            step(ev[k])
        sim.spin_synchronize()
        torch.cuda.synchronize()
        barrier()
        launches = sim.spin_kernel_launches() - launches0
        step_ms = [e[0].elapsed_time(e[2]) for e in ev]
        sweep_ms = [e[0].elapsed_time(e[1]) for e in ev]
        kernel = sim.spin_kernel_variant()
        if mode == "moments" and state.get("measure_launches") == 1:
            # the measured sweeps ran in one launch: the shared-memory-resident kernel with fused E / M / moments
            kernel += " (thermalisation) + ising_int8_resident (measured sweeps, reductions fused)"
        res = {"sim": sim, "step_ms": step_ms, "sweep_ms": sweep_ms, "launches": int(launches),
               "launches_per_sweep_call": state["per_call"], "kernel": kernel, "state": state,
               "host_enqueue_ms": list(state["host_ms"][:steps]),
               "step_fn": step}
        if e2e_steps:
            host_lat = torch.empty((w.batch, w.L, w.L), dtype=torch.int8).pin_memory()
            sim.spin_get_spins(host_lat.numpy())

            def e2e_step():
                sim.spin_set_spins_ptr(host_lat.data_ptr())
                if mode == "sweep":
                    sim.spin_sweep(w.beta, w.J, w.h, w.n_sweeps, state["offset"])
                    sim.spin_observables()
                else:
                    step()
            e2e_step()  # one untimed end-to-end step
            barrier()
            t0 = time.perf_counter()
            for _ in range(e2e_steps):
                e2e_step()
            dt = self.sharding.max_over_ranks(time.perf_counter() - t0, device="cuda")
            out_bytes = 2 * w.batch * 8 + 4
            if mode == "trace":
                out_bytes += 2 * w.n_sweeps * w.batch * 8
            if mode == "moments":
                out_bytes += 8 * w.batch * 8
            res["e2e"] = {"value": float(w.updates) * self.world * e2e_steps / (dt * 1e9), "unit": UNIT,
                          "h2d_bytes_per_step": int(host_lat.numel() + w.batch * 8 + w.batch * 32 * 4
                                                    + (8 * w.batch * 8 if mode == "moments" else 0)),
                          "d2h_bytes_per_step": int(out_bytes), "steps": e2e_steps}
        return res


def alu_peak(peaks):
    return INT32_LANES_PER_SM * N_SM * peaks["sm_max_mhz"] * 1e6 / 1e12


def summarise(w, res, peaks, measured_words_per_ns):
    """Per-config entry: throughput (mean, best, median over the timed steps) and the two ALU roofline fractions."""
    step_ms = np.array(res["step_ms"])
    sweep_ms = np.array(res["sweep_ms"])
    ops = OPS_PER_UPDATE[w.model]
    per_step = float(w.updates)
    vals = per_step / (step_ms * 1e6)
    sweep_rate = per_step / (float(np.mean(sweep_ms)) * 1e6)             # updates/ns over the sweep portion of the step
    frac = ops * sweep_rate * 1e9 / 1e12 / alu_peak(peaks)
    words = 1.0 if w.model == "ising" else 2.0
    d = {"workload": "%s: %s %dx%d^2, %d sweeps, layout %s" % (w.name, w.model, w.batch, w.L, w.n_sweeps, w.layout),
         "value": float(per_step * len(step_ms) / (step_ms.sum() * 1e6)), "unit": UNIT, "best": float(vals.max()),
         "median": float(np.median(vals)), "ms_per_step": float(step_ms.mean()), "kernel": res["kernel"],
         "gpu_launches_per_step": res["launches"] // len(step_ms),
         "roofline": {"bound": "alu", "frac": float(frac), "sweep_only_flips_per_ns": float(sweep_rate),
                      "frac_of_measured": (float(sweep_rate * words / measured_words_per_ns)
                                           if measured_words_per_ns else None)}}
    if "e2e" in res:
        d["e2e"] = res["e2e"]
    if res.get("host_enqueue_ms"):
        # host time of the spin_sweep call (it only enqueues): when this approaches ms_per_step the shape is bound by the
        # host's launch rate, not by the GPU
        d["host_enqueue_ms"] = float(np.mean(res["host_enqueue_ms"]))
    return d


def per_config_block(runner, sp, args, peaks, measured):
    """Every BASELINE.json configuration and the paper's Table III shapes, timed like the headline (N = 1 only)."""
    out = {}
    plan = [("C1", sp.workloads.config(1), "trace"), ("C2", sp.workloads.config(2), "sweep"),
            ("C3-bits", sp.workloads.config(3, layout="bits"), "sweep"),
            ("C3-int8", sp.workloads.config(3, layout="int8"), "sweep"),
            ("C4", sp.workloads.config(4), "sweep"), ("C5-sweep", sp.workloads.config(5), "sweep"),
            ("C5-measure", sp.workloads.config(5), "moments")]
    for key, w, mode in plan:
        if args.sweeps:
            w.n_sweeps = args.sweeps
            w.therm = min(w.therm, args.sweeps // 5)
        res = runner.run(w, mode, args.steps, args.warmup, e2e_steps=max(1, min(args.steps, 2)))
        out[key] = summarise(w, res, peaks, measured)
        out[key]["mode"] = {"sweep": "spin_sweep + spin_observables_dev", "trace": "spin_sweep_measure, E and M after every sweep",
                            "moments": "spin_sweep (thermalisation) + spin_sweep_measure with moments"}[mode]
        res["sim"].spin_destroy()
    # the paper's Table III corners: context shapes, launch/latency-bound on a B200
    paper = {"P_1x640": 0.89, "P_16x640": 1.70, "P_1x2560": 1.53, "P_16x2560": 1.71}
    for w in sp.workloads.paper_table3_shapes():
        if args.sweeps:
            w.n_sweeps = args.sweeps
        for layout in ("int8", "bits"):
            w.layout = layout
            res = runner.run(w, "sweep", args.steps, args.warmup)
            d = summarise(w, res, peaks, measured)
            d["paper_rtx3060_flips_per_ns"] = paper[w.name]
            out["%s-%s" % (w.name, layout)] = d
            res["sim"].spin_destroy()
        if w.name in ("P_1x2560", "P_16x640") and w.n_sweeps >= 64:
            # the same sweeps replayed from a CUDA graph (SPIN_POLICY_GRAPH): what it buys is host_enqueue_ms
            w.layout = "int8"
            res = runner.run(w, "sweep", args.steps, args.warmup, policy=sp.SPIN_POLICY_GRAPH)
            d = summarise(w, res, peaks, measured)
            d["mode"] = "SPIN_POLICY_GRAPH: one cudaGraphLaunch per 64 sweeps"
            out["%s-int8-graph" % w.name] = d
            res["sim"].spin_destroy()
    return out


def dmc_entries(runner, sp, args, peaks):
    """Differentiable Monte Carlo (Algorithm 2): forward only, and forward + backward (one training
    step of PAPER.md:308-332 without the optimiser), fp32, on a C2-shaped batch.  HBM-bound: the roofline is the
    algorithmic bytes per site per sweep over the measured copy bandwidth."""
    torch = runner.torch
    B, L, n_sweeps, seed, alpha, h = 64, 1024, 4, 7, 6.0, 0.0
    if args.sweeps:
        n_sweeps = max(1, min(n_sweeps, args.sweeps))
    gen = torch.Generator(device="cuda").manual_seed(seed)
    s0 = torch.rand((B, L, L), device="cuda", generator=gen) * 2 - 1
    Jh = torch.randn((B, L, L), device="cuda", generator=gen)
    Jv = torch.randn((B, L, L), device="cuda", generator=gen)
    target = torch.sign(torch.randn((B, L, L), device="cuda", generator=gen))
    beta = np.array([0.5 + 0.5 * b / (B - 1) for b in range(B)])
    out = torch.empty_like(s0)
    traj = torch.empty((2 * n_sweeps + 1, B, L, L), device="cuda")
    go, gs, gjh, gjv = (torch.empty_like(s0) for _ in range(4))
    stream = runner.stream
    F32 = sp.SPIN_DTYPE_F32

    def fwd(k):
        sp.spin_dmc_forward(B, L, F32, s0.data_ptr(), Jh.data_ptr(), Jv.data_ptr(), h, beta, alpha, seed, n_sweeps,
                            sweep_offset=k * n_sweeps, s_out_ptr=out.data_ptr(), cuda_stream=stream.cuda_stream)

    def train(k):
        sp.spin_dmc_forward(B, L, F32, s0.data_ptr(), Jh.data_ptr(), Jv.data_ptr(), h, beta, alpha, seed, n_sweeps,
                            sweep_offset=k * n_sweeps, s_out_ptr=out.data_ptr(), traj_ptr=traj.data_ptr(),
                            cuda_stream=stream.cuda_stream)
        with torch.cuda.stream(stream):
            torch.sub(out, target, out=go).mul_(2.0)                     # dLoss/ds of Eq. 8 (plumbing, not the product)
        sp.spin_dmc_backward(B, L, F32, traj.data_ptr(), Jh.data_ptr(), Jv.data_ptr(), h, beta, alpha, seed, n_sweeps,
                             go.data_ptr(), gs.data_ptr(), gjh.data_ptr(), gjv.data_ptr(), sweep_offset=k * n_sweeps,
                             cuda_stream=stream.cuda_stream, want_host=False)

    res = {}
    updates = float(B) * L * L * n_sweeps
    # algorithmic bytes per site and sweep, fp32: forward = read the lattice, write it, read both
    # coupling arrays once (16); with a stored trajectory the colour-0 state is written too (20); backward per half-sweep:
    # read s, Jh, Jv, g (16), write g_prev (4), read-modify-write dJh, dJv (16) = 36, i.e. 72 per sweep
    for key, fn, bytes_per_site_sweep, launches in (("DMC-forward", fwd, 16.0, n_sweeps),
                                                    ("DMC-forward+backward", train, 20.0 + 72.0, 3 * n_sweeps)):
        with torch.cuda.stream(stream):
            for k in range(args.warmup):
                fn(k)
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for k in range(args.steps):
            with torch.cuda.stream(stream):
                runner.flush.fill_(k)
            ev[k][0].record(stream)
            fn(args.warmup + k)
            ev[k][1].record(stream)
        torch.cuda.synchronize()
        ms = np.array([a.elapsed_time(b) for a, b in ev])
        vals = updates / (ms * 1e6)
        gbs = bytes_per_site_sweep * updates / (float(ms.mean()) * 1e-3) / 1e9
        res[key] = {"workload": "DMC: Ising +-J-glass couplings (normal), fp32, %dx%d^2, %d sweeps, alpha=%g" % (B, L, n_sweeps, alpha),
                    "value": float(updates * len(ms) / (ms.sum() * 1e6)), "unit": UNIT, "best": float(vals.max()),
                    "median": float(np.median(vals)), "ms_per_step": float(ms.mean()),
                    "kernel": "dmc_march_sweep_kernel" + ("" if key == "DMC-forward" else " + dmc_march_backward_kernel"),
                    "gpu_launches_per_step": launches, "dtype": "f32",
                    "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                 "frac": gbs / peaks["hbm_gbs"], "bytes_per_site_per_sweep": bytes_per_site_sweep,
                                 "peak_source": peaks["source"]}}
    return res


def general_entries(runner, sp, args, peaks, measured):
    """SURVEY.md 8(f) #2 shapes: real couplings + site fields (per-site thresholds, HBM-bound), the Potts field term
    (general kernel), and a +-J glass annealed by spin_sweep_schedule in one call (Fig. 9's Monte Carlo arm)."""
    from paper_2304_01772_b200.workloads import Workload
    out = {}
    n = args.sweeps or 40
    rng = np.random.default_rng(11)
    B, L = 16, 512
    w = Workload("F2-real-couplings", "ising", B, L, 8, np.full(B, 0.6), 1.0, 0.0, n)
    Jh, Jv, Bf = rng.normal(size=(B, L, L)), rng.normal(size=(B, L, L)), 0.3 * rng.normal(size=(B, L, L))
    res = runner.run(w, "sweep", args.steps, args.warmup, prepare=lambda sim: sim.spin_set_couplings(Jh, Jv, Bf))
    d = summarise(w, res, peaks, measured)
    rate = d["roofline"]["sweep_only_flips_per_ns"]
    # per site and sweep: one 4-byte threshold + the 4-byte always mask (each fetched as a 32-byte sector: 64 bytes of
    # DRAM traffic) + 3 bytes of spins
    d["kernel"] = "ising_int8_general_kernel"
    d["roofline"] = {"bound": "hbm", "achieved": 67.0 * rate, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                     "frac": 67.0 * rate / peaks["hbm_gbs"], "bytes_per_site_per_sweep": 67.0,
                     "note": "sector-granular bytes (2 x 32 B table sectors + 3 B of spins); useful bytes are 11 per site"}
    out[w.name] = d
    res["sim"].spin_destroy()
    q = np.array([3] * (B // 2) + [8] * (B // 2), dtype=np.int32)
    w = Workload("F2-potts-field", "potts", B, L, 9, np.full(B, 1.0), 1.0, 0.1, n, q=q)
    res = runner.run(w, "sweep", args.steps, args.warmup)
    d = summarise(w, res, peaks, measured)
    d["kernel"] = "potts_int8_rows_field_kernel"
    out[w.name] = d
    res["sim"].spin_destroy()
    B, L, n_steps, per = 4, 1024, 50, 4
    w = Workload("F2-anneal-schedule", "ising", B, L, 10, np.full(B, 1.0), 1.0, 0.0, n_steps * per, layout="bits")
    w.beta_steps = np.array([[0.1 + 2.9 * k / (n_steps - 1)] * B for k in range(n_steps)])
    sg = lambda: (2 * rng.integers(0, 2, size=(B, L, L)) - 1).astype(np.int8)
    Jh8, Jv8 = sg(), sg()
    res = runner.run(w, "schedule", args.steps, args.warmup, prepare=lambda sim: sim.spin_set_bonds(Jh8, Jv8))
    d = summarise(w, res, peaks, measured)
    d["mode"] = "spin_sweep_schedule: %d beta steps x %d sweeps in one call, +-J glass" % (n_steps, per)
    out[w.name] = d
    res["sim"].spin_destroy()
    return out


def _time_calls(runner, args, fn):
    """warm-up + timed steps of fn(k) on the runner's stream -> ms per step (numpy array)."""
    torch, stream = runner.torch, runner.stream
    for k in range(args.warmup):
        fn(k)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for k in range(args.steps):
        with torch.cuda.stream(stream):
            runner.flush.fill_(k)
        ev[k][0].record(stream)
        fn(args.warmup + k)
        ev[k][1].record(stream)
    torch.cuda.synchronize()
    return np.array([a.elapsed_time(b) for a, b in ev])


def _alu_entry(name, workload, updates, ms, ops, words, kernel, launches, peaks, measured):
    vals = updates / (ms * 1e6)
    rate = updates / (float(ms.mean()) * 1e6)
    return {"workload": workload, "value": float(updates * len(ms) / (ms.sum() * 1e6)), "unit": UNIT, "best": float(vals.max()),
            "median": float(np.median(vals)), "ms_per_step": float(ms.mean()), "kernel": kernel, "gpu_launches_per_step": launches,
            "roofline": {"bound": "alu", "frac": float(ops * rate * 1e9 / 1e12 / alu_peak(peaks)), "ops_per_update": ops,
                         "frac_of_measured": float(rate * words / measured) if measured else None}}


def stencil_cpm_entries(runner, sp, args, peaks, measured):
    """SURVEY.md 8(f) #4 (triangular, cubic, second-neighbour lattices) and #3 (cellular Potts, the paper's set-up)."""
    torch, stream = runner.torch, runner.stream
    out = {}
    n = args.sweeps or 20
    for key, stencil, B, L in (("F4-triangular", sp.SPIN_STENCIL_TRIANGULAR, 16, 768), ("F4-cubic", sp.SPIN_STENCIL_CUBIC, 8, 128),
                               ("F4-square-nnn", sp.SPIN_STENCIL_SQUARE_NNN, 16, 1024)):
        sites = sp.spin_stencil_sites(stencil, L)
        lat = torch.empty(B * sites, dtype=torch.int8, device="cuda")
        sp.spin_stencil_init(stencil, B, L, lat.data_ptr(), 21, cuda_stream=stream.cuda_stream)
        beta = np.full(B, 0.25 if stencil != sp.SPIN_STENCIL_SQUARE_NNN else 0.35)
        ms = _time_calls(runner, args, lambda k: sp.spin_stencil_sweep(stencil, B, L, lat.data_ptr(), beta, 1.0, 0.2, 0.0, 21, n,
                                                                       sweep_offset=k * n, cuda_stream=stream.cuda_stream))
        ncol = {sp.SPIN_STENCIL_TRIANGULAR: 3, sp.SPIN_STENCIL_CUBIC: 2, sp.SPIN_STENCIL_SQUARE_NNN: 4}[stencil]
        kern = {sp.SPIN_STENCIL_TRIANGULAR: "triangular_march_vec_kernel", sp.SPIN_STENCIL_CUBIC: "cubic_march_vec_kernel",
                sp.SPIN_STENCIL_SQUARE_NNN: "nnn_march_vec_kernel"}[stencil]
        out[key] = _alu_entry(key, "%s: Ising, batch %d, L = %d (%d sites per replica), %d sweeps" % (key, B, L, sites, n),
                              float(B) * sites * n, ms, 11.0, 1.0, kern, ncol * n, peaks, measured)
    B, L = 256, 64
    spins, tau, A = sp.workloads.cpm_initial(B, L, 6, 5, seed=5)
    lat = torch.from_numpy(spins.copy()).cuda()
    beta = np.full(B, 1.0 / 8.0)
    nc = args.sweeps or 50
    ms = _time_calls(runner, args, lambda k: sp.spin_cpm_sweep(B, L, lat.data_ptr(), tau, sp.workloads.CPM_TABLE_II, 1, A, beta, 5, nc,
                                                               sweep_offset=k * nc, cuda_stream=stream.cuda_stream))
    out["F3-cpm"] = _alu_entry("F3-cpm", "CPM: Table II, 36 cells + medium, k_B T = 8, A = 25, lambda = 1, batch %d x %d^2, %d sweeps "
                               "(copy attempts)" % (B, L, nc), float(B) * L * L * nc, ms, 21.0, 2.0,
                               "cpm_resident_kernel", 1, peaks, measured)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number 1..5 (default 2 = configs[1])")
    ap.add_argument("--layout", default=None, choices=[None, "int8", "bits"])
    ap.add_argument("--sweeps", type=int, default=None, help="override sweeps per step (diagnostics only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="headline workload only")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    import paper_2304_01772_b200 as sp
    from paper_2304_01772_b200 import sharding
    w = sp.workloads.config(args.config, layout=args.layout)
    if args.sweeps:
        w.n_sweeps = args.sweeps

    if args.impl == "reference":
        run_reference(args, w, rank, world)
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()

    runner = Runner(sp, torch, sharding, rank, world, local_rank)
    measured = sp.spin_measure_philox_compare_rate()        # stand-alone Philox + compare rate, random words per ns
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    res = runner.run(w, "sweep", args.steps, args.warmup, e2e_steps=max(1, min(args.steps, 3)), barrier=barrier)
    sim = res["sim"]
    if rank == 0 and len(sampler.lines) < 2:
        # the timed region was shorter than the sampling period (tiny workloads): keep the same load running,
        # untimed, until the sampler has seen it
        t_end = time.perf_counter() + 0.6
        while time.perf_counter() < t_end:
            sim.spin_sweep(w.beta, w.J, w.h, w.n_sweeps, res["state"]["offset"])
            sim.spin_synchronize()
    clocks = sampler.stop() if rank == 0 else None
    step_ms, sweep_ms = res["step_ms"], res["sweep_ms"]
    total_ms = sharding.max_over_ranks(sum(step_ms), device="cuda")      # the job is as slow as its slowest rank
    updates_per_step = float(w.updates) * world
    value = updates_per_step * args.steps / (total_ms * 1e6)  # flips per ns, whole job

    if rank == 0:
        peaks = _peaks()
        n_launch = res["launches_per_sweep_call"] or 2 * w.n_sweeps
        kern_ms = float(np.mean(sweep_ms)) / n_launch  # average launch duration incl. launch gaps
        upd_per_launch = float(w.updates) / n_launch
        ops = OPS_PER_UPDATE[w.model]
        achieved = ops * upd_per_launch / (kern_ms * 1e-3) / 1e12
        peak = alu_peak(peaks)
        bytes_per_site = 0.375 if w.layout == "bits" else 3.0  # per sweep, two launches
        if n_launch == 1:
            bytes_per_site = (0.25 if w.layout == "bits" else 2.0) / w.n_sweeps  # resident: one read + one write per call
        hbm_achieved = bytes_per_site * upd_per_launch / (kern_ms * 1e-3) / 1e9
        words = 1.0 if w.model == "ising" else 2.0
        measured_peak = measured * (ops / words) * 1e9 / 1e12           # Tint32op/s the stand-alone kernel sustains
        vals = float(w.updates) / (np.array(step_ms) * 1e6)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int8" if w.layout != "bits" else "u32 bit-packed", "data": "synthetic",
            "config": _config_dict(w, world),
            "clocks": clocks,
            "e2e": res["e2e"],
            "gpu_launches": res["launches"],
            "kernel": res["kernel"],
            "best": float(vals.max()), "median": float(np.median(vals)),
            "sweep_only_flips_per_ns": float(w.updates) / (float(np.mean(sweep_ms)) * 1e6),
            "roofline": {
                "bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tint32op/s", "frac": achieved / peak,
                "measured_peak": measured_peak, "frac_of_measured": achieved / measured_peak,
                "measured_peak_source": "spin_measure_philox_compare_rate(): register-only Philox-4x32-10 + 4 compares, "
                                        "%.1f random words/ns on this device in this run" % measured,
                "traffic": _ncu_traffic(res["kernel"], w),
                "algorithmic_bytes_per_launch": bytes_per_site * upd_per_launch,
                "launches_per_step": int(n_launch),
                "kernel_avg_launch_us": kern_ms * 1e3, "ops_per_update": ops,
                # > 1: the batch is swept as that many replica groups on their own streams, whose launches overlap
                # (csrc/spin_api.cu, streaming_groups): kernel_avg_launch_us is then sweep time / launches, not a duration
                "concurrent_chains": max(1, int(n_launch) // (2 * w.n_sweeps)),
                "peak_source": "derived: 64 INT32 lanes/SM/clk x 148 SMs x %.0f MHz (%s sm_max_mhz); DESIGN.md section 6"
                               % (peaks["sm_max_mhz"], peaks["source"]),
                "hbm": {"achieved_gbs": hbm_achieved, "peak_gbs": peaks["hbm_gbs"], "frac": hbm_achieved / peaks["hbm_gbs"],
                        "bytes_per_site_per_sweep": bytes_per_site, "peak_source": peaks["source"]},
            },
        }
        sim.spin_destroy()
        if world == 1 and not args.no_per_config:
            sampler2 = ClockSampler(local_rank)                 # clocks over the whole per_config part of the run
            sampler2.start()
            line["per_config"] = per_config_block(runner, sp, args, peaks, measured)
            line["per_config"].update(dmc_entries(runner, sp, args, peaks))
            line["per_config"].update(general_entries(runner, sp, args, peaks, measured))
            line["per_config"].update(stencil_cpm_entries(runner, sp, args, peaks, measured))
            line["per_config_clocks"] = sampler2.stop()
        if not args.no_cpu_baseline and world == 1:
            v, threads, sample, _ = oracle_throughput(w, 12.0)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                                    "note": "correctness oracle as it stands (one Philox call per site visit, natural "
                                            "layout, -O2): a checker, not a tuned CPU implementation"}
            v1, _, sample1, _ = oracle_throughput(w, 6.0, max_threads=1)
            line["cpu_baseline"]["single_thread"] = {"value": v1, "cores": 1, "sample": sample1}
        print(json.dumps(line), flush=True)
    else:
        sim.spin_destroy()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
