#!/usr/bin/env python
"""bench.py — throughput of the checkerboard Metropolis hot path on B200 (contract in the task statement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]

A "step" is one pass of the whole hot path over one batch: the acceptance-table build for the batch's betas,
all sweeps of the configuration (colour 0 + colour 1 each) and the per-replica E / M reductions.  At N = 1 the
workload is BASELINE.json configs[1] (C2: Ising 64 x 1024^2, 2000 sweeps).  With N > 1 (torchrun) every rank
runs the same number of replicas with replica_offset = rank * batch: replicas are independent, there is no
data-path collective ("weak" scaling).  Rank 0 prints ONE JSON line.
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
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "samples": len(sm)}


def _ncu_traffic(kernel_variant, w):
    """DRAM bytes per launch of the dominant kernel from the committed `ncu --set full` capture summary
    (profiles/r1_traffic.csv: kernel variant, workload, dram read + write bytes per launch), or None."""
    p = os.path.join(ROOT, "profiles", "r1_traffic.csv")
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

    stream = torch.cuda.Stream()
    lay = sp.SPIN_LAYOUT_BITPACKED if w.layout == "bits" else sp.SPIN_LAYOUT_INT8
    model = sp.SPIN_MODEL_POTTS if w.model == "potts" else sp.SPIN_MODEL_ISING
    nbytes = sp.spin_buffer_bytes(w.batch, w.L, model, lay)
    buf = torch.empty(nbytes, dtype=torch.int8, device="cuda")
    sim = sp.spin_create_ex(w.batch, w.L, model, q_per_replica=w.q, seed=w.seed, layout=lay,
                            replica_offset=sharding.replica_offset(rank, w.batch), device_buffer=buf.data_ptr(), buffer_bytes=nbytes,
                            cuda_stream=stream.cuda_stream, keepalive=buf)
    flush = torch.empty(256 << 20, dtype=torch.int8, device="cuda")
    E_dev = torch.zeros(w.batch, dtype=torch.int64, device="cuda")
    M_dev = torch.zeros(w.batch, dtype=torch.int64, device="cuda")

    # a step = the whole hot path with inputs resident in HBM: table build + upload, all sweeps, E/M reductions
    offset = 0
    launches_per_sweep_call = None
    for _ in range(args.warmup):
        l0 = sim.spin_kernel_launches()
        sim.spin_sweep(w.beta, w.J, w.h, w.n_sweeps, offset)
        launches_per_sweep_call = sim.spin_kernel_launches() - l0      # 2 per sweep (streaming) or 1 (resident)
        sim.spin_observables_dev(E_dev.data_ptr(), M_dev.data_ptr())
        offset += w.n_sweeps
    sim.spin_synchronize()
    torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    launches0 = sim.spin_kernel_launches()
    barrier()
    torch.cuda.synchronize()
    for k in range(args.steps):
        with torch.cuda.stream(stream):
            flush.fill_(k)  # L2 flush, outside the timed interval of the step
        ev[k][0].record(stream)
        sim.spin_sweep(w.beta, w.J, w.h, w.n_sweeps, offset)
        ev[k][1].record(stream)
        sim.spin_observables_dev(E_dev.data_ptr(), M_dev.data_ptr())
        ev[k][2].record(stream)
        offset += w.n_sweeps
    sim.spin_synchronize()
    torch.cuda.synchronize()
    barrier()
    launches = sim.spin_kernel_launches() - launches0
    if rank == 0 and len(sampler.lines) < 2:
        # the timed region was shorter than the sampling period (tiny workloads): keep the same load running,
        # untimed, until the sampler has seen it
        t_end = time.perf_counter() + 0.6
        while time.perf_counter() < t_end:
            sim.spin_sweep(w.beta, w.J, w.h, w.n_sweeps, offset)
            sim.spin_synchronize()
    clocks = sampler.stop() if rank == 0 else None
    step_ms = [e[0].elapsed_time(e[2]) for e in ev]
    sweep_ms = [e[0].elapsed_time(e[1]) for e in ev]
    total_ms = sharding.max_over_ranks(sum(step_ms), device="cuda")      # the job is as slow as its slowest rank
    updates_per_step = float(w.updates) * world
    value = updates_per_step * args.steps / (total_ms * 1e6)  # flips per ns, whole job

    # ---- end to end through the C ABI with HOST buffers: set_spins (H2D of the natural lattice) + sweeps +
    # observables to host.  Timed with the host clock around synchronising calls.
    host_lat = torch.empty((w.batch, w.L, w.L), dtype=torch.int8).pin_memory()
    sim.spin_get_spins(host_lat.numpy())
    e2e_steps = max(1, min(args.steps, 3))
    sim.spin_set_spins_ptr(host_lat.data_ptr())          # one untimed end-to-end step (same shape as the timed ones)
    sim.spin_sweep(w.beta, w.J, w.h, w.n_sweeps, offset)
    sim.spin_observables()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sim.spin_set_spins_ptr(host_lat.data_ptr())
        sim.spin_sweep(w.beta, w.J, w.h, w.n_sweeps, offset)
        Eh, Mh = sim.spin_observables()
    dt = sharding.max_over_ranks(time.perf_counter() - t0, device="cuda")
    e2e_value = updates_per_step * e2e_steps / (dt * 1e9)
    h2d = int(host_lat.numel() + w.batch * 8 + w.batch * 32 * 4)
    d2h = int(2 * w.batch * 8 + 4)

    if rank == 0:
        peaks = _peaks()
        n_launch = launches_per_sweep_call or 2 * w.n_sweeps
        kern_ms = float(np.mean(sweep_ms)) / n_launch  # average launch duration incl. launch gaps
        upd_per_launch = float(w.updates) / n_launch
        ops = OPS_PER_UPDATE[w.model]
        achieved = ops * upd_per_launch / (kern_ms * 1e-3) / 1e12
        peak = INT32_LANES_PER_SM * N_SM * peaks["sm_max_mhz"] * 1e6 / 1e12
        bytes_per_site = 0.375 if w.layout == "bits" else 3.0  # per sweep, two launches
        if n_launch == 1:
            bytes_per_site = (0.25 if w.layout == "bits" else 2.0) / w.n_sweeps  # resident: one read + one write per call
        hbm_achieved = bytes_per_site * upd_per_launch / (kern_ms * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int8" if w.layout != "bits" else "u32 bit-packed", "data": "synthetic",
            "config": _config_dict(w, world),
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps},
            "gpu_launches": int(launches),
            "kernel": sim.spin_kernel_variant(),
            "sweep_only_flips_per_ns": float(w.updates) / (float(np.mean(sweep_ms)) * 1e6),
            "roofline": {
                "bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tint32op/s", "frac": achieved / peak,
                "traffic": _ncu_traffic(sim.spin_kernel_variant(), w),
                "algorithmic_bytes_per_launch": bytes_per_site * upd_per_launch,
                "launches_per_step": int(n_launch),
                "kernel_avg_launch_us": kern_ms * 1e3, "ops_per_update": ops,
                "peak_source": "derived: 64 INT32 lanes/SM/clk x 148 SMs x %.0f MHz (%s sm_max_mhz); DESIGN.md section 6"
                               % (peaks["sm_max_mhz"], peaks["source"]),
                "hbm": {"achieved_gbs": hbm_achieved, "peak_gbs": peaks["hbm_gbs"], "frac": hbm_achieved / peaks["hbm_gbs"],
                        "bytes_per_site_per_sweep": bytes_per_site, "peak_source": peaks["source"]},
            },
        }
        if not args.no_cpu_baseline and world == 1:
            v, threads, sample, _ = oracle_throughput(w, 15.0)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample}
        print(json.dumps(line), flush=True)
    sim.spin_destroy()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
