#!/usr/bin/env python
"""bench.py -- HEOM RHS + RK4 throughput on B200 (BASELINE.json metric), one JSON line.

A "step" is one classical RK4 step of the whole hierarchy = 4 fused RHS+stage kernels
(all rows of SURVEY.md section 8(a) that recur; the hierarchy/coefficient build and
heom_set_state happen once, before the timed region).  Default workload: BASELINE.json
configs[1] (FMO-like 7 sites, K=1, D=8, 319 770 nodes, 250.7 MB per state buffer > L2).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg2] [--impl ours|reference]

N > 1 (torchrun): independent replicas of the same propagation (the paper's parameter-level
parallelism), no data-path collective, weak scaling; time = max over ranks.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
import workloads  # noqa: E402

METRIC = "heom_node_updates_per_s"
UNIT = "node-updates/s"


# FP64 peak of one B200: 148 SMs x 64 FP64 FMA/clk x 2 flop x 1.965 GHz (clocks.max.sm).
# MEASURED_PEAKS.json has no FP64 entry; a register-resident DMMA.8x8x4 probe on this pool measured 37.1 TFLOP/s.
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([s.strip() for s in line.split(",")])

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
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm),
                "reasons": sorted(reasons)}


def oracle_throughput(w, target_seconds=15.0):
    """The oracle as it stands, on the host cores, on a bounded sample of the same workload.
    States up to 2 GB: a whole number of RK4 steps of the full hierarchy sized to ~target_seconds.
    Larger states (configs 3 and 5: one oracle step would take minutes and 30-90 GB of host memory):
    right-hand-side evaluations (oracle_rhs_nodes) of a seeded sample of nodes of the full hierarchy,
    i.e. node-updates without the RK4 combination."""
    from oracle.oracle import Oracle
    o = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, bath_state=w.bath_state)
    o.set_state(w.sigma0())
    if w.state_bytes <= 2e9:
        t0 = time.perf_counter(); o.rk4_steps(w.dt_fs, 1); t1 = time.perf_counter() - t0
        n = int(max(1, min(w.steps, target_seconds / max(t1, 1e-6))))
        t0 = time.perf_counter(); o.rk4_steps(w.dt_fs, n); dt = time.perf_counter() - t0
        return {"value": 4.0 * w.nodes * n / dt, "unit": UNIT, "cores": o.threads, "kind": "oracle",
                "sample": f"{n} RK4 steps of the full {w.name} hierarchy ({w.nodes} nodes) after 1 warm-up step",
                "seconds": dt, "steps": n}
    rng = np.random.default_rng(7)
    probe = rng.integers(0, w.nodes, 64 * o.threads)
    t0 = time.perf_counter(); o.rhs_nodes(probe); t1 = time.perf_counter() - t0
    m = int(min(w.nodes, max(probe.size, probe.size * target_seconds / max(t1, 1e-6))))
    ids = rng.integers(0, w.nodes, m)
    t0 = time.perf_counter(); o.rhs_nodes(ids); dt = time.perf_counter() - t0
    return {"value": m / dt, "unit": UNIT, "cores": o.threads, "kind": "oracle",
            "sample": f"right-hand side of {m} seeded random nodes of the full {w.name} hierarchy ({w.nodes} nodes), "
                      f"sigma_0 = |1><1| state, no RK4 combination", "seconds": dt, "steps": 0}


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # each "step" of the reference arm is a bounded sample: one oracle RK4 step of the full hierarchy
    from oracle.oracle import Oracle
    o = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, bath_state=w.bath_state)
    o.set_state(w.sigma0())
    t0 = time.perf_counter(); o.rk4_steps(w.dt_fs, 1); t1 = time.perf_counter() - t0
    budget = 150.0
    warm = min(args.warmup, max(0, int(0.1 * budget / t1)))
    steps = max(1, min(args.steps, int(0.8 * budget / t1)))
    o.rk4_steps(w.dt_fs, warm)
    t0 = time.perf_counter(); o.rk4_steps(w.dt_fs, steps); dt = time.perf_counter() - t0
    val = 4.0 * w.nodes * steps / dt
    sample = (f"{steps} oracle RK4 steps of the full {w.name} hierarchy ({w.nodes} nodes) "
              f"after {warm + 1} warm-up steps (requested {args.steps}/{args.warmup}, bounded to ~{budget:.0f} s)")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": warm + 1, "ms_per_step": 1e3 * dt / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config_dict(w, 1),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": o.threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "rk4_steps_per_s": steps / dt}
    print(json.dumps(line))


def config_dict(w, n_gpus, shard=False):
    origin = (f"BASELINE.json configs[{list(workloads.CONFIGS).index(w.name[:4])}]" if w.name[:4] in workloads.CONFIGS
              else "linear-absorption variant of configs[1] (ground state + 7 sites, sigma_0(0) = mu_z|0><0|; not a BASELINE config)")
    return {"workload": f"{w.name}: {origin} "
                        f"N={w.N} K={w.K} D={w.D} T={w.T_kelvin:g}K nodes={w.nodes} dt={w.dt_fs}fs",
            "state_mb": round(w.state_bytes / 1e6, 1),
            "l2_policy": "state buffers (4 x %.0f MB) exceed the 126 MB L2; no flush needed" % (w.state_bytes / 1e6)
            if w.state_bytes > 130e6 else "state smaller than L2: L2 flushed by a 256 MB write between timed chunks",
            "parallelism": (f"one hierarchy sharded over {n_gpus} rank(s), halo all_to_all per stage (P:501)" if shard
                            else "single GPU" if n_gpus == 1
                            else f"{n_gpus} independent replicas (P:507), no collective"),
            "seed": workloads.SEED_FMO}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="cfg2", choices=list(workloads.CONFIGS) + list(workloads.EXTRA))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "shard"],
                    help="N > 1: independent replicas (default, weak scaling) or ONE hierarchy sharded over the "
                         "ranks with a halo exchange per stage (strong scaling; paper_1803_03498_b200/sharded.py)")
    ap.add_argument("--option", action="append", default=[], help="name=value library option")
    args = ap.parse_args()
    w = workloads.get(args.config)
    if args.impl == "reference":
        run_reference(args, w)
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_1803_03498_b200 import Heom
    from paper_1803_03498_b200 import replicas

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the HEOM path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    opts = dict(kv.split("=") for kv in args.option)
    stream = torch.cuda.Stream(device=local_rank)
    shard = args.parallel == "shard"
    if shard:
        from paper_1803_03498_b200.sharded import ShardedHeom
        g = ShardedHeom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, rank, world, device=local_rank,
                        bath_state=w.bath_state, **{k: int(v) for k, v in opts.items()})
    else:
        g = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, device=local_rank, bath_state=w.bath_state,
                 **{k: int(v) for k, v in opts.items()})
    g.bind(stream=stream)
    if w.sigma0_matrix is None and not shard:
        sigma0 = replicas.replica_sigma0(w, rank)
    elif args.config == "absorb" and not shard:
        sigma0 = workloads.absorption_fmo(p=(2 + rank) % 3).sigma0()   # replicas = polarisation directions (Eq. 55)
    else:
        sigma0 = w.sigma0()
    job = 1 if shard else world          # whole-job units: one hierarchy (shard) or one per rank (replicas)
    flush = None
    if w.state_bytes <= 130e6:
        flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=f"cuda:{local_rank}")

    # ---------------- kernel-resident timing: state already in HBM -----------------------
    g.set_state(sigma0)
    with torch.cuda.stream(stream):
        g.rk4_steps(w.dt_fs, args.warmup)
    g.sync()
    g.set_option("timing", 1)
    g.kernel_time()                      # reset the per-launch event list
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    replicas.barrier(world); torch.cuda.synchronize()
    n0 = g.launch_count()
    with torch.cuda.stream(stream):
        if flush is not None:
            flush.zero_()
        ev0.record(stream)
        g.rk4_steps(w.dt_fs, args.steps)
        ev1.record(stream)
    torch.cuda.synchronize(); replicas.barrier(world)
    launches = g.launch_count() - n0
    ms = replicas.max_over_ranks(ev0.elapsed_time(ev1), world)
    kern_ms, kern_n = g.kernel_time()
    g.set_option("timing", 0)
    clocks = sampler.stop() if rank == 0 else None
    pop, tr = g.populations()

    # ---------------- end to end through the C ABI with HOST buffers ---------------------
    # per step: heom_rk4_steps(dt, 1) then heom_populations -> HOST (the observable read-out of
    # every step); the region opens with heom_set_state from a HOST sigma_0.
    e_steps = args.steps
    replicas.barrier(world); torch.cuda.synchronize()
    t0 = time.perf_counter()
    g.set_state(sigma0)
    with torch.cuda.stream(stream):
        for _ in range(e_steps):
            g.rk4_steps(w.dt_fs, 1)
            pop_e, tr_e = g.populations()
    g.sync()
    e_dt = replicas.max_over_ranks(time.perf_counter() - t0, world)
    h2d = 16 * w.N * w.N / e_steps
    d2h = 8 * (w.N + 2)

    if rank == 0:
        peaks, which = measured_peaks()
        value = 4.0 * w.nodes * args.steps * job / (ms * 1e-3)
        launch_nodes = g.n_owned if shard else w.nodes             # shard: rank 0's owned nodes (ghost rows are overhead)
        alg_bytes_per_launch = 64.0 * w.N * w.N * launch_nodes     # 16 S per step / 4 launches
        alg_flops_per_launch = 8.0 * w.N ** 3 * launch_nodes       # real H: 8 N^3 per node-update
        avg_launch_s = (kern_ms / max(kern_n, 1)) * 1e-3
        kernel_name = g.kernel_name()
        ket_note = None
        if kernel_name == "rhs_ket_kernel":
            # column-sparse state (kernels_ket.cu): the state is one N-vector per node; Taylor-form RK4 moves
            # 3 + 4 + 4 + 3 = 14 ket sizes per step = 56 N bytes per node-update
            alg_bytes_per_launch = 56.0 * w.N * w.nodes
            ket_note = ("column-sparse state held as kets: 4 x %.0f MB; L2-resident where that fits 126 MB, so the "
                        "HBM roofline is context, not a bound" % (16e-6 * w.N * w.nodes))
        if kern_n < 4 * args.steps:
            # tiny hierarchy: the whole propagation ran in one launch (kernels_tiny.cu); quote the time of one
            # RHS evaluation + stage (a quarter of an RK4 step) so that the figures stay comparable
            avg_launch_s = kern_ms * 1e-3 / (4 * args.steps)
            kernel_name = "rk4_tiny_kernel (all steps in one launch; time per RK4 stage)"
        achieved = alg_bytes_per_launch / avg_launch_s / 1e9
        # dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full captures
        # (average over the 4 stage launches of one RK4 step), or null where no capture exists
        ncu_traffic = {"cfg2_fmo7": (964.6e6, "profiles/r1d_cfg2_hpipe.md"),
                       "cfg3_deep7": (36.6e9, "profiles/r1c_cfg3_hpipe.md"),
                       "cfg5_large96": (94.4e9, "profiles/r1c_cfg5_large.md")}.get(w.name, (None, None))
        if w.N >= 32:
            # arithmetic-bound (N/8 = 12 flop/B at N = 96): FP64 pipe (DMMA) roofline
            tf = alg_flops_per_launch / avg_launch_s / 1e12
            roof = {"bound": "alu", "achieved": tf, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                    "frac": tf / FP64_PEAK_TFLOPS, "traffic": ncu_traffic[0], "traffic_source": ncu_traffic[1],
                    "peak_source": "derived: 148 SMs x 64 FP64 FMA/clk x 2 x 1.965 GHz (DMMA probe measured 37.1)",
                    "kernel": kernel_name, "avg_launch_ms": avg_launch_s * 1e3, "launches_timed": kern_n,
                    "algorithmic_flops_per_launch": alg_flops_per_launch,
                    "algorithmic_bytes_per_launch": alg_bytes_per_launch,
                    "hbm_GBs_at_algorithmic_bytes": achieved}
        else:
            roof = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": achieved / peaks["hbm_gbs"], "traffic": ncu_traffic[0], "traffic_source": ncu_traffic[1],
                    "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({which})",
                    "kernel": kernel_name, "avg_launch_ms": avg_launch_s * 1e3,
                    "launches_timed": kern_n,
                    "algorithmic_bytes_per_launch": alg_bytes_per_launch,
                    "frac_of_nominal_8TBs": achieved / 8000.0}
        if ket_note:
            roof["note"] = ket_note
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong" if shard else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(w, world, shard),
            "rk4_steps_per_s": args.steps * job / (ms * 1e-3),
            "roofline": roof,
            "e2e": {"value": 4.0 * w.nodes * e_steps * job / e_dt, "unit": UNIT,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "what": "heom_set_state(HOST sigma_0) once, then per step heom_rk4_steps(dt,1) + "
                            "heom_populations -> HOST; host wall clock"},
            "gpu_launches": launches,
            "clocks": clocks,
            "check": {"trace": [tr.real, tr.imag], "rho11": float(pop[0])},
        }
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = oracle_throughput(w)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
