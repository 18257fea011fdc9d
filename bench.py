#!/usr/bin/env python
"""bench.py -- HEOM RHS + RK4 throughput on B200 (BASELINE.json metric), one JSON line.

A "step" is one RK4 step of the whole hierarchy = 4 fused RHS+stage kernels (all rows of SURVEY.md
section 8(a) that recur; the hierarchy/coefficient build and heom_set_state happen once, before the
timed region).  Headline workload: BASELINE.json configs[1] (FMO-like 7 sites, K=1, D=8, 319 770
nodes, 250.7 MB per state buffer > L2).  At N = 1 the line also carries `per_config`: a short run of
the other four BASELINE configs, each with its own roofline and oracle baseline.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg2] [--impl ours|reference]

Timing: a chunk = exactly K steps between two CUDA events on the launching stream, bracketed by a
barrier + synchronize; chunks are repeated until the timed region is >= --min-seconds long (so the
clock sampler sees it and the figure is the sustained one) and the MEDIAN chunk is reported.
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
# per_config: steps per chunk of the short runs of the non-headline configs
SHORT_STEPS = {"cfg1": 1000, "cfg2": 200, "cfg3": 8, "cfg4": 50, "cfg5": 2, "absorb": 200, "twoex": 50, "mid24": 20}
SEEDS = {"cfg1": None, "cfg2": workloads.SEED_FMO, "cfg3": workloads.SEED_FMO, "cfg4": workloads.SEED_LHCII,
         "cfg5": workloads.SEED_LARGE, "absorb": workloads.SEED_FMO, "twoex": workloads.SEED_FMO, "mid24": workloads.SEED_LHCII + 7}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0}, "fallback"


def ncu_traffic(name, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch (average over the four stage launches of one RK4
    step) from the committed `ncu --set full` captures, listed with their sources in profiles/traffic.csv;
    None if the capture is of another kernel than the one this run used."""
    import csv
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(p, newline="") as f:
            for row in csv.DictReader(f):
                if row["workload"] == name and row["kernel"] == kernel:
                    return int(row["bytes_per_launch"]), row["source"]
    except (OSError, ValueError, KeyError):
        pass
    return None, None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md).  Started before the
    warm-up (nvidia-smi needs a few hundred ms to deliver its first sample); only the samples that arrived
    inside [mark_start, mark_stop] count."""
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
            self.rows.append((time.perf_counter(), [s.strip() for s in line.split(",")]))

    def window(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": ["nvidia-smi unavailable"]}
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, r in list(self.rows):
            if t < t0 or t > t1 + 0.03 or len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()


def oracle_throughput(w, target_seconds=15.0):
    """The oracle as it stands, on the host cores, on a bounded sample of the same workload.
    States up to 2 GB: a whole number of RK4 steps of the full hierarchy sized to ~target_seconds.
    Larger states (configs 3 and 5: one oracle step would take minutes and 30-90 GB of host memory):
    right-hand-side evaluations (oracle_rhs_nodes) of a seeded sample of nodes of the full hierarchy,
    i.e. node-updates without the RK4 combination."""
    from oracle.oracle import Oracle
    o = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, bath_state=w.bath_state,
               bath_states=w.bath_states)
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
    o = Oracle(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, bath_state=w.bath_state,
               bath_states=w.bath_states)
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
            "data": "synthetic", "config": config_dict(w, args.config, 1),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": o.threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "rk4_steps_per_s": steps / dt}
    print(json.dumps(line))


def config_dict(w, key, n_gpus, shard=False):
    origin = (f"BASELINE.json configs[{list(workloads.CONFIGS).index(key)}]" if key in workloads.CONFIGS
              else "two-exciton space of configs[1]'s H (29 states, P:471-481, Eq. 54; not a BASELINE config)" if key == "twoex"
              else "mid-size site-map system, configs[3]'s generator at 24 sites (not a BASELINE config)" if key == "mid24"
              else "linear-absorption variant of configs[1] (ground state + 7 sites, sigma_0(0) = mu_z|0><0|; not a BASELINE config)")
    return {"workload": f"{w.name}: {origin} "
                        f"N={w.N} K={w.K} D={w.D} T={w.T_kelvin:g}K nodes={w.nodes} dt={w.dt_fs}fs",
            "state_mb": round(w.state_bytes / 1e6, 1),
            "l2_policy": "state buffers (3 x %.0f MB in use) exceed the 126 MB L2; no flush needed" % (w.state_bytes / 1e6)
            if w.state_bytes > 130e6 else "state smaller than L2: L2 flushed by a 256 MB write between timed chunks",
            "parallelism": (f"one hierarchy sharded over {n_gpus} rank(s), halo all_to_all per stage (P:501)" if shard
                            else "single GPU" if n_gpus == 1
                            else f"{n_gpus} independent replicas (P:507), no collective"),
            "seed": SEEDS.get(key)}


def fp64_peak(local_rank):
    """Measured in this process, on this GPU (heom_probe_peak): FP64 tensor-core and FP64 FMA rates."""
    from paper_1803_03498_b200.binding import probe_peak
    dmma, dfma = probe_peak("dmma", local_rank), probe_peak("dfma", local_rank)
    return {"dmma_tflops": dmma, "dfma_tflops": dfma, "hbm_copy_gbs": probe_peak("hbm", local_rank),
            "how": "heom_probe_peak (paper_1803_03498_b200/csrc/probe.cu): register-resident mma.sync.m8n8k4.f64 / "
                   "fma.f64 chains on 4 CTAs x 8 warps per SM, best of 5 after a warm-up; 1 GiB float4 copy kernel"}


def run_config(key, args, steps, ctx, with_e2e=True, with_cpu=True, options=None):
    """Time `steps`-step chunks of workload `key`; returns the fields of its bench block (rank 0) or None."""
    import torch
    from paper_1803_03498_b200 import Heom
    from paper_1803_03498_b200 import replicas

    world, rank, local_rank, stream, sampler = ctx["world"], ctx["rank"], ctx["local_rank"], ctx["stream"], ctx["sampler"]
    w = workloads.get(key)
    shard = args.parallel == "shard"
    opts = {k: int(v) for k, v in (options or {}).items()}
    if shard:
        from paper_1803_03498_b200.sharded import ShardedHeom
        g = ShardedHeom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, rank, world, device=local_rank,
                        bath_state=w.bath_state, **opts)
    else:
        g = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D, device=local_rank, bath_state=w.bath_state,
                 bath_states=w.bath_states, **opts)
    g.bind(stream=stream)
    if w.sigma0_matrix is None and not shard:
        sigma0 = replicas.replica_sigma0(w, rank)
    elif key == "absorb" and not shard:
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
    chunk_ms, launches = [], 0
    t_region0 = time.perf_counter()
    while True:
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        replicas.barrier(world); torch.cuda.synchronize()
        n0 = g.launch_count()
        with torch.cuda.stream(stream):
            if flush is not None:
                flush.zero_()
            ev0.record(stream)
            g.rk4_steps(w.dt_fs, steps)
            ev1.record(stream)
        torch.cuda.synchronize(); replicas.barrier(world)
        launches = g.launch_count() - n0
        chunk_ms.append(replicas.max_over_ranks(ev0.elapsed_time(ev1), world))
        done = sum(chunk_ms) >= 1e3 * args.min_seconds and len(chunk_ms) >= 3
        if replicas.max_over_ranks(1.0 if done or len(chunk_ms) >= args.max_chunks else 0.0, world) > 0:
            break
    t_region1 = time.perf_counter()
    ms = float(np.median(chunk_ms))
    clocks = sampler.window(t_region0, t_region1) if sampler else None

    # one more chunk with a CUDA event pair around every launch (kept out of the timed chunks): kernel-only time
    g.set_option("timing", 1)
    g.kernel_time()
    with torch.cuda.stream(stream):
        g.rk4_steps(w.dt_fs, min(steps, 25))
    kern_ms, kern_n = g.kernel_time()
    g.set_option("timing", 0)
    pop, tr = g.populations()

    # ---------------- end to end through the C ABI with HOST buffers ---------------------
    # per step: heom_rk4_steps(dt, 1) then heom_populations -> HOST (the observable read-out of
    # every step); the region opens with heom_set_state from a HOST sigma_0.
    e2e = None
    if with_e2e:
        e_steps = steps
        replicas.barrier(world); torch.cuda.synchronize()
        t0 = time.perf_counter()
        g.set_state(sigma0)
        with torch.cuda.stream(stream):
            for _ in range(e_steps):
                g.rk4_steps(w.dt_fs, 1)
                g.populations()
        g.sync()
        e_dt = replicas.max_over_ranks(time.perf_counter() - t0, world)
        e2e = {"value": 4.0 * w.nodes * e_steps * job / e_dt, "unit": UNIT,
               "h2d_bytes_per_step": 16 * w.N * w.N / e_steps, "d2h_bytes_per_step": 8 * (w.N + 2),
               "what": "heom_set_state(HOST sigma_0) once, then per step heom_rk4_steps(dt,1) + "
                       "heom_populations -> HOST; host wall clock"}
    stability = None
    if key == "cfg3" and not shard:
        # SURVEY.md 8(c) A7 / BASELINE.md: config 3 as specified (dt = 1 fs: dt * max d_u = 2.96 is outside RK4's
        # stability region, R8) with max|sigma| per hierarchy level logged, and the stable variant
        # (dt = 0.9 fs) alongside; same kernel, same launches, same throughput -- only the growth differs
        stability = {}
        for dt in (w.dt_fs, 0.9):
            g.set_state(sigma0)
            with torch.cuda.stream(stream):
                g.rk4_steps(dt, w.steps)
            lm = g.level_max()
            pop_s, tr_s = g.populations()
            stability[f"dt={dt}fs"] = {"steps": w.steps, "max_abs_per_level": [float(f"{v:.3e}") for v in lm],
                                       "trace_minus_1": tr_s.real - 1.0, "rho11": float(pop_s[0])}
    kernel_name = g.kernel_name()
    n_owned = g.n_owned if shard else w.nodes
    g.close()
    del g, flush
    torch.cuda.empty_cache()
    if rank != 0:
        return None

    peaks, which = measured_peaks()
    value = 4.0 * w.nodes * steps * job / (ms * 1e-3)
    horner = kernel_name in ("rhs_hpipe_kernel", "rhs_hpipe_general_kernel", "rhs_large_kernel", "rhs_ket_kernel",
                             "rhs_mma_kernel", "rhs_large_herm_kernel", "rhs_mma_herm_kernel") \
        and opts.get("rk4_form", -1) != 0
    # fused classical RK4 moves 16 state sizes per step = 64 N^2 bytes per node-update; the Horner form
    # the kernels run by default (R6) moves 2 + 3 + 3 + 3 = 11 state sizes = 44 N^2 bytes per node-update
    alg_bytes_per_launch = 64.0 * w.N * w.N * n_owned
    exe_bytes_per_launch = (44.0 if horner else 64.0) * w.N * w.N * n_owned
    alg_flops_per_launch = 8.0 * w.N ** 3 * n_owned            # real H: 8 N^3 per node-update
    tiny = launches < 4 * steps
    stage_launches = 4 * steps
    avg_launch_s = ms * 1e-3 / stage_launches                    # timed region / launches (launch gaps included)
    kernel_only_s = (kern_ms / max(kern_n, 1)) * 1e-3 if not tiny else None
    note = None
    if kernel_name == "rhs_ket_kernel":
        # column-sparse state (kernels_ket.cu): one N-vector per node; Horner-form RK4 moves 11 ket sizes per step
        alg_bytes_per_launch = 64.0 * w.N * w.nodes
        exe_bytes_per_launch = 44.0 * w.N * w.nodes
        note = ("column-sparse state held as kets: 3 x %.0f MB; L2-resident where that fits 126 MB, so the "
                "HBM roofline is context, not a bound" % (16e-6 * w.N * w.nodes))
    if tiny:
        kernel_name = "rk4_tiny_kernel (all steps in one launch; time per RK4 stage)"
    achieved = alg_bytes_per_launch / avg_launch_s / 1e9
    traffic, traffic_src = ncu_traffic(w.name, kernel_name if opts.get("rk4_form", -1) != 0 else None)
    common = {"kernel": kernel_name, "avg_launch_ms": avg_launch_s * 1e3,
              "kernel_only_launch_ms": kernel_only_s * 1e3 if kernel_only_s else None,
              "launches_timed": stage_launches * len(chunk_ms), "traffic": traffic, "traffic_source": traffic_src,
              "algorithmic_bytes_per_launch": alg_bytes_per_launch,
              "executed_form_bytes_per_launch": exe_bytes_per_launch,
              "rk4_form": "horner (11 state sizes per step)" if horner else "classical (16 state sizes per step)"}
    if w.N >= 32:
        # arithmetic-bound (N/8 = 12 flop/B at N = 96): FP64 tensor-core (DMMA) roofline, peak measured in this process
        fp = ctx["fp64"]
        tf = alg_flops_per_launch / avg_launch_s / 1e12
        # Hermitian states: the kernel forms H sigma only and takes k = Z + Z^dagger (4 N^3 executed flops)
        exe_flops = alg_flops_per_launch * (0.5 if kernel_name in ("rhs_large_herm_kernel", "rhs_mma_herm_kernel") else 1.0)
        roof = {"bound": "alu", "achieved": tf, "peak": fp["dmma_tflops"], "unit": "TFLOP/s",
                "frac": tf / fp["dmma_tflops"], "peak_source": "measured: " + fp["how"],
                "dfma_peak_tflops": fp["dfma_tflops"],
                "algorithmic_flops_per_launch": alg_flops_per_launch,
                "executed_flops_per_launch": exe_flops,
                "achieved_executed": exe_flops / avg_launch_s / 1e12,
                "frac_executed": exe_flops / avg_launch_s / 1e12 / fp["dmma_tflops"],
                "definition": "achieved = SURVEY 8(d) algorithmic flops (8 N^3 per node-update, real H) / launch time; "
                              "*_executed = tensor-core flops the kernel issues (4 N^3 when the state is Hermitian)",
                "hbm_GBs_at_executed_bytes": exe_bytes_per_launch / avg_launch_s / 1e9}
    else:
        exe = exe_bytes_per_launch / avg_launch_s / 1e9
        roof = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": achieved / peaks["hbm_gbs"],
                "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({which})",
                "achieved_executed_form": exe, "frac_executed_form": exe / peaks["hbm_gbs"],
                "frac_of_nominal_8TBs": achieved / 8000.0,
                "definition": "achieved = SURVEY 8(d) algorithmic bytes (64 N^2 per node-update, fused classical RK4) / "
                              "launch time; *_executed_form = compulsory bytes of the stage form the kernel runs"}
    roof.update(common)
    if note:
        roof["note"] = note
    block = {"value": value, "unit": UNIT, "steps": steps, "chunks": len(chunk_ms),
             "chunk_ms": [round(c, 4) for c in chunk_ms], "ms_per_step": ms / steps,
             "rk4_steps_per_s": steps * job / (ms * 1e-3), "config": config_dict(w, key, world, shard),
             "roofline": roof, "gpu_launches": launches * len(chunk_ms), "clocks": clocks,
             "check": {"trace": [tr.real, tr.imag], "rho11": float(pop[0])}}
    if e2e:
        block["e2e"] = e2e
    if stability:
        block["stability"] = stability
    if with_cpu and world == 1:
        block["cpu_baseline"] = oracle_throughput(w, target_seconds=args.cpu_seconds)
    return block


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="cfg2", choices=list(workloads.CONFIGS) + list(workloads.EXTRA))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the short runs of the other BASELINE configs")
    ap.add_argument("--min-seconds", type=float, default=0.6, help="repeat the timed chunk until the region is this long")
    ap.add_argument("--max-chunks", type=int, default=200)
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="oracle sample size (headline config)")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "shard"],
                    help="N > 1: independent replicas (default, weak scaling) or ONE hierarchy sharded over the "
                         "ranks with a halo exchange per stage (strong scaling; paper_1803_03498_b200/sharded.py)")
    ap.add_argument("--option", action="append", default=[], help="name=value library option")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args, workloads.get(args.config))
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the HEOM path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    opts = dict(kv.split("=") for kv in args.option)
    sampler = ClockSampler(local_rank) if rank == 0 else None
    if sampler:
        sampler.start()
    ctx = {"world": world, "rank": rank, "local_rank": local_rank, "sampler": sampler,
           "stream": torch.cuda.Stream(device=local_rank), "fp64": fp64_peak(local_rank) if rank == 0 else None}

    head = run_config(args.config, args, args.steps, ctx, with_cpu=not args.no_cpu_baseline, options=opts)
    per = {}
    if world == 1 and not args.no_per_config and args.config == "cfg2" and args.parallel == "replicas":
        args.cpu_seconds = min(args.cpu_seconds, 5.0)
        for key in workloads.CONFIGS:
            if key == args.config:
                continue
            blk = run_config(key, args, SHORT_STEPS[key], ctx, with_cpu=not args.no_cpu_baseline, options=opts)
            per[key] = blk
    if sampler:
        sampler.stop()
    if rank == 0:
        line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
                "scaling": "strong" if args.parallel == "shard" else "weak", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic"}
        for k in ("config", "rk4_steps_per_s", "chunks", "chunk_ms", "roofline", "e2e", "gpu_launches", "clocks",
                  "check", "cpu_baseline"):
            if k in head:
                line[k] = head[k]
        line["fp64_peak"] = ctx["fp64"]
        if per:
            line["per_config"] = per
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
