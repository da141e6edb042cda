#!/usr/bin/env python
"""bench.py -- particle pushes/sec (mover+arranger, fp64) of libpic on B200, with its HBM roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

One "step" is one pass of the whole hot path (gather, Boris update, x
advance, wall flag, per-cell histogram, scan, stable scatter + compaction, wall counters) over
every particle of the workload: one pic_push(species, 1) with arrange_every from the config.
Default workload: BASELINE.json configs[3], the 100 M-particle bandwidth-scale config the
metric's target is quoted on (3.6 GB of fp64 SoA per buffer set, far above the 126 MB L2, so
no L2 flush is needed between steps).  Inputs are seeded and synthetic (workloads.py).

N > 1: the path is single-GPU by BASELINE.json; ranks run independent replicas of the workload
("replicas only"), no data-path collective; value = sum of the ranks'
pushes / max-over-ranks device time.

Prints ONE JSON line (rank 0).  `value`: inputs resident in HBM, CUDA-event timed on the
library's stream.  `e2e`: the same metric through the C-ABI call pic_run_host with HOST
(pinned) buffers, H2D + the config's full step count + D2H inside the timed region.
`roofline`: the dominant kernel's algorithmic bytes / its mean launch duration measured with
CUDA events inside the timed region (pic_kernel_time), against MEASURED_PEAKS.json.
`cpu_baseline`: the CPU oracle (oracle/, as it stands) on the full-size workload for a reduced step
count: single thread (the authority), and `threaded`: its bit-identical OpenMP twin on all host cores.
`per_config` (default at --config 4 on one GPU; --no-per-config skips it): value, ms per step, dominant kernel and its
roofline fraction for the other four configs, each measured by this script in a subprocess (10 timed steps).
`fused_path`: how many timed steps took the fused kernel / were redone by the split kernels; a
decline inside the timed region marks the line "invalid" and the exit code is 3.

--impl reference: there is no reference implementation to install (the paper ships no code);
per the task contract this arm times the CPU oracle (threaded twin, all host cores) on the full-size
workload for a bounded number of steps.
"""
import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle pushes/sec (mover+arranger, fp64, 1 B200) and % of HBM peak"
UNIT = "pushes/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback

# Algorithmic bytes per particle per launch: what the step must move.
#   mover   : read x,vx,vy,vz (32) [+ cell (4) when flagged-dead particles may be present], write all five (36)
#   scatter : read all five (36), write all five (36)
#   fused   : read x,vx,vy,vz (32), write all five (36)
ALG_BYTES = {"mover": (68, 72), "scatter": (72, 72), "fused": (68, 68), "hist": (4, 4)}
DEPOSIT_BYTES = 8  # pic_deposit reads x only


def env_rank():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def committed_traffic(kernel, workload):
    """DRAM bytes per launch from the committed ncu --set full capture (profiles/traffic.json), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            t = json.load(f)
        return t.get(workload, {}).get(kernel)
    except Exception:
        return None


class ClockSampler(threading.Thread):
    """Samples SM clock / throttle reasons of one GPU through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, uuid, period=0.004):
        super().__init__(daemon=True)
        self.period, self.samples, self.reasons, self.power = period, [], set(), []
        self.stop_flag = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode() if isinstance(uuid, str) else uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # NVML missing: report that rather than invent clocks
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self.stop_flag.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(self.period)

    def result(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "note": "NVML unavailable: " + getattr(self, "err", "no samples")}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples), "power_w_max": max(self.power) if self.power else None}


# ----------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline of the main line; the whole of --impl reference)
# ----------------------------------------------------------------------------------------------
def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_run(inp, steps, threads):
    """Time `steps` steps of the oracle, as it stands, on the FULL workload `inp` (every species): threads=None is
    oracle/oracle.c (single thread, the authority), threads=0 its threaded twin oracle/oracle_omp.c on all host
    cores (pinned bit-identical to it by tests/test_oracle_omp.py).  Returns (pushes/s, seconds, pushes, cores)."""
    import oracle
    states = []
    for s in inp["species"]:
        states.append(oracle.State(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], nc=inp["nc"], dx=inp["dx"], dt=inp["dt"],
                                   boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"],
                                   arrange_every=inp["arrange_every"], threads=threads))
    oracle.lib()
    cores = 1 if threads is None else oracle.omp_max_threads()
    t0 = time.perf_counter()
    pushes = 0
    for _ in range(steps):
        for st in states:
            pushes += st.n
            st.push(1)
    dt = time.perf_counter() - t0
    return pushes / dt, dt, pushes, cores


# oracle steps timed by the cpu_baseline leg: the full-size workload with a reduced step count (SURVEY.md section
# 8(d): ">= 5 steps"; config 5 takes 10 so that one arrange is inside); configs 1 and 2 run their whole step count
CPU_STEPS = {1: 200, 2: 100, 3: 5, 4: 5, 5: 10}


def sample_text(config, inp, steps, what):
    n0 = sum(len(s["x"]) for s in inp["species"])
    return (f"BASELINE.json configs[{config - 1}] at full size ({n0} particles, {inp['nc']} cells, all species), "
            f"{steps} of its {inp['steps']} steps, arrange every {inp['arrange_every']}, {what}")


def cpu_baseline_block(config, inp):
    steps = min(CPU_STEPS[config], inp["steps"])
    v1, dt1, _, _ = oracle_run(inp, steps, None)
    vt, dtt, _, cores = oracle_run(inp, steps, 0)
    return {"value": v1, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt1,
            "sample": sample_text(config, inp, steps, "oracle/oracle.c single thread"),
            "threaded": {"value": vt, "unit": UNIT, "cores": cores, "kind": "oracle (threaded twin, bit-identical)",
                         "seconds": dtt, "cpu_model": cpu_model(),
                         "sample": sample_text(config, inp, steps, f"oracle/oracle_omp.c on {cores} threads")},
            "host_cores_available": os.cpu_count(), "same_config": True}


def run_reference(args, rank):
    """--impl reference: no reference code exists (the paper ships none); per the task contract this arm is the CPU
    oracle on the host cores: its threaded twin on all cores, on the full-size workload, for a bounded step count."""
    if rank != 0:
        return 0
    from paper_2603_24508_b200 import workloads
    kw = {}
    if args.scale != 1.0:
        kw["nc"] = max(8, int(workloads.CONFIGS[args.config]["nc"] * args.scale))
    inp = workloads.make(args.config, **kw)
    n0 = sum(len(s["x"]) for s in inp["species"])
    # each "step" of this arm = one oracle step over the whole workload; bound the CPU time to about a minute
    steps = max(1, min(args.steps, inp["steps"], int(6e9 // max(n0, 1)) or 1))
    for _ in range(max(0, min(args.warmup, 1))):
        oracle_run(workloads.make(args.config, nc=max(64, inp["nc"] // 64)), 1, 0)
    v, dt, pushes, cores = oracle_run(inp, steps, 0)
    desc = sample_text(args.config, inp, steps, f"oracle/oracle_omp.c on {cores} threads")
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args.config, inp),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle (threaded twin, bit-identical)",
                             "sample": desc, "cpu_model": cpu_model(), "same_config": True},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0,
            "note": "no reference code exists (paper only): this arm is the CPU oracle on the host cores"}
    if args.scale != 1.0:
        line["config"]["workload"] += f" SCALED x{args.scale} (debug, not a bench value)"
    print(json.dumps(line), flush=True)
    return 0


def aggregate_over_ranks(dist, seconds, pushes, device):
    """Whole-job figures of N independent replicas: (max over ranks of the time, sum over ranks of the pushes).
    dist is torch.distributed (initialised) or None for a single process.  No data-path collective exists on
    this path; this is the only exchange, and it happens outside the timed region."""
    if dist is None:
        return float(seconds), float(pushes)
    import torch
    t = torch.tensor([seconds, pushes], dtype=torch.float64, device=device)
    tmax = t.clone()
    dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(tmax[0]), float(t[1])


def workload_config(config, inp):
    from paper_2603_24508_b200 import workloads
    c = workloads.CONFIGS[config]
    out = {"workload": f"BASELINE.json configs[{config - 1}]: {c['name']}", "nc": c["nc"],
           "species": list(c["species"]), "boundary": "periodic" if c["boundary"] == 0 else "absorbing",
           "arrange_every": c["arrange_every"], "parallelism": "single GPU (replicas only for N>1)",
           "l2": "inputs (GBs of SoA) far exceed the 126 MB L2; no flush between steps"}
    if inp is not None:
        out["particles"] = int(sum(len(s["x"]) for s in inp["species"]))
    return out


def compact(line):
    r = line.get("roofline") or {}
    return {"value": line["value"], "ms_per_step": line["ms_per_step"], "kernel": r.get("kernel"), "frac": r.get("frac"),
            "step_frac": r.get("step_frac"), "kernel_ms_per_step": r.get("kernel_ms_per_step"),
            "particles": line["config"].get("particles"), "sm_mhz": (line.get("clocks") or {}).get("sm_mhz"),
            "reasons": (line.get("clocks") or {}).get("reasons"), "fused_path": line.get("fused_path"),
            "deposit_frac": (line.get("deposit") or {}).get("frac"), "invalid": line.get("invalid", False)}


def per_config_block(args, own_line):
    """The five configs in one place: this run's own, and the other four measured by this script in subprocesses
    (device-resident leg only: no e2e, no CPU baseline, no field legs), 10 timed steps after 3 warm-up steps each (config 1:
    200, its full run)."""
    import subprocess
    out = {str(args.config): compact(own_line)}
    for c in (1, 2, 3, 4, 5):
        if c == args.config:
            continue
        # config 1 is its full 200 steps: at 25 us per step ten steps are a timer-resolution measurement
        cmd = [sys.executable, os.path.abspath(__file__), "--config", str(c), "--steps", "200" if c == 1 else "10", "--warmup", "3", "--no-e2e",
               "--no-cpu", "--no-field", "--no-per-config"] + [a for o in args.option for a in ("--option", o)]
        r = subprocess.run(cmd, capture_output=True, text=True, cwd=ROOT)
        try:
            out[str(c)] = compact(json.loads(r.stdout.strip().splitlines()[-1]))
            out[str(c)]["exit_code"] = r.returncode
        except Exception as e:
            out[str(c)] = {"error": repr(e), "exit_code": r.returncode, "stderr": r.stderr[-500:]}
    return out


# ----------------------------------------------------------------------------------------------
# main arm
# ----------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the CPU-oracle baseline leg")
    ap.add_argument("--no-deposit", action="store_true", help="skip the separate timing of pic_deposit")
    ap.add_argument("--no-field", action="store_true", help="skip the separate timing of pic_solve_field and of the closed cycle")
    ap.add_argument("--all-configs", action="store_true",
                    help="append a compact per_config block: the other four configs, each run by this script in a "
                         "subprocess (the default at --config 4 on one GPU; this flag forces it for any --config)")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block")
    ap.add_argument("--option", action="append", default=[], help="pic_set_option key=value (e.g. fused=0)")
    ap.add_argument("--scale", type=float, default=1.0, help="scale nc (debug only; the line is then not a bench value)")
    ap.add_argument("--debug-fast-particle", type=float, default=None, metavar="VZ",
                    help="debug only (tests of the decline guard): give particle 7777 of species 0 the velocity (0, 0, VZ) "
                         "so that it jumps two cells after a few gyration steps and a fused step declines")
    args = ap.parse_args()
    rank, local_rank, world = env_rank()
    if args.impl == "reference":
        return run_reference(args, rank)

    import numpy as np
    import torch
    import paper_2603_24508_b200 as pic
    from paper_2603_24508_b200 import workloads
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    pic.lib()  # fails loudly if libpic.so is missing
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    warmup = max(3, args.warmup)

    kw = {}
    if args.scale != 1.0:
        kw["nc"] = max(8, int(workloads.CONFIGS[args.config]["nc"] * args.scale))
    inp = workloads.make(args.config, replica=rank, **kw)
    if args.debug_fast_particle is not None:
        s0 = inp["species"][0]
        s0["vx"][7777], s0["vy"][7777], s0["vz"][7777] = 0.0, 0.0, args.debug_fast_particle
    ae = inp["arrange_every"]
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        descs = [pic.make_species(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], qm=s["qm"], arrange_every=ae,
                                  device=dev) for s in inp["species"]]
    stream.synchronize()
    sim = pic.pic_create(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E_nodes=inp["E"],
                         B=inp["B"], species=descs, stream=stream)
    for kv in args.option:
        k, v = kv.split("=")
        pic.pic_set_option(sim, k, int(v))
    pic.pic_set_option(sim, "kernel_timing", 1)

    def step():
        pic.pic_push_all(sim, 1)  # = pic_push(sp, 1) per species; several species overlap on internal streams

    for _ in range(warmup):
        step()
    pic.pic_sync(sim)
    for k in ("mover", "hist", "scan", "scatter", "general", "fused"):
        pic.pic_kernel_time(sim, k)  # drop warm-up spans
    n_before = sum(pic.pic_n_slots(sp) for sp in sim.species)
    fused0 = [pic.pic_fused_info(sp) for sp in sim.species]
    launches0 = pic.pic_launch_count(sim)

    uuid = str(torch.cuda.get_device_properties(dev).uuid)
    sampler = ClockSampler(uuid if uuid.startswith("GPU-") else "GPU-" + uuid)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    # A fused step that declines on the device is redone by the split kernels in the next synchronising call:
    # force that call INSIDE the timed region, so that no skipped work can ever be timed as done.
    pic.pic_sync(sim)
    e1.record(stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    sampler.stop_flag.set()
    sampler.join()
    ms = e0.elapsed_time(e1)
    launches = pic.pic_launch_count(sim) - launches0
    n_after = sum(pic.pic_n_slots(sp) for sp in sim.species)
    pic.pic_sync(sim)  # raises on a deferred device-side error
    pushes = 0.5 * (n_before + n_after) * args.steps  # n_live changes only by wall absorption (negligible; exact if periodic)
    ktimes = {k: pic.pic_kernel_time(sim, k) for k in ("mover", "hist", "scan", "scatter", "general", "fused")}
    info = [pic.pic_arrange_info(sp) for sp in sim.species]
    fused1 = [pic.pic_fused_info(sp) for sp in sim.species]
    # which path the timed steps took: the fused step is expected whenever it was active at the start of the timed
    # region; every timed step must then have been one completed fused launch, none redone by the split mover
    expect_fused = all(f["active"] for f in fused0)
    fused_path = {"expected": bool(expect_fused), "fused_steps": int(ktimes["fused"][1]),
                  "split_mover_steps": int(ktimes["mover"][1]),
                  "decline_reasons_before": [f["decline_reasons"] for f in fused0],
                  "decline_reasons": [f["decline_reasons"] for f in fused1],
                  "active_after": [f["active"] for f in fused1]}
    invalid = None
    if expect_fused and (ktimes["mover"][1] != 0 or ktimes["fused"][1] != args.steps * len(sim.species)
                         or not all(f["active"] for f in fused1)
                         or any(a["decline_reasons"] != b["decline_reasons"] for a, b in zip(fused0, fused1))):
        invalid = "a fused step declined inside the timed region and was redone by the split kernels"

    ms_all, pushes_all = aggregate_over_ranks(dist, ms, pushes, dev)
    value = pushes_all / (ms_all * 1e-3)

    # roofline of the dominant kernel (this rank)
    peak, peak_src = measured_peak()
    dom = max(ktimes, key=lambda k: ktimes[k][0])
    dom_ms, dom_n = ktimes[dom]
    all_live = inp["boundary"] == workloads.PERIODIC
    per_particle = ALG_BYTES.get(dom, (72, 72))[0 if all_live else 1]
    n_per_launch = 0.5 * (n_before + n_after) / len(sim.species)
    roofline = None
    if dom_n:
        avg_ms = dom_ms / dom_n
        per_launch = n_per_launch
        concurrent = len(sim.species) > 1 and "species_streams=0" not in args.option
        if concurrent:
            # the species' launches of one step run concurrently on internal streams: their event pairs overlap, so
            # the unit is the group of launches of one step (all species' particles) and its duration the union of the
            # spans, bounded by the timed region itself
            avg_ms = min(dom_ms, ms) / args.steps
            per_launch = n_per_launch * len(sim.species)
        achieved = per_particle * per_launch / (avg_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "peak_source": peak_src, "avg_launch_ms": avg_ms,
                    "concurrent_species_launches": bool(concurrent),
                    "algorithmic_bytes_per_particle": per_particle, "particles_per_launch": per_launch,
                    "traffic": committed_traffic(dom, f"config{args.config}"),
                    "kernel_ms_per_step": {k: v[0] / args.steps for k, v in ktimes.items() if v[1]},
                    # kernels behind a fused step are guarded no-ops (they return at once): count a kernel's bytes only
                    # if its launches took at least a tenth of what those bytes cost at the peak
                    "step_algorithmic_GBps": sum(
                        ALG_BYTES[k][0 if all_live else 1] * n_per_launch * v[1] for k, v in ktimes.items()
                        if k in ALG_BYTES and v[1] and v[0] * 1e-3 / v[1] > 0.1 * ALG_BYTES[k][0] * n_per_launch / (peak * 1e9)
                    ) / (ms * 1e-3) / 1e9}
        roofline["step_frac"] = roofline["step_algorithmic_GBps"] / peak
    # the next row of the path, measured beside the step, outside its timed region:
    # charge deposition on the arranged state, 20 calls per species, device time from the library's event pairs
    deposit = None
    if ae == 1 and not args.no_deposit:
        rho = None
        for si, sp in enumerate(sim.species):  # warm-up: the first call allocates the per-cell sums
            rho = pic.pic_deposit(sp, -1.0 if si == 0 else 1.0, rho=rho, accumulate=si > 0)
        pic.pic_kernel_time(sim, "deposit")
        rho = None
        for _ in range(20):
            for si, sp in enumerate(sim.species):
                rho = pic.pic_deposit(sp, -1.0 if si == 0 else 1.0, rho=rho, accumulate=si > 0)
        dms, dn = pic.pic_kernel_time(sim, "deposit")
        if dn:
            d_ms = dms / dn
            d_gbs = DEPOSIT_BYTES * n_per_launch / (d_ms * 1e-3) / 1e9
            deposit = {"ms_per_call": d_ms, "calls": int(dn), "algorithmic_bytes_per_particle": DEPOSIT_BYTES,
                       "achieved": d_gbs, "unit": "GB/s", "frac": d_gbs / peak, "particles_per_call": n_per_launch,
                       "total_charge_check": float(rho[:-1].sum().item() if all_live else rho.sum().item())}
    # the row after that: the field solve on the device (two filter passes, Poisson,
    # E), and one whole PIC cycle with the field kept on the device: push + arrange, deposit (all species), solve
    field = None
    cycle = None
    if deposit is not None and not args.no_field:
        pic.pic_solve_field(sim, rho, smooth_passes=2)  # warm-up: the first call allocates the node scratch
        pic.pic_kernel_time(sim, "field")
        for _ in range(20):
            pic.pic_solve_field(sim, rho, smooth_passes=2)
        fms, fn = pic.pic_kernel_time(sim, "field")
        if fn:
            # algorithmic bytes of a solve: rho read once, E written once (phi is not asked for here) = 16 B per node;
            # the filter passes, the two prefix sums and the mean work on node arrays that stay in the 126 MB L2
            f_gbs = 16.0 * (inp["nc"] + 1) / (fms / fn * 1e-3) / 1e9
            field = {"ms_per_call": fms / fn, "calls": int(fn), "nodes": inp["nc"] + 1, "smooth_passes": 2,
                     "algorithmic_bytes_per_node": 16, "achieved": f_gbs, "unit": "GB/s", "frac": f_gbs / peak,
                     "note": "one cooperative kernel per solve (option field_fused=1, the default; 0 = six or seven "
                             "separate kernels); bound by its grid-wide barriers and launch latency, not by HBM: "
                             "8-24 MB of node data that stay in L2"}
        pic.pic_set_field(sim, inp["E"])  # the workload's own field again
        # macro-particle weights small enough that the self-consistent field stays of the order of the workload's own
        # (|E| <~ 0.05) even where nothing neutralises the charge (one species between absorbing walls)
        wts = [(-1.0 if s["qm"] < 0 else 1.0) * 0.1 / (max(1.0, n_per_launch / inp["nc"]) * inp["nc"] * inp["dx"])
               for s in inp["species"]]
        ncyc = 20

        def timed(fn):
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            c0.record(stream)
            fn()
            pic.pic_sync(sim)  # inside the timed region: a declined step would be redone here
            c1.record(stream)
            torch.cuda.synchronize()
            return c0.elapsed_time(c1) / ncyc

        def checked_calls():
            for _ in range(ncyc):
                r = None
                pic.pic_push_all(sim, 1)
                for si, sp in enumerate(sim.species):
                    r = pic.pic_deposit(sp, wts[si], rho=r, accumulate=si > 0)
                pic.pic_solve_field(sim, r, smooth_passes=2)

        rho_c = torch.empty(inp["nc"] + 1, dtype=torch.float64, device=dev)
        pic.pic_set_option(sim, "kernel_timing", 0)  # the cycles are timed from outside: no event pairs between their kernels
        pic.pic_cycle(sim, 2, wts, smooth_passes=2, rho=rho_c)  # warm-up
        cms = timed(lambda: pic.pic_cycle(sim, ncyc, wts, smooth_passes=2, rho=rho_c))
        cms_checked = timed(checked_calls)
        # algorithmic bytes of a cycle per particle: the fused step's 68 (read 32, write 36) + 8 for the deposition, which
        # reads x again (the node arrays add 16-40 B per NODE, i.e. < 1 % at 100 particles per cell)
        cyc_bytes = ALG_BYTES["fused"][0] if expect_fused else None
        cyc_gbs = ((cyc_bytes + DEPOSIT_BYTES) * n_per_launch * len(sim.species) / (cms * 1e-3) / 1e9) if cyc_bytes else None
        cycle = {"ms_per_cycle": cms, "cycles": ncyc, "pushes_per_s": n_per_launch * len(sim.species) / (cms * 1e-3),
                 "algorithmic_bytes_per_particle": (cyc_bytes + DEPOSIT_BYTES) if cyc_bytes else None,
                 "achieved": cyc_gbs, "unit": "GB/s", "frac": (cyc_gbs / peak) if cyc_gbs else None,
                 "what": "pic_cycle: push + arrange (all species), deposit, 2-pass filter, Poisson, E -- enqueued without a host "
                         "round trip; E never leaves the device",
                 "ms_per_cycle_checked_calls": cms_checked,
                 "checked_calls": "pic_push_all(1) + pic_deposit per species + pic_solve_field: one synchronisation per cycle",
                 "fused_declines": [pic.pic_fused_info(sp)["decline_reasons"] for sp in sim.species]}
    pic.pic_destroy(sim)
    del descs, sim
    torch.cuda.empty_cache()

    # e2e: the C-ABI call with HOST buffers (pic_run_host), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        cfg_steps = inp["steps"]
        host_species = []
        h2d = 0
        for s in inp["species"]:
            arrs = []
            for k in ("x", "vx", "vy", "vz", "cell"):
                t = torch.from_numpy(s[k]).pin_memory()
                arrs.append(t)
                h2d += t.numel() * t.element_size()
            host_species.append(dict(qm=s["qm"], arrays=arrs, arrange_every=ae))
        h2d += inp["E"].nbytes
        # three calls from the same pinned buffers (refilled outside the timed region: the call overwrites them with
        # the final state); the median is reported, all three are listed -- the first call of a process also pays the
        # one-off module load and allocator warm-up, and PCIe rates on a shared host vary from call to call
        samples = []
        for rep in range(3):
            if rep:
                for hs_, s in zip(host_species, inp["species"]):
                    for t, k in zip(hs_["arrays"], ("x", "vx", "vy", "vz", "cell")):
                        t.copy_(torch.from_numpy(s[k]))
            torch.cuda.synchronize()
            if dist is not None:
                dist.barrier()
            t0 = time.perf_counter()
            res = pic.pic_run_host(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E_nodes=inp["E"],
                                   B=inp["B"], species=host_species, nsteps=cfg_steps, stream=stream)
            torch.cuda.synchronize()
            samples.append(time.perf_counter() - t0)
        t_e2e = statistics.median(samples)
        n_out = sum(r[0] for r in res)
        d2h = n_out * 36 + 16 * len(res)
        n0_e = sum(len(s["x"]) for s in inp["species"])
        e_pushes = 0.5 * (n0_e + n_out) * cfg_steps
        t_e2e, e_pushes = aggregate_over_ranks(dist, t_e2e, e_pushes, dev)
        e2e = {"value": e_pushes / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d / cfg_steps,
               "d2h_bytes_per_step": d2h / cfg_steps, "steps": cfg_steps, "seconds": t_e2e, "seconds_all_calls": samples,
               "call": "pic_run_host (pinned host SoA in; device arena + H2D + pic_create + pic_push_all(nsteps) + D2H + "
                       "pic_destroy inside; the library keeps the arena and its small device objects for the next call "
                       "(pic_trim_memory releases them), so only the first of the 3 calls pays cudaMalloc; median of 3 calls)"}
        del host_species
        pic.pic_trim_memory()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_baseline_block(args.config, inp)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warmup,
                "ms_per_step": ms_all / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic", "config": workload_config(args.config, inp),
                "clocks": sampler.result(), "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
                "cpu_baseline": cpu, "deposit": deposit, "field_solve": field, "pic_cycle": cycle, "fused_path": fused_path,
                "path": {"arranger": ["general" if g else "fast" for (_, g) in info],
                         "options": args.option, "numpy": np.__version__}}
        if args.scale != 1.0:
            line["config"]["scaled_nc"] = inp["nc"]
            line["config"]["workload"] += f" SCALED x{args.scale} (debug, not a bench value)"
        if args.debug_fast_particle is not None:
            line["config"]["workload"] += " with an injected fast particle (debug, not a bench value)"
        # north_star asks for throughput on all five workloads: the headline run carries the other four too
        want_all = args.all_configs or (args.config == 4 and args.scale == 1.0 and args.debug_fast_particle is None)
        if want_all and not args.no_per_config and world == 1:
            line["per_config"] = per_config_block(args, line)
        if invalid:
            line["invalid"] = True
            line["invalid_reason"] = invalid
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 3 if invalid else 0


if __name__ == "__main__":
    sys.exit(main())
