#!/usr/bin/env python
"""bench.py -- throughput of the batched SRK two-phase flash on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n MIXTURES]

One "step" = one pass of the whole hot path (every SURVEY.md section-8(a) row: load, Wilson, probe,
stability SS + Newton, label, Rachford-Rice + split SS + Newton, store) over one batch of synthetic
mixtures.  Workload at N=1: BASELINE.json's 10-component CO2-rich configuration with 1,000,000
mixtures (configs[2], the one the >= 50 % roofline target is quoted on), seeded, inputs resident in HBM.
N>1 (torchrun, one rank per GPU): every rank flashes its own 1M-mixture shard (disjoint counter ranges of
the same generator), no collective on the data path -> "scaling": "weak".

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/) instead -- the only
place besides the cpu_baseline leg where this file executes anything under oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "two-phase flashes/sec (fp64, 1 B200) and % of FP64/HBM roofline"
UNIT = "flashes/s"
WORKLOADS = {
    2: "config2: 8-component n-alkane SRK flash (kij = 0), z~Dir(1), T~U[200,600]K, P~U[1,200]bar, seed 2205030902",
    4: "config4: the 10-component CO2-rich system with z~Dir(0.5), T~U[220,500]K, P~U[5,300]bar, seed 2205030904 (scaling sweep: --n 65536 .. 16777216)",
}
WORKLOAD = "config3: 10-component CO2-rich SRK flash (8 n-alkanes + CO2 + N2, kij per BASELINE.json), z=0.6*Dir(1)+0.4*e_CO2, T~U[220,500]K, P~U[5,300]bar, seed 2205030903"
# Algorithmic FP64 work per flash on this workload: thread-level predicated-on DADD + DMUL + 2*DFMA of
# all stage kernels, counted by ncu on the committed build (profiles/), per mixture.
# Per stage kernel, in flops per mixture of the batch (profiles/r01f_kernels.md; the two launches of the split kernels --
# probe-found and stability-found part -- are summed):
STAGES = ("k_init", "k2_probe", "k2_stab_ss", "k3_stab_newton", "k_stab_decide", "k2_split_ss", "k3_split_newton")
STAGE_FLOPS_PER_FLASH = {"k_init": 1.74e3, "k2_probe": 3.93e3, "k2_stab_ss": 10.85e3, "k3_stab_newton": 11.85e3,
                         "k_stab_decide": 0.69e3, "k2_split_ss": 4.93e3, "k3_split_newton": 1.86e3}
# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) per launch at N = 1e6 from the same ncu passes: whole call,
# and the dominant kernel k3_stab_newton from its `ncu --set full` capture (profiles/r01e_stab_newton_full.md)
TRAFFIC_CALL_1M = 4.507e9
TRAFFIC_STAB_NEWTON_1M = 7.65e8
FLOPS_PER_FLASH = float(os.environ.get("PTFLASH_FLOPS_PER_FLASH", sum(STAGE_FLOPS_PER_FLASH.values())))
BYTES_PER_FLASH_NC10 = 272.0   # 8(nc+2) in + 8(2nc+1)+8 out, SURVEY.md section 8(d)
FP64_PEAK_NOMINAL = 148 * 64 * 2 * 1.965e9   # SMs x DFMA lanes/clk x 2 flop x max SM clock


def _clock_sampler(path, gpu_index):
    q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    try:
        return subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "100",
                                 "-i", str(gpu_index)], stdout=open(path, "w"), stderr=subprocess.DEVNULL)
    except Exception:
        return None


def _parse_clocks(path):
    sm, mx, reasons = [], [], set()
    try:
        for line in open(path):
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
    except OSError:
        pass
    if not sm:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
    return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}


def _oracle_throughput(w, sample, threads=0):
    """Times the oracle as it stands on `sample` mixtures of workload w. Returns (flashes/s, threads used, seconds)."""
    from oracle import oracle as O
    O.build("double")
    orc = O.Oracle.from_system(w.system)
    z = np.ascontiguousarray(w.z[:, :sample]); P = w.P[:sample].copy(); T = w.T[:sample].copy()
    orc.flash(z[:, :2000], P[:2000], T[:2000], nthreads=threads)   # page in the library
    t0 = time.perf_counter()
    r = orc.flash(z, P, T, nthreads=threads)
    dt = time.perf_counter() - t0
    return sample / dt, int(r["threads"]), dt


def run_reference(args):
    """--impl reference: the CPU oracle on the box's host cores, same workload/metric (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2205_03090_b200 import workloads as W
    sample = min(args.n, args.ref_sample)
    w = W.config3(sample)
    for _ in range(min(args.warmup, 1)):
        _oracle_throughput(w, min(sample, 20000))
    vals, cores, secs = [], 1, 0.0
    for _ in range(args.steps):
        v, cores, dt = _oracle_throughput(w, sample)
        vals.append(v); secs += dt
    value = float(np.mean(vals))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "mixtures_per_step": sample, "nc": 10},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"first {sample} mixtures of the workload per step, OpenMP over mixtures"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=1_000_000, help="mixtures per GPU per step")
    ap.add_argument("--engine", type=int, default=1)
    ap.add_argument("--config", type=int, default=3, choices=[2, 3, 4],
                    help="BASELINE config to time (3 = the headline workload; 2 and 4 report throughput only: the flop count "
                         "behind the roofline fraction is config 3's)")
    ap.add_argument("--ref-sample", type=int, default=1_000_000)
    ap.add_argument("--cpu-sample", type=int, default=1_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_2205_03090_b200 import binding as B, workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    N = args.n
    w = W.CONFIGS[args.config](N, offset=rank * N)      # each rank: its own shard of the same seeded stream
    workload = WORKLOAD if args.config == 3 else WORKLOADS[args.config]
    nc = w.system.nc
    f = B.PTFlash.from_system(w.system, engine=args.engine)
    z, P, T = (torch.from_numpy(a).to(dev) for a in (w.z, w.P, w.T))
    f64 = dict(dtype=torch.float64, device=dev)
    i32 = dict(dtype=torch.int32, device=dev)
    out = dict(beta=torch.empty(N, **f64), x=torch.empty(nc, N, **f64), y=torch.empty(nc, N, **f64),
               phase=torch.empty(N, **i32), iters=torch.empty(N, **i32))

    def step():
        B.ptflash_flash(f.h, N, z, P, T, out["beta"], out["x"], out["y"], out["phase"], out["iters"])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing (inputs in HBM) ----
    for _ in range(args.warmup):
        step()
    barrier()
    clk_path = f"/tmp/ptflash_clocks_{os.getpid()}.csv"
    sampler = _clock_sampler(clk_path, local) if rank == 0 else None
    if sampler:
        time.sleep(0.25)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    # keep the sampler alive long enough to have at least a few samples under load for very short runs
    if sampler:
        t_extra = time.time()
        while ms_total < 400 and time.time() - t_extra < 0.5:
            step()
        torch.cuda.synchronize()
        sampler.terminate()
    stats = f.stats()
    # per-stage times of a few extra (untimed) calls: CUDA events recorded by the library on the call's stream between
    # the stage kernels (PTFLASH_OPT_STAGE_PROFILE) -- the live launch durations behind the dominant-kernel roofline
    stage_ms = None
    if args.engine == 1 and rank == 0:
        f.set_option("stage_profile", 1)
        acc = []
        for _ in range(5):
            step()
            acc.append(f.stage_ms()[:len(STAGES)])
        f.set_option("stage_profile", 0)
        if acc and len(acc[0]) == len(STAGES):
            stage_ms = [float(np.mean([a[i] for a in acc])) for i in range(len(STAGES))]
    t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    ms_step = ms_total / args.steps
    value = world * N / (ms_step * 1e-3)
    two_phase = float((out["phase"] == 2).double().mean().item())
    launches = int(stats["kernel_launches"]) * args.steps

    # ---- end to end: pinned host buffers -> C ABI (H2D + kernels + D2H inside the timed region) ----
    hz, hP, hT = (torch.from_numpy(a).pin_memory() for a in (w.z, w.P, w.T))
    hb = torch.empty(N, dtype=torch.float64).pin_memory()
    hx = torch.empty(nc, N, dtype=torch.float64).pin_memory()
    hy = torch.empty(nc, N, dtype=torch.float64).pin_memory()
    hph = torch.empty(N, dtype=torch.int32).pin_memory()
    hit = torch.empty(N, dtype=torch.int32).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        B.ptflash_flash_host(f.h, N, hz, hP, hT, hb, hx, hy, hph, hit)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        B.ptflash_flash_host(f.h, N, hz, hP, hT, hb, hx, hy, hph, hit)   # synchronises internally
    barrier()
    e2e_s = time.perf_counter() - t0
    te = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_value = world * N * e2e_steps / float(te.item())
    h2d = 8 * N * (nc + 2)
    d2h = 8 * N * (2 * nc + 1) + 4 * N * 2
    assert int((hph == 2).sum()) == int((out["phase"] == 2).sum().item())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline (ALU-bound: per-mixture scalar iteration, ~270 flop/B) ----
    try:
        peaks = json.load(open(ROOT / "MEASURED_PEAKS.json"))
    except Exception:
        peaks = {}
    fp64_live, _ = B.ptflash_fp64_peak(8192)
    flops_step = FLOPS_PER_FLASH * N
    achieved = flops_step / (ms_step * 1e-3) / 1e12
    peak = fp64_live / 1e12
    hbm = peaks.get("hbm_gbs", 6650.0)
    roofline = {
        "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
        "traffic": TRAFFIC_CALL_1M if (N == 1_000_000 and args.engine == 1) else None,
        "peak_source": "FP64 DFMA microbenchmark (ptflash_fp64_peak) measured live on this GPU; nominal %.1f TFLOP/s"
                       % (FP64_PEAK_NOMINAL / 1e12),
        "flops_per_flash": FLOPS_PER_FLASH,
        "hbm_frac": (BYTES_PER_FLASH_NC10 * N / (ms_step * 1e-3) / 1e9) / hbm,
        "hbm_peak_gbs": hbm, "hbm_peak_source": "MEASURED_PEAKS.json" if peaks else "fallback",
        "kernel": "all stage kernels of one ptflash_flash call (k_init .. k_split_newton)",
    }
    if args.config != 3:
        for k in ("achieved", "frac", "flops_per_flash", "traffic"):
            roofline[k] = None
        roofline["note"] = "flops per flash are counted for config 3 only"
    if stage_ms and args.config == 3:
        # the same figure per stage kernel; "dominant" = the kernel with the largest share of the step
        per = {}
        for name, ms in zip(STAGES, stage_ms):
            a = STAGE_FLOPS_PER_FLASH[name] * N / (ms * 1e-3) / 1e12 if ms > 0 else 0.0
            per[name] = {"ms": ms, "share": ms / sum(stage_ms), "achieved": a, "frac": a / peak}
        dom = max(per, key=lambda k: per[k]["ms"])
        roofline["stages"] = per
        roofline["dominant"] = dict(kernel=dom, **per[dom])
        if dom == "k3_stab_newton" and N == 1_000_000:
            roofline["dominant"]["traffic"] = TRAFFIC_STAB_NEWTON_1M

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        v, cores, dt = _oracle_throughput(w, min(N, args.cpu_sample))
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {min(N, args.cpu_sample)} mixtures of the workload, one pass, {dt:.2f} s wall, OpenMP over mixtures"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": workload, "mixtures_per_gpu_per_step": N, "nc": nc, "engine": args.engine,
                   "two_phase_fraction": two_phase,
                   "l2": ("inputs+outputs+workspace per step are %.0f MB > 126 MB L2, so every step streams from HBM" % (N * (16.0 * nc + 32 + 60.0 * nc) / 1e6)
                          if N * (16.0 * nc + 32 + 60.0 * nc) > 126e6 else
                          "working set %.0f MB fits the 126 MB L2 (small-N sweep point; no flush between steps)" % (N * (16.0 * nc + 32 + 60.0 * nc) / 1e6)),
                   "stats_last_step": stats},
        "clocks": _parse_clocks(clk_path),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "api": "ptflash_flash_host (pinned host buffers)"},
        "gpu_launches": launches,
        "roofline": roofline,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line))
    try:
        os.remove(clk_path)
    except OSError:
        pass
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
