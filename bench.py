#!/usr/bin/env python
"""bench.py -- throughput of the batched SRK two-phase flash on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n MIXTURES] [--config C]
    python bench.py --ncu-summary profiles/<tag>_kernels.csv [--ncu-tag <tag>]     (no GPU needed; see ncu_summary())

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
    "2": "config2: 8-component n-alkane SRK flash (kij = 0), z~Dir(1), T~U[200,600]K, P~U[1,200]bar, seed 2205030902",
    "3": "config3: 10-component CO2-rich SRK flash (8 n-alkanes + CO2 + N2, kij per BASELINE.json), z=0.6*Dir(1)+0.4*e_CO2, T~U[220,500]K, P~U[5,300]bar, seed 2205030903",
    "4": "config4: the 10-component CO2-rich system with z~Dir(0.5), T~U[220,500]K, P~U[5,300]bar, seed 2205030904 (scaling sweep: --n 65536 .. 16777216)",
    "5": "config5: warm-started, divergence-stressed flash of the 10-component CO2-rich system: (P,T,z) within 5% of each mixture's oracle-computed phase boundary, lnK0 = oracle lnK + N(0,0.05), skip-stability flags where the oracle label is two-phase (inputs built by tests/config5.py, seed 2205030905); value = the WARM call, config.cold = the same mixtures from Wilson",
    "paper2": "paper case study 1 (PAPER.md:117): CH4/C6H14, Table 1 constants (MPa), P~U[0.1,10]MPa, T~U[200,500]K, z~Dir(1)",
    "paper4": "paper case study 2 (PAPER.md:117): CH4..n-C4H10, Table 1 constants (MPa), P~U[0.1,10]MPa, T~U[200,500]K, z~Dir(1)",
    "paper9": "paper case study 3 (PAPER.md:117, Tables 1-3): 9 components, BIP(CH4-CO2)=0.0882, P~U[5,25]MPa, T~U[200,600]K, four reservoir-fluid types by Dirichlet(alpha of Table 3) rejected into Table 2's ranges, equally represented",
}
WORKLOAD = WORKLOADS["3"]
# Algorithmic FP64 work per flash on the headline workload (config 3, N = 1e6): thread-level predicated-on
# DADD + DMUL + 2*DFMA of all stage kernels, counted by ncu on the committed build, per mixture and
# per stage kernel (the two launches of the split kernels -- probe-found and stability-found part -- are summed), and the
# DRAM bytes per launch.  They live in profiles/<tag>_flops.json, written by `bench.py --ncu-summary` from the ncu CSV of
# that build together with a hash of the kernel sources; when the sources have changed since, the line says "flops_stale".
STAGES = ("k_init", "k2_probe", "k2_stab_ss", "k3_stab_newton", "k_stab_decide", "k2_split_ss", "k3_split_newton")
FLOPS_GLOB = "r0*_flops.json"   # the profile whose source hash matches the build, else the newest by name (marked stale)
BYTES_PER_FLASH_NC10 = 272.0   # 8(nc+2) in + 8(2nc+1)+8 out, SURVEY.md section 8(d)
FP64_PEAK_NOMINAL = 148 * 64 * 2 * 1.965e9   # SMs x DFMA lanes/clk x 2 flop x max SM clock
PAPER_TABLE4 = {"two_phase_share": 0.413442, "probe_proved_share": 0.3744, "seconds_per_1e6_on_RTX3080": 3.03,
                "stability_only_seconds_per_1e6": 2.0, "cite": "PAPER.md:243, 332-345 (another machine: context only)"}


def kernel_source_hash() -> str:
    """sha256 over the kernel sources (csrc/*.cu, *.cuh, *.h and include/ptflash.h), the key of profiles/*_flops.json."""
    import hashlib
    h = hashlib.sha256()
    files = sorted((ROOT / "paper_2205_03090_b200" / "csrc").glob("*.cu*")) + sorted((ROOT / "paper_2205_03090_b200" / "csrc").glob("*.h"))
    for f in files + [ROOT / "include" / "ptflash.h"]:
        h.update(f.name.encode())
        h.update(f.read_bytes())
    return h.hexdigest()[:16]


def load_flops():
    """-> (per-stage flops per flash, total, traffic per call, traffic of the dominant kernel, stale?, source)"""
    try:
        cands = [json.load(open(f)) | {"file": f.name} for f in sorted((ROOT / "profiles").glob(FLOPS_GLOB))]
    except Exception:
        return None
    if not cands:
        return None
    h = kernel_source_hash()
    match = [c for c in cands if c.get("csrc_hash") == h]
    d = match[-1] if match else cands[-1]
    d["stale"] = d.get("csrc_hash") != h
    return d


def ncu_summary(csv_path: str, tag: str):
    """Reads the raw CSV of the ncu per-kernel metrics pass (command in profiles/<tag>_kernels.md), prints the per-kernel
    table as markdown and writes profiles/<tag>_flops.json (flops per flash and DRAM bytes per stage kernel of the LAST
    profiled ptflash_flash call, N taken from the k_init grid's work) keyed by the hash of the kernel sources."""
    import collections
    import csv
    lines = open(csv_path).read().splitlines(keepends=True)
    start = next(i for i, l in enumerate(lines) if l.startswith('"ID"'))
    data = collections.OrderedDict()
    for r in csv.DictReader(lines[start:]):
        key = (int(r["ID"]), r["Kernel Name"].split("(")[0].split("<")[0].replace("void ", "").replace("ptf::", ""))
        v = r["Metric Value"].replace(",", "")
        try:
            v = float(v)
        except ValueError:
            pass
        data.setdefault(key, {})[r["Metric Name"]] = (v, r["Metric Unit"])
    first = max(i for (i, name) in data if name == "k_init")
    scale = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ms": 1e6, "msecond": 1e6, "us": 1e3, "usecond": 1e3, "second": 1e9}

    def g(m, k):
        if k not in m:
            return 0.0
        v, u = m[k]
        return v * scale.get(u, 1.0) if isinstance(v, float) else 0.0
    rows, cnt = [], collections.Counter()
    for (i, name), m in data.items():
        if i < first or name.startswith("at::") or "dfma_peak" in name:
            continue
        cnt[name] += 1
        fl = (g(m, "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum") + g(m, "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum")
              + 2 * g(m, "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum"))
        rows.append(dict(name=name, label=name if cnt[name] == 1 else f"{name} #{cnt[name]}", us=g(m, "gpu__time_duration.sum") / 1e3,
                         flops=fl, lanes=g(m, "smsp__thread_inst_executed_per_inst_executed.ratio"),
                         regs=g(m, "launch__registers_per_thread"), pipe=g(m, "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"),
                         warps=g(m, "sm__warps_active.avg.pct_of_peak_sustained_active"),
                         dr=g(m, "dram__bytes_read.sum"), dw=g(m, "dram__bytes_write.sum"),
                         ll=g(m, "l1tex__t_bytes_pipe_lsu_mem_local_op_ld.sum"), ls=g(m, "l1tex__t_bytes_pipe_lsu_mem_local_op_st.sum"),
                         inst=g(m, "smsp__inst_executed.sum")))
    print("| kernel | time us | lanes/32 | regs | GFLOP | TFLOP/s | fp64 pipe % | warps act % | dram MB r/w | local MB ld/st | inst M |")
    print("|---|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|")
    for r in rows:
        print(f"| {r['label']} | {r['us']:.0f} | {r['lanes']:.1f} | {r['regs']:.0f} | {r['flops'] / 1e9:.2f} | "
              f"{r['flops'] / r['us'] / 1e6 if r['us'] else 0:.2f} | {r['pipe']:.1f} | {r['warps']:.1f} | {r['dr'] / 1e6:.0f} / {r['dw'] / 1e6:.0f} | "
              f"{r['ll'] / 1e6:.0f} / {r['ls'] / 1e6:.0f} | {r['inst'] / 1e6:.0f} |")
    tot_us, tot_fl = sum(r["us"] for r in rows), sum(r["flops"] for r in rows)
    print(f"| total | {tot_us:.0f} | | | {tot_fl / 1e9:.2f} | {tot_fl / tot_us / 1e6:.2f} | | | {sum(r['dr'] for r in rows) / 1e6:.0f} / {sum(r['dw'] for r in rows) / 1e6:.0f} | | |")
    N = 1_000_000
    stage = {k: 0.0 for k in STAGES}
    traffic = {k: 0.0 for k in STAGES}
    for r in rows:
        if r["name"] in stage:
            stage[r["name"]] += r["flops"] / N
            traffic[r["name"]] += r["dr"] + r["dw"]
    out = {"tag": tag, "csv": os.path.basename(csv_path), "workload": "config3, N = 1000000 (bench.py --steps 1 --warmup 3 --no-cpu-baseline under ncu)",
           "csrc_hash": kernel_source_hash(), "stage_flops_per_flash": stage, "flops_per_flash": sum(stage.values()),
           "traffic_call_bytes": sum(r["dr"] + r["dw"] for r in rows), "stage_traffic_bytes": traffic,
           "launch_us_serialised": {r["label"]: r["us"] for r in rows}}
    path = ROOT / "profiles" / f"{tag}_flops.json"
    json.dump(out, open(path, "w"), indent=1)
    print(f"\nwrote {path}: {out['flops_per_flash']:.0f} flops per flash, {out['traffic_call_bytes'] / 1e9:.3f} GB per call, csrc hash {out['csrc_hash']}")


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


def _oracle_throughput(w, sample, threads=0, **kw):
    """Times the oracle as it stands on `sample` mixtures of workload w. Returns (flashes/s, threads used, seconds)."""
    from oracle import oracle as O
    O.build("double")
    orc = O.Oracle.from_system(w.system)
    z = np.ascontiguousarray(w.z[:, :sample]); P = w.P[:sample].copy(); T = w.T[:sample].copy()
    orc.flash(z[:, :2000], P[:2000], T[:2000], nthreads=threads)   # page in the library
    t0 = time.perf_counter()
    r = orc.flash(z, P, T, nthreads=threads, **kw)
    dt = time.perf_counter() - t0
    return sample / dt, int(r["threads"]), dt


def _load_workload(name: str, N: int, offset: int = 0):
    """-> (Workload, lnK0 or None, flags or None).  Config 5's inputs are DEFINED through the oracle (BASELINE.json: the
    oracle-computed phase boundary and converged ln K), so they are built by the test-side script tests/config5.py in a
    separate process and cached as a file of inputs only; this process never imports oracle/ for it."""
    from paper_2205_03090_b200 import workloads as W
    if name != "5":
        key = int(name) if name.isdigit() else name
        return W.CONFIGS[key](N, offset=offset), None, None
    import tempfile
    path = Path(tempfile.gettempdir()) / f"ptflash_config5_inputs_{N}.npz"
    if not path.exists():
        subprocess.run([sys.executable, str(ROOT / "tests" / "config5.py"), str(N), str(path)], check=True)
    d = np.load(path)
    w = W.Workload("config5_warm_near_boundary_10", W.system_co2_10(), d["P"], d["T"], np.ascontiguousarray(d["z"]), {})
    return w, np.ascontiguousarray(d["lnK0"]), np.ascontiguousarray(d["flags"])


def run_reference(args):
    """--impl reference: the CPU oracle on the box's host cores, same workload/metric (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sample = min(args.n, args.ref_sample)
    w, lnK0, flags = _load_workload(args.config, sample)
    kw = {} if lnK0 is None else dict(lnK0=lnK0, flags=flags)
    for _ in range(min(args.warmup, 1)):
        _oracle_throughput(w, min(sample, 20000))
    vals, cores, secs = [], 1, 0.0
    for _ in range(args.steps):
        v, cores, dt = _oracle_throughput(w, sample, **kw)
        vals.append(v); secs += dt
    value = float(np.mean(vals))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config], "mixtures_per_step": sample, "nc": w.system.nc},
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
    ap.add_argument("--n", "--mixtures", dest="n", type=int, default=1_000_000,
                    help="mixtures per GPU per step (under torchrun use --mixtures: its own parser claims the prefix --n)")
    ap.add_argument("--engine", type=int, default=1)
    ap.add_argument("--config", default="3", choices=sorted(WORKLOADS),
                    help="workload to time (3 = the headline: BASELINE.json configs[2]; the others report throughput only: "
                         "the flop count behind the roofline fraction is config 3's)")
    ap.add_argument("--ref-sample", type=int, default=1_000_000)
    ap.add_argument("--cpu-sample", type=int, default=1_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="library option for this run (binding.OPTIONS, e.g. early_split_ss=1); recorded in config.options")
    ap.add_argument("--ncu-summary", default="", help="raw CSV of the ncu per-kernel pass -> markdown table + profiles/<tag>_flops.json")
    ap.add_argument("--ncu-tag", default="r03")
    args = ap.parse_args()
    if args.ncu_summary:
        return ncu_summary(args.ncu_summary, args.ncu_tag)
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_2205_03090_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    # the process group exists whenever a launcher set one up (torchrun exports MASTER_PORT), also for a single rank: the same
    # NCCL init, barrier and max-over-ranks reduction then run at N = 1 as at N = 8, so that path is exercised on a 1-GPU box
    use_dist = world > 1 or ("MASTER_PORT" in os.environ and "RANK" in os.environ)
    if use_dist:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        try:
            dist.init_process_group("nccl", device_id=dev)
        except Exception:
            if world > 1:
                raise
            use_dist = False      # a single rank needs no group: leftover MASTER_* variables must not stop the N = 1 run

    N = args.n
    headline = args.config == "3"
    w, lnK0, flags = _load_workload(args.config, N, offset=rank * N)      # each rank: its own shard of the same seeded stream
    workload = WORKLOADS[args.config]
    nc = w.system.nc
    f = B.PTFlash.from_system(w.system, engine=args.engine)
    user_opts = {kv.split("=", 1)[0]: float(kv.split("=", 1)[1]) for kv in args.opt}
    for k, v in user_opts.items():
        f.set_option(k, v)
    z, P, T = (torch.from_numpy(a).to(dev) for a in (w.z, w.P, w.T))
    f64 = dict(dtype=torch.float64, device=dev)
    i32 = dict(dtype=torch.int32, device=dev)
    out = dict(beta=torch.empty(N, **f64), x=torch.empty(nc, N, **f64), y=torch.empty(nc, N, **f64),
               phase=torch.empty(N, **i32), iters=torch.empty(N, **i32))
    warm = lnK0 is not None
    if warm:
        d_l0, d_fl = torch.from_numpy(lnK0).to(dev), torch.from_numpy(flags).to(dev)
        out["status"] = torch.empty(N, **i32)

    def step(cold=False):
        if warm and not cold:
            B.ptflash_flash_ex(f.h, N, z, P, T, out["beta"], out["x"], out["y"], out["phase"], out["iters"],
                               lnK0=d_l0, flags=d_fl, out_status=out["status"])
        else:
            B.ptflash_flash(f.h, N, z, P, T, out["beta"], out["x"], out["y"], out["phase"], out["iters"])

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        barrier()
        return e0.elapsed_time(e1)

    # ---- device-resident timing (inputs in HBM) ----
    for _ in range(args.warmup):
        step()
    barrier()
    clk_path = f"/tmp/ptflash_clocks_{os.getpid()}.csv"
    sampler = _clock_sampler(clk_path, local) if rank == 0 else None
    if sampler:
        time.sleep(0.25)
    ms_total = timed(step, args.steps)
    # keep the sampler alive long enough to have at least a few samples under load for very short runs
    if sampler:
        t_extra = time.time()
        while ms_total < 400 and time.time() - t_extra < 0.5:
            step()
        torch.cuda.synchronize()
        sampler.terminate()
    stats = f.stats()
    two_phase = float((out["phase"] == 2).double().mean().item())
    mean_iters_two = float(out["iters"][out["phase"] == 2].double().mean().item()) if two_phase > 0 else 0.0
    n_two = int((out["phase"] == 2).sum().item())
    # per-stage times of a few extra (untimed) calls: CUDA events recorded by the library on the call's stream between
    # the stage kernels (PTFLASH_OPT_STAGE_PROFILE) -- the live launch durations behind the dominant-kernel roofline
    stage_ms = None
    if args.engine == 1 and rank == 0 and not warm:
        f.set_option("stage_profile", 1)
        acc = []
        for _ in range(5):
            step()
            acc.append(f.stage_ms()[:len(STAGES)])
        f.set_option("stage_profile", 0)
        if acc and len(acc[0]) == len(STAGES):
            stage_ms = [float(np.mean([a[i] for a in acc])) for i in range(len(STAGES))]
    t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
    if use_dist:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    ms_step = ms_total / args.steps
    value = world * N / (ms_step * 1e-3)
    launches = int(stats["kernel_launches"]) * args.steps

    # ---- extra legs (rank 0, one GPU): the cold call of config 5; the stability-only mode ----
    extra = {}
    if warm:
        for _ in range(3):
            step(cold=True)
        ms_cold = timed(lambda: step(cold=True), args.steps) / args.steps
        st_cold = f.stats()
        two_c = out["phase"] == 2
        extra["cold"] = {"ms_per_step": ms_cold, "flashes_per_s": world * N / (ms_cold * 1e-3),
                         "mean_ssi_iters_two_phase": float(out["iters"][two_c].double().mean().item()),
                         "two_phase_fraction": float(two_c.double().mean().item()), "stats": st_cold}
        extra["warm"] = {"ms_per_step": ms_step, "flashes_per_s": value, "mean_ssi_iters_two_phase": mean_iters_two,
                         "warm_restarts": int(stats["n_warm_restarts"]), "skip_stability_flags": int(flags.sum())}
    if rank == 0 and args.engine == 1 and not warm:
        f.set_option("stability_only", 1)
        for _ in range(3):
            step()
        ms_so = timed(step, max(3, args.steps // 2)) / max(3, args.steps // 2)
        f.set_option("stability_only", 0)
        extra["stability_only"] = {"ms_per_step": ms_so, "labels_per_s": N / (ms_so * 1e-3),
                                   "unstable_fraction": float((out["phase"] == 2).double().mean().item()),
                                   "note": "PTFLASH_OPT_STABILITY_ONLY: probe + stability analysis, no split (the paper labels 1e6 "
                                           "samples of its 9-component workload this way in about 2 s, PAPER.md:243)"}
        step()   # restore the outputs of the full flash

    # ---- end to end: pinned host buffers -> C ABI (H2D + kernels + D2H inside the timed region) ----
    # Every step copies its inputs from pinned host memory and its results back; the steps are submitted through the
    # pipelined call (up to PTFLASH_HOST_DEPTH batches in flight, one set of host output buffers per slot), which is how a
    # caller streams batches; the one-batch-at-a-time figure (ptflash_flash_host, returns after its results have landed) is
    # reported next to it.
    hz, hP, hT = (torch.from_numpy(a).pin_memory() for a in (w.z, w.P, w.T))
    depth = 3
    hout = [dict(b=torch.empty(N, dtype=torch.float64).pin_memory(), x=torch.empty(nc, N, dtype=torch.float64).pin_memory(),
                 y=torch.empty(nc, N, dtype=torch.float64).pin_memory(), ph=torch.empty(N, dtype=torch.int32).pin_memory(),
                 it=torch.empty(N, dtype=torch.int32).pin_memory()) for _ in range(depth)]

    def host_step(k, sync):
        o = hout[k % depth]
        (B.ptflash_flash_host if sync else B.ptflash_flash_host_async)(f.h, N, hz, hP, hT, o["b"], o["x"], o["y"], o["ph"], o["it"])

    def time_host(sync, steps):
        for k in range(depth):
            host_step(k, sync)
        B.ptflash_host_wait(f.h)
        barrier()
        t0 = time.perf_counter()
        for k in range(steps):
            host_step(k, sync)
        B.ptflash_host_wait(f.h)      # the last results have landed in host memory
        barrier()
        te = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
        if use_dist:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        return world * N * steps / float(te.item())

    e2e_steps = max(6, min(args.steps, 20))
    e2e_sync = time_host(True, max(3, e2e_steps // 2))
    e2e_value = time_host(False, e2e_steps)
    h2d = 8 * N * (nc + 2)
    d2h = 8 * N * (2 * nc + 1) + 4 * N * 2
    if not warm:
        for o in hout:
            assert int((o["ph"] == 2).sum()) == n_two

    if rank != 0:
        if use_dist:
            dist.destroy_process_group()
        return

    # ---- roofline (ALU-bound: per-mixture scalar iteration, ~130 flop/B) ----
    try:
        peaks = json.load(open(ROOT / "MEASURED_PEAKS.json"))
    except Exception:
        peaks = {}
    fp64_live, _ = B.ptflash_fp64_peak(8192)
    peak = fp64_live / 1e12
    hbm = peaks.get("hbm_gbs", 6650.0)
    fl = load_flops() if (headline and args.engine == 1) else None
    roofline = {
        "bound": "alu", "achieved": None, "peak": peak, "unit": "TFLOP/s", "frac": None, "traffic": None,
        "peak_source": "FP64 DFMA microbenchmark (ptflash_fp64_peak) measured live on this GPU; nominal %.1f TFLOP/s"
                       % (FP64_PEAK_NOMINAL / 1e12),
        "hbm_frac": (8.0 * (3 * nc + 4) * N / (ms_step * 1e-3) / 1e9) / hbm,
        "hbm_peak_gbs": hbm, "hbm_peak_source": "MEASURED_PEAKS.json" if peaks else "fallback",
        "kernel": "all stage kernels of one ptflash_flash call (k_init .. k_split_newton)",
    }
    if fl is None:
        roofline["note"] = "flops per flash are counted (ncu) for the headline workload, config 3 on engine 1, only"
    else:
        achieved = fl["flops_per_flash"] * N / (ms_step * 1e-3) / 1e12
        roofline.update(achieved=achieved, frac=achieved / peak, flops_per_flash=fl["flops_per_flash"],
                        traffic=fl["traffic_call_bytes"] if N == 1_000_000 else None,
                        flops_source=f"profiles/{fl['file']} (ncu count of build {fl['csrc_hash']})", flops_stale=bool(fl["stale"]))
        if stage_ms:
            # the same figure per stage kernel; "dominant" = the kernel with the largest share of the step
            per = {}
            for name, ms in zip(STAGES, stage_ms):
                a = fl["stage_flops_per_flash"][name] * N / (ms * 1e-3) / 1e12 if ms > 0 else 0.0
                per[name] = {"ms": ms, "share": ms / sum(stage_ms), "achieved": a, "frac": a / peak}
            dom = max(per, key=lambda k: per[k]["ms"])
            roofline["stages"] = per
            roofline["dominant"] = dict(kernel=dom, **per[dom])
            if N == 1_000_000:
                roofline["dominant"]["traffic"] = fl["stage_traffic_bytes"][dom]
    if stage_ms and fl is None:
        roofline["stages"] = {name: {"ms": ms, "share": ms / sum(stage_ms)} for name, ms in zip(STAGES, stage_ms)}

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        kw = {} if not warm else dict(lnK0=lnK0, flags=flags)
        v, cores, dt = _oracle_throughput(w, min(N, args.cpu_sample), **kw)
        one = min(N, 60_000)
        v1, c1, dt1 = _oracle_throughput(w, one, threads=1, **({} if not warm else dict(lnK0=lnK0[:, :one], flags=flags[:one])))
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {min(N, args.cpu_sample)} mixtures of the workload, one pass, {dt:.2f} s wall, OpenMP over mixtures",
               "one_core": {"value": v1, "unit": UNIT, "cores": c1, "sample": f"first {one} mixtures, one pass, {dt1:.2f} s wall"}}

    cfg = {"workload": workload, "mixtures_per_step": N, "nc": nc, "engine": args.engine, "two_phase_fraction": two_phase,
           "mean_ssi_iters_two_phase": mean_iters_two,
           "l2": ("inputs+outputs+workspace per step are %.0f MB > 126 MB L2, so every step streams from HBM" % (N * (16.0 * nc + 32 + 60.0 * nc) / 1e6)
                  if N * (16.0 * nc + 32 + 60.0 * nc) > 126e6 else
                  "working set %.0f MB fits the 126 MB L2 (small-N sweep point; no flush between steps)" % (N * (16.0 * nc + 32 + 60.0 * nc) / 1e6)),
           "stats_last_step": stats}
    cfg.update(extra)
    if user_opts:
        cfg["options"] = user_opts
    if args.config == "paper9":
        cfg["paper_table4"] = dict(PAPER_TABLE4, ours={"two_phase_share": stats["n_two_phase"] / N, "probe_proved_share": stats["n_probe_case3"] / N})
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": cfg,
        "clocks": _parse_clocks(clk_path),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps,
                "api": "ptflash_flash_host_async + ptflash_host_wait: pinned host buffers, every step's H2D and D2H copies inside the "
                       "timed region, up to 3 batches in flight" + ("; cold Wilson starts" if warm else ""),
                # the two host-buffer calls as peers: `value` above is the pipelined one, as in round 2; the figure
                # to hold against round 1's e2e.value (which timed ptflash_flash_host) is `sync`
                "pipelined": {"value": e2e_value, "unit": UNIT, "api": "ptflash_flash_host_async + ptflash_host_wait (3 batches in flight)"},
                "sync": {"value": e2e_sync, "unit": UNIT, "api": "ptflash_flash_host (returns after its results are in host memory)",
                         "note": "same API as BENCH_r01's e2e.value"},
                "one_batch_at_a_time": {"value": e2e_sync, "unit": UNIT, "api": "ptflash_flash_host (returns after its results are in host memory)"}},
        "gpu_launches": launches,
        "roofline": roofline,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line))
    try:
        os.remove(clk_path)
    except OSError:
        pass
    if use_dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
