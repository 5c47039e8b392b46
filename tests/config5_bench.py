"""BASELINE config 5 on the GPU: warm-started (caller lnK0 + skip-stability flags) against cold Wilson starts.

    python tests/config5_bench.py [N]          (needs a CUDA device; N defaults to 100000)

Lives under tests/ because the inputs need the CPU oracle (phase-boundary search, converged lnK: tests/config5.py); the
library itself never touches oracle/.  Prints one JSON line: flashes/s and mean iteration counts, warm vs cold.
"""
import json
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))
sys.path.insert(0, str(ROOT / "tests"))


def main():
    import torch
    import config5
    from oracle import oracle as O
    from paper_2205_03090_b200 import binding as B, workloads as W
    N = int(sys.argv[1]) if len(sys.argv) > 1 else 100_000
    O.build("double")
    orc = O.Oracle.from_system(W.system_co2_10())
    w, lnK0, flags, info = config5.build(orc, N)
    dev = torch.device("cuda:0")
    z, P, T = (torch.from_numpy(a).to(dev) for a in (w.z, w.P, w.T))
    l0 = torch.from_numpy(lnK0).to(dev)
    fl = torch.from_numpy(flags).to(dev)
    f = B.PTFlash.from_system(w.system)
    res = {}
    for name, kw in (("cold", {}), ("warm", dict(lnK0=l0, flags=fl))):
        for _ in range(3):
            out = f.flash(z, P, T, **kw)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        K = 10
        for _ in range(K):
            out = f.flash(z, P, T, **kw)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / K
        two = (out["phase"] == 2)
        res[name] = {"ms_per_step": ms, "flashes_per_s": N / (ms * 1e-3), "two_phase_fraction": float(two.double().mean()),
                     "mean_iters_two_phase": float(out["iters"][two].double().mean()),
                     "mean_stab_iters": float(out["stab_iters"].double().mean()),
                     "warm_restarts": int(((out["status"] & 64) != 0).sum())}
    print(json.dumps({"workload": "config5: warm start near the phase boundary (tests/config5.py)", "N": N,
                      "oracle_two_phase_fraction": info["two_phase_fraction"], **res}))


if __name__ == "__main__":
    main()
