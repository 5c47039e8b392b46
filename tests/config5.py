"""BASELINE.json config 5: warm-started, divergence-stressed flash (test-side input builder).

Emulates the paper's network-provided K estimates (section 4.3) without trained weights: same
10-component system and kij as config 3; (P, T, z) within 5 % of each mixture's ORACLE-computed phase boundary so
iteration counts are high and varied; initial lnK = oracle-converged lnK + N(0, 0.05) and stability skipped for
mixtures whose oracle label is two-phase.

This builder calls the oracle, so it lives with the tests and not in the (oracle-free) workloads module.
Recipe: candidates c = 0, 1, 2, ... draw (T, z) like config 3
under seed 2205030905; oracle labels on 28 log-spaced pressures in [5, 300] bar; candidates without a label change are
skipped; one label change is picked with a seeded uniform and bisected in P to |dP|/P < 1e-6 -> P_b;
P = P_b (1 + 0.05 (2u - 1)) clipped to [5, 300].
"""
from __future__ import annotations

import sys
from pathlib import Path

import numpy as np

sys.path.insert(0, str(Path(__file__).resolve().parents[1]))   # also runnable as a script (see the bottom of the file)
from paper_2205_03090_b200 import workloads as W  # noqa: E402

SEED = W.SEEDS[5]
N_GRID = 28


def build(oracle, N: int, batch: int = 4096, nthreads: int = 0):
    """Returns (Workload, lnK0 [nc, N], flags [N] uint8, info dict)."""
    sysm = W.system_co2_10()
    nc = sysm.nc
    grid = np.exp(np.linspace(np.log(5.0), np.log(300.0), N_GRID))
    Ts, zs, Ps = [], [], []
    c0 = 0
    tried = 0
    while sum(len(t) for t in Ts) < N:
        n = np.arange(c0, c0 + batch)
        c0 += batch
        tried += batch
        T = 220.0 + 280.0 * W.uniform(SEED, n, 0)
        d = W._dirichlet1(SEED, n, nc, k0=2)
        z = 0.6 * d
        z[8] += 0.4
        z = z / z.sum(axis=0, keepdims=True)
        upick = W.uniform(SEED, n, 40)
        ujit = W.uniform(SEED, n, 41)
        # labels on the pressure grid
        lab = np.empty((N_GRID, batch), dtype=np.int32)
        for g, Pg in enumerate(grid):
            lab[g] = oracle.flash(z, np.full(batch, Pg), T, nthreads=nthreads)["phase"]
        change = lab[1:] != lab[:-1]                       # [27, batch]
        nch = change.sum(axis=0)
        ok = nch > 0
        # pick the k-th change, k = floor(u * nch)
        kth = np.minimum((upick * np.maximum(nch, 1)).astype(int), np.maximum(nch - 1, 0))
        cum = np.cumsum(change, axis=0)
        sel = np.argmax((cum == (kth + 1)[None, :]) & change, axis=0)   # index g with boundary between g and g+1
        idx = np.where(ok)[0]
        lo, hi = grid[sel[idx]].copy(), grid[sel[idx] + 1].copy()
        lab_lo = lab[sel[idx], idx]
        zi, Ti = np.ascontiguousarray(z[:, idx]), T[idx].copy()
        for _ in range(60):
            mid = np.sqrt(lo * hi)
            if np.all((hi - lo) / mid < 1e-6):
                break
            lm = oracle.flash(zi, mid, Ti, nthreads=nthreads)["phase"]
            same = lm == lab_lo
            lo = np.where(same, mid, lo)
            hi = np.where(same, hi, mid)
        Pb = np.sqrt(lo * hi)
        P = np.clip(Pb * (1.0 + 0.05 * (2.0 * ujit[idx] - 1.0)), 5.0, 300.0)
        Ts.append(Ti); zs.append(zi); Ps.append(P)
    T = np.concatenate(Ts)[:N]
    z = np.ascontiguousarray(np.concatenate(zs, axis=1)[:, :N])
    P = np.concatenate(Ps)[:N]
    w = W.Workload("config5_warm_near_boundary_10", sysm, P, T, z, {"seed": SEED, "candidates_tried": tried})
    cold = oracle.flash(z, P, T, nthreads=nthreads)
    two = cold["phase"] == 2
    m = np.arange(N)
    noise = np.stack([0.05 * W.normal(SEED + 1, m, 2 * i) for i in range(nc)])
    lnK0 = np.where(two[None, :], cold["lnK"] + noise, 0.0)
    flags = np.where(two, 1, 0).astype(np.uint8)
    return w, np.ascontiguousarray(lnK0), flags, {"cold": cold, "two_phase_fraction": float(two.mean()),
                                                  "acceptance": float(N) / tried}


def build_cached(oracle, N: int, cache_dir: str = ""):
    """build() with the result kept in the system's temporary directory (scratch; gpurun_out/ is limited to 64 MiB): the
    boundary search costs ~60 oracle flashes per accepted mixture (SURVEY.md section 8(d) allows caching it).  The cache
    holds inputs only; the oracle's cold answers are recomputed, so a stale cache can never supply an expected value, and
    nothing depends on the cache being there."""
    import tempfile
    from pathlib import Path
    path = Path(cache_dir or tempfile.gettempdir()) / f"ptflash_config5_inputs_{N}.npz"
    sysm = W.system_co2_10()
    if path.exists():
        d = np.load(path)
        w = W.Workload("config5_warm_near_boundary_10", sysm, d["P"], d["T"], np.ascontiguousarray(d["z"]), {"seed": SEED})
        cold = oracle.flash(w.z, w.P, w.T)
        two = cold["phase"] == 2
        if np.array_equal(two, d["two"]):
            return w, np.ascontiguousarray(d["lnK0"]), d["flags"], {"cold": cold, "two_phase_fraction": float(two.mean())}
    w, lnK0, flags, info = build(oracle, N, batch=min(65536, max(4096, N // 8)))
    try:
        path.parent.mkdir(exist_ok=True)
        np.savez(path, P=w.P, T=w.T, z=w.z, lnK0=lnK0, flags=flags, two=info["cold"]["phase"] == 2)
    except OSError:
        pass
    return w, lnK0, flags, info


if __name__ == "__main__":
    # python tests/config5.py N OUT.npz -- writes the INPUTS of config 5 (P, T, z, lnK0, flags; no expected values) for
    # `bench.py --config 5`, which runs this script in a process of its own so that the benchmark process never imports oracle/.
    from oracle import oracle as O
    O.build("double")
    n_mix, out_path = int(sys.argv[1]), sys.argv[2]
    w_, l0_, fl_, info_ = build(O.Oracle.from_system(W.system_co2_10()), n_mix, batch=min(65536, max(4096, n_mix // 8)))
    np.savez(out_path, P=w_.P, T=w_.T, z=w_.z, lnK0=l0_, flags=fl_, two=info_["cold"]["phase"] == 2)
    print(f"config 5: {n_mix} mixtures, two-phase share {info_['two_phase_fraction']:.4f}, acceptance {info_['acceptance']:.3f} -> {out_path}")
