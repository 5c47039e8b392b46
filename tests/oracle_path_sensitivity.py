"""Which phase labels depend on the SCHEDULE of the stability analysis rather than on the mixture?  (oracle only)

    python tests/oracle_path_sensitivity.py [--configs 3,4] [--n 1000000] [--threads 0]

The paper's stability test is a heuristic: two local searches from Wilson-based starts, nine successive
substitutions then a trust-region Newton, with the restricted-step details left to a citation (B.1b
PAPER.md:468; reading C11 of DESIGN.md fills them in: eta grows x8, geometric bisection to a bracket ratio of 1.5).  The
label "stable" is therefore "neither search found a negative tangent-plane distance", and for a few mixtures which
stationary point a search reaches depends on those schedule constants.  This script

  1. flashes a workload with the default schedule and with perturbed ones (stab_ss_iters 6 / 12, eta growth x4 / x16,
     bisection ratio 1.25 / 2.0) and lists every mixture whose LABEL changes (outside the |tpd_min| < 1e-9 band of C9);
  2. adjudicates each of them -- and, as a control, a seeded sample of ordinary mixtures -- with many more starts
     (Wilson K to the powers +-1/3, +-2/3, +-1, +-4/3; every pure-component-rich trial 0.9 e_i + 0.1 z): a negative
     tpd found from ANY start proves the mixture unstable (eq. 3), so the adjudicated label is the true one
     as far as those starts can tell.

It calls only oracle/ (never the CUDA path); its numbers are quoted in DESIGN.md section 3 and pinned at a reduced size by
tests/test_oracle_pins.py::test_path_sensitivity_set.
"""
from __future__ import annotations

import argparse
import json
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[1]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

VARIANTS = {
    "stab_ss_iters=6": dict(stab_ss_iters=6), "stab_ss_iters=12": dict(stab_ss_iters=12),
    "eta_growth=4": dict(eta_growth=4.0), "eta_growth=16": dict(eta_growth=16.0),
    "eta_ratio=1.25": dict(eta_ratio=1.25), "eta_ratio=2": dict(eta_ratio=2.0),
}
BAND = 1e-9


def label_changes(orc, w, nthreads=0):
    """Returns (base result, {n: {variant: (label, tpd_min)}}) for mixtures whose label differs from the default's."""
    base = orc.flash(w.z, w.P, w.T, nthreads=nthreads)
    in_band = np.isfinite(base["tpd_min"]) & (base["tpd_min"] != 0) & (np.abs(base["tpd_min"]) < BAND)
    changed = {}
    for name, opts in VARIANTS.items():
        r = orc.flash(w.z, w.P, w.T, opts=opts, nthreads=nthreads)
        for n in np.where((r["phase"] != base["phase"]) & ~in_band)[0]:
            changed.setdefault(int(n), {})[name] = (int(r["phase"][n]), float(r["tpd_min"][n]))
    return base, changed


def adjudicate(orc, P, T, z):
    """Minimum tpd over many starts.  Returns (tpd_min over non-trivial stationary points or 0.0, number of starts that
    found a negative tpd, number of starts)."""
    z = np.asarray(z, dtype=np.float64)
    act = z > 0
    lnz = np.where(act, np.log(np.where(act, z, 1.0)), 0.0)
    wil = orc.wilson(P, T)
    starts = [(wil * p, s) for p in (1.0 / 3.0, 2.0 / 3.0, 1.0, 4.0 / 3.0) for s in (+1, -1)]
    for i in np.where(act)[0]:
        c = 0.1 * z
        c[i] += 0.9
        starts.append((np.where(act, np.log(np.where(act, c, 1.0)) - lnz, 0.0), +1))
    best, neg = 0.0, 0
    for lnK, side in starts:
        t = orc.stability_trial(P, T, z, lnK, side)
        if not t["trivial"] and not t["capped"]:
            best = min(best, t["tpd"])
            neg += t["tpd"] < -BAND
    return best, neg, len(starts)


def report(orc, w, nthreads=0, control=2000, seed=11):
    base, changed = label_changes(orc, w, nthreads)
    rows = []
    for n, var in sorted(changed.items()):
        tpd, neg, ns = adjudicate(orc, w.P[n], w.T[n], w.z[:, n])
        rows.append(dict(n=n, default_label=int(base["phase"][n]), default_tpd_min=float(base["tpd_min"][n]),
                         variants={k: dict(label=v[0], tpd_min=v[1]) for k, v in var.items()},
                         adjudicated_tpd_min=float(tpd), starts_negative=int(neg), starts=ns,
                         true_label_unstable=bool(tpd < -BAND),
                         default_is_true_label=bool((tpd < -BAND) == (base["tpd_min"][n] < 0 or base["probe_case"][n] == 3))))
    # control: how often do many starts overturn the two-start verdict on ordinary mixtures?
    rng = np.random.default_rng(seed)
    went = np.where((base["probe_case"] == 1) | (base["probe_case"] == 2))[0]     # decided by the stability analysis
    pick = rng.choice(went, size=min(control, len(went)), replace=False)
    overturned = []
    for n in pick:
        tpd, neg, ns = adjudicate(orc, w.P[n], w.T[n], w.z[:, n])
        if (tpd < -BAND) != (base["tpd_min"][n] < 0):
            overturned.append(dict(n=int(n), default_tpd_min=float(base["tpd_min"][n]), adjudicated_tpd_min=float(tpd)))
    return dict(workload=w.name, N=int(w.N), variants=list(VARIANTS), label_changes=len(rows), mixtures=rows,
                control_sample=int(len(pick)), control_overturned=overturned)


def main():
    from oracle import oracle as O
    from paper_2205_03090_b200 import workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="3,4")
    ap.add_argument("--n", type=int, default=1_000_000)
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--control", type=int, default=2000)
    a = ap.parse_args()
    O.build("double")
    for cfg in (int(c) for c in a.configs.split(",")):
        w = W.CONFIGS[cfg](a.n)
        print(json.dumps(report(O.Oracle.from_system(w.system), w, a.threads, a.control)))


if __name__ == "__main__":
    main()
