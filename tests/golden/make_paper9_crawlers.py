"""Writes tests/golden/paper9_crawlers.json: the INPUTS (P, T, z) of the few mixtures of the paper's 9-component workload
(workloads.paper9, first 10^6 mixtures) whose phase split is a "crawler" -- still outside 0 < theta < 1 after the nine
successive substitutions of PAPER.md:92, so that the substitution continues (reading C13) -- as found by the
oracle (split SS iteration count > split_ss_iters).  Inputs only, no expected values: the GPU test flashes them and compares
with the oracle at run time.  They are stored because generating mixture 927885 of the rejection-sampled workload takes a
minute of numpy time.

    python tests/golden/make_paper9_crawlers.py        (calls only workloads.py and oracle/)
"""
from __future__ import annotations

import json
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))

from oracle import oracle as O                                  # noqa: E402
from paper_2205_03090_b200 import workloads as W               # noqa: E402


def main():
    N = 1_000_000
    w = W.paper9(N)
    o = O.Oracle.from_system(w.system).flash(w.z, w.P, w.T)
    ss = o["stage"][5]                                           # split SS iterations (oracle/ptflash_oracle.cpp, orc_flash_batch)
    idx = np.where(ss > 9)[0]
    out = {"workload": "paper9", "N": N, "criterion": "oracle split SS iterations > 9",
           "n": [int(n) for n in idx], "oracle_split_ss_iters": [int(ss[n]) for n in idx],
           "P": [float.hex(float(w.P[n])) for n in idx], "T": [float.hex(float(w.T[n])) for n in idx],
           "z": [[float.hex(float(v)) for v in w.z[:, n]] for n in idx]}
    path = Path(__file__).with_name("paper9_crawlers.json")
    path.write_text(json.dumps(out, indent=1) + "\n")
    print(f"wrote {path}: {len(idx)} mixtures, SS iterations {sorted(out['oracle_split_ss_iters'])}")


if __name__ == "__main__":
    main()
