#!/usr/bin/env python
"""Writes tests/golden/oracle_energies.json: the CPU oracle's own values on BASELINE.json's seeded configs.

    python tests/golden/make_golden.py

The paper prints no worked numerical example of E(T) (Table 1, gives deviations from an external
program only), so absolute values are "parity unpinned by the paper" (P10).  These numbers are
regression goldens: after the pins P1-P9 of tests/test_oracle_pins.py pass, the oracle's results on the seeded
synthetic inputs are frozen here.  This script calls ONLY ``oracle/`` and the seeded input generator -- never the
CUDA path.  Stored: tiny (nocc=8, nvirt=40) full E(T), E[4], E[5] and all per-triplet energies (C loops, restricted
mode, reading Q4); small (16, 120) and medium (24, 240): sampled triplets incl. the forced edge cases, numpy
restatement (Eq. (2.2.2)-(2.2.5), one triplet at a time).  Values are printed with 17 significant digits.
"""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import oracle  # noqa: E402
from paper_1609_08094_b200 import synth  # noqa: E402

SAMPLES = {"small": 10, "medium": 7}


def main():
    out = {"_citation": "arXiv:1609.08094 Eq. (2.2.1)-(2.2.5) (PAPER.md L87-L109), readings Q1/Q4 of DESIGN.md; "
                        "inputs: BASELINE.json configs, seed 0, paper_1609_08094_b200/synth.py",
           "_writer": "tests/golden/make_golden.py (oracle only)"}
    inp = synth.make_config("tiny", seed=0)
    E, et = oracle.energy_restricted(inp.nocc, inp.nvirt, *inp.arrays(), with_triplets=True)
    out["tiny"] = {"nocc": inp.nocc, "nvirt": inp.nvirt, "E": [float(x) for x in E],
                   "triplets": [[float(x) for x in row] for row in et]}
    for name, n in SAMPLES.items():
        o, v, naux = synth.CONFIGS[name]
        inp = synth.make_config(name, seed=0)
        trips = [t for t in synth.sample_triplets(o, n, seed=0)]
        a = inp.arrays()
        e = oracle.energy_subset_numpy(a[0], a[1], a[2], a[3], a[4], a[5], a[6], trips)
        out[name] = {"nocc": o, "nvirt": v, "triplets_ijk": [list(map(int, t)) for t in trips],
                     "energies": [[float(x) for x in row] for row in e]}
        print(name, "done", file=sys.stderr)
    with open(os.path.join(HERE, "oracle_energies.json"), "w") as f:
        json.dump(out, f, indent=0, separators=(",", ":"))
        f.write("\n")


if __name__ == "__main__":
    main()
