#!/usr/bin/env python
"""Writes the stored oracle values under tests/golden/: the CPU oracle's own results on BASELINE.json's seeded configs.

    python tests/golden/make_golden.py legacy                 # oracle_energies.json (tiny full; small / medium samples)
    python tests/golden/make_golden.py small_full             # all 816 triplets of configs[1]
    python tests/golden/make_golden.py medium_full            # all 2600 triplets of configs[2] (hours on 8 cores)
    python tests/golden/make_golden.py medium_t1              # configs[2] with t1 ~ N(0,1): sampled triplets, pins E[5]
    python tests/golden/make_golden.py large_sample           # configs[3]: 6 forced + 32 seeded triplets
    python tests/golden/make_golden.py largest_sample         # configs[4]: 6 forced + 32 seeded triplets
    python tests/golden/make_golden.py paper_ala4_sample      # the paper's (nocc 81, nvirt 323) size: 6 forced + 10 seeded
        [--procs N] [--threads M]   worker processes over independent triplets x BLAS threads each

The paper prints no worked numerical example of E(T) (Table 1, gives deviations from an external
program only), so absolute values are "parity unpinned by the paper" (P10).  These numbers are
regression goldens: after the pins P1-P9 of tests/test_oracle_pins.py pass, the oracle's results on the seeded
synthetic inputs are frozen here.  This script calls ONLY ``oracle/`` and the seeded input generator -- never the
CUDA path.  Every value is the oracle's numpy restatement of Eq. (2.2.2)-(2.2.5), one triplet at a time
(``oracle.triplet_energy_numpy``), except the tiny config (C loops, restricted mode, reading Q4).  At configs[3..4]
the 16-35 GB vvvo tensor is never built: the oracle gets the slices vvvo[:, :, :, r] of its triplet, rebuilt on the
host from the B factors (``synth.vvvo_slice``).  Files are written incrementally and the run resumes from what a file
already holds.  Values are printed with 17 significant digits.
"""
import argparse
import json
import math
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from oracle import oracle  # noqa: E402
from paper_1609_08094_b200 import synth  # noqa: E402

CITATION = ("arXiv:1609.08094 Eq. (2.2.1)-(2.2.5) (PAPER.md L87-L109), readings Q1/Q4 of DESIGN.md; "
            "inputs: BASELINE.json configs, paper_1609_08094_b200/synth.py")
LEGACY_SAMPLES = {"small": 10, "medium": 7}

# name -> (config, t1_sigma, input seed, triplets: "full" or sample size incl. the 6 forced cases)
JOBS = {
    "small_full": ("small", 1e-3, 0, "full"),
    "medium_full": ("medium", 1e-3, 0, "full"),
    "medium_t1": ("medium", 1.0, 0, 22),
    "large_sample": ("large", 1e-3, 0, 38),
    "largest_sample": ("largest", 1e-3, 0, 38),
    # the paper's [ala]-4/cc-pVDZ size, naux = 3 nvirt, same generator: the only multi-tile ODD nvirt
    "paper_ala4_sample": (("paper_ala4", 81, 323, 969), 1e-3, 0, 16),
}


def legacy():
    out = {"_citation": CITATION, "_writer": "tests/golden/make_golden.py legacy (oracle only)"}
    inp = synth.make_config("tiny", seed=0)
    E, et = oracle.energy_restricted(inp.nocc, inp.nvirt, *inp.arrays(), with_triplets=True)
    out["tiny"] = {"nocc": inp.nocc, "nvirt": inp.nvirt, "E": [float(x) for x in E],
                   "triplets": [[float(x) for x in row] for row in et]}
    for name, n in LEGACY_SAMPLES.items():
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


# ---- worker state (inherited by fork): the small tensors, the B factors, a bounded cache of vvvo slices
_G = {}


def _slice(r):
    cache = _G["cache"]
    if r not in cache:
        while len(cache) >= _G["max_slices"]:
            cache.pop(next(iter(cache)))
        cache[r] = synth.vvvo_slice(_G["B"], _G["o"], _G["v"], r)
    return cache[r]


def _one(t):
    if "threads" in _G and not _G.get("limited"):
        try:
            from threadpoolctl import threadpool_limits

            _G["limiter"] = threadpool_limits(limits=_G["threads"])
        except Exception:
            pass
        _G["limited"] = True
    i, j, k = t
    X = {r: _slice(r) for r in (i, j, k)}
    return t, oracle.triplet_energy_numpy(_G["eps_o"], _G["eps_v"], _G["t1"], _G["t2"], X, _G["ovoo"], _G["ovov"],
                                          i, j, k)


def run(name, procs, threads):
    config, t1_sigma, seed, which = JOBS[name]
    if isinstance(config, tuple):                     # a size outside BASELINE.json's configs: (label, nocc, nvirt, naux)
        config, o, v, naux = config
    else:
        o, v, naux = synth.CONFIGS[config]
    path = os.path.join(HERE, f"{name}.json")
    trips = synth.triplet_list(o) if which == "full" else synth.sample_triplets(o, which, seed=0)
    trips = [tuple(int(x) for x in t) for t in trips]
    doc = {"_citation": CITATION, "_writer": f"tests/golden/make_golden.py {name} (oracle only)", "config": config,
           "nocc": o, "nvirt": v, "naux": naux, "seed": seed, "t1_sigma": t1_sigma,
           "mode": "full" if which == "full" else "sample",
           "layout": "energies[n] = [w*(e4+e5), w*e4, w*e5] of triplets_ijk[n], w = 2 - d_ij - d_jk",
           "triplets_ijk": [], "energies": [], "complete": False}
    done = {}
    if os.path.exists(path):
        with open(path) as f:
            old = json.load(f)
        if all(old.get(k) == doc[k] for k in ("config", "nocc", "nvirt", "naux", "seed", "t1_sigma", "mode")):
            done = {tuple(t): e for t, e in zip(old["triplets_ijk"], old["energies"])}
    todo = [t for t in trips if t not in done]
    print(f"{name}: {len(done)} of {len(trips)} triplets stored, {len(todo)} to do", file=sys.stderr, flush=True)

    def flush():
        have = [t for t in trips if t in done]
        doc["triplets_ijk"] = [list(t) for t in have]
        doc["energies"] = [[float(x) for x in done[t]] for t in have]
        doc["complete"] = len(have) == len(trips)
        if doc["complete"] and which == "full":      # E(T) = sum of the weighted per-triplet energies, Eq. (2.2.1)
            e4 = math.fsum(done[t][1] for t in trips)
            e5 = math.fsum(done[t][2] for t in trips)
            doc["E"] = [e4 + e5, e4, e5]
        with open(path + ".tmp", "w") as f:
            json.dump(doc, f, indent=0, separators=(",", ":"))
            f.write("\n")
        os.replace(path + ".tmp", path)

    if todo:
        eps_o, eps_v, t1, t2, ovoo, ovov, B = synth.make_inputs_sliced(o, v, naux, seed, t1_sigma)
        # slices kept per worker: all of them while that stays below ~6 GB, else the three of the running triplet
        max_slices = max(3, min(o, int(6e9 / (8.0 * v ** 3))))
        _G.update(dict(o=o, v=v, eps_o=eps_o, eps_v=eps_v, t1=t1, t2=t2, ovoo=ovoo, ovov=ovov, B=B, cache={},
                       max_slices=max_slices, threads=threads))
        # a worker holds its slice cache plus ~14 v^3 arrays of temporaries: keep the sum below ~40 GB of host memory
        procs = max(1, min(procs, int(40e9 / (8.0 * v ** 3 * (14 + max_slices)))))
        t0 = time.time()
        last = t0
        if procs > 1:
            import multiprocessing as mp

            pool = mp.get_context("fork").Pool(procs)
            it = pool.imap_unordered(_one, todo, chunksize=1)
        else:
            it = map(_one, todo)
        for n, (t, e) in enumerate(it):
            done[t] = [float(x) for x in e]
            if time.time() - last > 120 or n + 1 == len(todo):
                flush()
                last = time.time()
                print(f"{name}: {n + 1}/{len(todo)} in {time.time() - t0:.0f} s", file=sys.stderr, flush=True)
        if procs > 1:
            pool.close()
            pool.join()
    flush()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("what", nargs="+", choices=["legacy"] + list(JOBS))
    ap.add_argument("--procs", type=int, default=1)
    ap.add_argument("--threads", type=int, default=max(1, (os.cpu_count() or 1)))
    args = ap.parse_args()
    for w in args.what:
        if w == "legacy":
            legacy()
        else:
            run(w, args.procs, args.threads)


if __name__ == "__main__":
    main()
