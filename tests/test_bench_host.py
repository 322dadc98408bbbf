"""Host-side logic of bench.py (no GPU): the rank reduction used for multi-process runs (world size 2, gloo, CPU),
the flop formula of the metric, and the reference arm (the CPU oracle timed on a bounded sample)."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank = dist.get_rank()
t, u = bench.reduce_over_ranks(1.0 + rank, 10.0 * (rank + 1), dist.get_world_size())
# triplet-sharded mode: every rank holds its shard's partial (E(T), E[4], E[5]); the ordered sum is the total
import paper_1609_08094_b200 as tb
o, v = 9, 40
_, sot, jps = tb.triples_plan_shards(o, v, tb.FP64, dist.get_world_size())
fake = [1e-3 * (n + 1) * (1 + 1e-7 * n) for n in range(len(sot))]          # a stand-in energy per triplet
mine = sum(fake[n] for n in range(len(sot)) if sot[n] == rank)
tot = bench.combine_shard_partials((mine, mine, 0.0), dist.get_world_size())
print(json.dumps({{"rank": rank, "t": t, "u": u, "tot": tot, "mine": mine, "covered": int((sot == rank).sum()),
                  "all": int((sot >= 0).sum()), "jobs": [int(x) for x in jps],
                  "single": sum(fake[n] for n in range(len(sot)) if sot[n] >= 0)}}), flush=True)
dist.destroy_process_group()
"""


def test_reduce_over_ranks_world_size_2_gloo():
    """Replicas-only multi-GPU path: MAX of the per-rank times, SUM of the per-rank units."""
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", _WORKER.format(root=ROOT)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["t"] == 2.0 and o["u"] == 30.0       # max(1, 2) seconds, 10 + 20 units on every rank
    # sharded mode: the two ranks cover every non-diagonal triplet exactly once, both ranks get
    # the same rank-ordered total, and it equals the single-rank sum to rounding
    assert outs[0]["covered"] + outs[1]["covered"] == outs[0]["all"] and min(o["covered"] for o in outs) > 0
    assert outs[0]["tot"] == outs[1]["tot"]
    by_rank = sorted(outs, key=lambda o: o["rank"])
    assert outs[0]["tot"][0] == by_rank[0]["mine"] + by_rank[1]["mine"]
    assert abs(outs[0]["tot"][0] - outs[0]["single"]) <= 1e-13 * abs(outs[0]["single"])
    assert max(outs[0]["jobs"]) <= 1.6 * min(outs[0]["jobs"])          # whole window blocks, near-equal task weight (L198)


def test_reduce_over_ranks_single_process_is_identity():
    assert bench.reduce_over_ranks(1.5, 7.0, 1) == (1.5, 7.0)


@pytest.mark.parametrize("o,v", [(8, 40), (24, 240), (40, 480)])
def test_formula_flops_is_the_papers_task_count_times_the_gemm_flops(o, v):
    # PAPER.md Eq. (5.0.7b): T = No(No+1)(No+2)/6 equal-weight tasks; 12 v^4 + 12 o v^3 flop each
    T = sum((o - i) * (1 + (o - i)) // 2 for i in range(o))
    assert bench.formula_flops(o, v) == T * (12.0 * v ** 4 + 12.0 * o * v ** 3)


def test_measured_peaks_has_the_roofline_denominators():
    peaks, kind = bench.measured_peaks()
    assert kind in ("measured", "fallback")
    assert peaks["hbm_gbs"] > 1000 and peaks["bf16_tflops_sustained"] > 100


def _run_reference(extra_env):
    env = dict(os.environ, **extra_env)
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "tiny",
                           "--steps", "1", "--warmup", "1", "--ref-triplets", "2"], env=env, capture_output=True,
                          text=True, timeout=600)


def test_reference_arm_times_the_oracle_and_prints_one_json_line():
    res = _run_reference({})
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "TFLOP/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["cpu_baseline"]["kind"].startswith("oracle") and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["gpu_launches"] == 0 and "tiny" in d["config"]["workload"]


def test_reference_arm_other_ranks_exit_quietly():
    res = _run_reference({"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"})
    assert res.returncode == 0 and res.stdout.strip() == ""


def test_parity_vs_golden_compares_the_stored_oracle_values():
    """bench.py's parity figure: the run's per-triplet energies against tests/golden/ (no oracle run, no GPU)."""
    import numpy as np
    g = bench.load_golden("small")
    o = g["nocc"]
    trip = [(i, j, k) for i in range(o) for j in range(i, o) for k in range(j, o)]
    index = {t: n for n, t in enumerate(trip)}
    et = np.zeros((len(trip), 3))
    for t, e in zip(g["triplets_ijk"], g["energies"]):
        et[index[tuple(t)]] = e
    exact = bench.parity_vs_golden("small", et, index, 1e-10)
    assert exact["ok"] and exact["max_rel_err"] == 0.0 and exact["triplets_compared"] == len(trip) - o
    n = index[(0, 1, 2)]
    et[n, 0] *= 1 + 3e-9
    off = bench.parity_vs_golden("small", et, index, 1e-10)
    assert not off["ok"] and 2e-9 < off["max_rel_err"] < 4e-9
    assert bench.load_golden("nonexistent") is None
    assert len(bench.load_golden("tiny")["triplets_ijk"]) == 120            # configs[0]: the C-loop golden


def test_final_bench_line_stays_small_whatever_the_legs_carry():
    """Round 2's default command printed one 22 KB line; the driver keeps ~3 KB of stdout and recorded `parsed: null`.
    The last line is now a digest: the contract's keys, numbers and short strings, under bench.LINE_LIMIT bytes, however
    much the legs and notes of the full document grow (that document goes to stdout leg by leg and to a file)."""
    with open(os.path.join(ROOT, "profiles", "r02_bench_default.json")) as f:
        full = json.load(f)                                      # the 22 KB document itself
    assert len(json.dumps(full)) > 20000
    full["legs"]["largest"]["fp64"] = dict(full["legs"]["large"]["fp64"])
    full["roofline"]["peak_note"] = "x" * 5000                    # notes of any length never reach the line
    full["config"]["why_this_config"] = "y" * 3000
    full["detail"] = "legs: one JSON line each above this one; whole document: gpurun_out/bench_detail.json"
    text = bench.compact_line(full)
    assert len(text) < bench.LINE_LIMIT <= 2500 and "\n" not in text
    d = json.loads(text)
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "gpu_launches", "roofline", "roofline_reduction",
                "cpu_baseline", "e2e", "parity"):
        assert key in d, key
    assert d["value"] > 0 and d["config"]["workload"].startswith("medium")
    for r in (d["roofline"], d["roofline_reduction"]):
        assert set(r) <= set(bench.ROOF_KEYS) and r["frac"] == pytest.approx(r["achieved"] / r["peak"], rel=1e-4)
    assert set(d["e2e"]) == {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "api"}
    assert set(d["cpu_baseline"]) == {"value", "unit", "cores", "kind", "sample"}
    assert d["legs"]["largest.fp64"][0] == pytest.approx(full["legs"]["large"]["fp64"]["value"], rel=1e-5)
    assert len(d["legs"]["large.mixed"]) == len(d["legs_columns"].split(","))
    # a line that would still be too long loses its digest rather than its contract keys
    full["legs"] = {f"cfg{n}": {"fp64": full["legs"]["large"]["fp64"]} for n in range(60)}
    d2 = json.loads(bench.compact_line(full))
    assert "legs" not in d2 and d2["roofline"]["frac"] == d["roofline"]["frac"]
