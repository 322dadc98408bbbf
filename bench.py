#!/usr/bin/env python
"""Benchmark of the B200 closed-shell (T) energy path (arXiv:1609.08094 section 2.2).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config medium] [--precision fp64|mixed|emu64]
    python bench.py --impl reference ...          # the CPU oracle, timed on the host cores

A "step" is one pass of the whole hot path -- repack, every contraction batch, every fused reduction batch,
the per-triplet finalize and the total -- i.e. one E(T) of the workload.  Prints ONE JSON line (rank 0).

Metric: (T) TFLOP/s = T*(12 v^4 + 12 o v^3) / seconds per E(T), T = o(o+1)(o+2)/6 (Eq. (5.0.7b)),
the paper's task count; `executed_value` counts the flops the kernels really execute (i=j=k tasks skipped,
coinciding contractions of i=j / j=k tasks computed once) and is the figure to hold against the hardware peak.

The default line (medium, FP64) also carries: the mixed-precision path on the same workload (`mixed_path`), the
RI-direct and out-of-core variants (`ri_direct`, `streamed`), and short legs on the two largest single-GPU
configs (`legs.large`: FP64 + mixed + emulated FP64 + streamed, `legs.largest`: mixed + emulated FP64; `emu64_path`:
FP64-class results from the INT8 tensor cores on the default workload), each with its own roofline fractions
and its parity against the stored oracle values of tests/golden/.  --no-legs / --no-variants skip them.

Multi-GPU: north_star builds a single-GPU path ("replicas only"): --gpus N runs N
independent replicas, one process per GPU, no data-path collective.  --sharded instead cuts the restricted loop
into N contiguous ranges of window blocks (triples_energy_sharded) and adds the three partial sums of every rank in
rank order: the triplet-sharded mode of SURVEY 8(f) NEXT-3 ("scaling": "strong").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

NAMES = ("eps_o", "eps_v", "t1", "t2", "vvvo", "ovoo", "ovov")
MIXED_DTYPE = "fp16 split x = h + l (f32 accumulate), f64 reduction"
EMU_DTYPE = "f64 emulated: 6 base-256 int8 digits per operand, 21 exact s8 x s8 -> s32 products, f64 recombination and reduction"
GOLDEN_OF = {"small": "small_full", "medium": "medium_full", "large": "large_sample", "largest": "largest_sample"}


def formula_flops(o: int, v: int) -> float:
    T = o * (o + 1) * (o + 2) // 6
    return float(T) * (12.0 * v ** 4 + 12.0 * o * v ** 3)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        keys = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.lines:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for k, val in zip(keys, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(k)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample_seconds(host, trips):
    """Time the CPU oracle (numpy restatement of Eq. (2.2.1)-(2.2.5), one triplet at a time) on `trips`."""
    from oracle import oracle

    t0 = time.perf_counter()
    e = oracle.energy_subset_numpy(host["eps_o"], host["eps_v"], host["t1"], host["t2"], host["vvvo"], host["ovoo"],
                                   host["ovov"], trips)
    return time.perf_counter() - t0, e


def oracle_c_loops_rate():
    """The plain C-loop oracle (oracle/triples_oracle.c, no BLAS) as SURVEY 8(d) asks for it: oracle_triples_subset is
    OpenMP-parallel over triplets, so it gets one triplet of configs[1] (small) per host core (at least 4)."""
    from oracle import oracle
    from paper_1609_08094_b200 import synth

    o, v, _ = synth.CONFIGS["small"]
    inp = synth.make_config("small", seed=0)
    cores = oracle.num_threads()
    trips = [t for t in synth.triplet_list(o) if len(set(t)) == 3][: max(cores, 4)]
    t0 = time.perf_counter()
    oracle.energy_subset(o, v, *inp.arrays(), trips)
    dt = time.perf_counter() - t0
    return {"value": len(trips) * (12.0 * v ** 4 + 12.0 * o * v ** 3) / dt / 1e12, "unit": "TFLOP/s", "cores": cores,
            "kind": "oracle (plain C loops, OpenMP over triplets)",
            "sample": f"{len(trips)} triplets of small (16,120), {dt:.1f} s"}


def blas_threads():
    try:
        from threadpoolctl import threadpool_info

        n = [p.get("num_threads", 1) for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else os.cpu_count()
    except Exception:
        return os.cpu_count()


def reduce_over_ranks(local_seconds: float, local_units: float, world: int):
    """MAX of the per-rank times, SUM of the per-rank units (torch.distributed when world > 1)."""
    if world == 1:
        return local_seconds, local_units
    import torch
    import torch.distributed as dist

    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([local_seconds], dtype=torch.float64, device=dev)
    u = torch.tensor([local_units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def combine_shard_partials(partial, world: int):
    """Sharded mode: the only exchange step of the method -- all-gather of (E(T), E[4], E[5]) of every rank, added
    in RANK ORDER on every rank (bitwise reproducible for a fixed world size)."""
    if world == 1:
        return tuple(float(x) for x in partial)
    import torch
    import torch.distributed as dist

    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    mine = torch.tensor(list(partial), dtype=torch.float64, device=dev)
    parts = [torch.zeros(3, dtype=torch.float64, device=dev) for _ in range(world)]
    dist.all_gather(parts, mine)
    tot = [0.0, 0.0, 0.0]
    for p in parts:                       # rank order
        for n in range(3):
            tot[n] += float(p[n].item())
    return tuple(tot)


def run_reference(args, rank, world):
    """--impl reference: the oracle as it stands on the host cores, each step a bounded sample of the workload."""
    if rank != 0:
        return
    from paper_1609_08094_b200 import synth

    o, v, naux = synth.CONFIGS[args.config]
    inp = synth.make_config(args.config, seed=0)
    host = dict(zip(NAMES, inp.arrays()))
    trips = [t for t in synth.sample_triplets(o, 16, seed=0) if not (t[0] == t[1] == t[2])][: args.ref_triplets]
    for _ in range(args.warmup):
        oracle_sample_seconds(host, trips[:1])
    times = []
    for _ in range(args.steps):
        dt, _ = oracle_sample_seconds(host, trips)
        times.append(dt)
    per_step = float(np.mean(times))
    flops = len(trips) * (12.0 * v ** 4 + 12.0 * o * v ** 3)
    value = flops / per_step / 1e12
    sample = f"{len(trips)} of {o*(o+1)*(o+2)//6} triplets per step ({trips}), oracle.energy_subset_numpy"
    kind = "oracle (numpy restatement of Eq. (2.2.1)-(2.2.5), BLAS einsum)"
    line = {
        "impl": "reference", "metric": "(T) TFLOP/s", "value": value, "unit": "TFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": per_step * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, args.precision, o, v, naux), "sample": sample},
        "s_per_ET_extrapolated": formula_flops(o, v) / (value * 1e12),
        "cpu_baseline": {"value": value, "unit": "TFLOP/s", "cores": blas_threads(), "kind": kind, "sample": sample},
        "e2e": {"value": value, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# The timed headline stays on configs[2]: --steps 20 --warmup 5 means ~47 FP64 steps (with the e2e leg); a large /
# largest FP64 step takes 54 s / 215 s, so those configs are one-step legs of the same command (all five configs x
# FP64 are driver-run: tiny/small by the tests, medium here, large and largest as legs).
WHY_MEDIUM = "20+5 steps of large/largest FP64 (54 s / 215 s each) exceed the run limit: they are 1-step legs"


def workload_name(config, precision, o, v, naux):
    return f"{config}: nocc={o} nvirt={v} naux={naux} seed=0, {precision}, full E(T) over all i<=j<=k"


def load_golden(config):
    if config == "tiny":         # configs[0]: all 120 triplets, written by the C-loop oracle (oracle_energies.json)
        with open(os.path.join(ROOT, "tests", "golden", "oracle_energies.json")) as f:
            g = json.load(f)["tiny"]
        o = g["nocc"]
        trips = [[i, j, k] for i in range(o) for j in range(i, o) for k in range(j, o)]
        return {"triplets_ijk": trips, "energies": g["triplets"], "mode": "full", "file": "oracle_energies.json"}
    path = os.path.join(ROOT, "tests", "golden", GOLDEN_OF.get(config, "") + ".json")
    if not os.path.exists(path):
        return None
    with open(path) as f:
        return json.load(f)


def parity_vs_golden(config, et, triplet_index, tol):
    """Largest deviation of the timed run's per-triplet energies from the oracle's stored values (tests/golden/,
    written by tests/golden/make_golden.py from oracle/ only), relative to |w e4| of the triplet."""
    g = load_golden(config)
    if g is None or not g["triplets_ijk"]:
        return None
    want = np.array(g["energies"])
    worst, n_cmp = 0.0, 0
    for n, t in enumerate(g["triplets_ijk"]):
        if t[0] == t[1] == t[2]:
            continue
        got = et[triplet_index[tuple(t)]]
        worst = max(worst, abs(got[0] - want[n, 0]) / abs(want[n, 1]), abs(got[1] - want[n, 1]) / abs(want[n, 1]))
        n_cmp += 1
    return {"max_rel_err": worst, "triplets_compared": n_cmp, "tolerance": tol, "ok": bool(worst <= tol),
            "source": f"tests/golden/{g.get('file', GOLDEN_OF.get(config, '') + '.json')} ({g['mode']}; oracle values), "
                      "against the timed run's e_triplet_out"}


ROOF_KEYS = ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic", "share_of_step", "avg_launch_ms")
LINE_LIMIT = 2500            # bytes: the driver keeps only the last ~3 KB of stdout, and the final line must be whole


def _short(x):
    """Numbers to 6 significant digits, everything else unchanged (keeps the final line small)."""
    if isinstance(x, float):
        return float(f"{x:.6g}")
    if isinstance(x, dict):
        return {k: _short(val) for k, val in x.items()}
    if isinstance(x, (list, tuple)):
        return [_short(val) for val in x]
    return x


def _pick(d, keys):
    return None if d is None else {k: d.get(k) for k in keys if k in d}


def leg_digest(leg):
    """[TFLOP/s, s per E(T), contraction roofline frac, reduction roofline frac, parity max rel err] of one leg."""
    par = leg.get("parity") or {}
    return [leg.get("value"), leg.get("s_per_ET"), (leg.get("roofline") or {}).get("frac"),
            (leg.get("roofline_reduction") or {}).get("frac"), par.get("max_rel_err")]


def compact_line(full):
    """The LAST stdout line: the contract's keys as numbers and short strings only (explanations live in DESIGN.md
    section 10 and in the detail document, which is printed leg by leg before this line and written to a file)."""
    keep = ("metric", "value", "executed_value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
            "scaling", "vs_baseline", "dtype", "data", "gpu_launches", "detail")
    line = {k: full[k] for k in keep if k in full}
    line["config"] = _pick(full.get("config"), ("workload", "parallelism", "l2"))
    line["clocks"] = _pick(full.get("clocks"), ("sm_mhz", "sm_max_mhz", "reasons"))
    line["roofline"] = _pick(full.get("roofline"), ROOF_KEYS)
    line["roofline_reduction"] = _pick(full.get("roofline_reduction"), ROOF_KEYS)
    line["cpu_baseline"] = _pick(full.get("cpu_baseline"), ("value", "unit", "cores", "kind", "sample"))
    line["e2e"] = _pick(full.get("e2e"), ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "api"))
    line["parity"] = _pick(full.get("parity"), ("max_rel_err", "tolerance", "ok", "triplets_compared"))
    digest = {}
    for name in ("mixed_path", "emu64_path", "ri_direct", "streamed"):
        if full.get(name):
            digest[name] = leg_digest(full[name])
    for cfg, legs in (full.get("legs") or {}).items():
        for name, leg in legs.items():
            if isinstance(leg, dict) and "value" in leg:
                digest[f"{cfg}.{name}"] = leg_digest(leg)
    if digest:
        line["legs"] = digest
        line["legs_columns"] = "TFLOP/s, s_per_ET, roofline.frac, roofline_reduction.frac, parity_max_rel_err"
    line = _short(line)
    text = json.dumps(line, separators=(",", ":"))
    if len(text) > LINE_LIMIT:                  # never let an over-long line reach the driver: drop the digest first
        line.pop("legs", None)
        line.pop("legs_columns", None)
        text = json.dumps(line, separators=(",", ":"))
    assert len(text) <= LINE_LIMIT, f"final bench line is {len(text)} bytes (limit {LINE_LIMIT})"
    return text


def emit_leg(name, leg, detail_path=None):
    """One JSON line per leg, printed as soon as the leg is measured (the final line only carries a digest)."""
    print(json.dumps({"leg": name, **leg}), flush=True)


def write_detail(full, path):
    """The whole document (every leg, every note) as a file next to the run; failure to write is not an error."""
    try:
        os.makedirs(os.path.dirname(path) or ".", exist_ok=True)
        with open(path, "w") as f:
            json.dump(full, f, indent=1)
        return path
    except OSError:
        return None


def rooflines(tb, prec, prof, peaks, peak_kind, fp64_peak, traffic):
    """Contraction (tensor pipe) and fused reduction (HBM) rooflines from one profiled step."""
    gemm_tflops = prof["contraction_flops"] / (prof["contraction_ms"] * 1e-3) / 1e12
    red_gbs = prof["reduction_bytes"] / (prof["reduction_ms"] * 1e-3) / 1e9
    step_ms = prof["prepare_ms"] + prof["contraction_ms"] + prof["reduction_ms"] + prof["other_ms"] + prof["slices_ms"]
    nl = max(prof["contraction_launches"], 1)
    # Denominators: FP64 = the DMMA peak probed in this run.  The two tcgen05 kernels: the
    # tcgen05.mma issue-loop rate of their own instruction kind and shape probed in this run (triples_probe_tc_peak,
    # ~2 s = under the power cap, like the kernels inside a long step) divided by the MMAs one product costs: 3 FP16
    # MMAs per FP32-class product (mixed), 21 int8 digit products per FP64-class product (emulated FP64).  The round-2
    # nominal-ratio figures (0.5 x / 2 x sustained cuBLAS bf16) stay beside them as peak_nominal.
    tc = peaks.get("tc_probe")
    if prec == tb.FP64:
        kernel, peak, peak_src, nominal = "gemm_f64_kernel", fp64_peak["tflops"], "dmma probe, this run", None
    elif prec == tb.EMU64:
        kernel, nominal = "gemm_emu64_kernel", peaks["bf16_tflops_sustained"] * 2.0 / 21.0
        peak, peak_src = (tc["i8_sustained"] / 21.0, "tcgen05 kind::i8 probe (sustained), this run / 21") if tc else \
                         (nominal, f"2 x bf16 sustained ({peak_kind}) / 21")
    else:
        kernel, nominal = "gemm_f16split_kernel", peaks["bf16_tflops_sustained"] * 0.5
        peak, peak_src = (tc["f16_sustained"] / 3.0, "tcgen05 kind::f16 probe (sustained), this run / 3") if tc else \
                         (nominal, f"0.5 x bf16 sustained ({peak_kind})")
    roof = {"bound": "tensor", "kernel": kernel, "achieved": gemm_tflops, "peak": peak, "unit": "TFLOP/s",
            "frac": gemm_tflops / peak, "traffic": None, "peak_src": peak_src, "peak_nominal": nominal,
            "share_of_step": prof["contraction_ms"] / step_ms, "launches_per_step": prof["contraction_launches"],
            "flops_per_launch": prof["contraction_flops"] / nl, "avg_launch_ms": prof["contraction_ms"] / nl}
    if prec == tb.MIXED:
        roof["tensor_pipe_fp16"] = 3.0 * gemm_tflops          # FP16-rate work the tensor pipe executes
    if prec == tb.EMU64:
        roof["tensor_pipe_int8"] = 21.0 * gemm_tflops
        roof["vs_native_fp64_peak"] = gemm_tflops / fp64_peak["tflops"]
    nr = max(prof["reduction_launches"], 1)
    red = {"bound": "hbm", "kernel": "reduce_kernel<float>" if prec == tb.MIXED else "reduce_kernel<double>",
           "achieved": red_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": red_gbs / peaks["hbm_gbs"],
           "traffic": None, "peak_src": f"copy bandwidth ({peak_kind})",
           "bytes_per_launch": prof["reduction_bytes"] / nr, "avg_launch_ms": prof["reduction_ms"] / nr}
    for r in (roof, red):
        t = (traffic or {}).get(r["kernel"])
        if t:
            r["traffic"] = t["dram_bytes"]
    return roof, red


def load_traffic(config):
    """ncu --set full DRAM bytes per launch of the dominant kernels (profiles/rNN_ncu_traffic.json; newest round wins)."""
    out = {}
    for rnd in ("r02", "r03"):
        path = os.path.join(ROOT, "profiles", f"{rnd}_ncu_traffic.json")
        if os.path.exists(path):
            with open(path) as f:
                out.update(json.load(f).get(config, {}))
    return out


def timed_steps(fn, steps, warmup, stream, torch):
    """`warmup` untimed calls, then `steps` calls between CUDA events on `stream`; seconds per step and last result."""
    out = None
    for _ in range(warmup):
        out = fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(steps):
        out = fn()
    e1.record(stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / 1e3 / steps, out


def profiled_step(tb, fn):
    tb.triples_set_profiling(True)
    try:
        fn()
        return tb.triples_last_profile()
    finally:
        tb.triples_set_profiling(False)


def precision_leg(tb, torch, config, prec, o, v, dargs, ws, stream, steps, warmup, peaks, peak_kind, fp64_peak, index):
    """One precision of one config: whole-step rate, rooflines of the two dominant kernels, parity vs goldens."""
    T = tb.triples_triplet_count(o)
    et = torch.zeros((T, 3), dtype=torch.float64, device="cuda")
    sampler = ClockSampler(torch.cuda.current_device()).start()
    sec, E = timed_steps(lambda: tb.triples_energy(o, v, *dargs, prec, ws, stream=stream, e_triplet_out=et), steps, warmup,
                         stream, torch)
    clocks = sampler.stop()
    prof = profiled_step(tb, lambda: tb.triples_energy(o, v, *dargs, prec, ws, stream=stream))
    roof, red = rooflines(tb, prec, prof, peaks, peak_kind, fp64_peak, load_traffic(config))
    tol = 1e-5 if prec == tb.MIXED else 1e-10
    leg = {"value": formula_flops(o, v) / sec / 1e12, "executed_value": prof["contraction_flops"] / sec / 1e12,
           "unit": "TFLOP/s", "s_per_ET": sec, "steps": steps, "warmup": warmup,
           "dtype": dtype_name(tb, prec), "E_T": E[0], "E4": E[1], "E5": E[2],
           "roofline": roof, "roofline_reduction": red, "clocks": clocks,
           "parity": parity_vs_golden(config, et.cpu().numpy(), index, tol)}
    return leg, E


def dtype_name(tb, prec):
    return "f64" if prec == tb.FP64 else (MIXED_DTYPE if prec == tb.MIXED else EMU_DTYPE)


def streamed_leg(tb, torch, o, v, d, prec, stream, nslots, win, resident_sec, E_resident, scan=False):
    """Out-of-core run (NEXT-1): vvvo in pinned host memory (slice-major), a device cache of `nslots` slices; the
    H2D copies of the slices are inside the timed region.  One warm-up-free timed call (the copies ARE the point).
    scan: packed precisions only -- pass vvvo_absmax = 0, i.e. what a caller pays who does not know the largest
    |(ab|ck)| of a tensor that is not on the device: the library's own scan pass (one more H2D pass) is then timed too."""
    vv = d["vvvo"]
    host = torch.empty((o, v, v, v), dtype=torch.float64, pin_memory=True)
    for k in range(o):                                  # generator-side reshuffle to the slice-major layout
        host[k].copy_(vv[:, :, :, k])
    torch.cuda.synchronize()
    absmax = float(vv.abs().max().item()) if (prec != tb.FP64 and not scan) else 0.0
    nbytes = tb.triples_workspace_bytes_streamed(o, v, prec, nslots, win)
    slots, w = tb.triples_cache_slots(o, v, 0, prec, 1, nbytes)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    call = lambda: tb.triples_energy_streamed(o, v, d["eps_o"], d["eps_v"], d["t1"], d["t2"], host.numpy(), d["ovoo"],
                                              d["ovov"], prec, ws, stream=stream, vvvo_absmax=absmax)
    torch.cuda.synchronize()
    tb.triples_set_profiling(True)          # per-batch CUDA events of the timed call itself (counts slices and bytes)
    try:
        t0 = time.perf_counter()
        E = call()
        torch.cuda.synchronize()
        sec = time.perf_counter() - t0
        prof = tb.triples_last_profile()
    finally:
        tb.triples_set_profiling(False)
    del ws, host
    return {"api": "triples_energy_streamed (C ABI; vovv_host pinned, slice-major)", "value": formula_flops(o, v) / sec / 1e12,
            "unit": "TFLOP/s", "s_per_ET": sec, "cache_slots": slots, "slices": o, "window": w,
            "device_workspace_bytes": nbytes, "vvvo_bytes": 8 * v ** 3 * o,
            "h2d_bytes_per_step": prof["h2d_bytes"] + 8 * (o + v + o * v), "slices_loaded": prof["slices_loaded"],
            "vs_resident": resident_sec / sec, "bitwise_equal_to_resident": bool(E == E_resident),
            "vvvo_absmax": "n/a (fp64)" if prec == tb.FP64 else ("scanned by the library inside the timed call" if scan
                                                                 else "supplied by the caller"),
            "note": "copies of batch b+2 run on a copy stream while batch b+1 computes; vs_resident = resident s / streamed s "
                    "(1.0 = transfer fully hidden)"}


def paper_size_leg(tb, torch, synth, prec, stream, nslots):
    """--paper-leg: the paper's [ala]-4/cc-pVDZ size (nocc=81, nvirt=323), naux = 3 nvirt, same generator:
    one resident E(T) and one out-of-core E(T) (vvvo 21.8 GB in pinned host memory, `nslots` of 81 slices cached)."""
    o, v, naux = 81, 323, 969
    d = synth.make_inputs_device(o, v, naux, seed=0)
    args_ = [d[k] for k in NAMES]
    ws = torch.empty(tb.triples_workspace_bytes(o, v, prec), dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    E = tb.triples_energy(o, v, *args_, prec, ws, stream=stream)
    torch.cuda.synchronize()
    sec = time.perf_counter() - t0
    del ws
    torch.cuda.empty_cache()
    st = streamed_leg(tb, torch, o, v, d, prec, stream, nslots, 0, sec, E)
    return {"workload": f"paper [ala]-4/cc-pVDZ size: nocc={o} nvirt={v} naux={naux} seed=0, {dtype_name(tb, prec)}",
            "resident": {"value": formula_flops(o, v) / sec / 1e12, "unit": "TFLOP/s", "s_per_ET": sec, "E_T": E[0],
                         "note": "one call, no warm-up (first-call overheads included)"},
            "streamed": st}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", default="medium", choices=["tiny", "small", "medium", "large", "largest"])
    ap.add_argument("--precision", default="fp64", choices=["fp64", "mixed", "emu64"])
    ap.add_argument("--ref-triplets", type=int, default=2, help="triplets per step of the reference arm")
    ap.add_argument("--cpu-triplets", type=int, default=4, help="triplets of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-mixed-leg", action="store_true",
                    help="FP64 runs only: skip the extra mixed-precision measurement reported under 'mixed_path'")
    ap.add_argument("--no-variants", action="store_true", help="skip the RI-direct and streamed measurements")
    ap.add_argument("--no-legs", action="store_true", help="skip the short legs on the large / largest configs")
    ap.add_argument("--no-tc-probe", action="store_true", help="use the nominal-ratio tcgen05 peaks instead of probing them")
    ap.add_argument("--no-largest-fp64", action="store_true", help="legs: skip the one-step native-FP64 E(T) at largest (~215 s)")
    ap.add_argument("--detail-out", default=os.path.join(ROOT, "gpurun_out", "bench_detail.json"),
                    help="file that receives the whole document (all legs and notes); the last stdout line is a digest")
    ap.add_argument("--sharded", action="store_true", help="--gpus N: triplet-sharded run instead of N replicas")
    ap.add_argument("--paper-leg", action="store_true",
                    help="only the paper-size (81,323) resident + out-of-core leg in --precision (minutes; not in the default line)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch

    import paper_1609_08094_b200 as tb
    from paper_1609_08094_b200 import synth

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the (T) hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    prec = {"fp64": tb.FP64, "mixed": tb.MIXED, "emu64": tb.EMU64}[args.precision]
    if args.paper_leg:
        leg = paper_size_leg(tb, torch, synth, prec, torch.cuda.current_stream(), 27)
        print(json.dumps({"metric": "(T) TFLOP/s", "unit": "TFLOP/s", "paper_size_leg": leg, "data": "synthetic",
                          "value": leg["streamed"]["value"], "n_gpus": 1, "higher_is_better": True}), flush=True)
        return
    tol = 1e-5 if prec == tb.MIXED else 1e-10
    o, v, naux = synth.CONFIGS[args.config]
    default_line = args.config == "medium" and prec == tb.FP64 and world == 1
    # ---- synthetic inputs: host copies (pinned, for the e2e leg and the oracle) and device-resident copies
    need_host = (not args.no_e2e) or (rank == 0 and not args.no_cpu_baseline)
    if need_host and args.config in ("tiny", "small", "medium"):
        inp = synth.make_config(args.config, seed=0)
        host = dict(zip(NAMES, inp.arrays()))
        dev = {k: torch.from_numpy(a).cuda() for k, a in host.items()}
        B_host = None
    else:
        d = synth.make_inputs_device(o, v, naux, seed=0)
        dev = {k: d[k] for k in NAMES}
        B_host = d["B_host"]
        host = None
        if need_host:
            host = {k: dev[k].cpu().numpy() for k in NAMES}
    dargs = [dev[k] for k in NAMES]
    mixed_leg = prec == tb.FP64 and world == 1 and not args.no_mixed_leg and args.config in ("tiny", "small", "medium")
    emu_leg = mixed_leg
    ws_bytes = tb.triples_workspace_bytes_host(o, v, prec)
    if mixed_leg:
        ws_bytes = max(ws_bytes, tb.triples_workspace_bytes(o, v, tb.MIXED), tb.triples_workspace_bytes(o, v, tb.EMU64))
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    T = tb.triples_triplet_count(o)
    index = {t: n for n, t in enumerate(synth.triplet_list(o))}

    def barrier():
        if world > 1:
            import torch.distributed as dist

            dist.barrier()
        torch.cuda.synchronize()

    # ---- roofline denominators measured in this run / on this pool
    peaks, peak_kind = measured_peaks()
    fp64_peak = {"tflops": tb.triples_probe_fp64_peak(ws, stream=stream)}     # DMMA issue loop on all SMs, best of 3

    def probe_tc():
        """tcgen05.mma issue loops: 50 ms (burst) and 2 s (under the power cap) per kind -> peaks["tc_probe"]."""
        if args.no_tc_probe or "tc_probe" in peaks:
            return
        tc = {}
        for kind, name in ((0, "f16"), (1, "i8")):
            tc[name + "_burst"], tc[name + "_burst_mhz"] = tb.triples_probe_tc_peak(kind, 0.05, ws, stream=stream)
            tc[name + "_sustained"], tc[name + "_sustained_mhz"] = tb.triples_probe_tc_peak(kind, 2.0, ws, stream=stream)
        tc["unit"] = "Tera-op/s of tcgen05.mma cta_group::2 (f16: M256 N256 K16; i8: M256 N80 K32), SM MHz during the loop"
        peaks["tc_probe"] = tc
        if rank == 0:
            emit_leg("tc_probe", tc)

    peaks = dict(peaks)
    if prec != tb.FP64:          # an FP64 headline does not need them: they run after its timed region (4 s at 1 kW)
        probe_tc()

    # ---- device-resident timing: W warm-up steps, then exactly K steps between CUDA events
    sharded = args.sharded and world > 1
    et = torch.zeros((T, 3), dtype=torch.float64, device="cuda")

    def step():
        if sharded:
            part = tb.triples_energy_sharded(o, v, *dargs, prec, rank, world, ws, stream=stream, e_triplet_out=et)
            return combine_shard_partials(part, world)
        return tb.triples_energy(o, v, *dargs, prec, ws, stream=stream, e_triplet_out=et)

    tb.triples_set_profiling(False)
    E = None
    for _ in range(args.warmup):
        E = step()
    sampler = ClockSampler(local_rank)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    ev0.record(stream)
    for _ in range(args.steps):
        E = step()
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    launches = tb.triples_last_launch_count() * args.steps
    sec = ev0.elapsed_time(ev1) / 1e3
    units = formula_flops(o, v) * args.steps
    sec_max, flops_all = reduce_over_ranks(sec, units / world if sharded else units, world)
    value = flops_all / sec_max / 1e12
    ms_per_step = sec_max / args.steps * 1e3
    et_timed = et.cpu().numpy()

    # ---- per-kernel roofline: one extra profiled step (CUDA events around every launch, on the same stream)
    prof = profiled_step(tb, step)
    roofline, roofline_reduction = rooflines(tb, prec, prof, peaks, peak_kind, fp64_peak, load_traffic(args.config))
    executed_local = prof["contraction_flops"] / (sec / args.steps) / 1e12
    _, executed_value = reduce_over_ranks(sec, executed_local, world)
    if not sharded and world > 1:
        pass                                             # replicas: the sum over ranks is the whole-job rate
    if prec == tb.FP64:                                  # sanity: executed work cannot beat the measured peak
        assert executed_local <= 1.02 * fp64_peak["tflops"], (executed_local, fp64_peak)

    # ---- end-to-end: host (pinned) inputs through triples_energy_host, copies inside the timed region
    e2e = None
    if not args.no_e2e and not sharded:
        pinned = {k: torch.from_numpy(np.ascontiguousarray(host[k])).pin_memory() for k in NAMES}
        hargs = [pinned[k].numpy() for k in NAMES]
        h2d = int(sum(a.nbytes for a in hargs))
        tb.triples_energy_host(o, v, *hargs, prec, ws, stream=stream)          # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            Eh = tb.triples_energy_host(o, v, *hargs, prec, ws, stream=stream)
        torch.cuda.synchronize()
        sec_e = time.perf_counter() - t0
        sec_e_max, flops_e = reduce_over_ranks(sec_e, formula_flops(o, v) * args.steps, world)
        assert Eh == E, "host and device entry points disagree"
        e2e = {"value": flops_e / sec_e_max / 1e12, "unit": "TFLOP/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": 24, "s_per_ET": sec_e_max / args.steps,
               "api": "triples_energy_host (C ABI, host buffers pinned)"}
        del pinned, hargs

    probe_tc()

    # ---- the paper's other precision beside the headline one (its single/double study): same workload
    mixed = None
    if mixed_leg:
        mixed, Em = precision_leg(tb, torch, args.config, tb.MIXED, o, v, dargs, ws, stream, args.steps, 1, peaks,
                                  peak_kind, fp64_peak, index)
        mixed["rel_dev_from_fp64"] = {
            "E_T": abs(Em[0] - E[0]) / abs(E[0]), "E4": abs(Em[1] - E[1]) / abs(E[1]),
            "E5_abs_dev_over_abs_E4": abs(Em[2] - E[2]) / abs(E[1]),
            "note": "tolerance 1e-5 on E(T); E5 is 1e-7..1e-4 of E4 with the generator's t1 ~ N(0,1e-3^2) and a sum of both "
                    "signs, so its deviation is given on the scale of E4 (tests pin E5 with t1 ~ N(0,1))"}
        if rank == 0:
            emit_leg("mixed_path", mixed)

    # ---- FP64-class results from the INT8 tensor cores: same workload, FP64 tolerance
    emu = None
    if emu_leg:
        emu, Ee = precision_leg(tb, torch, args.config, tb.EMU64, o, v, dargs, ws, stream, args.steps, 1, peaks, peak_kind,
                                fp64_peak, index)
        emu["rel_dev_from_fp64"] = {"E_T": abs(Ee[0] - E[0]) / abs(E[0]), "E4": abs(Ee[1] - E[1]) / abs(E[1]),
                                    "E5": abs(Ee[2] - E[2]) / abs(E[2])}
        emu["speedup_over_fp64_path"] = (sec / args.steps) / emu["s_per_ET"]
        if rank == 0:
            emit_leg("emu64_path", emu)

    # ---- CPU baseline: the oracle as it stands on the host cores, bounded sample (rank 0, N=1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        trips = [t for t in synth.sample_triplets(o, 16, seed=0) if not (t[0] == t[1] == t[2])][: args.cpu_triplets]
        dt, e_or = oracle_sample_seconds(host, trips)
        e_gpu = et_timed[[index[t] for t in trips]]            # the TIMED run's per-triplet energies
        parity = float(np.max(np.abs(e_gpu[:, 0] - e_or[:, 0]) / np.abs(e_or[:, 1])))
        cpu_flops = len(trips) * (12.0 * v ** 4 + 12.0 * o * v ** 3)
        cpu = {"value": cpu_flops / dt / 1e12, "unit": "TFLOP/s", "cores": blas_threads(),
               "kind": "oracle", "oracle_form": "numpy restatement of Eq. (2.2.1)-(2.2.5), BLAS einsum",
               "sample": f"{len(trips)} of {T} triplets, oracle.energy_subset_numpy, {dt:.1f} s "
                         f"(full E(T) would take {formula_flops(o, v)/(cpu_flops/dt):.0f} s)",
               "sample_triplets": trips,
               "parity_max_rel_err_on_sample": parity, "parity_ok": bool(parity <= tol),
               "parity_source": "the timed run's e_triplet_out against the oracle run here",
               "c_loops": oracle_c_loops_rate()}
    parity_golden = parity_vs_golden(args.config, et_timed, index, tol) if rank == 0 else None

    # ---- SURVEY 8(f) variants on the same workload: RI-direct slices (NEXT-2) and out-of-core slices (NEXT-1)
    ri = streamed = None
    if default_line and not args.no_variants:
        if B_host is None:
            _, _, B_host, _ = synth.draw_factors(o, v, naux, seed=0)
        Bd = torch.from_numpy(B_host).cuda()
        nb_ri = tb.triples_workspace_bytes_ri(o, v, naux, prec, o, 0)
        ws_ri = ws if nb_ri <= ws.numel() else torch.empty(nb_ri, dtype=torch.uint8, device="cuda")
        call = lambda: tb.triples_energy_ri(o, v, naux, dev["eps_o"], dev["eps_v"], dev["t1"], dev["t2"], Bd, dev["ovoo"],
                                            dev["ovov"], prec, ws_ri, stream=stream)
        sec_ri, Eri = timed_steps(call, 1, 1, stream, torch)
        pri = profiled_step(tb, call)
        ri = {"api": "triples_energy_ri (C ABI; B[naux,n,n] instead of vvvo)", "value": formula_flops(o, v) / sec_ri / 1e12,
              "unit": "TFLOP/s", "s_per_ET": sec_ri, "naux": naux, "cache_slots": o,
              "slices_built": pri["slices_loaded"], "ri_flops": pri["ri_flops"], "ri_ms": pri["slices_ms"],
              "ri_flops_over_contraction_flops": pri["ri_flops"] / pri["contraction_flops"],
              "device_workspace_bytes": nb_ri, "input_bytes_B": int(B_host.nbytes), "vvvo_bytes_not_needed": 8 * v ** 3 * o,
              "rel_dev_from_resident": abs(Eri[0] - E[0]) / abs(E[0]),
              "note": "value counts the method's flops T(12v^4+12ov^3); the slice GEMMs (2 naux v^3 each) are extra work, "
                      "listed as ri_flops; a full cache builds every slice once"}
        del Bd, ws_ri
        d_ = dict(dev)
        streamed = streamed_leg(tb, torch, o, v, d_, prec, stream, 12, 2, sec / args.steps, E)
        emit_leg("ri_direct", ri)
        emit_leg("streamed", streamed)

    # ---- short legs on the two largest single-GPU configs (the driver times only this default command)
    legs = None
    if default_line and not args.no_legs:
        legs = {}
        del dargs, dev, ws, et
        host = None
        import gc
        largest_precs = (tb.MIXED, tb.EMU64) if args.no_largest_fp64 else (tb.MIXED, tb.EMU64, tb.FP64)
        for cfg, precs in (("large", (tb.FP64, tb.MIXED, tb.EMU64)), ("largest", largest_precs)):
            gc.collect()
            torch.cuda.empty_cache()
            lo, lv, lnaux = synth.CONFIGS[cfg]
            t0 = time.perf_counter()
            d = synth.make_inputs_device(lo, lv, lnaux, seed=0)
            torch.cuda.synchronize()
            gen_s = time.perf_counter() - t0
            largs = [d[k] for k in NAMES]
            lws = torch.empty(max(tb.triples_workspace_bytes(lo, lv, p) for p in precs), dtype=torch.uint8, device="cuda")
            lindex = {t: n for n, t in enumerate(synth.triplet_list(lo))}
            pname = {tb.FP64: "fp64", tb.MIXED: "mixed", tb.EMU64: "emu64"}
            leg = {"workload": workload_name(cfg, "+".join(pname[p] for p in precs), lo, lv, lnaux),
                   "input_generation_s": gen_s}
            for p in precs:
                key = pname[p]
                # steps of 7-70 s: one untimed warm-up only where a step is short (large mixed); a first call's
                # one-off costs (module load, attribute calls) are milliseconds
                short = cfg == "large" and p == tb.MIXED
                leg[key], El = precision_leg(tb, torch, cfg, p, lo, lv, largs, lws, stream, 2 if short else 1,
                                             1 if short else 0, peaks, peak_kind, fp64_peak, lindex)
                if cfg == "large" and p in (tb.FP64, tb.EMU64) and not args.no_variants:
                    del lws
                    torch.cuda.empty_cache()
                    leg["streamed_" + key] = streamed_leg(tb, torch, lo, lv, d, p, stream, 16, 2, leg[key]["s_per_ET"], El,
                                                          scan=(p == tb.EMU64))
                    lws = torch.empty(max(tb.triples_workspace_bytes(lo, lv, q) for q in precs), dtype=torch.uint8,
                                      device="cuda")
            legs[cfg] = leg
            emit_leg("legs." + cfg, leg)
            del d, largs, lws

    if rank == 0:
        line = {
            "metric": "(T) TFLOP/s", "value": value, "executed_value": executed_value, "unit": "TFLOP/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "s_per_ET": ms_per_step / 1e3,
            "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
            "dtype": dtype_name(tb, prec), "data": "synthetic",
            "config": {"workload": workload_name(args.config, args.precision, o, v, naux),
                       "parallelism": (f"triplet-sharded x{world}" if sharded else f"replicas x{world}"),
                       "l2": f"inputs larger than L2 (vvvo {8*v**3*o/1e6:.0f} MB, U buffers re-written every batch)",
                       "why_this_config": WHY_MEDIUM if default_line else None},
            "E_T": E[0], "E4": E[1], "E5": E[2],
            "clocks": clocks, "gpu_launches": int(launches),
            "roofline": roofline, "roofline_reduction": roofline_reduction,
            "phase_ms": {k: prof[k] for k in ("prepare_ms", "contraction_ms", "reduction_ms", "other_ms")},
            "fp64_peak_probe": fp64_peak, "tc_probe": peaks.get("tc_probe"),
            "parity": parity_golden, "e2e": e2e, "cpu_baseline": cpu,
        }
        if mixed is not None:
            line["mixed_path"] = mixed
        if emu is not None:
            line["emu64_path"] = emu
        if ri is not None:
            line["ri_direct"] = ri
        if streamed is not None:
            line["streamed"] = streamed
        if legs is not None:
            line["legs"] = legs
        line["detail"] = "legs: one JSON line each above this one"
        path = write_detail(line, args.detail_out)
        if path:
            line["detail"] += "; whole document: " + os.path.relpath(path, ROOT)
        print(compact_line(line), flush=True)
    if world > 1:
        import torch.distributed as dist

        dist.destroy_process_group()


if __name__ == "__main__":
    main()
