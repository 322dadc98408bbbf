#!/usr/bin/env python
"""Benchmark of the B200 closed-shell (T) energy path (arXiv:1609.08094 section 2.2).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config medium] [--precision fp64|mixed]
    python bench.py --impl reference ...          # the CPU oracle, timed on the host cores

A "step" is one pass of the whole hot path -- repack, every contraction batch, every fused reduction batch,
the per-triplet finalize and the total -- i.e. one E(T) of the workload.  Prints ONE JSON line (rank 0).

Metric: (T) TFLOP/s = T*(12 v^4 + 12 o v^3) / seconds per E(T), T = o(o+1)(o+2)/6 (Eq. (5.0.7b)),
the paper's task count (i=j=k tasks included although they contribute zero and are skipped).
Multi-GPU: the path is single-GPU by north_star ("replicas only"): --gpus N runs N independent
replicas of the same workload, one process per GPU; no data-path collective.
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
FP64_DMMA_PEAK_TFLOPS = 37.0   # measured, profiles/r01_fp64_peak_probe.txt (148 SM x 128 flop/clk x 1.965 GHz = 37.2)


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
    line = {
        "impl": "reference", "metric": "(T) TFLOP/s", "value": value, "unit": "TFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": per_step * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args, o, v, naux), "sample": sample},
        "s_per_ET_extrapolated": formula_flops(o, v) / (value * 1e12),
        "cpu_baseline": {"value": value, "unit": "TFLOP/s", "cores": blas_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_name(args, o, v, naux):
    return f"{args.config}: nocc={o} nvirt={v} naux={naux} seed=0, {args.precision}, full E(T) over all i<=j<=k"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", default="medium", choices=["tiny", "small", "medium", "large", "largest"])
    ap.add_argument("--precision", default="fp64", choices=["fp64", "mixed"])
    ap.add_argument("--ref-triplets", type=int, default=2, help="triplets per step of the reference arm")
    ap.add_argument("--cpu-triplets", type=int, default=4, help="triplets of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-mixed-leg", action="store_true",
                    help="FP64 runs only: skip the extra mixed-precision measurement reported under 'mixed_path'")
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

    prec = tb.FP64 if args.precision == "fp64" else tb.MIXED
    o, v, naux = synth.CONFIGS[args.config]
    # ---- synthetic inputs: host copies (pinned, for the e2e leg and the oracle) and device-resident copies
    need_host = (not args.no_e2e) or (rank == 0 and not args.no_cpu_baseline)
    if need_host and args.config in ("tiny", "small", "medium"):
        inp = synth.make_config(args.config, seed=0)
        host = dict(zip(NAMES, inp.arrays()))
        dev = {k: torch.from_numpy(a).cuda() for k, a in host.items()}
    else:
        d = synth.make_inputs_device(o, v, naux, seed=0)
        dev = {k: d[k] for k in NAMES}
        host = None
        if need_host:
            host = {k: dev[k].cpu().numpy() for k in NAMES}
    dargs = [dev[k] for k in NAMES]
    mixed_leg = prec == tb.FP64 and world == 1 and not args.no_mixed_leg and args.config in ("tiny", "small", "medium")
    ws_bytes = tb.triples_workspace_bytes_host(o, v, prec)
    if mixed_leg:
        ws_bytes = max(ws_bytes, tb.triples_workspace_bytes(o, v, tb.MIXED))
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            import torch.distributed as dist

            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then exactly K steps between CUDA events
    tb.triples_set_profiling(False)
    E = None
    for _ in range(args.warmup):
        E = tb.triples_energy(o, v, *dargs, prec, ws, stream=stream)
    sampler = ClockSampler(local_rank)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    ev0.record(stream)
    for _ in range(args.steps):
        E = tb.triples_energy(o, v, *dargs, prec, ws, stream=stream)
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    launches = tb.triples_last_launch_count() * args.steps
    sec = ev0.elapsed_time(ev1) / 1e3
    sec_max, flops_all = reduce_over_ranks(sec, formula_flops(o, v) * args.steps, world)
    value = flops_all / sec_max / 1e12
    ms_per_step = sec_max / args.steps * 1e3

    # ---- per-kernel roofline: one extra profiled step (CUDA events around every launch, on the same stream)
    tb.triples_set_profiling(True)
    tb.triples_energy(o, v, *dargs, prec, ws, stream=stream)
    prof = tb.triples_last_profile()
    tb.triples_set_profiling(False)
    peaks, peak_kind = measured_peaks()
    gemm_tflops = prof["contraction_flops"] / (prof["contraction_ms"] * 1e-3) / 1e12
    red_gbs = prof["reduction_bytes"] / (prof["reduction_ms"] * 1e-3) / 1e9
    if prec == tb.FP64:
        peak, peak_note = FP64_DMMA_PEAK_TFLOPS, ("FP64 DMMA peak measured on this pool's B200 with a register-resident "
                                                  "mma.sync.m8n8k4.f64 loop (profiles/r01_fp64_peak_probe.txt)")
    else:
        peak = peaks["bf16_tflops_sustained"] * 0.5
        peak_note = (f"TF32 dense = 0.5 x bf16 sustained cuBLAS ({peak_kind}, MEASURED_PEAKS.json; nominal ratio of the "
                     "profiling guide). achieved = ALGORITHMIC flops (12v^4+12ov^3 per executed job triple); the split "
                     "h*h' + h*l' + l*h' runs as three FP16 MMAs (K=16), i.e. 1.5x that many TF32-rate flops of "
                     "tensor-pipe time: see tensor_pipe_tf32_equiv / frac_tensor_pipe")
    roofline = {
        "bound": "tensor", "kernel": "gemm_f64_kernel" if prec == tb.FP64 else "gemm_tf32_kernel",
        "achieved": gemm_tflops, "peak": peak, "unit": "TFLOP/s", "frac": gemm_tflops / peak, "traffic": None,
        "peak_note": peak_note,
        "share_of_step": prof["contraction_ms"] / (prof["prepare_ms"] + prof["contraction_ms"] + prof["reduction_ms"] +
                                                   prof["other_ms"]),
        "launches_per_step": prof["contraction_launches"],
        "flops_per_launch": prof["contraction_flops"] / max(prof["contraction_launches"], 1),
        "avg_launch_ms": prof["contraction_ms"] / max(prof["contraction_launches"], 1),
    }
    if prec != tb.FP64:
        roofline["tensor_pipe_tf32_equiv"] = 1.5 * gemm_tflops
        roofline["frac_tensor_pipe"] = 1.5 * gemm_tflops / peak
    roofline_reduction = {
        "bound": "hbm", "kernel": "reduce_kernel", "achieved": red_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
        "frac": red_gbs / peaks["hbm_gbs"], "traffic": None, "peak_note": f"{peak_kind} copy bandwidth",
        "bytes_per_launch": prof["reduction_bytes"] / max(prof["reduction_launches"], 1),
        "avg_launch_ms": prof["reduction_ms"] / max(prof["reduction_launches"], 1),
    }

    # DRAM traffic per launch of the captured batch (ncu --set full summary committed under profiles/; medium only)
    tpath = os.path.join(ROOT, "profiles", "r01_ncu_traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as f:
            tr = json.load(f).get(args.config, {})
        g = tr.get(roofline["kernel"])
        r = tr.get("reduce_kernel<double>" if prec == tb.FP64 else "reduce_kernel<float>")
        if g:
            roofline["traffic"] = g["dram_bytes"]
            roofline["traffic_note"] = (f"ncu dram bytes of one captured launch ({g.get('jobs_in_launch')} jobs, "
                                        "profiles/r01_ncu_full_medium.md); launches differ in size")
        if r:
            roofline_reduction["traffic"] = r["dram_bytes"]
            roofline_reduction["traffic_note"] = "ncu dram bytes of one captured launch (profiles/r01_ncu_full_medium.md)"

    # ---- end-to-end: host (pinned) inputs through triples_energy_host, copies inside the timed region
    e2e = None
    if not args.no_e2e:
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

    # ---- the paper's other precision beside the headline one (its single/double study): same workload
    mixed = None
    if mixed_leg:
        tb.triples_energy(o, v, *dargs, tb.MIXED, ws, stream=stream)            # warm-up
        m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        m0.record(stream)
        for _ in range(args.steps):
            Em = tb.triples_energy(o, v, *dargs, tb.MIXED, ws, stream=stream)
        m1.record(stream)
        torch.cuda.synchronize()
        msec = m0.elapsed_time(m1) / 1e3 / args.steps
        tb.triples_set_profiling(True)
        tb.triples_energy(o, v, *dargs, tb.MIXED, ws, stream=stream)
        mp = tb.triples_last_profile()
        tb.triples_set_profiling(False)
        mg = mp["contraction_flops"] / (mp["contraction_ms"] * 1e-3) / 1e12
        mr = mp["reduction_bytes"] / (mp["reduction_ms"] * 1e-3) / 1e9
        tf32_peak = peaks["bf16_tflops_sustained"] * 0.5
        mixed = {"value": formula_flops(o, v) / msec / 1e12, "unit": "TFLOP/s", "s_per_ET": msec,
                 "dtype": "fp16 split x = h + l (f32 accumulate), f64 reduction",
                 "E_T": Em[0], "E4": Em[1], "E5": Em[2],
                 "rel_dev_from_fp64": {"E_T": abs(Em[0] - E[0]) / abs(E[0]), "E4": abs(Em[1] - E[1]) / abs(E[1]),
                                       "E5_abs_dev_over_abs_E4": abs(Em[2] - E[2]) / abs(E[1]),
                                       "note": "tolerance 1e-5 on E(T); E5 is 1e-7..1e-4 of E4 with the generator's "
                                               "t1 ~ N(0,1e-3^2) and a sum of both signs, so its deviation is "
                                               "given on the scale of E4 (tests pin E5 with t1 ~ N(0,1))"},
                 "contraction": {"kernel": "gemm_tf32_kernel", "achieved": mg, "peak": tf32_peak, "unit": "TFLOP/s",
                                 "frac": mg / tf32_peak, "frac_tensor_pipe": 1.5 * mg / tf32_peak,
                                 "peak_note": "0.5 x measured sustained bf16; frac = algorithmic flops, "
                                              "frac_tensor_pipe = TF32-rate-equivalent tensor work (DESIGN.md 7.2)"},
                 "reduction": {"kernel": "reduce_kernel<float>", "achieved": mr, "peak": peaks["hbm_gbs"],
                               "unit": "GB/s", "frac": mr / peaks["hbm_gbs"]}}

    # ---- CPU baseline: the oracle as it stands on the host cores, bounded sample (rank 0, N=1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        trips = [t for t in synth.sample_triplets(o, 16, seed=0) if not (t[0] == t[1] == t[2])][: args.cpu_triplets]
        dt, e_or = oracle_sample_seconds(host, trips)
        e_gpu = tb.triples_energy_subset(o, v, *dargs, prec, trips, ws, stream=stream)
        tol = 1e-10 if prec == tb.FP64 else 1e-5
        parity = float(np.max(np.abs(e_gpu[:, 0] - e_or[:, 0]) / np.abs(e_or[:, 1])))
        cpu_flops = len(trips) * (12.0 * v ** 4 + 12.0 * o * v ** 3)
        cpu = {"value": cpu_flops / dt / 1e12, "unit": "TFLOP/s", "cores": blas_threads(), "kind": "oracle",
               "sample": f"{len(trips)} of {o*(o+1)*(o+2)//6} triplets ({trips}) via oracle.energy_subset_numpy, "
                         f"{dt:.1f} s; full E(T) extrapolated {formula_flops(o, v)/(cpu_flops/dt):.0f} s",
               "parity_max_rel_err_on_sample": parity, "parity_ok": bool(parity <= tol)}

    if rank == 0:
        line = {
            "metric": "(T) TFLOP/s", "value": value, "unit": "TFLOP/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "s_per_ET": ms_per_step / 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if prec == tb.FP64 else "fp16 split x = h + l (f32 accumulate), f64 reduction", "data": "synthetic",
            "config": {"workload": workload_name(args, o, v, naux), "parallelism": f"replicas x{world}",
                       "l2": f"inputs larger than L2 (vvvo {8*v**3*o/1e6:.0f} MB, U buffers re-written every batch)",
                       "flop_count": "T*(12v^4+12ov^3), T=o(o+1)(o+2)/6 (paper's task count, Eq. 5.0.7b)"},
            "E_T": E[0], "E4": E[1], "E5": E[2],
            "clocks": clocks, "gpu_launches": int(launches),
            "roofline": roofline, "roofline_reduction": roofline_reduction,
            "phase_ms": {k: prof[k] for k in ("prepare_ms", "contraction_ms", "reduction_ms", "other_ms")},
            "e2e": e2e, "cpu_baseline": cpu,
        }
        if mixed is not None:
            line["mixed_path"] = mixed
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist

        dist.destroy_process_group()


if __name__ == "__main__":
    main()
