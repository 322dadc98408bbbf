"""triples_energy_noalloc: the (T) energy for callers that cannot allocate device memory.

Every other compute entry point wants a caller-allocated workspace.  A plug-in running inside a host program
that has already taken the GPU's memory for its own pool, or code that may not stall on cudaMalloc's device-wide
synchronisation, has no way to produce one; triples_energy_noalloc therefore works out of a 32 MiB array that is
part of the library's device image (include/triples_b200.h states the limit, the first-call set-up and the
sharing rules).  It runs the same kernels as triples_energy, so its results are checked against that path here,
on consecutive calls, because the array is shared and keeps whatever the previous call wrote into it.

This file sorts after the other test files on purpose: under `pytest -x` a failure here hides nothing else.
It passes alone in a fresh process (the first call does the per-device set-up) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest
import torch

import paper_1609_08094_b200 as tb
from paper_1609_08094_b200 import binding, build, synth

# the tolerances of tests/test_parity_gpu.py and tests/test_variants_gpu.py, relative to the reference value
TOL = {tb.FP64: 1e-10, tb.MIXED: 1e-5, tb.EMU64: 1e-10}


def dev(inp):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in inp.arrays()]


def with_workspace(inp, d, prec):
    """The existing path: triples_energy on a workspace the caller allocated."""
    o, v = inp.nocc, inp.nvirt
    et = torch.zeros((tb.triples_triplet_count(o), 3), dtype=torch.float64, device="cuda")
    ws = torch.empty(tb.triples_workspace_bytes(o, v, prec), dtype=torch.uint8, device="cuda")
    E = tb.triples_energy(o, v, *d, prec, ws, e_triplet_out=et)
    return np.array(E), et.cpu().numpy()


def without_workspace(inp, d, prec):
    o, v = inp.nocc, inp.nvirt
    et = torch.full((tb.triples_triplet_count(o), 3), np.nan, dtype=torch.float64, device="cuda")
    E = tb.triples_energy_noalloc(o, v, *d, prec, e_triplet_out=et)
    return np.array(E), et.cpu().numpy()


def close(got, want, tol):
    got, want = np.asarray(got), np.asarray(want)
    return bool(np.all(np.abs(got - want) <= tol * np.max(np.abs(want))))


@pytest.mark.gpu
@pytest.mark.parametrize("prec", [tb.FP64, tb.MIXED, tb.EMU64], ids=["fp64", "mixed", "emu64"])
def test_noalloc_matches_the_workspace_path_on_consecutive_calls(prec):
    """Calls in a row on the shared array: BASELINE.json configs[0], then a smaller odd shape whose buffers overlap
    the first call's leftovers at other offsets, then configs[0] again.  Each must agree with triples_energy
    (E(T), E[4], E[5] and every per-triplet row), and the repeat must reproduce the first call bit for bit."""
    big = synth.make_config("tiny", seed=0)                      # nocc 8, nvirt 40: close to the 32 MiB limit
    odd = synth.make_inputs(6, 27, 40, seed=5, t1_sigma=0.2)     # ragged tiles, padded rows
    runs = []
    for inp in (big, odd, big):
        d = dev(inp)
        want_E, want_et = with_workspace(inp, d, prec)
        got_E, got_et = without_workspace(inp, d, prec)
        assert np.all(np.isfinite(got_et)), "a per-triplet row was never written"
        assert close(got_E, want_E, TOL[prec]), (got_E, want_E)
        assert close(got_et, want_et, TOL[prec])
        runs.append((got_E, got_et))
    assert np.array_equal(runs[0][0], runs[2][0]) and np.array_equal(runs[0][1], runs[2][1])


@pytest.mark.gpu
def test_noalloc_really_does_not_allocate():
    """Device memory in use (driver view, outside torch's cache) is the same before and after a warmed-up call."""
    inp = synth.make_config("tiny", seed=1)
    d = dev(inp)
    tb.triples_energy_noalloc(inp.nocc, inp.nvirt, *d, tb.FP64)      # set-up + module load happen here
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for prec in (tb.FP64, tb.MIXED, tb.EMU64):
        tb.triples_energy_noalloc(inp.nocc, inp.nvirt, *d, prec)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    # first launches of the tcgen05 kernels may still make the driver load code lazily; nothing near a workspace
    assert free0 - free1 < (8 << 20), f"device memory in use grew by {free0 - free1} bytes"


def test_noalloc_refuses_what_does_not_fit():
    """Sizes are checked on the host before any GPU work (so this runs without a GPU): BASELINE.json configs[1]
    needs ~0.5 GB even at the narrowest window and is turned away with EWORKSPACE and both byte counts."""
    build.build()
    L = binding.lib()
    null = ctypes.c_void_p(None)
    e = (ctypes.c_double * 3)()
    for prec in (tb.FP64, tb.MIXED, tb.EMU64):
        rc = L.triples_energy_noalloc(16, 120, null, null, null, null, null, null, null, prec, null, e, null)
        msg = L.triples_last_error().decode()
        assert rc == 2, (rc, msg)                                     # TRIPLES_EWORKSPACE
        assert str(binding.NOALLOC_SCRATCH_BYTES) in msg and "triples_energy" in msg
    assert L.triples_energy_noalloc(0, 40, null, null, null, null, null, null, null, 0, null, e, null) == 1
    assert L.triples_energy_noalloc(8, 40, null, null, null, null, null, null, null, 9, null, e, null) == 1
    # configs[0] fits in every precision: the call gets past the size check and stops at the null pointers
    for prec in (tb.FP64, tb.MIXED, tb.EMU64):
        assert L.triples_energy_noalloc(8, 40, null, null, null, null, null, null, null, prec, null, e, null) == 1
        assert "null pointer" in L.triples_last_error().decode()
