"""GPU tests of the SURVEY.md 8(f) rows built on the same kernels as triples_energy: out-of-core streaming of the
(vv|vo) slices (NEXT-1), the RI-direct slice build (NEXT-2; Eq. (2.1.3)) and the
triplet-sharded run (NEXT-3; L119-L121).  Each is compared with the CPU oracle and with the resident run."""
import numpy as np
import pytest
import torch

import paper_1609_08094_b200 as tb
from oracle import oracle
from paper_1609_08094_b200 import synth

pytestmark = pytest.mark.gpu

TOL = {tb.FP64: 1e-10, tb.MIXED: 1e-5, tb.EMU64: 1e-10}
STREAMED, RI = 1, 2


def dev(inp):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in inp.arrays()]


def ws_bytes(n):
    return torch.empty(n, dtype=torch.uint8, device="cuda")


def resident(inp, prec):
    o, v = inp.nocc, inp.nvirt
    d = dev(inp)
    et = torch.zeros((tb.triples_triplet_count(o), 3), dtype=torch.float64, device="cuda")
    E = tb.triples_energy(o, v, *d, prec, ws_bytes(tb.triples_workspace_bytes(o, v, prec)), e_triplet_out=et)
    return E, et.cpu().numpy(), d


def slice_major_host(inp):
    """vovv_host[k,a,b,c] = (ab|ck), pinned (the layout triples_energy_streamed reads; generator-side reshuffle)."""
    t = torch.from_numpy(np.ascontiguousarray(inp.vvvo.transpose(3, 0, 1, 2))).pin_memory()
    return t, t.numpy()


@pytest.mark.parametrize("prec", [tb.FP64, tb.MIXED, tb.EMU64], ids=["fp64", "mixed", "emu64"])
@pytest.mark.parametrize("o,v,naux,win,extra", [(6, 24, 40, 1, 0), (7, 33, 40, 1, 1), (9, 40, 50, 2, 0), (14, 64, 70, 2, 2),
                                                (5, 17, 30, 0, 0)])
def test_streamed_is_bitwise_the_resident_run(o, v, naux, win, extra, prec):
    """A device budget that holds only a few slices: per-triplet energies equal the resident path bit for bit."""
    inp = synth.make_inputs(o, v, naux, seed=11, t1_sigma=0.2)
    E, et, d = resident(inp, prec)
    keep, host = slice_major_host(inp)
    lo = tb.triples_workspace_bytes_streamed(o, v, prec, 0, win)
    n0, _ = tb.triples_cache_slots(o, v, 0, prec, STREAMED, lo)
    nbytes = tb.triples_workspace_bytes_streamed(o, v, prec, n0 + extra, win)
    nslots, w = tb.triples_cache_slots(o, v, 0, prec, STREAMED, nbytes)
    assert nslots == min(o, n0 + extra)
    if nslots < o:
        loads, _, _ = tb.triples_plan_slices(o, v, prec, STREAMED, nslots, w)
        assert len(loads) > o                                  # slices really are evicted and re-loaded
    ets = torch.zeros_like(torch.from_numpy(et)).cuda()
    for absmax in ([0.0] if prec == tb.FP64 else [0.0, float(np.abs(inp.vvvo).max())]):
        Es = tb.triples_energy_streamed(o, v, d[0], d[1], d[2], d[3], host, d[5], d[6], prec, ws_bytes(nbytes),
                                        e_triplet_out=ets, vvvo_absmax=absmax)
        assert Es == E
        assert np.array_equal(ets.cpu().numpy(), et)
    Eo = oracle.energy_restricted(o, v, *inp.arrays())
    assert abs(E[0] - Eo[0]) <= TOL[prec] * abs(Eo[0])


def test_streamed_profile_counts_slices_and_bytes():
    o, v, naux = 9, 40, 50
    inp = synth.make_inputs(o, v, naux, seed=2)
    d = dev(inp)
    keep, host = slice_major_host(inp)
    nbytes = tb.triples_workspace_bytes_streamed(o, v, tb.FP64, 0, 1)
    loads, _, info = tb.triples_plan_slices(o, v, tb.FP64, STREAMED, 0, 1)
    tb.triples_set_profiling(True)
    try:
        tb.triples_energy_streamed(o, v, d[0], d[1], d[2], d[3], host, d[5], d[6], tb.FP64, ws_bytes(nbytes))
        p = tb.triples_last_profile()
    finally:
        tb.triples_set_profiling(False)
    assert p["slices_loaded"] == len(loads) and p["h2d_bytes"] == len(loads) * 8 * v ** 3


@pytest.mark.parametrize("prec", [tb.FP64, tb.MIXED, tb.EMU64], ids=["fp64", "mixed", "emu64"])
@pytest.mark.parametrize("o,v,naux,slots", [(3, 5, 9, 0), (6, 24, 37, 0), (8, 40, 120, 0), (7, 33, 50, 7), (9, 48, 130, 4),
                                            (5, 130, 40, 0)])
def test_ri_direct_matches_the_oracle(o, v, naux, slots, prec):
    """No vvvo tensor on the device: slices rebuilt from B.  Full E(T), E[4], E[5] and every triplet vs the oracle
    (which is fed the B-built integrals of the same generator)."""
    inp = synth.make_inputs(o, v, naux, seed=4, t1_sigma=0.3)
    _, _, B, _ = synth.draw_factors(o, v, naux, seed=4, t1_sigma=0.3)
    d = dev(inp)
    Bd = torch.from_numpy(B).cuda()
    nbytes = tb.triples_workspace_bytes_ri(o, v, naux, prec, slots, 0)
    et = torch.zeros((tb.triples_triplet_count(o), 3), dtype=torch.float64, device="cuda")
    tb.triples_set_profiling(True)
    try:
        E = tb.triples_energy_ri(o, v, naux, d[0], d[1], d[2], d[3], Bd, d[5], d[6], prec, ws_bytes(nbytes), e_triplet_out=et)
        p = tb.triples_last_profile()
    finally:
        tb.triples_set_profiling(False)
    (Eo, et_o) = oracle.energy_restricted(o, v, *inp.arrays(), with_triplets=True)
    scale = abs(Eo[1])
    for n in range(3):
        assert abs(E[n] - Eo[n]) <= TOL[prec] * max(abs(Eo[n]), 1e-3 * scale), (n, E, Eo)
    assert np.abs(et.cpu().numpy() - et_o).max() <= TOL[prec] * np.abs(et_o).max()
    assert p["slices_loaded"] >= o - (1 if o == 1 else 0) and p["ri_flops"] == p["slices_loaded"] * 2.0 * naux * v ** 3
    if prec == tb.FP64:       # same contraction kernels, operands equal up to the rounding order of the slice build
        Er, etr, _ = resident(inp, prec)
        assert abs(E[0] - Er[0]) <= 1e-12 * abs(Er[0])


@pytest.mark.parametrize("prec", [tb.FP64, tb.MIXED, tb.EMU64], ids=["fp64", "mixed", "emu64"])
@pytest.mark.parametrize("o,v,naux,nshards", [(6, 24, 40, 2), (9, 40, 50, 3), (8, 40, 120, 8), (3, 9, 12, 5)])
def test_sharded_partials_add_up_to_the_full_run(o, v, naux, nshards, prec):
    inp = synth.make_inputs(o, v, naux, seed=8, t1_sigma=0.2)
    E, et, d = resident(inp, prec)
    ws = ws_bytes(tb.triples_workspace_bytes(o, v, prec))
    _, sot, _ = tb.triples_plan_shards(o, v, prec, nshards)
    tot = np.zeros(3)
    seen = np.zeros_like(et)
    for s in range(nshards):
        ets = torch.zeros((len(et), 3), dtype=torch.float64, device="cuda")
        part = tb.triples_energy_sharded(o, v, *d, prec, s, nshards, ws, e_triplet_out=ets)
        ets = ets.cpu().numpy()
        mine = sot == s
        assert np.array_equal(ets[mine], et[mine]) and np.all(ets[~mine] == 0.0)     # bitwise the full run's rows
        seen += ets
        tot += np.array(part)                                                         # added in shard order
    assert np.array_equal(seen, et)
    for n in range(3):
        assert abs(tot[n] - E[n]) <= 1e-13 * abs(E[1])
    # ... and against the oracle, not only against the library's own resident run: the union of the shards' rows
    # and the rank-ordered total (a wrong row index after the shard selection would be common to both GPU paths)
    (Eo, et_o) = oracle.energy_restricted(o, v, *inp.arrays(), with_triplets=True)
    assert np.abs(seen - et_o).max() <= TOL[prec] * np.abs(et_o).max()
    for n in range(3):
        assert abs(tot[n] - Eo[n]) <= TOL[prec] * max(abs(Eo[n]), 1e-3 * abs(Eo[1])), (n, tot, Eo)


@pytest.mark.parametrize("prec", [tb.FP64, tb.MIXED, tb.EMU64], ids=["fp64", "mixed", "emu64"])
def test_sharded_small_config_against_oracle_goldens(prec):
    """BASELINE.json configs[1] (nocc 16, nvirt 120) cut into three shards: every triplet row, collected from the
    shard that owns it, against the stored oracle values of tests/golden/small_full.json, and the rank-ordered sum of
    the three partials against the stored E(T), E[4], E[5] (the cycles are independent)."""
    import json
    import os
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "small_full.json")) as f:
        g = json.load(f)
    o, v, naux = synth.CONFIGS["small"]
    assert (g["nocc"], g["nvirt"], g["naux"], g["seed"], g["complete"]) == (o, v, naux, 0, True)
    inp = synth.make_config("small", seed=0)
    d = dev(inp)
    ws = ws_bytes(tb.triples_workspace_bytes(o, v, prec))
    nshards = 3
    _, sot, jobs = tb.triples_plan_shards(o, v, prec, nshards)
    assert jobs.min() > 0 and jobs.max() <= 1.35 * jobs.min()
    T = tb.triples_triplet_count(o)
    seen = np.zeros((T, 3))
    tot = np.zeros(3)
    for s in range(nshards):
        ets = torch.zeros((T, 3), dtype=torch.float64, device="cuda")
        part = tb.triples_energy_sharded(o, v, *d, prec, s, nshards, ws, e_triplet_out=ets)
        ets = ets.cpu().numpy()
        assert np.all(ets[sot != s] == 0.0)
        seen += ets
        tot += np.array(part)
    index = {t: n for n, t in enumerate(synth.triplet_list(o))}
    want = np.array(g["energies"])
    for n, t in enumerate(g["triplets_ijk"]):
        got = seen[index[tuple(t)]]
        if t[0] == t[1] == t[2]:
            assert np.all(got == 0.0)
            continue
        s4 = abs(want[n, 1])
        assert abs(got[0] - want[n, 0]) <= TOL[prec] * s4 and abs(got[1] - want[n, 1]) <= TOL[prec] * s4, (t, got, want[n])
        assert abs(got[2] - want[n, 2]) <= max(TOL[prec] * s4, 100 * TOL[prec] * abs(want[n, 2])), (t, got, want[n])
    for n in range(2):
        assert abs(tot[n] - g["E"][n]) <= TOL[prec] * abs(g["E"][n]), (n, tot, g["E"])


@pytest.mark.parametrize("prec", [tb.MIXED, tb.EMU64], ids=["mixed", "emu64"])
def test_streamed_run_rejects_a_vvvo_absmax_that_is_too_small(prec):
    """The caller's vvvo_absmax fixes the operand scale of both packed paths.  Too large only costs precision; too
    small used to overflow FP16 (mixed) / wrap the top digit (emulated FP64) silently: now TRIPLES_EINVAL."""
    o, v = 7, 33
    inp = synth.make_inputs(o, v, 40, seed=3, t1_sigma=0.2)
    # (vv|vo) and (ov|oo) share one scale (the integral class); the generator's largest (ov|oo) exceeds its largest
    # (vv|vo) and would hide an under-stated vvvo_absmax, so the (ov|oo) block is shrunk for this test
    inp.ovoo = np.ascontiguousarray(inp.ovoo / 64.0)
    assert np.abs(inp.ovoo).max() < np.abs(inp.vvvo).max() / 8.0
    E, et, d = resident(inp, prec)
    keep, host = slice_major_host(inp)
    nbytes = tb.triples_workspace_bytes_streamed(o, v, prec, 0, 1)
    true_max = float(np.abs(inp.vvvo).max())
    call = lambda m: tb.triples_energy_streamed(o, v, d[0], d[1], d[2], d[3], host, d[5], d[6], prec, ws_bytes(nbytes),
                                                vvvo_absmax=m)
    assert call(true_max) == E
    Ebig = call(true_max * 5.0)                         # two to three bits of headroom wasted, nothing else
    assert abs(Ebig[0] - E[0]) <= 8 * TOL[prec] * abs(E[0])
    for too_small in (true_max / 2.5, true_max / 7.0):
        with pytest.raises(tb.TriplesError) as err:
            call(too_small)
        assert err.value.status == 1 and "vvvo_absmax" in str(err.value)
    assert call(0.0) == E                               # the library stays usable, and its own scan gives the same scale


def test_host_pointer_where_a_device_pointer_is_expected_is_einval():
    """cudaPointerGetAttributes check (no sticky CUDA fault): the library stays usable afterwards."""
    import ctypes
    inp = synth.make_inputs(3, 8, 10, seed=0)
    o, v = inp.nocc, inp.nvirt
    d = dev(inp)
    ws = ws_bytes(tb.triples_workspace_bytes(o, v, tb.FP64))
    L = tb.binding.lib()
    host_t2 = np.ascontiguousarray(inp.t2)
    e_out = (ctypes.c_double * 3)()
    ptrs = [ctypes.c_void_p(t.data_ptr()) for t in d]
    ptrs[3] = ctypes.c_void_p(host_t2.ctypes.data)
    rc = L.triples_energy(o, v, *ptrs, tb.FP64, ctypes.c_void_p(ws.data_ptr()), ws.numel(), None, e_out, None)
    assert rc == 1 and b"not a device pointer" in L.triples_last_error()
    E = tb.triples_energy(o, v, *d, tb.FP64, ws)
    Eo = oracle.energy_restricted(o, v, *inp.arrays())
    assert abs(E[0] - Eo[0]) <= 1e-10 * abs(Eo[0])


def test_binding_rejects_wrong_sizes():
    inp = synth.make_inputs(3, 8, 10, seed=0)
    o, v = inp.nocc, inp.nvirt
    d = dev(inp)
    ws = ws_bytes(tb.triples_workspace_bytes(o, v, tb.FP64))
    with pytest.raises(ValueError):
        tb.triples_energy(v, o, *d, tb.FP64, ws)                      # swapped o / v
    with pytest.raises(ValueError):
        tb.triples_energy(o, v, *d, tb.FP64, ws, e_triplet_out=torch.zeros(5, dtype=torch.float64, device="cuda"))


def test_fp64_peak_probe():
    ws = ws_bytes(1 << 20)
    tf = tb.triples_probe_fp64_peak(ws, iters=4000)
    assert 20.0 < tf < 60.0, tf           # B200: 148 SM x 128 flop/clk x ~1.9 GHz = ~37 TFLOP/s


# ------------------------------------------------------------------------------------------------------------------
# BASELINE.json configs at full size through the NEXT-1 / NEXT-2 entry points, against the stored oracle values
# ------------------------------------------------------------------------------------------------------------------
def _golden(name):
    import json
    import os
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name + ".json")) as f:
        return json.load(f)


def _check_against_golden(g, et, o, tol):
    index = {t: n for n, t in enumerate(synth.triplet_list(o))}
    want = np.array(g["energies"])
    n_cmp = 0
    for n, t in enumerate(g["triplets_ijk"]):
        if t[0] == t[1] == t[2]:
            continue
        got = et[index[tuple(t)]]
        assert abs(got[0] - want[n, 0]) <= tol * abs(want[n, 1]) and abs(got[1] - want[n, 1]) <= tol * abs(want[n, 1]), (t, got, want[n])
        n_cmp += 1
    return n_cmp


@pytest.mark.parametrize("prec", [tb.FP64, tb.MIXED, tb.EMU64], ids=["fp64", "mixed", "emu64"])
def test_medium_streamed_with_a_budget_below_vvvo_is_bitwise_the_resident_run(prec):
    """configs[2] (vvvo 2.65 GB) with a device workspace SMALLER than what it streams -- the vvvo tensor (FP64) or the
    packed X / XT operands of all slices (mixed 2.8 GB, emulated FP64 4.2 GB): window 1, six cache slots, 2576 batches,
    ~3000 slice loads; on the packed paths every load goes through the FP64 staging ring and is split / digitised on
    the device.  Per-triplet energies bitwise equal to the resident run, and within the precision's tolerance of the
    oracle's stored values."""
    o, v, naux = synth.CONFIGS["medium"]
    d = synth.make_inputs_device(o, v, naux, seed=0)
    args = [d[k] for k in ("eps_o", "eps_v", "t1", "t2", "vvvo", "ovoo", "ovov")]
    T = tb.triples_triplet_count(o)
    et = torch.zeros((T, 3), dtype=torch.float64, device="cuda")
    ws = ws_bytes(tb.triples_workspace_bytes(o, v, prec))
    E = tb.triples_energy(o, v, *args, prec, ws, e_triplet_out=et)
    del ws
    host = torch.empty((o, v, v, v), dtype=torch.float64, pin_memory=True)
    for k in range(o):
        host[k].copy_(d["vvvo"][:, :, :, k])
    torch.cuda.synchronize()
    nbytes = tb.triples_workspace_bytes_streamed(o, v, prec, 0, 1)
    vk = {tb.MIXED: (v + 31) // 32 * 32, tb.EMU64: (v + 63) // 64 * 96}
    streamed_bytes = 8 * v ** 3 * o if prec == tb.FP64 else 2 * o * v * v * vk[prec] * 4
    assert nbytes < streamed_bytes, "the budget must be smaller than the operands that are streamed"
    assert tb.triples_cache_slots(o, v, 0, prec, STREAMED, nbytes) == (6, 1)
    ets = torch.zeros_like(et)
    Es = tb.triples_energy_streamed(o, v, d["eps_o"], d["eps_v"], d["t1"], d["t2"], host.numpy(), d["ovoo"], d["ovov"],
                                    prec, ws_bytes(nbytes), e_triplet_out=ets)
    assert Es == E and torch.equal(ets, et)
    g = _golden("medium_full")
    assert _check_against_golden(g, ets.cpu().numpy(), o, TOL[prec]) >= 64


@pytest.mark.parametrize("name,prec", [("small", tb.FP64), ("small", tb.MIXED), ("small", tb.EMU64), ("medium", tb.FP64)],
                         ids=["small-fp64", "small-mixed", "small-emu64", "medium-fp64"])
def test_ri_direct_at_config_size_against_oracle_goldens(name, prec):
    """configs[1..2] without a vvvo tensor on the device: every stored triplet of the oracle's full goldens."""
    o, v, naux = synth.CONFIGS[name]
    eps_o, eps_v, t1, t2, ovoo, ovov, B = synth.make_inputs_sliced(o, v, naux, seed=0)
    dv = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (eps_o, eps_v, t1, t2, B, ovoo, ovov)]
    T = tb.triples_triplet_count(o)
    et = torch.zeros((T, 3), dtype=torch.float64, device="cuda")
    nbytes = tb.triples_workspace_bytes_ri(o, v, naux, prec, o // 2, 0)          # half the slices cached: rebuilds happen
    E = tb.triples_energy_ri(o, v, naux, *dv, prec, ws_bytes(nbytes), e_triplet_out=et)
    g = _golden(name + "_full")
    tol = TOL[prec]
    n_cmp = _check_against_golden(g, et.cpu().numpy(), o, tol)
    assert n_cmp >= 64
    if g["complete"]:
        assert abs(E[0] - g["E"][0]) <= tol * abs(g["E"][0]) and abs(E[1] - g["E"][1]) <= tol * abs(g["E"][1])


def test_mixed_run_is_bitwise_repeatable_on_a_ragged_size():
    """Stress of the CTA-pair hand-offs of the mixed contraction (TMA of both CTAs on the leader's barrier, relaxed
    remote arrives for the TMEM buffers): 25 repeats of a ragged-size run must agree bit for bit."""
    inp = synth.make_inputs(7, 75, 40, seed=13, t1_sigma=0.1)
    o, v = inp.nocc, inp.nvirt
    d = dev(inp)
    ws = ws_bytes(tb.triples_workspace_bytes(o, v, tb.MIXED))
    T = tb.triples_triplet_count(o)
    ref = None
    for _ in range(25):
        et = torch.zeros((T, 3), dtype=torch.float64, device="cuda")
        E = tb.triples_energy(o, v, *d, tb.MIXED, ws, e_triplet_out=et)
        if ref is None:
            ref = (E, et.clone())
        else:
            assert E == ref[0] and torch.equal(et, ref[1])
