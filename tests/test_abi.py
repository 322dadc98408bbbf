"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol include/*.h declares,
and its host logic (triplet enumeration, workspace planner, argument validation) behaves as documented.
No compute call needs a GPU here; the one that would returns an error instead of falling back."""
import ctypes
import glob
import os
import re

import numpy as np
import pytest

import paper_1609_08094_b200 as tb
from paper_1609_08094_b200 import binding, build, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def declared_functions():
    names = []
    for h in glob.glob(os.path.join(ROOT, "include", "*.h")):
        text = re.sub(r"/\*.*?\*/", "", open(h).read(), flags=re.S)
        names += re.findall(r"\b(triples_\w+)\s*\(", text)
    return sorted(set(names))


def test_header_declares_the_survey_entry_points():
    names = declared_functions()
    for need in ("triples_energy", "triples_workspace_bytes", "triples_last_error", "triples_energy_host",
                 "triples_energy_subset", "triples_w_block", "triples_triplet_list"):
        assert need in names


def test_library_exports_every_declared_symbol(lib):
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} declared in include/*.h but not exported"
    assert binding.triples_abi_version() == 2


def test_binding_has_the_same_names():
    for name in declared_functions():
        if name in ("triples_last_error",):
            continue
        assert hasattr(binding, name), f"binding lacks {name}"


@pytest.mark.parametrize("o", [1, 2, 3, 8, 16, 24, 32, 40])
def test_triplet_enumeration_matches_eq_5_0_7b(o):
    # PAPER.md Eq. (5.0.7b): T = sum_i (No-i)(1+(No-i))/2 = No(No+1)(No+2)/6
    T = tb.triples_triplet_count(o)
    assert T == sum((o - i) * (1 + (o - i)) // 2 for i in range(o)) == o * (o + 1) * (o + 2) // 6
    lst = tb.triples_triplet_list(o)
    assert lst.shape == (T, 3)
    assert [tuple(x) for x in lst.tolist()] == synth.triplet_list(o)


def test_triplet_count_invalid():
    assert tb.triples_triplet_count(0) == 0
    assert tb.triples_triplet_count(-3) == 0


def test_workspace_bytes_planner():
    # invalid arguments -> 0
    assert tb.triples_workspace_bytes(0, 10, tb.FP64) == 0
    assert tb.triples_workspace_bytes(4, 0, tb.FP64) == 0
    assert tb.triples_workspace_bytes(4, 10, 7) == 0
    assert tb.triples_workspace_bytes(4, 5000, tb.FP64) == 0
    for name, (o, v, _) in synth.CONFIGS.items():
        w = tb.triples_workspace_bytes(o, v, tb.FP64)
        wh = tb.triples_workspace_bytes_host(o, v, tb.FP64)
        x_bytes = 2 * o * v ** 3 * 8          # X and XT repacks
        inputs = 8 * (o + v + o * v + 2 * o * o * v * v + v ** 3 * o + o ** 3 * v)
        assert w > x_bytes, name
        assert wh >= w + inputs, name
        assert wh < 180e9, f"{name}: must fit the 180 GB of HBM"
    # monotone in both sizes
    assert tb.triples_workspace_bytes(9, 40, tb.FP64) > tb.triples_workspace_bytes(8, 40, tb.FP64)
    assert tb.triples_workspace_bytes(8, 48, tb.FP64) > tb.triples_workspace_bytes(8, 40, tb.FP64)


def test_null_and_bad_arguments_return_einval(lib):
    e_out = (ctypes.c_double * 3)()
    rc = lib.triples_energy(4, 8, None, None, None, None, None, None, None, 0, None, 0, None, e_out, None)
    assert rc == 1 and b"null" in lib.triples_last_error()
    rc = lib.triples_energy(0, 8, None, None, None, None, None, None, None, 0, None, 0, None, e_out, None)
    assert rc == 1 and b"invalid" in lib.triples_last_error()
    rc = lib.triples_triplet_list(0, None)
    assert rc == 1
    out = (ctypes.c_double * 10)()
    assert lib.triples_last_profile(out) == 1          # no profiled call yet on this thread


def test_no_cpu_fallback_without_a_gpu(lib):
    """With valid host-side arguments but no usable device the call must fail loudly, not compute on the CPU."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present; the fallback check is for the CPU box")
    o, v = 2, 4
    inp = synth.make_inputs(o, v, 6, seed=0)
    bufs = [np.ascontiguousarray(a) for a in inp.arrays()]
    ptrs = [ctypes.c_void_p(b.ctypes.data) for b in bufs]
    ws = np.zeros(tb.triples_workspace_bytes_host(o, v, tb.FP64) + 512, dtype=np.uint8)
    wp = (ws.ctypes.data + 255) & ~255
    e_out = (ctypes.c_double * 3)(7.0, 7.0, 7.0)
    rc = lib.triples_energy_host(o, v, *ptrs, 0, ctypes.c_void_p(wp), ws.size - 256, None, e_out, None)
    assert rc in (3, 4), "expected TRIPLES_ECUDA/EARCH without a device"
    assert list(e_out) == [7.0, 7.0, 7.0]
    assert len(lib.triples_last_error()) > 0


def test_product_does_not_import_the_oracle():
    """The product path (package + bench's default arm) must not route through oracle/."""
    for path in glob.glob(os.path.join(ROOT, "paper_1609_08094_b200", "**", "*"), recursive=True):
        if os.path.isfile(path) and path.endswith((".py", ".cu", ".cuh", ".h")):
            text = open(path).read()
            assert "import oracle" not in text and "from oracle" not in text and "liboracle" not in text, path
    for path in glob.glob(os.path.join(ROOT, "oracle", "*")):
        if os.path.isfile(path) and path.endswith((".py", ".c")):
            text = open(path).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1609_08094_b200", text, flags=re.M), path
            assert "libtriples_b200" not in text and "triples_b200.h" not in text, path


# ------------------------------------------------------------------------------------------------------------------
# host planner (S1): batches = blocks of occupied-index windows, contraction jobs grouped by (q,r)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("o,v,prec", [(1, 6, 0), (2, 3, 0), (8, 40, 0), (8, 40, 1), (16, 120, 1), (24, 240, 0),
                                      (24, 240, 1), (13, 50, 1), (40, 480, 1), (40, 480, 0), (32, 400, 0)])
def test_batches_cover_every_triplet_once_and_jobs_are_grouped(o, v, prec):
    nb, bot, jobs = tb.triples_plan_batches(o, v, prec)
    trips = tb.triples_triplet_list(o)
    T = len(trips)
    diag = np.array([i == j == k for i, j, k in trips])
    # i=j=k cycles contribute exactly zero (Q5) and are in no batch; every other cycle is in exactly one
    assert np.all(bot[diag] == -1) and np.all(bot[~diag] >= 0)
    if T == int(diag.sum()):
        assert nb == 0 and len(jobs) == 0
        return
    assert set(bot[~diag].tolist()) == set(range(nb))
    # a batch is one block of index windows of one width, at most 64 triplets
    sizes = np.bincount(bot[~diag], minlength=nb)
    assert sizes.max() <= 64
    for w in (1, 2, 3, 4):
        key = (trips[:, 0] // w) * 10000 + (trips[:, 1] // w) * 100 + trips[:, 2] // w
        if all(len(set(key[(bot == b)].tolist())) == 1 for b in range(nb)) and \
                len(set(zip(key[~diag].tolist(), bot[~diag].tolist()))) == nb:
            break
    else:
        raise AssertionError("batches are not the blocks of any window width 1..4")
    # jobs: every triplet gets G(i,j,k), G(j,i,k), G(k,i,j), coinciding ones once
    want = {}
    for n, (i, j, k) in enumerate(trips.tolist()):
        if i == j == k:
            continue
        for g in {(i, j, k), (j, i, k), (k, i, j)}:
            want[(int(bot[n]),) + g] = want.get((int(bot[n]),) + g, 0) + 1
    got = {}
    for b, p, q, r, gs, gn in jobs.tolist():
        got[(b, p, q, r)] = got.get((b, p, q, r), 0) + 1
    assert got == want
    # launch order: batch by batch; inside a batch sorted by (q,r); group fields describe the runs of equal (q,r)
    assert np.all(np.diff(jobs[:, 0]) >= 0)
    for b in range(nb):
        jb = jobs[jobs[:, 0] == b]
        qr = [tuple(x) for x in jb[:, 2:4].tolist()]
        assert qr == sorted(qr)
        n = 0
        while n < len(jb):
            gs, gn = int(jb[n, 4]), int(jb[n, 5])
            assert gs == n and gn >= 1
            assert all(tuple(x) == qr[n] for x in jb[n:n + gn, 2:4].tolist())
            assert np.all(jb[n:n + gn, 4] == gs) and np.all(jb[n:n + gn, 5] == gn)
            assert n + gn == len(jb) or qr[n + gn] != qr[n]
            n += gn


def test_window_batches_share_operand_slices():
    """medium config: blocks of width-4 windows, so a (q,r) group has up to 4 jobs (the (vv|vo) slices X_r, XT_q
    are fetched once per group instead of once per job)."""
    nb, bot, jobs = tb.triples_plan_batches(24, 240, 1)
    assert nb == 56                                   # 6 windows: 6*7*8/6 blocks
    gsz = jobs[:, 5]
    assert gsz.max() == 4 and gsz.mean() > 3.0


def test_plan_batches_rejects_bad_sizes(lib):
    import ctypes
    assert lib.triples_plan_batches(0, 5, 0, None, None, None) == -1
    assert lib.triples_plan_batches(3, 5, 7, None, None, None) == -1
    assert b"invalid" in lib.triples_last_error()
    assert lib.triples_plan_batches(3, 5, 0, None, None, None) > 0


def test_decaying_generator_keeps_draws_and_symmetries():
    """synth decay option (dynamic-range tests of the packed precisions): decay = 0 is the default generator bit for
    bit; decay > 0 keeps the symmetries the kernels rely on and spreads the integrals over many orders of magnitude."""
    flat = synth.make_inputs(4, 9, 12, seed=1)
    same = synth.make_inputs(4, 9, 12, seed=1, decay=0.0)
    for a, b in zip(flat.arrays(), same.arrays()):
        assert np.array_equal(a, b)
    dec = synth.make_inputs(4, 9, 12, seed=1, decay=0.6)
    assert np.array_equal(dec.eps_o, flat.eps_o) and np.array_equal(dec.t1, flat.t1)
    sym = lambda x, perm: np.abs(x - x.transpose(*perm)).max() <= 1e-13 * np.abs(x).max()   # up to GEMM rounding order
    assert sym(dec.t2, (1, 0, 3, 2))                                                    # t2[i,j,a,b] = t2[j,i,b,a]
    assert sym(dec.vvvo, (1, 0, 2, 3))                                                  # (ab|ck) = (ba|ck)
    assert sym(dec.ovov, (2, 3, 0, 1))                                                  # (ia|jb) = (jb|ia)
    spread = lambda x: np.abs(x).max() / np.median(np.abs(x))
    assert spread(dec.vvvo) > 30 * spread(flat.vvvo)
    assert all(np.all((dec.eps_o[i] + dec.eps_o[j] - dec.eps_v[:, None] - dec.eps_v[None, :]) < 0)
               for i in range(4) for j in range(4))
