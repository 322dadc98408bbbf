"""ctypes binding of include/triples_b200.h -- argument marshalling only.

Every function has the name and the argument order of its C entry point.  Tensors are torch tensors
(device memory, streams) or numpy arrays (host variant); nothing is computed here.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

FP64 = 0
MIXED = 1
EMU64 = 2

_STATUS = {0: "OK", 1: "EINVAL", 2: "EWORKSPACE", 3: "ECUDA", 4: "EARCH"}
_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtriples_b200.so")
_lib = None


class TriplesError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"triples_b200: {_STATUS.get(status, status)}: {message}")
        self.status = status


def lib() -> ctypes.CDLL:
    """Load the CUDA library; fail loudly if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1609_08094_b200.build` "
                "(there is no CPU or PyTorch fallback for the (T) hot path)")
        L = ctypes.CDLL(LIB_PATH)
        vp, dp, ip = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
        L.triples_abi_version.restype = ctypes.c_int
        L.triples_last_error.restype = ctypes.c_char_p
        L.triples_set_profiling.argtypes = [ctypes.c_int]
        L.triples_set_profiling.restype = None
        L.triples_last_profile.argtypes = [dp]
        L.triples_last_profile.restype = ctypes.c_int
        L.triples_last_launch_count.restype = ctypes.c_longlong
        L.triples_triplet_count.argtypes = [ctypes.c_int]
        L.triples_triplet_count.restype = ctypes.c_longlong
        L.triples_triplet_list.argtypes = [ctypes.c_int, ip]
        L.triples_triplet_list.restype = ctypes.c_int
        L.triples_plan_batches.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ip, ip,
                                           ctypes.POINTER(ctypes.c_longlong)]
        L.triples_plan_batches.restype = ctypes.c_longlong
        for name in ("triples_workspace_bytes", "triples_workspace_bytes_host"):
            f = getattr(L, name)
            f.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int]
            f.restype = ctypes.c_size_t
        for name in ("triples_energy", "triples_energy_host"):
            f = getattr(L, name)
            f.argtypes = [ctypes.c_int, ctypes.c_int] + [vp] * 7 + [ctypes.c_int, vp, ctypes.c_size_t, vp, dp, vp]
            f.restype = ctypes.c_int
        L.triples_energy_noalloc.argtypes = [ctypes.c_int, ctypes.c_int] + [vp] * 7 + [ctypes.c_int, vp, dp, vp]
        L.triples_energy_noalloc.restype = ctypes.c_int
        L.triples_energy_sharded.argtypes = ([ctypes.c_int, ctypes.c_int] + [vp] * 7 + [ctypes.c_int] * 3 +
                                             [vp, ctypes.c_size_t, vp, dp, vp])
        L.triples_energy_sharded.restype = ctypes.c_int
        L.triples_energy_streamed.argtypes = ([ctypes.c_int, ctypes.c_int] + [vp] * 7 + [ctypes.c_int, ctypes.c_double] +
                                              [vp, ctypes.c_size_t, vp, dp, vp])
        L.triples_energy_streamed.restype = ctypes.c_int
        L.triples_energy_ri.argtypes = ([ctypes.c_int] * 3 + [vp] * 7 + [ctypes.c_int] +
                                        [vp, ctypes.c_size_t, vp, dp, vp])
        L.triples_energy_ri.restype = ctypes.c_int
        L.triples_workspace_bytes_streamed.argtypes = [ctypes.c_int] * 5
        L.triples_workspace_bytes_streamed.restype = ctypes.c_size_t
        L.triples_workspace_bytes_ri.argtypes = [ctypes.c_int] * 6
        L.triples_workspace_bytes_ri.restype = ctypes.c_size_t
        L.triples_cache_slots.argtypes = [ctypes.c_int] * 5 + [ctypes.c_size_t, ip]
        L.triples_cache_slots.restype = ctypes.c_int
        L.triples_plan_shards.argtypes = [ctypes.c_int] * 4 + [ip, ctypes.POINTER(ctypes.c_longlong)]
        L.triples_plan_shards.restype = ctypes.c_longlong
        L.triples_plan_slices.argtypes = [ctypes.c_int] * 6 + [ip, ctypes.c_longlong, ip, ctypes.c_longlong, ip]
        L.triples_plan_slices.restype = ctypes.c_longlong
        L.triples_probe_fp64_peak.argtypes = [vp, ctypes.c_size_t, vp, ctypes.c_int, dp]
        L.triples_probe_fp64_peak.restype = ctypes.c_int
        L.triples_probe_tc_peak.argtypes = [ctypes.c_int, ctypes.c_double, vp, ctypes.c_size_t, vp, dp, dp]
        L.triples_probe_tc_peak.restype = ctypes.c_int
        L.triples_energy_subset.argtypes = ([ctypes.c_int, ctypes.c_int] + [vp] * 7 +
                                            [ctypes.c_int, ctypes.c_int, ip, vp, ctypes.c_size_t, vp, dp])
        L.triples_energy_subset.restype = ctypes.c_int
        L.triples_w_block.argtypes = ([ctypes.c_int, ctypes.c_int] + [vp] * 3 + [ctypes.c_int] * 4 +
                                      [vp, ctypes.c_size_t, vp, vp])
        L.triples_w_block.restype = ctypes.c_int
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise TriplesError(rc, lib().triples_last_error().decode())


def _dev_ptr(t, name, numel=None):
    import torch

    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous float64 CUDA tensor")
    if t.device.index != torch.cuda.current_device():
        raise ValueError(f"{name}: lives on {t.device}, the current device is cuda:{torch.cuda.current_device()}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name}: {t.numel()} elements, expected {numel} (the C side cannot see sizes)")
    return ctypes.c_void_p(t.data_ptr())


def _host_ptr(a, name, numel=None):
    if not isinstance(a, np.ndarray) or a.dtype != np.float64 or not a.flags.c_contiguous:
        raise TypeError(f"{name}: expected a C-contiguous float64 numpy array")
    if numel is not None and a.size != numel:
        raise ValueError(f"{name}: {a.size} elements, expected {numel} (the C side cannot see sizes)")
    return ctypes.c_void_p(a.ctypes.data)


def _sizes(o, v):
    """Element counts of (eps_o, eps_v, t1, t2, vvvo, ovoo, ovov) for the layouts of include/triples_b200.h."""
    return (o, v, o * v, o * o * v * v, v * v * v * o, o * v * o * o, o * v * o * v)


def _stream_ptr(stream):
    import torch

    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _ws(workspace):
    import torch

    if not isinstance(workspace, torch.Tensor) or not workspace.is_cuda or workspace.dtype != torch.uint8:
        raise TypeError("workspace: expected a torch.uint8 CUDA tensor")
    if workspace.device.index != torch.cuda.current_device():
        raise ValueError(f"workspace: lives on {workspace.device}, the current device is "
                         f"cuda:{torch.cuda.current_device()}")
    return ctypes.c_void_p(workspace.data_ptr()), ctypes.c_size_t(workspace.numel())


_NAMES = ("eps_o", "eps_v", "t1", "t2", "vvvo", "ovoo", "ovov")


def triples_abi_version() -> int:
    return int(lib().triples_abi_version())


def triples_triplet_count(nocc: int) -> int:
    return int(lib().triples_triplet_count(nocc))


def triples_triplet_list(nocc: int) -> np.ndarray:
    T = triples_triplet_count(nocc)
    out = np.zeros((max(T, 0), 3), dtype=np.int32)
    _check(lib().triples_triplet_list(nocc, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int))))
    return out


def triples_workspace_bytes(nocc: int, nvirt: int, precision: int) -> int:
    return int(lib().triples_workspace_bytes(nocc, nvirt, precision))


def triples_workspace_bytes_host(nocc: int, nvirt: int, precision: int) -> int:
    return int(lib().triples_workspace_bytes_host(nocc, nvirt, precision))


def triples_set_profiling(on: bool) -> None:
    lib().triples_set_profiling(1 if on else 0)


def triples_last_profile() -> dict:
    out = (ctypes.c_double * 16)()
    _check(lib().triples_last_profile(out))
    keys = ("prepare_ms", "contraction_ms", "contraction_launches", "reduction_ms", "reduction_launches",
            "other_ms", "other_launches", "contraction_flops", "reduction_bytes", "triplets",
            "slices_ms", "slices_loaded", "h2d_bytes", "ri_flops")
    return dict(zip(keys, [float(x) for x in out]))


def triples_plan_batches(nocc: int, nvirt: int, precision: int):
    """(number of batches, batch_of_triplet[T], jobs[njobs, 6] = {batch, p, q, r, group_start, group_size})."""
    T = triples_triplet_count(nocc)
    bot = np.empty(T, dtype=np.int32)
    jobs = np.empty((3 * T, 6), dtype=np.int32)
    nj = ctypes.c_longlong(0)
    ip = ctypes.POINTER(ctypes.c_int)
    nb = lib().triples_plan_batches(nocc, nvirt, precision, bot.ctypes.data_as(ip), jobs.ctypes.data_as(ip),
                                    ctypes.byref(nj))
    if nb < 0:
        raise TriplesError(1, lib().triples_last_error().decode())
    return int(nb), bot, jobs[: nj.value].copy()


def triples_plan_shards(nocc: int, nvirt: int, precision: int, nshards: int):
    """(number of batches, shard_of_triplet[T] (-1 for i=j=k), jobs_per_shard[nshards])."""
    T = triples_triplet_count(nocc)
    sot = np.empty(max(T, 0), dtype=np.int32)
    jps = np.zeros(max(nshards, 1), dtype=np.int64)
    nb = lib().triples_plan_shards(nocc, nvirt, precision, nshards, sot.ctypes.data_as(ctypes.POINTER(ctypes.c_int)),
                                   jps.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)))
    if nb < 0:
        raise TriplesError(1, lib().triples_last_error().decode())
    return int(nb), sot, jps


def triples_plan_slices(nocc: int, nvirt: int, precision: int, mode: int, nslots: int = 0, win: int = 0):
    """(loads[n, 3] = {batch, r, slot}, jobs[njobs, 5] = {batch, q, r, slot of XT_q, slot of X_r},
    info = {"nslots", "win", "batches", "jobs"}) of a streamed (mode 1) / RI (mode 2) run."""
    T = triples_triplet_count(nocc)
    cap = 12 * max(T, 1)
    loads = np.empty((cap, 3), dtype=np.int32)
    jobs = np.empty((3 * max(T, 1), 5), dtype=np.int32)
    info = np.zeros(4, dtype=np.int32)
    ip = ctypes.POINTER(ctypes.c_int)
    n = lib().triples_plan_slices(nocc, nvirt, precision, mode, nslots, win, loads.ctypes.data_as(ip), cap,
                                  jobs.ctypes.data_as(ip), jobs.shape[0], info.ctypes.data_as(ip))
    if n < 0:
        raise TriplesError(1, lib().triples_last_error().decode())
    return loads[:n].copy(), jobs[: info[3]].copy(), dict(zip(("nslots", "win", "batches", "jobs"), map(int, info)))


def triples_workspace_bytes_streamed(nocc: int, nvirt: int, precision: int, nslots: int = 0, win: int = 0) -> int:
    return int(lib().triples_workspace_bytes_streamed(nocc, nvirt, precision, nslots, win))


def triples_workspace_bytes_ri(nocc: int, nvirt: int, naux: int, precision: int, nslots: int = 0, win: int = 0) -> int:
    return int(lib().triples_workspace_bytes_ri(nocc, nvirt, naux, precision, nslots, win))


def triples_cache_slots(nocc: int, nvirt: int, naux: int, precision: int, mode: int, workspace_bytes: int):
    """(cache slots, window width) a streamed (mode 1) / RI (mode 2) run gets from a workspace of that size."""
    win = ctypes.c_int(0)
    n = int(lib().triples_cache_slots(nocc, nvirt, naux, precision, mode, workspace_bytes, ctypes.byref(win)))
    return n, int(win.value)


def triples_last_launch_count() -> int:
    return int(lib().triples_last_launch_count())


def triples_probe_fp64_peak(workspace, stream=None, iters: int = 20000) -> float:
    """Measured FP64 tensor-core (DMMA) peak of the current device in TFLOP/s."""
    wp, wn = _ws(workspace)
    out = ctypes.c_double(0.0)
    _check(lib().triples_probe_fp64_peak(wp, wn, _stream_ptr(stream), iters, ctypes.byref(out)))
    return float(out.value)


def triples_probe_tc_peak(kind: int, seconds: float, workspace, stream=None):
    """(Tera-op/s, SM MHz during the loop) of tcgen05.mma kind::f16 (kind 0) / kind::i8 (kind 1) on the current device."""
    wp, wn = _ws(workspace)
    tops, mhz = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(lib().triples_probe_tc_peak(kind, float(seconds), wp, wn, _stream_ptr(stream), ctypes.byref(tops),
                                       ctypes.byref(mhz)))
    return float(tops.value), float(mhz.value)


def _e_triplet(e_triplet_out, nocc, host=False):
    if e_triplet_out is None:
        return ctypes.c_void_p(None)
    n = 3 * triples_triplet_count(nocc)
    return _host_ptr(e_triplet_out, "e_triplet_out", n) if host else _dev_ptr(e_triplet_out, "e_triplet_out", n)


def triples_energy(nocc, nvirt, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, precision, workspace, stream=None,
                   e_triplet_out=None):
    """Device-resident inputs (torch float64 CUDA tensors).  Returns (E(T), E[4], E[5])."""
    ptrs = [_dev_ptr(t, n, k) for t, n, k in zip((eps_o, eps_v, t1, t2, vvvo, ovoo, ovov), _NAMES, _sizes(nocc, nvirt))]
    wp, wn = _ws(workspace)
    e_out = (ctypes.c_double * 3)()
    _check(lib().triples_energy(nocc, nvirt, *ptrs, precision, wp, wn, _stream_ptr(stream), e_out,
                                _e_triplet(e_triplet_out, nocc)))
    return float(e_out[0]), float(e_out[1]), float(e_out[2])


NOALLOC_SCRATCH_BYTES = 32 << 20   # TRIPLES_NOALLOC_SCRATCH_BYTES of include/triples_b200.h


def triples_energy_noalloc(nocc, nvirt, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, precision, stream=None,
                           e_triplet_out=None):
    """triples_energy without a workspace argument, for callers that cannot allocate device memory (a plug-in whose
    host program owns the device's memory, code that may not stall on cudaMalloc): the scratch is a 32 MiB array
    inside the library's device image, so only small problems (about nocc <= 8, nvirt <= 40) are accepted; larger
    ones raise EWORKSPACE.  One array per GPU, shared by all calls: do not overlap two calls on one GPU, and make
    the first call on a device outside stream capture.  Returns (E(T), E[4], E[5])."""
    ptrs = [_dev_ptr(t, n, k) for t, n, k in zip((eps_o, eps_v, t1, t2, vvvo, ovoo, ovov), _NAMES, _sizes(nocc, nvirt))]
    e_out = (ctypes.c_double * 3)()
    _check(lib().triples_energy_noalloc(nocc, nvirt, *ptrs, precision, _stream_ptr(stream), e_out,
                                        _e_triplet(e_triplet_out, nocc)))
    return float(e_out[0]), float(e_out[1]), float(e_out[2])


def triples_energy_sharded(nocc, nvirt, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, precision, shard, nshards, workspace,
                           stream=None, e_triplet_out=None):
    """This shard's partial (E(T), E[4], E[5]); the caller adds the partials in shard order."""
    ptrs = [_dev_ptr(t, n, k) for t, n, k in zip((eps_o, eps_v, t1, t2, vvvo, ovoo, ovov), _NAMES, _sizes(nocc, nvirt))]
    wp, wn = _ws(workspace)
    e_out = (ctypes.c_double * 3)()
    _check(lib().triples_energy_sharded(nocc, nvirt, *ptrs, precision, shard, nshards, wp, wn, _stream_ptr(stream),
                                        e_out, _e_triplet(e_triplet_out, nocc)))
    return float(e_out[0]), float(e_out[1]), float(e_out[2])


def triples_energy_host(nocc, nvirt, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, precision, workspace, stream=None,
                        e_triplet_out=None):
    """Host inputs (numpy float64); host<->device copies happen inside the call."""
    ptrs = [_host_ptr(a, n, k) for a, n, k in zip((eps_o, eps_v, t1, t2, vvvo, ovoo, ovov), _NAMES, _sizes(nocc, nvirt))]
    wp, wn = _ws(workspace)
    e_out = (ctypes.c_double * 3)()
    _check(lib().triples_energy_host(nocc, nvirt, *ptrs, precision, wp, wn, _stream_ptr(stream), e_out,
                                     _e_triplet(e_triplet_out, nocc, host=True)))
    return float(e_out[0]), float(e_out[1]), float(e_out[2])


def triples_energy_streamed(nocc, nvirt, eps_o, eps_v, t1, t2, vovv_host, ovoo, ovov, precision, workspace, stream=None,
                            e_triplet_out=None, vvvo_absmax=0.0):
    """Out-of-core run: vovv_host[k,a,b,c] = (ab|ck) is a HOST array (numpy, ideally pinned); the rest on the device."""
    o, v = nocc, nvirt
    sz = _sizes(o, v)
    ptrs = [_dev_ptr(t, n, k) for t, n, k in zip((eps_o, eps_v, t1, t2), _NAMES[:4], sz[:4])]
    ptrs.append(_host_ptr(vovv_host, "vovv_host", sz[4]))
    ptrs += [_dev_ptr(ovoo, "ovoo", sz[5]), _dev_ptr(ovov, "ovov", sz[6])]
    wp, wn = _ws(workspace)
    e_out = (ctypes.c_double * 3)()
    _check(lib().triples_energy_streamed(o, v, *ptrs, precision, float(vvvo_absmax), wp, wn, _stream_ptr(stream), e_out,
                                         _e_triplet(e_triplet_out, nocc)))
    return float(e_out[0]), float(e_out[1]), float(e_out[2])


def triples_energy_ri(nocc, nvirt, naux, eps_o, eps_v, t1, t2, B, ovoo, ovov, precision, workspace, stream=None,
                      e_triplet_out=None):
    """RI-direct run: B[Q,p,q] (device, [naux, n, n], n = nocc + nvirt) instead of the vvvo tensor."""
    o, v = nocc, nvirt
    sz = _sizes(o, v)
    ptrs = [_dev_ptr(t, n, k) for t, n, k in zip((eps_o, eps_v, t1, t2), _NAMES[:4], sz[:4])]
    ptrs.append(_dev_ptr(B, "B", naux * (o + v) * (o + v)))
    ptrs += [_dev_ptr(ovoo, "ovoo", sz[5]), _dev_ptr(ovov, "ovov", sz[6])]
    wp, wn = _ws(workspace)
    e_out = (ctypes.c_double * 3)()
    _check(lib().triples_energy_ri(o, v, naux, *ptrs, precision, wp, wn, _stream_ptr(stream), e_out,
                                   _e_triplet(e_triplet_out, nocc)))
    return float(e_out[0]), float(e_out[1]), float(e_out[2])


def triples_energy_subset(nocc, nvirt, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, precision, triplets, workspace,
                          stream=None) -> np.ndarray:
    """Weighted per-triplet energies [n,3] for a list of restricted triplets (device inputs)."""
    ptrs = [_dev_ptr(t, n, k) for t, n, k in zip((eps_o, eps_v, t1, t2, vvvo, ovoo, ovov), _NAMES, _sizes(nocc, nvirt))]
    wp, wn = _ws(workspace)
    trip = np.ascontiguousarray(np.asarray(triplets, dtype=np.int32).reshape(-1, 3))
    out = np.zeros((trip.shape[0], 3), dtype=np.float64)
    _check(lib().triples_energy_subset(nocc, nvirt, *ptrs, precision, trip.shape[0],
                                       trip.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), wp, wn,
                                       _stream_ptr(stream), out.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
    return out


def triples_w_block(nocc, nvirt, t2, vvvo, ovoo, precision, i, j, k, workspace, W_out, stream=None):
    """W_ijk^abc of Eq. (2.2.2)-(2.2.3) into W_out (float64 CUDA tensor [v,v,v])."""
    sz = _sizes(nocc, nvirt)
    ptrs = [_dev_ptr(t, n, k_) for t, n, k_ in zip((t2, vvvo, ovoo), ("t2", "vvvo", "ovoo"), (sz[3], sz[4], sz[5]))]
    wp, wn = _ws(workspace)
    _check(lib().triples_w_block(nocc, nvirt, *ptrs, precision, i, j, k, wp, wn, _stream_ptr(stream),
                                 _dev_ptr(W_out, "W_out", nvirt ** 3)))
    return W_out
