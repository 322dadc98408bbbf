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


def _dev_ptr(t, name):
    import torch

    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous float64 CUDA tensor")
    return ctypes.c_void_p(t.data_ptr())


def _host_ptr(a, name):
    if not isinstance(a, np.ndarray) or a.dtype != np.float64 or not a.flags.c_contiguous:
        raise TypeError(f"{name}: expected a C-contiguous float64 numpy array")
    return ctypes.c_void_p(a.ctypes.data)


def _stream_ptr(stream):
    import torch

    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _ws(workspace):
    import torch

    if not isinstance(workspace, torch.Tensor) or not workspace.is_cuda or workspace.dtype != torch.uint8:
        raise TypeError("workspace: expected a torch.uint8 CUDA tensor")
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
    out = (ctypes.c_double * 10)()
    _check(lib().triples_last_profile(out))
    keys = ("prepare_ms", "contraction_ms", "contraction_launches", "reduction_ms", "reduction_launches",
            "other_ms", "other_launches", "contraction_flops", "reduction_bytes", "triplets")
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


def triples_last_launch_count() -> int:
    return int(lib().triples_last_launch_count())


def triples_energy(nocc, nvirt, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, precision, workspace, stream=None,
                   e_triplet_out=None):
    """Device-resident inputs (torch float64 CUDA tensors).  Returns (E(T), E[4], E[5])."""
    ptrs = [_dev_ptr(t, n) for t, n in zip((eps_o, eps_v, t1, t2, vvvo, ovoo, ovov), _NAMES)]
    wp, wn = _ws(workspace)
    e_out = (ctypes.c_double * 3)()
    et = ctypes.c_void_p(None) if e_triplet_out is None else _dev_ptr(e_triplet_out, "e_triplet_out")
    _check(lib().triples_energy(nocc, nvirt, *ptrs, precision, wp, wn, _stream_ptr(stream), e_out, et))
    return float(e_out[0]), float(e_out[1]), float(e_out[2])


def triples_energy_host(nocc, nvirt, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, precision, workspace, stream=None,
                        e_triplet_out=None):
    """Host inputs (numpy float64); host<->device copies happen inside the call."""
    ptrs = [_host_ptr(a, n) for a, n in zip((eps_o, eps_v, t1, t2, vvvo, ovoo, ovov), _NAMES)]
    wp, wn = _ws(workspace)
    e_out = (ctypes.c_double * 3)()
    et = ctypes.c_void_p(None) if e_triplet_out is None else _host_ptr(e_triplet_out, "e_triplet_out")
    _check(lib().triples_energy_host(nocc, nvirt, *ptrs, precision, wp, wn, _stream_ptr(stream), e_out, et))
    return float(e_out[0]), float(e_out[1]), float(e_out[2])


def triples_energy_subset(nocc, nvirt, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, precision, triplets, workspace,
                          stream=None) -> np.ndarray:
    """Weighted per-triplet energies [n,3] for a list of restricted triplets (device inputs)."""
    ptrs = [_dev_ptr(t, n) for t, n in zip((eps_o, eps_v, t1, t2, vvvo, ovoo, ovov), _NAMES)]
    wp, wn = _ws(workspace)
    trip = np.ascontiguousarray(np.asarray(triplets, dtype=np.int32).reshape(-1, 3))
    out = np.zeros((trip.shape[0], 3), dtype=np.float64)
    _check(lib().triples_energy_subset(nocc, nvirt, *ptrs, precision, trip.shape[0],
                                       trip.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), wp, wn,
                                       _stream_ptr(stream), out.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
    return out


def triples_w_block(nocc, nvirt, t2, vvvo, ovoo, precision, i, j, k, workspace, W_out, stream=None):
    """W_ijk^abc of Eq. (2.2.2)-(2.2.3) into W_out (float64 CUDA tensor [v,v,v])."""
    ptrs = [_dev_ptr(t, n) for t, n in zip((t2, vvvo, ovoo), ("t2", "vvvo", "ovoo"))]
    wp, wn = _ws(workspace)
    _check(lib().triples_w_block(nocc, nvirt, *ptrs, precision, i, j, k, wp, wn, _stream_ptr(stream),
                                 _dev_ptr(W_out, "W_out")))
    return W_out
