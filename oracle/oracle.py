"""Python face of the CPU oracle -- TEST INFRASTRUCTURE, not the product.

Two independent evaluations of PAPER.md Eq. (2.2.1)-(2.2.5) (L87-L109):

* the C loops of oracle/triples_oracle.c (the definition written out; modes (i) and (ii)),
  reached through ctypes;
* ``triplet_energy_numpy`` / ``w_block_numpy``: the same definition per triplet with
  ``numpy.einsum``/``matmul`` as the contraction step (a library primitive as a step, no
  blocking or fusion beyond the definition), used where the loops are too slow (sampled
  triplets of configs[1..4]).  tests/test_oracle_pins.py checks it against the C loops.

Readings Q1 (sign) and Q4 (restricted weights) are documented in triples_oracle.c and DESIGN.md.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import build_oracle

_lib = None


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build_oracle.build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        L.oracle_triples_unrestricted.argtypes = [ctypes.c_int, ctypes.c_int] + [dp] * 8
        L.oracle_triples_unrestricted.restype = ctypes.c_int
        L.oracle_triples_restricted.argtypes = [ctypes.c_int, ctypes.c_int] + [dp] * 9
        L.oracle_triples_restricted.restype = ctypes.c_int
        L.oracle_triples_subset.argtypes = [ctypes.c_int, ctypes.c_int] + [dp] * 7 + [ctypes.c_int, ip, dp]
        L.oracle_triples_subset.restype = ctypes.c_int
        L.oracle_w_block.argtypes = [ctypes.c_int, ctypes.c_int] + [dp] * 3 + [ctypes.c_int] * 3 + [dp]
        L.oracle_w_block.restype = ctypes.c_int
        L.oracle_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def _pack(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov):
    assert eps_o.shape == (o,) and eps_v.shape == (v,) and t1.shape == (o, v)
    assert t2.shape == (o, o, v, v) and vvvo.shape == (v, v, v, o)
    assert ovoo.shape == (o, v, o, o) and ovov.shape == (o, v, o, v)
    keep, ptrs = [], []
    for a in (eps_o, eps_v, t1, t2, vvvo, ovoo, ovov):
        arr, p = _c(a)
        keep.append(arr)
        ptrs.append(p)
    return keep, ptrs


def energy_unrestricted(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov):
    """Mode (i): literal sum over all ordered i,j,k.  Returns (E(T), E[4], E[5])."""
    keep, ptrs = _pack(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov)
    out_arr, out_p = _c(np.zeros(3))
    rc = lib().oracle_triples_unrestricted(o, v, *ptrs, out_p)
    if rc != 0:
        raise RuntimeError(f"oracle_triples_unrestricted rc={rc}")
    return tuple(float(x) for x in out_arr)


def energy_restricted(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, with_triplets=False):
    """Mode (ii): i<=j<=k, weight 2-d_ij-d_jk.  Returns (E(T), E[4], E[5])[, e_triplet[T,3]]."""
    keep, ptrs = _pack(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov)
    T = o * (o + 1) * (o + 2) // 6
    out_arr, out_p = _c(np.zeros(3))
    et_arr, et_p = _c(np.zeros((T, 3)))
    rc = lib().oracle_triples_restricted(o, v, *ptrs, out_p, et_p)
    if rc != 0:
        raise RuntimeError(f"oracle_triples_restricted rc={rc}")
    res = tuple(float(x) for x in out_arr)
    return (res, et_arr) if with_triplets else res


def energy_subset(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, triplets):
    """Weighted per-triplet energies [n,3] = (w*(e4+e5), w*e4, w*e5) for restricted triplets."""
    keep, ptrs = _pack(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov)
    trip = np.ascontiguousarray(np.asarray(triplets, dtype=np.int32).reshape(-1, 3))
    n = trip.shape[0]
    e_arr, e_p = _c(np.zeros((n, 3)))
    rc = lib().oracle_triples_subset(o, v, *ptrs, n, trip.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), e_p)
    if rc != 0:
        raise RuntimeError(f"oracle_triples_subset rc={rc}")
    return e_arr


def w_block(o, v, t2, vvvo, ovoo, i, j, k):
    """W_ijk^abc (numerator of Eq. (2.2.2) after P, Eq. (2.2.3)) by the C loops: [v,v,v]."""
    t2a, t2p = _c(t2)
    va, vp = _c(vvvo)
    oa, op = _c(ovoo)
    W, Wp = _c(np.zeros((v, v, v)))
    rc = lib().oracle_w_block(o, v, t2p, vp, op, i, j, k, Wp)
    if rc != 0:
        raise RuntimeError(f"oracle_w_block rc={rc}")
    return W


# ----------------------------------------------------------------------------------------------
# numpy restatement, per triplet (library contraction as a step)
# ----------------------------------------------------------------------------------------------

def _x_numpy(t2, X, ovoo, p, q, r):
    """x_pqr^{a'b'c'} = sum_d t_pq^{a'd} (b'd|c'r) - sum_l t_pl^{a'b'} (c'r|lq), Eq. (2.2.2), L94.

    ``X[r]`` is the slice vvvo[:, :, :, r] (indexed [b', d, c']).
    """
    virt = np.einsum("ad,bdc->abc", t2[p, q], X[r], optimize=True)
    occ = np.einsum("lab,cl->abc", t2[p], ovoo[r, :, :, q], optimize=True)
    return virt - occ


def w_block_numpy(t2, vvvo_slices, ovoo, i, j, k):
    """W_ijk^abc = P_ijk^abc x_ijk^abc, Eq. (2.2.3), L99.  ``vvvo_slices[r] = vvvo[:, :, :, r]``."""
    X = vvvo_slices
    return (
        _x_numpy(t2, X, ovoo, i, j, k)
        + _x_numpy(t2, X, ovoo, i, k, j).transpose(0, 2, 1)   # x_ikj^acb
        + _x_numpy(t2, X, ovoo, j, i, k).transpose(1, 0, 2)   # x_jik^bac
        + _x_numpy(t2, X, ovoo, j, k, i).transpose(2, 0, 1)   # x_jki^bca -> [b,c,a] stored, want [a,b,c]
        + _x_numpy(t2, X, ovoo, k, i, j).transpose(1, 2, 0)   # x_kij^cab
        + _x_numpy(t2, X, ovoo, k, j, i).transpose(2, 1, 0)   # x_kji^cba
    )


def triplet_energy_numpy(eps_o, eps_v, t1, t2, vvvo_slices, ovoo, ovov, i, j, k):
    """Weighted (w*(e4+e5), w*e4, w*e5) of one restricted triplet i<=j<=k, reading Q4."""
    assert i <= j <= k
    W = w_block_numpy(t2, vvvo_slices, ovoo, i, j, k)
    # Eq. (2.2.4): Vd^abc = t_i^a (jb|kc) + t_j^b (ia|kc) + t_k^c (ia|jb)
    Vd = (
        t1[i][:, None, None] * ovov[j, :, k, :][None, :, :]
        + t1[j][None, :, None] * ovov[i, :, k, :][:, None, :]
        + t1[k][None, None, :] * ovov[i, :, j, :][:, :, None]
    )
    D = (eps_o[i] + eps_o[j] + eps_o[k]) - (
        eps_v[:, None, None] + eps_v[None, :, None] + eps_v[None, None, :]
    )
    Z = (
        4.0 * W + W.transpose(2, 0, 1) + W.transpose(1, 2, 0)          # W^abc, W^bca, W^cab
        - 2.0 * W.transpose(0, 2, 1) - 2.0 * W.transpose(2, 1, 0) - 2.0 * W.transpose(1, 0, 2)
    )
    w = 2.0 - (1.0 if i == j else 0.0) - (1.0 if j == k else 0.0)
    e4 = w * float(np.sum(Z * W / D, dtype=np.longdouble))
    e5 = w * float(np.sum(Z * Vd / D, dtype=np.longdouble))
    return e4 + e5, e4, e5


def energy_subset_numpy(eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, triplets, vvvo_slices=None):
    """[n,3] weighted per-triplet energies via the numpy path.

    ``vvvo_slices`` may be a dict {r: vvvo[:, :, :, r]} (for configs where the caller only holds
    the slices the sampled triplets need); otherwise slices are taken from ``vvvo``.
    """
    out = np.zeros((len(triplets), 3))
    cache = {} if vvvo_slices is None else vvvo_slices
    for n, (i, j, k) in enumerate(triplets):
        for r in (i, j, k):
            if r not in cache:
                cache[r] = np.ascontiguousarray(vvvo[:, :, :, r])
        out[n] = triplet_energy_numpy(eps_o, eps_v, t1, t2, cache, ovoo, ovov, i, j, k)
    return out
