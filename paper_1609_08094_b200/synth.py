"""Seeded synthetic inputs for the closed-shell (T) kernel.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's
tests/bench.  It holds none of the (T) method's arithmetic: it only draws random
numbers and builds input tensors the way BASELINE.json ``configs`` prescribes
(section 4: the paper itself initialises all tensors with "unique, yet
arbitrary" numbers).  The recipe:

    rng      = numpy PCG64(seed); draw order: eps_o, eps_v, B, t1
    eps_o    ~ U(-1.5, -0.3) Eh, sorted ascending            [nocc]
    eps_v    ~ U( 0.1,  5.0) Eh, sorted ascending            [nvirt]
    B[Q,p,q] ~ N(0, 0.05^2) over n = nocc + nvirt orbitals (occupied first),
               symmetrised (B + B^T)/2 in (p,q)              [naux, n, n]
    (pq|rs)  = sum_Q B[Q,p,q] B[Q,r,s]                       (Mulliken)
    vvvo[a,b,c,k] = (ab|ck)   ovoo[i,a,j,k] = (ia|jk)   ovov[i,a,j,b] = (ia|jb)
    t2[i,j,a,b]   = ovov[i,a,j,b] / (e_i + e_j - e_a - e_b)  (MP2-like)
    t1[i,a]  ~ N(0, t1_sigma^2), t1_sigma = 1e-3

All arrays are C-ordered float64.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

# (nocc, nvirt, naux) of BASELINE.json configs[0..4]
CONFIGS = {
    "tiny": (8, 40, 120),
    "small": (16, 120, 360),
    "medium": (24, 240, 720),
    "large": (32, 400, 1200),
    "largest": (40, 480, 1440),
}
CONFIG_ORDER = ["tiny", "small", "medium", "large", "largest"]


@dataclass
class TriplesInputs:
    nocc: int
    nvirt: int
    eps_o: np.ndarray  # [o]
    eps_v: np.ndarray  # [v]
    t1: np.ndarray  # [o, v]
    t2: np.ndarray  # [o, o, v, v]
    vvvo: np.ndarray  # [v, v, v, o]
    ovoo: np.ndarray  # [o, v, o, o]
    ovov: np.ndarray  # [o, v, o, v]

    def arrays(self):
        return (self.eps_o, self.eps_v, self.t1, self.t2, self.vvvo, self.ovoo, self.ovov)


def draw_factors(nocc: int, nvirt: int, naux: int, seed: int = 0, t1_sigma: float = 1e-3, decay: float = 0.0):
    """Random draws only (fixed order): eps_o, eps_v, symmetrised B, t1.

    decay > 0 gives the integrals the structure real ones have and the flat default lacks: B[Q,p,q] is multiplied by
    exp(-decay |p - q|) (orbital pairs far apart overlap little), so (pq|rs) spans many orders of magnitude instead of
    one.  The draws are the same; decay = 0 leaves every stored golden value untouched."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = nocc + nvirt
    eps_o = np.sort(rng.uniform(-1.5, -0.3, size=nocc))
    eps_v = np.sort(rng.uniform(0.1, 5.0, size=nvirt))
    B = rng.normal(0.0, 0.05, size=(naux, n, n))
    B = 0.5 * (B + B.transpose(0, 2, 1))
    if decay > 0.0:
        idx = np.arange(n)
        B = B * np.exp(-decay * np.abs(idx[:, None] - idx[None, :]))[None, :, :]
    t1 = rng.normal(0.0, t1_sigma, size=(nocc, nvirt))
    return eps_o, eps_v, np.ascontiguousarray(B), t1


def make_inputs(nocc: int, nvirt: int, naux: int, seed: int = 0, t1_sigma: float = 1e-3,
                decay: float = 0.0) -> TriplesInputs:
    """Full float64 input set on the host (numpy)."""
    o, v = nocc, nvirt
    eps_o, eps_v, B, t1 = draw_factors(o, v, naux, seed, t1_sigma, decay)
    Boo = np.ascontiguousarray(B[:, :o, :o]).reshape(naux, o * o)
    Bov = np.ascontiguousarray(B[:, :o, o:]).reshape(naux, o * v)
    Bvo = np.ascontiguousarray(B[:, o:, :o]).reshape(naux, v * o)
    Bvv = np.ascontiguousarray(B[:, o:, o:]).reshape(naux, v * v)
    vvvo = (Bvv.T @ Bvo).reshape(v, v, v, o)
    ovoo = (Bov.T @ Boo).reshape(o, v, o, o)
    ovov = (Bov.T @ Bov).reshape(o, v, o, v)
    denom = (
        eps_o[:, None, None, None]
        + eps_o[None, :, None, None]
        - eps_v[None, None, :, None]
        - eps_v[None, None, None, :]
    )
    t2 = np.ascontiguousarray(ovov.transpose(0, 2, 1, 3)) / denom
    return TriplesInputs(o, v, eps_o, eps_v, np.ascontiguousarray(t1), np.ascontiguousarray(t2),
                         np.ascontiguousarray(vvvo), np.ascontiguousarray(ovoo), np.ascontiguousarray(ovov))


def make_config(name: str, seed: int = 0, t1_sigma: float = 1e-3, decay: float = 0.0) -> TriplesInputs:
    o, v, naux = CONFIGS[name]
    return make_inputs(o, v, naux, seed, t1_sigma, decay)


def make_inputs_device(nocc: int, nvirt: int, naux: int, seed: int = 0, t1_sigma: float = 1e-3,
                       device: str = "cuda", chunk: int = 64):
    """Same recipe, same random draws, but the integral contractions run with torch on
    ``device`` (harness only; needed at configs[3..4] where vvvo is 16-35 GB).

    Returns a dict of float64 torch tensors on ``device`` plus the host B factors (so a
    test can rebuild any integral slice on the host independently).  vvvo is contracted in
    chunks of ``chunk`` leading virtual indices to bound the temporaries.
    """
    import torch

    o, v = nocc, nvirt
    eps_o, eps_v, B, t1 = draw_factors(o, v, naux, seed, t1_sigma)
    Bd = torch.from_numpy(B).to(device)
    Boo = Bd[:, :o, :o].reshape(naux, o * o)
    Bov = Bd[:, :o, o:].reshape(naux, o * v)
    Bvo = Bd[:, o:, :o].reshape(naux, v * o).contiguous()
    # (ab|ck) = (ba|ck): only the blocks b >= a0 of every a-chunk go through the GEMM (half the generator's flops,
    # which at configs[4] are 1.3e16 in FP64); the rest is their mirror image
    vvvo = torch.empty((v, v, v, o), dtype=torch.float64, device=device)
    for a0 in range(0, v, chunk):
        a1 = min(v, a0 + chunk)
        Bvv = Bd[:, o + a0:o + a1, o + a0:].reshape(naux, (a1 - a0) * (v - a0))
        blk = (Bvv.T @ Bvo).reshape(a1 - a0, v - a0, v, o)
        vvvo[a0:a1, a0:] = blk
        if a1 < v:
            vvvo[a1:, a0:a1] = blk[:, a1 - a0:].permute(1, 0, 2, 3)
        del blk
    ovoo = (Bov.T @ Boo).reshape(o, v, o, o).contiguous()
    ovov = (Bov.T @ Bov).reshape(o, v, o, v).contiguous()
    eo = torch.from_numpy(eps_o).to(device)
    ev = torch.from_numpy(eps_v).to(device)
    denom = eo[:, None, None, None] + eo[None, :, None, None] - ev[None, None, :, None] - ev[None, None, None, :]
    t2 = (ovov.permute(0, 2, 1, 3) / denom).contiguous()
    return {
        "nocc": o, "nvirt": v,
        "eps_o": eo, "eps_v": ev, "t1": torch.from_numpy(t1).to(device).contiguous(), "t2": t2,
        "vvvo": vvvo, "ovoo": ovoo, "ovov": ovov, "B_host": B,
    }


def make_inputs_sliced(nocc: int, nvirt: int, naux: int, seed: int = 0, t1_sigma: float = 1e-3):
    """Host inputs WITHOUT the full vvvo tensor (16-35 GB at configs[3..4]): the small tensors plus the B factors.

    Returns (eps_o, eps_v, t1, t2, ovoo, ovov, B); any slice vvvo[:, :, :, r] follows from ``vvvo_slice``.
    Same random draws and the same formulas as ``make_inputs``.
    """
    o, v = nocc, nvirt
    eps_o, eps_v, B, t1 = draw_factors(o, v, naux, seed, t1_sigma)
    Boo = np.ascontiguousarray(B[:, :o, :o]).reshape(naux, o * o)
    Bov = np.ascontiguousarray(B[:, :o, o:]).reshape(naux, o * v)
    ovoo = (Bov.T @ Boo).reshape(o, v, o, o)
    ovov = (Bov.T @ Bov).reshape(o, v, o, v)
    denom = (eps_o[:, None, None, None] + eps_o[None, :, None, None]
             - eps_v[None, None, :, None] - eps_v[None, None, None, :])
    t2 = np.ascontiguousarray(ovov.transpose(0, 2, 1, 3)) / denom
    return (eps_o, eps_v, np.ascontiguousarray(t1), np.ascontiguousarray(t2), np.ascontiguousarray(ovoo),
            np.ascontiguousarray(ovov), B)


def vvvo_slice(B: np.ndarray, nocc: int, nvirt: int, r: int) -> np.ndarray:
    """vvvo[:, :, :, r] = (ab|cr) = sum_Q B[Q,a,b] B[Q,c,r] as a C-ordered [v,v,v] array (generator only)."""
    o, v = nocc, nvirt
    naux = B.shape[0]
    Bvv = np.ascontiguousarray(B[:, o:, o:]).reshape(naux, v * v)
    Bvr = np.ascontiguousarray(B[:, o:, r])                       # [naux, v]
    return np.ascontiguousarray((Bvv.T @ Bvr).reshape(v, v, v))


def triplet_list(nocc: int):
    """Enumeration order of the restricted loop, i<=j<=k (Eq. (5.0.7b))."""
    return [(i, j, k) for i in range(nocc) for j in range(i, nocc) for k in range(j, nocc)]


def sample_triplets(nocc: int, n: int, seed: int = 0):
    """Seeded sample of restricted triplets incl. the forced edge cases of SURVEY 8(c)."""
    o = nocc
    forced = [(0, 0, 0), (0, 0, 1), (0, 1, 1), (0, 1, 2), (o - 3, o - 2, o - 1), (o - 1, o - 1, o - 1)]
    forced = [t for t in forced if min(t) >= 0 and max(t) < o and t[0] <= t[1] <= t[2]]
    allt = triplet_list(o)
    rng = np.random.Generator(np.random.PCG64(seed + 12345))
    picks = [allt[x] for x in rng.permutation(len(allt))]
    out = []
    for t in forced + picks:
        if t not in out:
            out.append(t)
        if len(out) >= max(n, len(forced)):
            break
    return out
