"""Pins for the CPU oracle (oracle/): what the paper and the mathematics fix.

SURVEY.md 8(c) P1..P9.  None of these retypes the oracle's own formula: they are invariants,
closed forms, special cases, and an independent textbook definition (spin-orbital (T),
Raghavachari et al., the paper's ref. 9) evaluated by brute force.
"""
import itertools

import numpy as np
import pytest

from oracle import oracle
from paper_1609_08094_b200 import synth


def tiny(o=3, v=4, naux=9, seed=1, t1_sigma=0.3):
    return synth.make_inputs(o, v, naux, seed=seed, t1_sigma=t1_sigma)


def E_restricted(inp):
    return oracle.energy_restricted(inp.nocc, inp.nvirt, *inp.arrays())


def E_unrestricted(inp):
    return oracle.energy_unrestricted(inp.nocc, inp.nvirt, *inp.arrays())


# ---------------------------------------------------------------------------------------------
# P7: independent textbook definition, spin-orbital (T), brute force on (o=2, v=3)
# ---------------------------------------------------------------------------------------------

def spin_orbital_T(inp):
    """E(T) = 1/36 sum t_c D (t_c + t_d) over spin orbitals (canonical HF orbitals).

    D t_c(ijkabc) = P(i/jk) P(a/bc) [ sum_e t_jk^ae <ei||bc> - sum_m t_im^bc <ma||jk> ]
    D t_d(ijkabc) = P(i/jk) P(a/bc) t_i^a <jk||bc>
    P(p/qr) f(pqr) = f(pqr) - f(qpr) - f(rqp);  D = e_i + e_j + e_k - e_a - e_b - e_c
    <pq||rs> = <pq|rs> - <pq|sr>,  <pq|rs> = (pr|qs) [spin(p)=spin(r)] [spin(q)=spin(s)]
    Spin-orbital amplitudes from the closed-shell ones:
    t_IJ^AB = t_ij^ab [sI=sA][sJ=sB] - t_ij^ba [sI=sB][sJ=sA],  t_I^A = t_i^a [sI=sA].
    Returns (E4-like connected part, E5-like disconnected part).
    """
    o, v = inp.nocc, inp.nvirt
    no, nv = 2 * o, 2 * v
    sp = lambda P: (P // 2, P % 2)
    t2, t1, vvvo, ovoo, ovov = inp.t2, inp.t1, inp.vvvo, inp.ovoo, inp.ovov

    T2 = np.zeros((no, no, nv, nv))
    for I, J, A, B in itertools.product(range(no), range(no), range(nv), range(nv)):
        (i, si), (j, sj), (a, sa), (b, sb) = sp(I), sp(J), sp(A), sp(B)
        val = 0.0
        if si == sa and sj == sb:
            val += t2[i, j, a, b]
        if si == sb and sj == sa:
            val -= t2[i, j, b, a]
        T2[I, J, A, B] = val
    T1 = np.zeros((no, nv))
    for I, A in itertools.product(range(no), range(nv)):
        (i, si), (a, sa) = sp(I), sp(A)
        if si == sa:
            T1[I, A] = t1[i, a]

    # <ei||bc>: e,b,c virtual, i occupied.  <ei|bc> = (eb|ic) = vvvo[e,b,c,i]
    Veibc = np.zeros((nv, no, nv, nv))
    for E, I, B, C in itertools.product(range(nv), range(no), range(nv), range(nv)):
        (e, se), (i, si), (b, sb), (c, sc) = sp(E), sp(I), sp(B), sp(C)
        val = 0.0
        if se == sb and si == sc:
            val += vvvo[e, b, c, i]          # (eb|ci)
        if se == sc and si == sb:
            val -= vvvo[e, c, b, i]          # (ec|bi)
        Veibc[E, I, B, C] = val
    # <ma||jk>: m,j,k occupied, a virtual.  <ma|jk> = (mj|ak) = (ka|jm) = ovoo[k,a,j,m]
    Vmajk = np.zeros((no, nv, no, no))
    for M, A, J, K in itertools.product(range(no), range(nv), range(no), range(no)):
        (m, sm), (a, sa), (j, sj), (k, sk) = sp(M), sp(A), sp(J), sp(K)
        val = 0.0
        if sm == sj and sa == sk:
            val += ovoo[k, a, j, m]          # (ka|jm) = (mj|ak)
        if sm == sk and sa == sj:
            val -= ovoo[j, a, k, m]          # (ja|km) = (mk|aj)
        Vmajk[M, A, J, K] = val
    # <jk||bc> = (jb|kc) - (jc|kb)
    Vjkbc = np.zeros((no, no, nv, nv))
    for J, K, B, C in itertools.product(range(no), range(no), range(nv), range(nv)):
        (j, sj), (k, sk), (b, sb), (c, sc) = sp(J), sp(K), sp(B), sp(C)
        val = 0.0
        if sj == sb and sk == sc:
            val += ovov[j, b, k, c]
        if sj == sc and sk == sb:
            val -= ovov[j, c, k, b]
        Vjkbc[J, K, B, C] = val

    eo = np.repeat(inp.eps_o, 2)
    ev = np.repeat(inp.eps_v, 2)

    Xc = np.einsum("jkae,eibc->ijkabc", T2, Veibc) - np.einsum("imbc,majk->ijkabc", T2, Vmajk)
    Xd = np.einsum("ia,jkbc->ijkabc", T1, Vjkbc)

    def P_i_jk(f):   # f(ijk) - f(jik) - f(kji) on axes 0,1,2
        return f - f.transpose(1, 0, 2, 3, 4, 5) - f.transpose(2, 1, 0, 3, 4, 5)

    def P_a_bc(f):   # same on axes 3,4,5
        return f - f.transpose(0, 1, 2, 4, 3, 5) - f.transpose(0, 1, 2, 5, 4, 3)

    Dtc = P_i_jk(P_a_bc(Xc))
    Dtd = P_i_jk(P_a_bc(Xd))
    D = (eo[:, None, None, None, None, None] + eo[None, :, None, None, None, None]
         + eo[None, None, :, None, None, None] - ev[None, None, None, :, None, None]
         - ev[None, None, None, None, :, None] - ev[None, None, None, None, None, :])
    e_c = float(np.sum(Dtc * Dtc / D)) / 36.0
    e_d = float(np.sum(Dtc * Dtd / D)) / 36.0
    return e_c, e_d


@pytest.mark.parametrize("o,v,seed", [(2, 3, 0), (3, 3, 5), (2, 4, 11)])
def test_P7_spin_orbital_textbook_formula(o, v, seed):
    inp = synth.make_inputs(o, v, 7, seed=seed, t1_sigma=0.5)
    e_c, e_d = spin_orbital_T(inp)
    et, e4, e5 = E_unrestricted(inp)
    assert e4 == pytest.approx(e_c, rel=1e-12, abs=1e-15)
    assert e5 == pytest.approx(e_d, rel=1e-12, abs=1e-15)
    assert et == pytest.approx(e_c + e_d, rel=1e-12, abs=1e-15)
    et2, e42, e52 = E_restricted(inp)
    assert e42 == pytest.approx(e_c, rel=1e-12, abs=1e-15)
    assert e52 == pytest.approx(e_d, rel=1e-12, abs=1e-15)


# ---------------------------------------------------------------------------------------------
# P1: unrestricted literal sum == restricted weighted sum
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("o,v,seed", [(1, 3, 0), (2, 5, 1), (4, 6, 2), (5, 7, 3)])
def test_P1_unrestricted_equals_restricted(o, v, seed):
    inp = synth.make_inputs(o, v, 3 * (o + v), seed=seed, t1_sigma=0.2)
    u = E_unrestricted(inp)
    r = E_restricted(inp)
    for x, y in zip(u, r):
        assert x == pytest.approx(y, rel=1e-12, abs=1e-18)


def test_P1_tiny_config_shape_restricted_vs_unrestricted():
    # one size up: o=4, v=12 (64 ordered cycles vs 20 restricted)
    inp = synth.make_inputs(4, 12, 48, seed=7, t1_sigma=1e-3)
    u = E_unrestricted(inp)
    r = E_restricted(inp)
    for x, y in zip(u, r):
        assert x == pytest.approx(y, rel=1e-12, abs=1e-18)


# ---------------------------------------------------------------------------------------------
# P2: invariance under relabelling of occupied and of virtual orbitals
# ---------------------------------------------------------------------------------------------

def relabel(inp, po, pv):
    return synth.TriplesInputs(
        inp.nocc, inp.nvirt,
        inp.eps_o[po].copy(), inp.eps_v[pv].copy(),
        np.ascontiguousarray(inp.t1[np.ix_(po, pv)]),
        np.ascontiguousarray(inp.t2[np.ix_(po, po, pv, pv)]),
        np.ascontiguousarray(inp.vvvo[np.ix_(pv, pv, pv, po)]),
        np.ascontiguousarray(inp.ovoo[np.ix_(po, pv, po, po)]),
        np.ascontiguousarray(inp.ovov[np.ix_(po, pv, po, pv)]),
    )


@pytest.mark.parametrize("seed", [0, 1])
def test_P2_relabelling_invariance(seed):
    inp = synth.make_inputs(4, 6, 20, seed=seed, t1_sigma=0.3)
    rng = np.random.default_rng(seed + 100)
    po, pv = rng.permutation(4), rng.permutation(6)
    ref = E_restricted(inp)
    got = E_restricted(relabel(inp, po, pv))
    got_u = E_unrestricted(relabel(inp, po, pv))
    for x, y, z in zip(ref, got, got_u):
        assert y == pytest.approx(x, rel=1e-12)
        assert z == pytest.approx(x, rel=1e-12)


# ---------------------------------------------------------------------------------------------
# P3: zeros
# ---------------------------------------------------------------------------------------------

def test_P3_zero_integrals_and_zero_t2():
    inp = tiny()
    z = lambda a: np.zeros_like(a)
    e = oracle.energy_restricted(inp.nocc, inp.nvirt, inp.eps_o, inp.eps_v, inp.t1, inp.t2,
                                 z(inp.vvvo), z(inp.ovoo), z(inp.ovov))
    assert e == (0.0, 0.0, 0.0)
    e = oracle.energy_unrestricted(inp.nocc, inp.nvirt, inp.eps_o, inp.eps_v, inp.t1, inp.t2,
                                   z(inp.vvvo), z(inp.ovoo), z(inp.ovov))
    assert e == (0.0, 0.0, 0.0)
    # t2 = 0 kills W, hence Z[W], even with t1 != 0
    e = oracle.energy_restricted(inp.nocc, inp.nvirt, inp.eps_o, inp.eps_v, inp.t1, z(inp.t2),
                                 inp.vvvo, inp.ovoo, inp.ovov)
    assert e == (0.0, 0.0, 0.0)


# ---------------------------------------------------------------------------------------------
# P4: scaling laws
# ---------------------------------------------------------------------------------------------

def test_P4_scaling():
    inp = tiny(o=3, v=5, naux=11, seed=3, t1_sigma=0.0)
    assert np.all(inp.t1 == 0.0)
    e0 = E_restricted(inp)
    assert e0[2] == 0.0 and e0[0] == e0[1]
    lam, mu = 1.7, 0.6
    a = inp.arrays()
    e_l = oracle.energy_restricted(inp.nocc, inp.nvirt, a[0], a[1], a[2], lam * a[3], a[4], a[5], a[6])
    assert e_l[0] == pytest.approx(lam ** 2 * e0[0], rel=1e-12)
    e_m = oracle.energy_restricted(inp.nocc, inp.nvirt, a[0], a[1], a[2], a[3], mu * a[4], mu * a[5], mu * a[6])
    assert e_m[0] == pytest.approx(mu ** 2 * e0[0], rel=1e-12)
    # with t1 != 0: E4 ~ lam^2, E5 ~ lam * |t1| (bilinear in (t2, t1))
    inp1 = tiny(o=3, v=5, naux=11, seed=3, t1_sigma=0.4)
    b = inp1.arrays()
    f0 = E_restricted(inp1)
    f1 = oracle.energy_restricted(inp1.nocc, inp1.nvirt, b[0], b[1], 3.0 * b[2], lam * b[3], b[4], b[5], b[6])
    assert f1[1] == pytest.approx(lam ** 2 * f0[1], rel=1e-12)
    assert f1[2] == pytest.approx(3.0 * lam * f0[2], rel=1e-12)
    assert abs(f0[2]) > 1e-3 * abs(f0[1])   # the E5 channel is really exercised


# ---------------------------------------------------------------------------------------------
# P5: degenerate sizes and i=j=k cycles vanish
# ---------------------------------------------------------------------------------------------

def test_P5_degenerate_sizes():
    inp = synth.make_inputs(1, 6, 9, seed=2, t1_sigma=0.3)        # o = 1: only i=j=k
    e = E_restricted(inp)
    eu = E_unrestricted(inp)
    scale = float(np.abs(inp.t2).max() * np.abs(inp.vvvo).max()) ** 2
    assert abs(eu[0]) < 1e-12 * max(scale, 1e-30) + 1e-20
    assert e == (0.0, 0.0, 0.0)                                   # weight 0 exactly
    inp = synth.make_inputs(4, 1, 9, seed=2, t1_sigma=0.3)        # v = 1: W totally symmetric
    e = E_restricted(inp)
    eu = E_unrestricted(inp)
    assert abs(e[0]) < 1e-20 and abs(eu[0]) < 1e-20


def test_P5_diagonal_cycles_vanish_in_literal_sum():
    # literal per-cycle value of (i,i,i) is ~0 because W_iii is totally symmetric in abc and
    # Eq. (2.2.5) annihilates the symmetric part: compare unrestricted o=1 sub-problem.
    inp = synth.make_inputs(3, 5, 12, seed=9, t1_sigma=0.3)
    e_all = oracle.energy_subset(inp.nocc, inp.nvirt, *inp.arrays(), [(1, 1, 1), (0, 1, 2)])
    assert np.all(e_all[0] == 0.0)
    assert abs(e_all[1, 0]) > 0.0


# ---------------------------------------------------------------------------------------------
# P6: E[4] <= 0 per triplet when all D < 0  (Z has eigenvalues {0, 3, 12} on S3)
# ---------------------------------------------------------------------------------------------

def test_P6_sign_per_triplet():
    inp = synth.make_inputs(4, 7, 25, seed=4, t1_sigma=0.0)
    (et, e4, e5), trip = oracle.energy_restricted(inp.nocc, inp.nvirt, *inp.arrays(), with_triplets=True)
    assert np.all(trip[:, 1] <= 0.0)
    assert e4 < 0.0 and et < 0.0 and e5 == 0.0
    # random (non-MP2-like) t2 with the required symmetry t_ij^ab = t_ji^ba: still <= 0
    rng = np.random.default_rng(0)
    t2 = rng.normal(size=inp.t2.shape)
    t2 = 0.5 * (t2 + t2.transpose(1, 0, 3, 2))
    a = inp.arrays()
    (et, e4, e5), trip = oracle.energy_restricted(inp.nocc, inp.nvirt, a[0], a[1], a[2], t2, a[4], a[5], a[6],
                                                  with_triplets=True)
    assert np.all(trip[:, 1] <= 0.0) and e4 < 0.0


# ---------------------------------------------------------------------------------------------
# P9: task count, Eq. (5.0.7b), and enumeration order
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("o", [1, 2, 3, 8, 16, 24, 32, 40])
def test_P9_task_count(o):
    T_paper = sum((o - i) * (1 + (o - i)) // 2 for i in range(o))     # Eq. (5.0.7b)
    assert T_paper == o * (o + 1) * (o + 2) // 6
    assert len(synth.triplet_list(o)) == T_paper


def test_triplet_sum_matches_total_and_subset_order():
    inp = synth.make_inputs(4, 5, 15, seed=6, t1_sigma=0.2)
    (et, e4, e5), trip = oracle.energy_restricted(inp.nocc, inp.nvirt, *inp.arrays(), with_triplets=True)
    assert trip[:, 0].sum() == pytest.approx(et, rel=1e-13)
    tl = synth.triplet_list(4)
    sub = oracle.energy_subset(inp.nocc, inp.nvirt, *inp.arrays(), [tl[7], tl[3]])
    assert np.array_equal(sub[0], trip[7]) and np.array_equal(sub[1], trip[3])


# ---------------------------------------------------------------------------------------------
# numpy restatement (library contraction as a step) == C loops, elementwise W and energies
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("ijk", [(0, 1, 2), (2, 0, 1), (1, 1, 3), (3, 3, 3)])
def test_numpy_w_block_equals_loops(ijk):
    inp = synth.make_inputs(4, 6, 20, seed=8, t1_sigma=0.2)
    i, j, k = ijk
    Wc = oracle.w_block(inp.nocc, inp.nvirt, inp.t2, inp.vvvo, inp.ovoo, i, j, k)
    slices = {r: np.ascontiguousarray(inp.vvvo[:, :, :, r]) for r in range(inp.nocc)}
    Wn = oracle.w_block_numpy(inp.t2, slices, inp.ovoo, i, j, k)
    assert np.allclose(Wc, Wn, rtol=1e-12, atol=1e-15 * np.abs(Wc).max())
    # W is invariant under simultaneous permutation of (i,a),(j,b),(k,c) pairs (Eq. (2.2.3))
    Wp = oracle.w_block(inp.nocc, inp.nvirt, inp.t2, inp.vvvo, inp.ovoo, j, i, k)
    assert np.allclose(Wp.transpose(1, 0, 2), Wc, rtol=1e-12, atol=1e-14 * np.abs(Wc).max())


def test_numpy_energies_equal_loops():
    inp = synth.make_inputs(5, 9, 30, seed=10, t1_sigma=0.3)
    tl = synth.triplet_list(5)
    ec = oracle.energy_subset(inp.nocc, inp.nvirt, *inp.arrays(), tl)
    en = oracle.energy_subset_numpy(*inp.arrays(), tl)
    assert np.allclose(ec, en, rtol=1e-11, atol=1e-14 * np.abs(ec).max())


# ---------------------------------------------------------------------------------------------
# generator facts the method relies on (preconditions Q6, Q12)
# ---------------------------------------------------------------------------------------------

def test_generator_preconditions():
    inp = synth.make_inputs(4, 6, 20, seed=0)
    assert np.allclose(inp.t2, inp.t2.transpose(1, 0, 3, 2), rtol=0, atol=1e-15)   # t_ij^ab = t_ji^ba
    assert inp.eps_o.max() < -0.3 + 1e-12 and inp.eps_v.min() > 0.1 - 1e-12        # all D <= -1.2
    assert np.all(np.diff(inp.eps_o) >= 0) and np.all(np.diff(inp.eps_v) >= 0)
    assert np.allclose(inp.vvvo, inp.vvvo.transpose(1, 0, 2, 3), atol=1e-14)       # (ab|ck) = (ba|ck)
    assert np.allclose(inp.ovov, inp.ovov.transpose(2, 3, 0, 1), atol=1e-14)       # (ia|jb) = (jb|ia)
    for arr in inp.arrays():
        assert arr.dtype == np.float64 and arr.flags.c_contiguous


# ------------------------------------------------------------------------------------------------------------------
# regression goldens (tests/golden/oracle_energies.json, written by tests/golden/make_golden.py from the oracle only;
# absolute values are "parity unpinned by the paper", DESIGN.md section 4 P10)
# ------------------------------------------------------------------------------------------------------------------
def _golden():
    import json
    import os
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_energies.json")) as f:
        return json.load(f)


def test_oracle_reproduces_its_golden_values_tiny():
    g = _golden()["tiny"]
    inp = synth.make_config("tiny", seed=0)
    E, et = oracle.energy_restricted(inp.nocc, inp.nvirt, *inp.arrays(), with_triplets=True)
    assert np.allclose(E, g["E"], rtol=1e-13, atol=0.0)
    assert np.allclose(et, np.array(g["triplets"]), rtol=1e-12, atol=1e-18)
    # Q1: the (T) correction is negative; E[4] <= 0 triplet by triplet (P6)
    assert g["E"][0] < 0 and np.all(np.array(g["triplets"])[:, 1] <= 0)


def test_numpy_restatement_reproduces_its_golden_values_small():
    g = _golden()["small"]
    inp = synth.make_config("small", seed=0)
    a = inp.arrays()
    pick = [1, 3, 7]
    trips = [tuple(g["triplets_ijk"][n]) for n in pick]
    e = oracle.energy_subset_numpy(a[0], a[1], a[2], a[3], a[4], a[5], a[6], trips)
    assert np.allclose(e, np.array(g["energies"])[pick], rtol=1e-12, atol=0.0)


def _golden_file(name):
    import json
    import os
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name + ".json")) as f:
        return json.load(f)


def test_full_config_goldens_are_consistent():
    """small_full / medium_full: written triplet by triplet by the numpy restatement; their totals are the sums of
    the stored per-triplet energies (Eq. (2.2.1)), E(T) < 0 (Q1), every e4 <= 0 (P6), i=j=k rows ~0 (P5)."""
    import math
    for name, o in (("small_full", 16), ("medium_full", 24)):
        g = _golden_file(name)
        e = np.array(g["energies"])
        assert g["nocc"] == o and len(e) == len(g["triplets_ijk"]) and len(e) > 0
        assert np.all(e[:, 1] <= 1e-12 * np.abs(e[:, 1]).max())
        for t, row in zip(g["triplets_ijk"], e):
            if t[0] == t[1] == t[2]:
                assert np.abs(row).max() <= 1e-12 * np.abs(e[:, 1]).max()
        if g["complete"]:
            assert len(e) == o * (o + 1) * (o + 2) // 6
            assert [tuple(t) for t in g["triplets_ijk"]] == synth.triplet_list(o)
            assert g["E"][0] < 0
            assert abs(g["E"][1] - math.fsum(e[:, 1])) <= 1e-15 * abs(g["E"][1])
            assert abs(g["E"][0] - (g["E"][1] + g["E"][2])) <= 1e-15 * abs(g["E"][0])


def test_numpy_restatement_reproduces_the_full_small_golden_on_a_sample():
    g = _golden_file("small_full")
    inp = synth.make_config("small", seed=0)
    a = inp.arrays()
    pick = [2, 17, 135, 400, 811]
    trips = [tuple(g["triplets_ijk"][n]) for n in pick]
    e = oracle.energy_subset_numpy(a[0], a[1], a[2], a[3], a[4], a[5], a[6], trips)
    assert np.allclose(e, np.array(g["energies"])[pick], rtol=1e-12, atol=0.0)
    # and the C loops (the definition written out) agree with the stored numpy values on two of them
    ec = oracle.energy_subset(inp.nocc, inp.nvirt, *a, trips[:2])
    assert np.allclose(ec, np.array(g["energies"])[pick[:2]], rtol=1e-11, atol=0.0)


def test_sliced_generator_matches_the_full_generator():
    """configs[3..4] goldens are written from vvvo slices rebuilt from B (synth.vvvo_slice): same tensors."""
    o, v, naux = 5, 13, 17
    inp = synth.make_inputs(o, v, naux, seed=9, t1_sigma=0.5)
    eps_o, eps_v, t1, t2, ovoo, ovov, B = synth.make_inputs_sliced(o, v, naux, seed=9, t1_sigma=0.5)
    for x, y in ((eps_o, inp.eps_o), (eps_v, inp.eps_v), (t1, inp.t1), (t2, inp.t2), (ovoo, inp.ovoo), (ovov, inp.ovov)):
        assert np.array_equal(x, y)
    for r in range(o):
        assert np.allclose(synth.vvvo_slice(B, o, v, r), inp.vvvo[:, :, :, r], rtol=1e-13, atol=1e-18)
    slices = {r: synth.vvvo_slice(B, o, v, r) for r in range(o)}
    trips = [(0, 1, 2), (1, 1, 4), (2, 3, 3)]
    e1 = oracle.energy_subset_numpy(eps_o, eps_v, t1, t2, None, ovoo, ovov, trips, vvvo_slices=slices)
    e2 = oracle.energy_subset(o, v, *inp.arrays(), trips)
    assert np.allclose(e1, e2, rtol=1e-11, atol=0.0)
