"""Pins for the oracle's descriptor (Eq. 12-13, 17-19): closed forms for dimer/trimer,
the addition-theorem identity through scipy's complex Y_lm, invariances, perfect diamond.
PAPER.md:117-173."""
import math
import os

import numpy as np
import pytest

from paper_2107_08119_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")
BIG = np.array([60.0, 60.0, 60.0])


def _hyper(oracle, ntypes=1, nr=7, na=7, lmax=4, neu=30, rcr=5.0, rca=4.0):
    return oracle.Hyper(rcr, rca, nr, na, lmax, neu, ntypes)


def _cluster_q(oracle, h, pts, types=None, znum=(14,), i=0):
    """Descriptor of atom i of an open cluster (big box), lists by brute force."""
    pos = np.ascontiguousarray(np.asarray(pts, dtype=np.float64).T)
    n = pos.shape[1]
    types = np.zeros(n, dtype=np.int32) if types is None else np.asarray(types, dtype=np.int32)
    cR, iR, _ = oracle.neighbors(pos, BIG, h.rc_r, 64)
    cA, iA, _ = oracle.neighbors(pos, BIG, h.rc_a, 64)
    return oracle.descriptor_atom(h, np.asarray(znum, dtype=np.int32), types, pos, BIG, i,
                                  iR[i, :cR[i]], iA[i, :cA[i]])


def test_dimer_closed_form(oracle):
    h = _hyper(oracle)
    r = 2.7
    q = _cluster_q(oracle, h, [[10, 10, 10], [10 + r, 10, 10]])
    gR, _ = oracle.radial(r, 5.0, 7)
    gA, _ = oracle.radial(r, 4.0, 7)          # r_c^A in x and f_c of the angular family (Q3)
    assert np.allclose(q[:8], gR, atol=1e-15)
    for n in range(8):
        for l in range(1, 5):                  # P_l(1) = 1, j = k term only (Q2)
            assert q[8 + 4 * n + (l - 1)] == pytest.approx(gA[n] ** 2, abs=1e-15)


def test_dimer_between_cutoffs_has_no_angular_part(oracle):
    h = _hyper(oracle)
    q = _cluster_q(oracle, h, [[10, 10, 10], [10, 14.5, 10]])    # r_c^A <= 4.5 < r_c^R
    assert np.all(q[:8] > 0) and np.all(q[8:] == 0.0)
    q = _cluster_q(oracle, h, [[10, 10, 10], [10, 15.5, 10]])    # beyond both: isolated atom (Q14)
    assert np.all(q == 0.0)


def test_trimer_closed_form(oracle):
    h = _hyper(oracle)
    ra, rb, th = 2.4, 3.1, 1.91
    pts = [[20, 20, 20], [20 + ra, 20, 20], [20 + rb * math.cos(th), 20 + rb * math.sin(th), 20]]
    q = _cluster_q(oracle, h, pts)
    ga, _ = oracle.radial(ra, 4.0, 7); gb, _ = oracle.radial(rb, 4.0, 7)
    gRa, _ = oracle.radial(ra, 5.0, 7); gRb, _ = oracle.radial(rb, 5.0, 7)
    P, _ = oracle.legendre(math.cos(th), 4)
    assert np.allclose(q[:8], gRa + gRb, atol=1e-14)
    for n in range(8):
        for l in range(1, 5):
            expect = ga[n] ** 2 + gb[n] ** 2 + 2 * ga[n] * gb[n] * P[l]
            assert q[8 + 4 * n + (l - 1)] == pytest.approx(expect, abs=1e-14)


def test_multicomponent_weighting_eq19(oracle):
    h = _hyper(oracle, ntypes=2)
    ra, rb, th = 2.4, 3.1, 1.2
    pts = [[20, 20, 20], [20 + ra, 20, 20], [20 + rb * math.cos(th), 20 + rb * math.sin(th), 20]]
    Z = (82, 52)
    q = _cluster_q(oracle, h, pts, types=[0, 1, 0], znum=Z)
    wa, wb = math.sqrt(82 * 52), math.sqrt(82 * 82)
    ga, _ = oracle.radial(ra, 4.0, 7); gb, _ = oracle.radial(rb, 4.0, 7)
    gRa, _ = oracle.radial(ra, 5.0, 7); gRb, _ = oracle.radial(rb, 5.0, 7)
    P, _ = oracle.legendre(math.cos(th), 4)
    assert np.allclose(q[:8], wa * gRa + wb * gRb, rtol=1e-14)
    for n in range(8):
        for l in range(1, 5):
            expect = (wa * ga[n]) ** 2 + (wb * gb[n]) ** 2 + 2 * wa * wb * ga[n] * gb[n] * P[l]
            assert q[8 + 4 * n + (l - 1)] == pytest.approx(expect, rel=1e-13)
    # central-atom information: swapping the centre's species changes q
    q2 = _cluster_q(oracle, h, pts, types=[1, 1, 0], znum=Z)
    assert not np.allclose(q, q2)


def _random_cluster(seed, n=9, spread=2.6):
    u = inputs.uniform01(seed, 3 * n).reshape(n, 3)
    pts = 30.0 + (u - 0.5) * 2 * spread
    pts[0] = 30.0
    return pts


def test_addition_theorem_eq17_18(oracle):
    """q_nl = 4 pi/(2l+1) sum_m |c_nlm|^2, c_nlm = sum_j g_n(r_ij) Y*_lm."""
    from scipy.special import sph_harm_y
    h = _hyper(oracle)
    pts = _random_cluster(21)
    q = _cluster_q(oracle, h, pts)
    d = pts[1:] - pts[0]
    r = np.linalg.norm(d, axis=1)
    keep = r < h.rc_a
    assert keep.sum() >= 4
    d, r = d[keep], r[keep]
    theta = np.arccos(d[:, 2] / r); phi = np.arctan2(d[:, 1], d[:, 0])
    G = np.array([oracle.radial(float(t), h.rc_a, 7)[0] for t in r])      # (nbr, n)
    for n in range(8):
        for l in range(1, 5):
            tot = 0.0
            for m in range(-l, l + 1):
                c = np.sum(G[:, n] * np.conj(sph_harm_y(l, m, theta, phi)))
                tot += (c * np.conj(c)).real
            assert q[8 + 4 * n + (l - 1)] == pytest.approx(4 * math.pi / (2 * l + 1) * tot, rel=1e-12)


def _rotation(seed):
    u = inputs.normal(seed, 9).reshape(3, 3)
    Q, R = np.linalg.qr(u)
    Q = Q * np.sign(np.diag(R))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    return Q


def test_invariances(oracle):
    """translation, rotation, inversion, permutation of same-species atoms."""
    h = _hyper(oracle, ntypes=2)
    Z = (82, 52)
    pts = _random_cluster(5, n=10)
    types = np.array([0, 1, 0, 1, 1, 0, 0, 1, 0, 1], dtype=np.int32)
    q0 = _cluster_q(oracle, h, pts, types, Z)
    assert np.abs(q0).max() > 1.0
    c = pts[0].copy()
    Rm = _rotation(3)
    for new in (pts + np.array([1.3, -2.2, 0.7]),                 # translation
                (pts - c) @ Rm.T + c,                             # rotation about atom 0
                -(pts - c) + c):                                  # inversion
        assert np.allclose(_cluster_q(oracle, h, new, types, Z), q0, rtol=1e-12, atol=1e-12)
    perm = np.array([0, 3, 2, 1, 7, 5, 6, 4, 8, 9])              # swaps Te<->Te (1<->3, 4<->7)
    assert np.array_equal(types[perm], types)
    assert np.allclose(_cluster_q(oracle, h, pts[perm], types[perm], Z), q0, rtol=1e-12, atol=1e-12)
    # swapping atoms of DIFFERENT species is not a symmetry
    perm2 = np.array([0, 2, 1, 3, 4, 5, 6, 7, 8, 9])
    assert not np.allclose(_cluster_q(oracle, h, pts[perm2], types, Z), q0, rtol=1e-6)


def test_perfect_diamond(oracle):
    """Perfect diamond 3x3x3 cells: shells 4/12/12/6 -> 28 radial and 16 angular neighbours at
    5.0 / 4.0 A; every atom has the same descriptor; forces vanish; W_i identical and isotropic."""
    a = 5.431
    shells = [(float(s[1]), int(s[2])) for s in
              (l.split() for l in open(os.path.join(GOLD, "diamond_shells.txt")) if l[0] != "#")]
    expect_R = sum(m for d2, m in shells if math.sqrt(d2) * a < 5.0)
    expect_A = sum(m for d2, m in shells if math.sqrt(d2) * a < 4.0)
    assert (expect_R, expect_A) == (28, 16)
    w = inputs.si_cells((3, 3, 3), sigma=0.0)
    h = _hyper(oracle)
    cR, iR, _ = oracle.neighbors(w.pos, w.box, 5.0, 64)
    cA, iA, _ = oracle.neighbors(w.pos, w.box, 4.0, 64)
    assert np.all(cR == expect_R) and np.all(cA == expect_A)
    out = oracle.compute(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, cR, iR, cA, iA,
                         want_internals=True)
    assert np.allclose(out["q"], out["q"][0], rtol=1e-11, atol=1e-11)
    assert np.abs(out["F"]).max() < 1e-12
    assert np.allclose(out["U"], out["U"][0], atol=1e-13)
    W = out["W"].T.reshape(-1, 3, 3)
    assert np.allclose(W, W[0], atol=1e-10)
    assert np.allclose(W[0], np.eye(3) * W[0][0, 0], atol=1e-10) and abs(W[0][0, 0]) > 1e-3
