"""Pins for the oracle's variants of SURVEY.md 8(f) f-4: more hidden layers ("generalization to more hidden
layers is straightforward") and the SOAP-like descriptor q_nn'l of Eq. 17-18."""
import math

import numpy as np
import pytest

from paper_2107_08119_b200 import inputs
from test_oracle_descriptor import BIG, _cluster_q, _random_cluster


def _h(oracle, nr=7, na=7, lmax=4, neu=30, nlayers=0, neu2=0, neu3=0, kind=0, ntypes=1, rcr=5.0, rca=4.0):
    h = oracle.Hyper(rcr, rca, nr, na, lmax, neu, ntypes)
    h.nlayers, h.nneu2, h.nneu3, h.kind = nlayers, neu2, neu3, kind
    return h


def test_dimensions(oracle):
    assert oracle.descriptor_dim(_h(oracle, 7, 7, 4, kind=1)) == 8 + 36 * 4            # pairs n <= n'
    assert oracle.descriptor_dim(_h(oracle, 15, 3, 2, kind=1)) == 16 + 10 * 2
    assert oracle.num_params(_h(oracle, nlayers=1)) == oracle.num_params(_h(oracle)) == 1261
    # 40 -> 30 -> 20 -> 1: (40+1)*30 + (30+1)*20 + 20 + 1
    assert oracle.num_params(_h(oracle, nlayers=2, neu2=20)) == 41 * 30 + 31 * 20 + 21
    assert oracle.num_params(_h(oracle, nlayers=3, neu2=20, neu3=7)) == 41 * 30 + 31 * 20 + 21 * 7 + 8


def test_deep_network_hand_case_and_gradient(oracle):
    # 1 -> 1 -> 1 -> 1 by hand: U = w3 tanh(w2 tanh(w1 q - b1) - b2) - b3  (minus biases as in Eq. 21-22)
    h = _h(oracle, nr=0, na=0, lmax=0, neu=1, nlayers=2, neu2=1)
    h.lmax = 0
    assert oracle.descriptor_dim(h) == 1 and oracle.num_params(h) == 6
    w1, b1, w2, b2, w3, b3 = 0.7, -0.2, -1.3, 0.4, 2.1, 0.5
    q = 0.9
    U, Fp = oracle.network(h, [w1, b1, w2, b2, w3, b3], [q])
    x1 = math.tanh(w1 * q - b1); x2 = math.tanh(w2 * x1 - b2)
    assert U == pytest.approx(w3 * x2 - b3, abs=1e-15)
    assert Fp[0] == pytest.approx(w3 * (1 - x2 * x2) * w2 * (1 - x1 * x1) * w1, abs=1e-15)
    wrong = w3 * math.tanh(w2 * math.tanh(w1 * q + b1) + b2) + b3       # plus biases: must differ
    assert abs(U - wrong) > 1e-2
    # general widths: dU/dq against central differences of U, and the forward pass against plain numpy
    for (nl, n2, n3) in ((2, 17, 0), (3, 11, 5)):
        h = _h(oracle, nlayers=nl, neu2=n2, neu3=n3)
        D = oracle.descriptor_dim(h)
        par = inputs.make_params(D, 30, 5)[:0]
        par = 0.3 * (2 * inputs.uniform01(9, oracle.num_params(h)) - 1)
        q = inputs.normal(10, D)
        U, Fp = oracle.network(h, par, q)
        widths = [30, n2, n3][:nl]
        x = q.copy(); o = 0; nin = D
        for wdt in widths:
            W = par[o:o + wdt * nin].reshape(wdt, nin); o += wdt * nin
            b = par[o:o + wdt]; o += wdt
            x = np.tanh(W @ x - b); nin = wdt
        assert U == pytest.approx(par[o:o + nin] @ x - par[o + nin], abs=1e-13)
        for v in (0, 7, D - 1):
            e = 1e-6
            qp = q.copy(); qp[v] += e; qm = q.copy(); qm[v] -= e
            fd = (oracle.network(h, par, qp)[0] - oracle.network(h, par, qm)[0]) / (2 * e)
            assert Fp[v] == pytest.approx(fd, rel=1e-7, abs=1e-10)


def test_soap_like_descriptor_through_complex_harmonics(oracle):
    """q_nn'l = sum_m c_nlm (c_n'lm)^*, c_nlm = sum_j g_n(r_ij) Y*_lm (Eq. 17-18), with scipy's orthonormal Y_lm;
    its diagonal is (2l+1)/(4 pi) times the q_nl of Eq. 13."""
    from scipy.special import sph_harm_y
    h1 = _h(oracle, kind=1)
    h0 = _h(oracle, kind=0)
    pts = _random_cluster(21)
    q1 = _cluster_q(oracle, h1, pts)
    q0 = _cluster_q(oracle, h0, pts)
    d = pts[1:] - pts[0]
    r = np.linalg.norm(d, axis=1)
    keep = r < h1.rc_a
    d, r = d[keep], r[keep]
    theta = np.arccos(d[:, 2] / r); phi = np.arctan2(d[:, 1], d[:, 0])
    G = np.array([oracle.radial(float(t), h1.rc_a, 7)[0] for t in r])
    assert np.array_equal(q1[:8], q0[:8])                    # the radial part is unchanged
    v = 8
    for n in range(8):
        for n2 in range(n, 8):
            for l in range(1, 5):
                tot = 0.0
                for m in range(-l, l + 1):
                    Y = sph_harm_y(l, m, theta, phi)
                    tot += (np.sum(G[:, n] * np.conj(Y)) * np.conj(np.sum(G[:, n2] * np.conj(Y)))).real
                assert q1[v] == pytest.approx(tot, rel=1e-11, abs=1e-14), (n, n2, l)
                if n2 == n:
                    assert q1[v] == pytest.approx((2 * l + 1) / (4 * math.pi) * q0[8 + 4 * n + l - 1], rel=1e-12)
                v += 1
    assert v == oracle.descriptor_dim(h1)


@pytest.mark.parametrize("variant", ["deep", "soap", "both"])
def test_force_is_minus_gradient_for_the_variants(oracle, variant):
    w = inputs.config0()
    h = _h(oracle, nr=5, na=3, lmax=3, neu=12, nlayers=2 if variant != "soap" else 0, neu2=9 if variant != "soap" else 0,
           kind=1 if variant != "deep" else 0)
    par = 0.4 * (2 * inputs.uniform01(33, oracle.num_params(h)) - 1)
    ev = lambda p: oracle.evaluate(h, w.atomic_numbers, par, p, None, w.types, w.box)
    out = ev(w.pos)
    F = out["F"]
    frms = math.sqrt((F ** 2).mean())
    eps = 1e-5
    for (a, i) in [(0, 0), (1, 7), (2, 13), (0, 31), (2, 63)]:
        def U_at(t):
            pp = w.pos.copy(); pp[a, i] += t
            return ev(pp)["U"].sum()
        num = -(8 * (U_at(eps) - U_at(-eps)) - (U_at(2 * eps) - U_at(-2 * eps))) / (12 * eps)
        assert F[a, i] == pytest.approx(num, abs=1e-6 * max(frms, 1e-3)), (a, i)
    assert np.abs(F.sum(axis=1)).max() < 1e-10 * max(1.0, np.abs(F).max())
    Wtot = out["W"].sum(axis=1).reshape(3, 3)
    assert np.allclose(Wtot, Wtot.T, atol=1e-9 * np.abs(Wtot).max())
