"""Pins for the oracle's elementary functions: what the paper and mathematics fix.
PAPER.md:129-140 (Eq. 14-15), 148-151 (Eq. 16), 223 (Eq. 26), 484-496 (App. A)."""
import math
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            out.append(line.split())
    return out


def test_paper_dims(oracle):
    for mat, nr, na, lm, neu, ndes, npar in _rows("paper_dims.txt"):
        h = oracle.Hyper(5.0, 4.0, int(nr), int(na), int(lm), int(neu), 1)
        assert oracle.descriptor_dim(h) == int(ndes), mat
        assert oracle.num_params(h) == int(npar), mat


def test_chebyshev_trig_identities(oracle):
    for phi in np.linspace(0.05, 3.0, 23):
        T, U = oracle.chebyshev(math.cos(phi), 16)
        for n in range(17):
            assert T[n] == pytest.approx(math.cos(n * phi), abs=1e-12)
            assert U[n] == pytest.approx(math.sin((n + 1) * phi) / math.sin(phi), abs=1e-10)


def test_chebyshev_derivative_A2(oracle):
    # dT_n/dx = n U_{n-1}: central differences of T against U
    h = 1e-6
    for x in (-0.9, -0.3, 0.0, 0.4, 0.85):
        Tp, _ = oracle.chebyshev(x + h, 12)
        Tm, _ = oracle.chebyshev(x - h, 12)
        _, U = oracle.chebyshev(x, 12)
        for n in range(1, 13):
            assert (Tp[n] - Tm[n]) / (2 * h) == pytest.approx(n * U[n - 1], rel=1e-7, abs=1e-7)


def test_cutoff_function(oracle):
    rc = 5.0
    assert oracle.cutoff(0.0, rc)[0] == 1.0
    assert oracle.cutoff(rc / 2, rc)[0] == pytest.approx(0.5, abs=1e-15)
    assert oracle.cutoff(rc, rc) == (0.0, 0.0)
    assert oracle.cutoff(rc + 1.0, rc) == (0.0, 0.0)
    # vanishes smoothly: value and slope -> 0 at r_c
    fc, dfc = oracle.cutoff(rc * (1 - 1e-6), rc)
    assert abs(fc) < 1e-11 and abs(dfc) < 1e-5
    h = 1e-6
    for r in (0.3, 1.7, 4.2):
        num = (oracle.cutoff(r + h, rc)[0] - oracle.cutoff(r - h, rc)[0]) / (2 * h)
        assert oracle.cutoff(r, rc)[1] == pytest.approx(num, rel=1e-8)


def test_radial_special_values(oracle):
    rc = 4.0
    g0, _ = oracle.radial(0.0, rc, 8)
    assert np.allclose(g0, 1.0)                      # x(0) = 1, T_n(1) = 1, f_c(0) = 1
    for n, val in _rows("radial_half_cutoff.txt"):
        g, _ = oracle.radial(rc / 2, rc, 8)
        assert g[int(n)] == pytest.approx(float(val), abs=1e-14)
    g, dg = oracle.radial(rc * (1 - 1e-7), rc, 8)
    assert np.all(np.abs(g) < 1e-12) and np.all(np.abs(dg) < 1e-5)   # C^1 at the cutoff
    for r in np.linspace(0.05, rc - 0.05, 31):
        g, _ = oracle.radial(r, rc, 12)
        fc, _ = oracle.cutoff(r, rc)
        assert g[0] == pytest.approx(fc, abs=1e-15)                  # g_0 = f_c
        assert np.all(g >= 0.0) and np.all(g <= 1.0 + 1e-15)         # "positive definite"
        x = 2 * (r / rc - 1) ** 2 - 1
        assert -1.0 <= x <= 1.0


def test_radial_weight_and_derivative(oracle):
    rc = 5.0
    h = 1e-6
    omega = math.sqrt(82 * 52)
    for r in (0.7, 2.35, 3.84, 4.9):
        g, dg = oracle.radial(r, rc, 10, omega)
        g1, _ = oracle.radial(r, rc, 10, 1.0)
        assert np.allclose(g, omega * g1, rtol=1e-15)                # Eq. 19 is a plain factor
        gp, _ = oracle.radial(r + h, rc, 10, omega)
        gm, _ = oracle.radial(r - h, rc, 10, omega)
        assert np.allclose(dg, (gp - gm) / (2 * h), rtol=1e-6, atol=1e-6)


def test_radial_fig1_shapes(oracle):
    # Fig. 1: g_0 decreases monotonically from 1 to 0; g_n has n interior
    # zeros of (T_n+1), i.e. touches zero where T_n(x) = -1.
    rc = 1.0
    r = np.linspace(0.0, 1.0, 2001)
    G = np.array([oracle.radial(float(t), rc, 3)[0] for t in r])
    assert np.all(np.diff(G[:, 0]) <= 1e-15)
    # T_1 = x = -1 only at r = r_c; T_2 = -1 at x = 0 -> r/r_c = 1 - 1/sqrt(2)
    k = np.argmin(np.abs(r - (1 - 1 / math.sqrt(2))))
    assert G[k, 2] < 1e-6 and G[k, 1] > 0.05
    # T_3 = -1 at x = 1/2 (and x = -1): r/r_c = 1 - sqrt(3)/2
    k = np.argmin(np.abs(r - (1 - math.sqrt(3) / 2)))
    assert G[k, 3] < 1e-5


def test_legendre_closed_forms(oracle):
    for c in np.linspace(-1.0, 1.0, 41):
        P, dP = oracle.legendre(float(c), 4)
        assert P[1] == pytest.approx(c, abs=1e-15)
        assert P[2] == pytest.approx((3 * c * c - 1) / 2, abs=1e-14)
        assert P[3] == pytest.approx((5 * c ** 3 - 3 * c) / 2, abs=1e-14)
        assert P[4] == pytest.approx((35 * c ** 4 - 30 * c * c + 3) / 8, abs=1e-14)
        assert dP[2] == pytest.approx(3 * c, abs=1e-14)
        assert dP[3] == pytest.approx((15 * c * c - 3) / 2, abs=1e-14)
        assert dP[4] == pytest.approx((140 * c ** 3 - 60 * c) / 8, abs=1e-13)
    P, dP = oracle.legendre(1.0, 6)
    assert np.allclose(P, 1.0) and np.allclose(dP, [l * (l + 1) / 2 for l in range(7)])
    P, _ = oracle.legendre(-1.0, 6)
    assert np.allclose(P, [(-1) ** l for l in range(7)])
    from scipy.special import eval_legendre, legendre as legendre_poly
    for l in range(7):
        assert oracle.legendre(0.3731, 6)[0][l] == pytest.approx(eval_legendre(l, 0.3731), abs=1e-14)
    # up to l = 8, the largest l_max the GPU's general-l kernel is judged at: values and derivatives
    for c in (-0.9137, -0.25, 0.0, 0.3731, 0.77, 0.999):
        P, dP = oracle.legendre(c, 8)
        for l in range(9):
            assert P[l] == pytest.approx(eval_legendre(l, c), abs=2e-14)
            assert dP[l] == pytest.approx(float(legendre_poly(l).deriv()(c)), abs=1e-11)
    P, dP = oracle.legendre(1.0, 8)
    assert np.allclose(P, 1.0) and np.allclose(dP, [l * (l + 1) / 2 for l in range(9)])


def test_network_hand_case(oracle):
    # D = 3 (n_max_R = 0, n_max_A = 0, l_max = 2), H = 2, computed by hand from Eq. 21-22
    h = oracle.Hyper(5.0, 4.0, 0, 0, 2, 2, 1)
    assert oracle.descriptor_dim(h) == 3 and oracle.num_params(h) == 11
    w1 = np.array([[0.5, -1.0, 0.25], [2.0, 0.0, -0.5]])
    b1 = np.array([0.1, -0.2]); w2 = np.array([1.5, -0.7]); b2 = 0.3
    params = np.concatenate([w1.ravel(), b1, w2, [b2]])
    q = np.array([0.2, 0.4, -0.6])
    a = w1 @ q - b1                                           # minus bias, Eq. 21
    x = np.tanh(a)
    U, Fp = oracle.network(h, params, q)
    assert U == pytest.approx(w2 @ x - b2, abs=1e-15)         # minus bias, Eq. 22
    assert np.allclose(Fp, (w2 * (1 - x * x)) @ w1, atol=1e-15)
    # a plus-sign mistake in either bias would change U
    assert abs(U - (w2 @ np.tanh(w1 @ q + b1) - b2)) > 1e-3
    # q = 0: isolated atom (reading Q14)
    U0, _ = oracle.network(h, params, np.zeros(3))
    assert U0 == pytest.approx(w2 @ np.tanh(-b1) - b2, abs=1e-15)


def test_network_gradient_fd(oracle):
    from paper_2107_08119_b200 import inputs
    h = oracle.Hyper(5.0, 4.0, 7, 7, 4, 30, 1)
    params = inputs.make_params(40, 30, 1)
    q = inputs.uniform01(11, 40) * 3.0
    _, Fp = oracle.network(h, params, q)
    eps = 1e-6
    for v in range(40):
        qp = q.copy(); qp[v] += eps
        qm = q.copy(); qm[v] -= eps
        num = (oracle.network(h, params, qp)[0] - oracle.network(h, params, qm)[0]) / (2 * eps)
        assert Fp[v] == pytest.approx(num, rel=1e-7, abs=1e-9)
