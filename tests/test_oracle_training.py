"""Pins for the oracle's training side: the loss of Eq. 29-34 and one generation of the separable
natural evolution strategy, Eq. 35-39."""
import math

import numpy as np
import pytest

from paper_2107_08119_b200 import inputs


def _h(oracle):
    return oracle.Hyper(5.0, 4.0, 3, 2, 2, 6, 1)          # a small model keeps the O(M^2) oracle quick


def _targets(oracle, h, ts, z):
    """Per-structure energy and virial PER ATOM (reading Q23) and all forces, from the oracle's plain evaluation."""
    e, v = [], []
    f = np.zeros((3, ts.n_atoms))
    comp = [0, 4, 8, 1, 5, 6]                              # xx yy zz xy yz zx (reading Q24)
    for n in range(ts.n_structures):
        a0, a1 = ts.first[n], ts.first[n + 1]
        out = oracle.evaluate(h, [14], z, np.ascontiguousarray(ts.pos[:, a0:a1]), None, ts.types[a0:a1], ts.boxes[n])
        e.append(out["U"].sum() / (a1 - a0))
        v.append(out["W"].sum(axis=1)[comp] / (a1 - a0))
        f[:, a0:a1] = out["F"]
    return np.array(e), f, np.array(v)


def test_loss_closed_forms(oracle):
    h = _h(oracle)
    ts = inputs.training_set(5, seed=51)
    npar = oracle.num_params(h)
    z = 0.5 * (2 * inputs.uniform01(52, npar) - 1)
    e, f, v = _targets(oracle, h, ts, z)
    lam = [1.0, 1.0, 1.0, 0.05, 0.03]
    L = oracle.loss(h, [14], z, ts.first, ts.pos, ts.types, ts.boxes, e, f, v, lam)
    assert L[0] < 1e-13 and L[1] < 1e-13 and L[2] < 1e-13                    # its own outputs as targets
    assert L[3] == pytest.approx(np.abs(z).mean(), rel=1e-14)                # Eq. 33
    assert L[4] == pytest.approx(math.sqrt((z ** 2).mean()), rel=1e-14)      # Eq. 34
    assert L[5] == pytest.approx(0.05 * L[3] + 0.03 * L[4], rel=1e-14)       # Eq. 29
    # known offsets: RMSE of a constant shift is its magnitude
    L = oracle.loss(h, [14], z, ts.first, ts.pos, ts.types, ts.boxes, e + 0.02, f - 0.3, v, lam)
    assert L[0] == pytest.approx(0.02, rel=1e-10) and L[1] == pytest.approx(0.3, rel=1e-10) and L[2] < 1e-13
    v2 = v.copy(); v2[:, 3] += 0.6                                           # one of six components of every structure
    L = oracle.loss(h, [14], z, ts.first, ts.pos, ts.types, ts.boxes, e, f, v2, lam)
    assert L[2] == pytest.approx(0.6 / math.sqrt(6.0), rel=1e-10)            # Eq. 32: 1 / (6 N_str)
    # a single force component of a single atom: Eq. 31's 1 / (3N)
    f2 = f.copy(); f2[1, 7] += 0.9
    L = oracle.loss(h, [14], z, ts.first, ts.pos, ts.types, ts.boxes, e, f2, v, lam)
    assert L[1] == pytest.approx(0.9 / math.sqrt(3.0 * ts.n_atoms), rel=1e-10)


def test_energy_and_virial_are_per_atom(oracle):
    """Reading Q23: doubling a structure along x (same per-atom energy and virial) must leave L_e and L_v unchanged;
    with total energies it would not."""
    h = _h(oracle)
    ts = inputs.training_set(2, seed=53)
    z = 0.5 * (2 * inputs.uniform01(54, oracle.num_params(h)) - 1)
    e, f, v = _targets(oracle, h, ts, z)
    a0, a1 = ts.first[0], ts.first[1]
    p0 = ts.pos[:, a0:a1]
    shifted = p0 + np.array([[ts.boxes[0][0]], [0.0], [0.0]])
    pos2 = np.ascontiguousarray(np.concatenate([p0, shifted, ts.pos[:, a1:]], axis=1))
    first2 = np.array([0, 2 * (a1 - a0), 2 * (a1 - a0) + ts.first[2] - a1])
    boxes2 = ts.boxes.copy(); boxes2[0, 0] *= 2
    f2 = np.concatenate([f[:, a0:a1], f[:, a0:a1], f[:, a1:]], axis=1)
    L = oracle.loss(h, [14], z, first2, pos2, np.zeros(pos2.shape[1], dtype=np.int32), boxes2, e + 0.01, f2, v, [1, 1, 1, 0, 0])
    assert L[0] == pytest.approx(0.01, rel=1e-8) and L[1] < 1e-12 and L[2] < 1e-12


def test_utilities_and_two_member_update_by_hand(oracle):
    u = oracle.snes_utilities([0.3, 0.1, 0.7, 0.2, 0.9, 0.5])
    assert abs(u.sum()) < 1e-15
    order = np.argsort([0.3, 0.1, 0.7, 0.2, 0.9, 0.5])
    assert np.all(np.diff(u[order]) <= 1e-15)                                # better members never get less
    assert np.array_equal(oracle.snes_utilities([0.1, 0.3, 0.2]), oracle.snes_utilities([1.0, 30.0, 2.0]))   # ranks only
    # N_pop = 2: u = (+1/2, -1/2) -- ln(2) - ln(1) normalised to 1, minus 1/2; ln(2) - ln(2) = 0, minus 1/2
    r = np.array([[0.8, -1.1, 0.2], [-0.3, 0.4, 1.5]])
    m, s = np.array([0.1, 0.2, 0.3]), np.array([0.1, 0.2, 0.05])
    z = oracle.snes_sample(m, s, r)
    assert np.allclose(z, m + s * r, atol=0, rtol=1e-16)                     # Eq. 35
    m2, s2 = oracle.snes_update(m, s, r, [2.0, 5.0], 1.0, 0.7)
    gm = 0.5 * r[0] - 0.5 * r[1]
    gs = 0.5 * (r[0] ** 2 - 1) - 0.5 * (r[1] ** 2 - 1)
    assert np.allclose(m2, m + s * gm, rtol=1e-15) and np.allclose(s2, s * np.exp(0.35 * gs), rtol=1e-15)
    m3, s3 = oracle.snes_update(m, s, r[::-1].copy(), [5.0, 2.0], 1.0, 0.7)  # relabelling the members changes nothing
    assert np.allclose(m3, m2, rtol=1e-15) and np.allclose(s3, s2, rtol=1e-15)


def test_a_member_with_a_non_finite_loss_ranks_last(oracle):
    """Reading Q25 (the paper gives no rule; a NaN compares false with everything, so a literal rank count would put the
    broken member FIRST and pull m, s towards it): NaN and +-inf losses count as +inf, ties among them by index."""
    good = [0.3, 0.1, 0.7, 0.2, 0.9, 0.5, 0.4, 0.6]
    for bad in (float("nan"), float("inf"), float("-inf")):
        l = list(good); l[3] = bad
        as_huge = list(good); as_huge[3] = 1e300
        u = oracle.snes_utilities(l)
        assert np.array_equal(u, oracle.snes_utilities(as_huge))
        assert u[3] == u.min() == pytest.approx(-1.0 / len(good)) and abs(u.sum()) < 1e-15
    two = list(good); two[1] = float("nan"); two[6] = float("inf")
    ref = list(good); ref[1] = 1e300; ref[6] = 2e300                          # the earlier index ranks first among the broken
    assert np.array_equal(oracle.snes_utilities(two), oracle.snes_utilities(ref))
    assert np.array_equal(oracle.snes_utilities(good), oracle.snes_utilities([2 * x for x in good]))     # finite losses as before


def test_snes_minimises_a_quadratic(oracle):
    """The update follows the natural gradient: on L(z) = |z - z*|^2 the mean converges to z* (PAPER.md:273)."""
    npar, npop = 12, 20
    zstar = inputs.normal(60, npar)
    m = np.zeros(npar); s = np.full(npar, 0.5)
    eta_s = (3 + math.log(npar)) / (5 * math.sqrt(npar))
    d0 = np.linalg.norm(m - zstar)
    for g in range(150):
        r = inputs.normal(61 + g, npop * npar).reshape(npop, npar)
        z = oracle.snes_sample(m, s, r)
        m, s = oracle.snes_update(m, s, r, ((z - zstar) ** 2).sum(axis=1), 1.0, eta_s)
    assert np.linalg.norm(m - zstar) < 0.05 * d0
    assert s.max() < 0.5                                                      # the search distribution contracts
