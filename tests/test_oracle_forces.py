"""Pins for the oracle's partial forces, force, virial, heat current, neighbours and MD.
PAPER.md:68-92 (Eq. 4-7), 202-215 (Eq. 23-25); BASELINE.json north_star (finite differences,
zero net force, brute-force neighbours, NVE)."""
import math

import numpy as np
import pytest

from paper_2107_08119_b200 import inputs


def _hyper(oracle, w):
    return oracle.Hyper(w.rc_r, w.rc_a, w.n_max_r, w.n_max_a, w.l_max, w.n_neurons, len(w.atomic_numbers))


def _total_U(oracle, h, w, pos, box=None):
    box = w.box if box is None else box
    return oracle.evaluate(h, w.atomic_numbers, w.params, pos, None, w.types, box)["U"].sum()


def _small_pbte():
    w = inputs.config3(cells=(2, 2, 2))          # 64 atoms, box 12.92 > 2 * 6.0
    return w


@pytest.mark.parametrize("which", ["si", "pbte"])
def test_force_is_minus_gradient(oracle, which):
    w = inputs.config0() if which == "si" else _small_pbte()
    h = _hyper(oracle, w)
    out = oracle.evaluate(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box)
    F = out["F"]
    eps = 1e-5
    frms = math.sqrt((F ** 2).mean())
    for (a, i) in [(0, 0), (1, 7), (2, 13), (0, 31), (1, 50), (2, 63)]:
        def U_at(t):
            pp = w.pos.copy(); pp[a, i] += t
            return _total_U(oracle, h, w, pp)
        # 4th-order central difference (the Eq. 19 PbTe surface is stiff: large 3rd derivative)
        num = -(8 * (U_at(eps) - U_at(-eps)) - (U_at(2 * eps) - U_at(-2 * eps))) / (12 * eps)
        assert F[a, i] == pytest.approx(num, abs=1e-6 * max(frms, 1e-3)), (a, i)
    # zero net force: F_ij = -F_ji
    assert np.abs(F.sum(axis=1)).max() < 1e-10 * max(1.0, np.abs(F).max())


@pytest.mark.parametrize("l_max,n_max_a", [(6, 5), (8, 3)])
def test_force_is_minus_gradient_for_l_max_above_four(oracle, l_max, n_max_a):
    """The literal Legendre double sum of Eq. 13 / 25 at l_max = 6 and 8 -- what the GPU's general-l kernel is compared
    with (the finite-difference pin stopped at l_max = 4)."""
    w = inputs.config0()
    h = oracle.Hyper(w.rc_r, w.rc_a, w.n_max_r, n_max_a, l_max, 30, 1)
    dim = oracle.descriptor_dim(h)
    par = (2.0 * inputs.uniform01(43, oracle.num_params(h)) - 1.0) / math.sqrt(float(dim))
    F = oracle.evaluate(h, w.atomic_numbers, par, w.pos, w.vel, w.types, w.box)["F"]
    frms = math.sqrt((F ** 2).mean())
    eps = 1e-5
    for (a, i) in [(0, 0), (1, 7), (2, 13), (0, 31), (1, 50), (2, 63)]:
        def U_at(t):
            pp = w.pos.copy(); pp[a, i] += t
            return oracle.evaluate(h, w.atomic_numbers, par, pp, None, w.types, w.box)["U"].sum()
        num = -(8 * (U_at(eps) - U_at(-eps)) - (U_at(2 * eps) - U_at(-2 * eps))) / (12 * eps)
        assert F[a, i] == pytest.approx(num, abs=1e-6 * max(frms, 1e-3)), (a, i)
    assert np.abs(F.sum(axis=1)).max() < 1e-10 * max(1.0, np.abs(F).max())


@pytest.mark.parametrize("which", ["si", "pbte"])
def test_total_virial_is_minus_strain_derivative(oracle, which):
    w = inputs.config0() if which == "si" else _small_pbte()
    h = _hyper(oracle, w)
    out = oracle.evaluate(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box)
    Wtot = out["W"].sum(axis=1).reshape(3, 3)
    assert np.allclose(Wtot, Wtot.T, atol=1e-9 * np.abs(Wtot).max())         # total symmetric
    Wi = out["W"].T.reshape(-1, 3, 3)
    assert np.abs(Wi - Wi.transpose(0, 2, 1)).max() > 1e-6 * np.abs(Wi).max()  # per-atom is not
    eps = 1e-6
    for a in range(3):                      # diagonal strain keeps the box orthorhombic
        sp = np.ones(3); sp[a] += eps
        sm = np.ones(3); sm[a] -= eps
        Up = _total_U(oracle, h, w, w.pos * sp[:, None], w.box * sp)
        Um = _total_U(oracle, h, w, w.pos * sm[:, None], w.box * sm)
        assert Wtot[a, a] == pytest.approx(-(Up - Um) / (2 * eps), rel=1e-6, abs=1e-7)


def test_offdiagonal_virial_and_heat_current_on_open_cluster(oracle):
    """Open (non-periodic) cluster in a big box.  (i) sum_i W_i = -dU/d(eps) for a shear strain;
    (ii) sum_i W_i . v_i = sum_i r_i (dU_i/dt + F_i . v_i), which fixes the index orientation of
    Eq. 6-7 (reading Q13): the transposed contraction fails this identity."""
    n = 14
    u = inputs.uniform01(77, 3 * n).reshape(n, 3)
    pts = 40.0 + (u - 0.5) * 6.0
    box = np.array([80.0, 80.0, 80.0])
    pos = np.ascontiguousarray(pts.T)
    vel = np.ascontiguousarray((inputs.normal(78, 3 * n).reshape(n, 3) * 0.01).T)
    types = np.zeros(n, dtype=np.int32)
    w = inputs.config0()
    h = _hyper(oracle, w)
    ev = lambda p, v=None: oracle.evaluate(h, w.atomic_numbers, w.params, p, v, types, box)
    out = ev(pos, vel)
    W = out["W"].T.reshape(n, 3, 3)
    Wtot = W.sum(0)
    eps = 1e-6
    for (a, b) in [(0, 1), (1, 2), (2, 0), (1, 0)]:
        S = np.zeros((3, 3)); S[a, b] = eps
        Up = ev(np.ascontiguousarray(((np.eye(3) + S) @ pos)))["U"].sum()
        Um = ev(np.ascontiguousarray(((np.eye(3) - S) @ pos)))["U"].sum()
        assert Wtot[a, b] == pytest.approx(-(Up - Um) / (2 * eps), rel=1e-6, abs=1e-8)
    hh = 1e-4
    dUdt = (ev(pos + hh * vel)["U"] - ev(pos - hh * vel)["U"]) / (2 * hh)
    Fv = (out["F"] * vel).sum(0)
    rhs = (pos * (dUdt + Fv)[None, :]).sum(1)
    J = out["J"].sum(1)
    assert np.allclose(J, rhs, rtol=1e-6, atol=1e-9 * np.abs(rhs).max())
    J_transposed = np.einsum("iba,ib->a", W, vel.T)
    assert not np.allclose(J_transposed, rhs, rtol=1e-2)
    # Eq. 7 per atom
    assert np.allclose(out["J"].T, np.einsum("iab,ib->ia", W, vel.T), atol=1e-15)


def test_partial_force_structure(oracle):
    """p_ij for r_c^A <= r < r_c^R is purely radial (parallel to r_ij); Eq. 4-6 rebuild F and W
    from the stored partial forces."""
    w = inputs.config0()
    h = _hyper(oracle, w)
    cR, iR, _ = oracle.neighbors(w.pos, w.box, w.rc_r, 64)
    cA, iA, _ = oracle.neighbors(w.pos, w.box, w.rc_a, 64)
    out = oracle.compute(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, cR, iR, cA, iA, True)
    p = out["p"]
    n = w.n_atoms
    F = np.zeros((3, n)); Wt = np.zeros((n, 3, 3))
    checked = 0
    for i in range(n):
        for s in range(cR[i]):
            j = iR[i, s]
            d = w.pos[:, j] - w.pos[:, i]
            d -= w.box * np.rint(d / w.box)
            back = list(iR[j, :cR[j]]).index(i)
            F[:, i] += p[i, s] - p[j, back]
            Wt[i] += np.outer(d, p[j, back])
            if np.linalg.norm(d) >= w.rc_a:
                assert np.linalg.norm(np.cross(d, p[i, s])) < 1e-14
                checked += 1
    assert checked > 100
    assert np.allclose(F, out["F"], atol=1e-14)
    assert np.allclose(Wt.reshape(n, 9).T, out["W"], atol=1e-13)


def test_dimer_force_along_bond(oracle):
    w = inputs.config0()
    h = _hyper(oracle, w)
    box = np.array([50.0, 50.0, 50.0]); types = np.zeros(2, dtype=np.int32)

    def U_of(r):
        pos = np.array([[10.0, 10.0 + r], [10.0, 10.0], [10.0, 10.0]])
        return oracle.evaluate(h, w.atomic_numbers, w.params, pos, None, types, box)

    r, e = 2.9, 1e-6
    out = U_of(r)
    dUdr = (U_of(r + e)["U"].sum() - U_of(r - e)["U"].sum()) / (2 * e)
    assert out["F"][0, 1] == pytest.approx(-dUdr, rel=1e-7)
    assert out["F"][0, 0] == pytest.approx(dUdr, rel=1e-7)
    assert np.abs(out["F"][1:]).max() < 1e-15


def test_neighbors_brute_vs_cell_and_symmetry(oracle):
    for w, caps in ((inputs.config0(), (64, 32)), (inputs.si_cells((4, 4, 4)), (64, 32)),
                    (inputs.config3(cells=(3, 3, 3)), (96, 48))):
        for rc, cap in ((w.rc_r, caps[0]), (w.rc_a, caps[1])):
            cb, ib, nb = oracle.neighbors(w.pos, w.box, rc, cap, "brute")
            cc, ic, nc = oracle.neighbors(w.pos, w.box, rc, cap, "cell")
            assert np.array_equal(cb, cc) and np.array_equal(ib, ic)
            assert nb == 0 and nc == 0                       # no borderline pairs for these seeds (Q9)
            # independent numpy brute force
            d = w.pos[:, None, :] - w.pos[:, :, None]        # d[a,i,j] = r_j - r_i
            d -= w.box[:, None, None] * np.rint(d / w.box[:, None, None])
            r2 = (d ** 2).sum(0)
            np.fill_diagonal(r2, np.inf)
            adj = r2 < rc * rc
            assert np.array_equal(adj, adj.T)
            assert np.array_equal(adj.sum(1), cb)
            for i in (0, 5, w.n_atoms - 1):
                assert np.array_equal(np.nonzero(adj[i])[0], ib[i, :cb[i]])


def test_nve_conservation_and_dt_scaling(oracle):
    w = inputs.config0()
    h = _hyper(oracle, w)

    def run(dt, steps):
        out = oracle.md(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, dt, steps)
        E = out["thermo"][:, 0] + out["thermo"][:, 1]
        return out, E

    out1, E1 = run(1.0, 40)
    out2, E2 = run(0.5, 80)
    fl1 = np.abs(E1 - E1[0]).max() / w.n_atoms
    fl2 = np.abs(E2 - E2[0]).max() / w.n_atoms
    assert fl1 < 2e-5                                          # no drift: bounded fluctuation
    assert fl2 < fl1 / 2.5                                     # ~ dt^2
    # kinetic energy at step 0 is 300 K with 3N-3 degrees of freedom
    assert 2 * out1["thermo"][0, 1] / ((3 * 64 - 3) * inputs.KB_EV_PER_K) == pytest.approx(300.0, rel=1e-9)
    # time reversibility: flip velocities, integrate back
    back = oracle.md(h, w.atomic_numbers, w.params, out1["pos"], -out1["vel"], w.types, w.box, w.masses, 1.0, 40)
    assert np.abs(back["pos"] - w.pos).max() < 1e-9
    assert np.abs(back["vel"] + w.vel).max() < 1e-11
    # accumulated heat current equals the sum of per-step J (steps 1..n)
    assert np.allclose(out1["Jsum"].sum(1), out1["thermo"][1:, 2:5].sum(0), rtol=1e-10)


def _per_atom_virial_fd(ev, pos, box, periodic, atoms, eps=1e-5):
    """W_i^{ab} = sum_{j != i} r_ij^a dU_j/dr_i^b (Eq. 6 with dU_j/dr_ji == dU_j/dr_i):
    the derivative by 4th-order central differences of the oracle's PER-ATOM energies U_j as atom i moves.
    Also returns the 'wrong partial force' variant sum_j r_ij^a dU_i/dr_j^b (p_ij in place of p_ji)."""
    n = pos.shape[1]
    W = {}; Wwrong = {}
    for i in atoms:
        d = pos - pos[:, [i]]                                 # r_ij = r_j - r_i  (Eq. 3)
        if periodic:
            d -= box[:, None] * np.rint(d / box[:, None])
        dUj_dri = np.zeros((n, 3))
        for b in range(3):
            def U_at(t):
                pp = pos.copy(); pp[b, i] += t
                return ev(pp)["U"]
            dUj_dri[:, b] = (8 * (U_at(eps) - U_at(-eps)) - (U_at(2 * eps) - U_at(-2 * eps))) / (12 * eps)
        dUj_dri[i] = 0.0                                      # j != i
        W[i] = np.einsum("aj,jb->ab", d, dUj_dri)
        # negative control: dU_i/dr_j (what Eq. 6 would be with p_ij instead of p_ji)
        dUi_drj = np.zeros((n, 3))
        for j in range(n):
            if j == i or np.linalg.norm(d[:, j]) > 6.0:
                continue
            for b in range(3):
                pp = pos.copy(); pp[b, j] += eps
                pm = pos.copy(); pm[b, j] -= eps
                dUi_drj[j, b] = (ev(pp)["U"][i] - ev(pm)["U"][i]) / (2 * eps)
        Wwrong[i] = np.einsum("aj,jb->ab", d, dUi_drj)
    return W, Wwrong


@pytest.mark.parametrize("which", ["open_cluster", "c0_periodic"])
def test_per_atom_virial_and_heat_current_from_site_energy_derivatives(oracle, which):
    """Pins the PER-ATOM split of W_i (Eq. 6) and J_i (Eq. 7) with something other than the oracle's own
    formula: dU_j/dr_ji == dU_j/dr_i, so W_i^{ab} = sum_j r_ij^a dU_j/dr_i^b follows from central
    differences of the per-atom energies.  Negative controls: the transposed index order and p_ij in
    place of p_ji both fail."""
    w = inputs.config0()
    h = _hyper(oracle, w)
    if which == "open_cluster":
        n = 14
        u = inputs.uniform01(77, 3 * n).reshape(n, 3)
        pos = np.ascontiguousarray((40.0 + (u - 0.5) * 6.0).T)
        box = np.array([80.0, 80.0, 80.0])
        vel = np.ascontiguousarray((inputs.normal(78, 3 * n).reshape(n, 3) * 0.01).T)
        types = np.zeros(n, dtype=np.int32)
        atoms = list(range(n)); periodic = False
    else:
        pos, box, vel, types = w.pos, w.box, w.vel, w.types
        atoms = [0, 7, 13, 31, 50, 63]; periodic = True
    ev = lambda p, v=None: oracle.evaluate(h, w.atomic_numbers, w.params, p, v, types, box)
    out = ev(pos, vel)
    Wfd, Wwrong = _per_atom_virial_fd(ev, pos, box, periodic, atoms)
    scale = np.sqrt((out["W"] ** 2).mean())
    worst_T = 0.0; worst_P = 0.0
    for i in atoms:
        Wi = out["W"][:, i].reshape(3, 3)
        assert np.abs(Wi - Wfd[i]).max() < 1e-6 * max(scale, np.abs(Wi).max()), i
        Ji = Wfd[i] @ vel[:, i]                                # Eq. 7: J^a = sum_b W^{ab} v^b
        assert np.abs(out["J"][:, i] - Ji).max() < 1e-6 * max(np.abs(out["J"]).max(), 1e-12), i
        worst_T = max(worst_T, np.abs(Wi.T - Wfd[i]).max() / scale)
        worst_P = max(worst_P, np.abs(Wi - Wwrong[i]).max() / scale)
    assert worst_T > 1e-2        # transposed indices: off by O(1)
    assert worst_P > 1e-2        # p_ij in place of p_ji: off by O(1)
