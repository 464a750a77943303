"""Pins for the oracle's HNEMD step (Eq. 8-11): the driving force F_i^ext = F_e . W_i and the
virial-velocity correlation K(t) = sum_i W_i(0) . v_i(t)."""
import numpy as np
import pytest

from paper_2107_08119_b200 import inputs


def _hyper(oracle, w):
    return oracle.Hyper(w.rc_r, w.rc_a, w.n_max_r, w.n_max_a, w.l_max, w.n_neurons, len(w.atomic_numbers))


def test_zero_driving_force_is_nve_bit_for_bit(oracle):
    w = inputs.config0()
    h = _hyper(oracle, w)
    a = oracle.md(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, 1.0, 12)
    b = oracle.md_driven(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, 1.0, 12, Fe=None)
    c = oracle.md_driven(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, 1.0, 12, Fe=[0.0, 0.0, 0.0])
    for k in ("pos", "vel", "U", "F", "W", "J", "Jsum", "thermo"):
        assert np.array_equal(a[k], b[k]), k
        assert np.array_equal(a[k], c[k]), k


def test_work_of_the_driving_force_equals_energy_change(oracle):
    """dE/dt = sum_i F_i^ext . v_i = F_e . J  (J = sum_i W_i . v_i, Eq. 7) holds only for the index reading
    (F^ext)^b = sum_a F_e^a W^{ab}.  Checked as E(t_n) - E(0) = integral of F_e . J dt (trapezoid); halving dt
    shrinks the residual ~4x (the integrator's and the quadrature's O(dt^2)); the transposed reading misses."""
    w = inputs.config0()
    h = _hyper(oracle, w)
    Fe = np.array([1.0e-2, -5.0e-3, 7.5e-3])            # 1/A: large enough that the work dominates the NVE fluctuation

    def run(dt, n):
        o = oracle.md_driven(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, dt, n, Fe=Fe)
        E = o["thermo"][:, 0] + o["thermo"][:, 1]
        P = o["thermo"][:, 2:5] @ Fe                    # F_e . J(t)
        work = dt * (0.5 * P[0] + P[1:-1].sum() + 0.5 * P[-1])
        return o, E[-1] - E[0], work

    o1, dE1, w1 = run(1.0, 40)
    o2, dE2, w2 = run(0.5, 80)
    o4, dE4, w4 = run(0.25, 160)
    r1, r2, r4 = abs(dE1 - w1), abs(dE2 - w2), abs(dE4 - w4)
    print("dE", dE1, dE2, dE4, "work", w1, w2, w4)
    assert abs(w4) > 3e-4                                 # the driven run really exchanges energy
    assert r4 < 0.05 * abs(w4)                            # energy balance closes ...
    assert 3.0 < r1 / r2 < 5.0 and 3.0 < r2 / r4 < 5.0    # ... at the integrator's O(dt^2)
    # negative control: the transposed contraction (F^ext)^b = sum_a F_e^a W^{ba} gives another power
    W = o1["W"]; v = o1["vel"]
    p_right = np.einsum("a,abi,bi->", Fe, W.reshape(3, 3, -1), v)
    p_wrong = np.einsum("a,bai,bi->", Fe, W.reshape(3, 3, -1), v)
    assert abs(p_right - o1["thermo"][-1, 2:5] @ Fe) < 1e-12 * max(1.0, abs(p_right))
    assert abs(p_wrong - p_right) > 1e-2 * abs(p_right)


def test_virial_velocity_correlation(oracle):
    """K(t) of Eq. 11 with the default W_i(0): K(0) = sum_i W_i(0) . v_i(0) = J(0); a supplied W0 is used as given;
    transposing W0 changes K."""
    w = inputs.config0()
    h = _hyper(oracle, w)
    o = oracle.md_driven(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, 1.0, 6, Fe=[1e-3, 0, 0])
    assert np.allclose(o["Kt"][0], o["thermo"][0, 2:5], rtol=1e-12, atol=1e-15)
    ev = oracle.evaluate(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box)
    o2 = oracle.md_driven(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, 1.0, 6, Fe=[1e-3, 0, 0], W0=ev["W"])
    assert np.array_equal(o["Kt"], o2["Kt"])
    # independent numpy evaluation at the last step
    K = np.einsum("abi,bi->a", ev["W"].reshape(3, 3, -1), o["vel"])
    assert np.allclose(o["Kt"][-1], K, rtol=1e-12)
    Kt = np.einsum("bai,bi->a", ev["W"].reshape(3, 3, -1), o["vel"])
    assert not np.allclose(Kt, K, rtol=1e-3)
