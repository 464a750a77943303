"""GPU parity on the BASELINE.json configs that round 1 left uncovered:
C4 at 262,144 / 884,736 / 1,048,576 atoms over ALL atoms with bit-exact lists; the MD legs of C2 (100 steps),
C3 at its full 64,000 atoms and C4-32768 (with an in-loop rebuild) against orc_md; D = 45 on C2.
All at the north-star bars (tests/test_gpu_parity.py)."""
import numpy as np
import pytest

from paper_2107_08119_b200 import inputs
from test_gpu_parity import TOL_REL, TOL_U, _gpu, _hyper, check_lists, compare_outputs, run_config

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_atoms", [262144, 884736, 1048576])
def test_c4_full_arrays(oracle, n_atoms):
    """Every atom of the large C4 sizes (1,048,576 = the launch configuration bench.py times): radial and
    angular lists bit-exact against the oracle's cell list, U, F, W, J element by element."""
    torch, api = _gpu()
    w = inputs.config4(n_atoms)
    model, system, pos, vel = api.from_workload(w, 64, 32, 1.0)
    system.neighbors(pos, w.box)
    out = system.compute(pos, vel)
    system.status()
    check_lists(oracle, w, system, 64, 32)
    ref = oracle.evaluate(_hyper(oracle, w), w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, 64, 32)
    compare_outputs(out, ref, label=w.name)
    F = out[1].double().cpu().numpy()
    frms = np.sqrt((ref["F"] ** 2).mean())
    assert np.abs(F.sum(1)).max() < 1e-4 * frms * np.sqrt(n_atoms)       # zero net force


def test_c2_d45(oracle):
    """The second reading of Q1 (n_max = 8, D = 45) on the irregular amorphous cell."""
    run_config(oracle, inputs.config2(n_max=8), cap_r=80, cap_a=40)


def _md_leg(oracle, w, n_steps, cap_r, cap_a, min_rebuilds, label, traj_tol, path=1):
    """n_steps of nep_md_step against orc_md: (i) the trajectories stay together, (ii) the energy record
    follows the oracle's, (iii) the outputs of the last step meet the north-star bars against the oracle
    evaluated at the SAME final state (so trajectory divergence does not enter the comparison),
    (iv) the filtered lists at the final positions are bit-exact."""
    torch, api = _gpu()
    model, system, pos, vel = api.from_workload(w, cap_r, cap_a, 1.0, path=path)
    system.neighbors(pos, w.box)
    heat_sum = torch.zeros((3, w.n_atoms), dtype=torch.float64, device="cuda")
    thermo = torch.zeros((n_steps, 5), dtype=torch.float64, device="cuda")
    out = system.md_step(pos, vel, w.masses, w.dt, n_steps, heat_sum=heat_sum, thermo=thermo)
    system.status()
    st = system.stats()
    assert st["rebuilds"] >= min_rebuilds, st
    h = _hyper(oracle, w)
    ref = oracle.md(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, w.dt, n_steps, 96, 64)
    gpos, gvel = pos.cpu().numpy(), vel.cpu().numpy()
    th = thermo.cpu().numpy()
    E = th[:, 0] + th[:, 1]
    Eref = ref["thermo"][1:, 0] + ref["thermo"][1:, 1]
    drift, drift_ref = np.abs(E - E[0]).max() / w.n_atoms, np.abs(Eref - Eref[0]).max() / w.n_atoms
    dpos = np.abs(gpos - ref["pos"]).max()
    print("%s: %d steps, rebuilds %d, |E-E0|/N gpu %.3g oracle %.3g, max|E-Eref|/N %.3g, max|dpos| %.3g A"
          % (label, n_steps, st["rebuilds"], drift, drift_ref, np.abs(E - Eref).max() / w.n_atoms, dpos))
    assert dpos < traj_tol
    assert np.abs(E - Eref).max() / w.n_atoms < 1e-5
    assert drift < 2 * drift_ref + 2e-5
    # outputs at the GPU's own final state
    w2 = inputs.Workload(w.name, gpos, gvel, w.types, w.box, w.rc_r, w.rc_a, w.n_max_r, w.n_max_a, w.l_max,
                         w.n_neurons, w.atomic_numbers, w.masses, w.params)
    check_lists(oracle, w2, system, cap_r, cap_a)
    ref2 = oracle.evaluate(h, w.atomic_numbers, w.params, gpos, gvel, w.types, w.box, 96, 64)
    compare_outputs(out, ref2, label=label + " final state")
    hs = heat_sum.cpu().numpy()
    assert np.abs(hs - ref["Jsum"]).max() < 5e-3 * np.abs(ref["Jsum"]).max()


def test_md_c2_amorphous_100_steps(oracle):
    _md_leg(oracle, inputs.config2(), 100, 80, 40, 2, "C2 a-Si 8000", 2e-3)


@pytest.mark.parametrize("path", [1, 2])
def test_md_c3_pbte_64000(oracle, path):
    _md_leg(oracle, inputs.config3(), 20, 80, 40, 1, "C3 PbTe 64000 path %d" % path, 1e-4, path=path)


def test_md_c4_32768_with_rebuild(oracle):
    _md_leg(oracle, inputs.config4(32768), 60, 64, 32, 2, "C4 Si 32768", 1e-4)


def _md_final_state(oracle, w, n_steps, cap_r, cap_a, min_rebuilds, label, oracle_md_steps=0, max_drift=2e-5, ocaps=(96, 64)):
    """MD above 65,536 atoms, where launch_build takes its third form: the ten-kernel device-gated chain that re-sorts
    an already sorted state (first = 0, gated = 2), with k_main's per-SM parking slots and the kick+drift fused into
    k_assemble (npad >= 262144) -- the configuration bench.py times.
    After n_steps with at least min_rebuilds in-loop rebuilds: filtered lists bit-exact and U, F, W, J at the
    north-star bars against the oracle evaluated at the GPU's OWN final state; the energy record stays flat.  With
    oracle_md_steps > 0 the first steps are also followed against orc_md (energies, trajectory, accumulated J)."""
    torch, api = _gpu()
    model, system, pos, vel = api.from_workload(w, cap_r, cap_a, 1.0)
    assert system.path == 1
    system.neighbors(pos, w.box)
    heat_sum = torch.zeros((3, w.n_atoms), dtype=torch.float64, device="cuda")
    thermo = torch.zeros((n_steps, 5), dtype=torch.float64, device="cuda")
    h = _hyper(oracle, w)
    done = 0
    if oracle_md_steps:
        system.md_step(pos, vel, w.masses, w.dt, oracle_md_steps, heat_sum=heat_sum, thermo=thermo[:oracle_md_steps])
        system.status()
        ref = oracle.md(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, w.dt, oracle_md_steps, 96, 64)
        th = thermo[:oracle_md_steps].cpu().numpy()
        E, Eref = th[:, 0] + th[:, 1], ref["thermo"][1:, 0] + ref["thermo"][1:, 1]
        dpos = np.abs(pos.cpu().numpy() - ref["pos"]).max()
        print("%s: first %d steps vs orc_md: max|E-Eref|/N %.3g, max|dpos| %.3g A" % (label, oracle_md_steps,
                                                                                 np.abs(E - Eref).max() / w.n_atoms, dpos))
        assert dpos < 1e-4 and np.abs(E - Eref).max() / w.n_atoms < 1e-5
        assert np.abs(heat_sum.cpu().numpy() - ref["Jsum"]).max() < 5e-3 * np.abs(ref["Jsum"]).max()
        done = oracle_md_steps
    out = system.md_step(pos, vel, w.masses, w.dt, n_steps - done, heat_sum=heat_sum, thermo=thermo[done:])
    system.status()
    st = system.stats()
    th = thermo.cpu().numpy()
    E = th[:, 0] + th[:, 1]
    drift = np.abs(E - E[0]).max() / w.n_atoms
    print("%s: %d steps, rebuilds %d, |E-E0|/N %.3g eV" % (label, n_steps, st["rebuilds"], drift))
    assert st["rebuilds"] >= min_rebuilds + 1, st          # the initial nep_neighbors counts as one
    assert max_drift is None or drift < max_drift
    gpos, gvel = pos.cpu().numpy(), vel.cpu().numpy()
    w2 = inputs.Workload(w.name, gpos, gvel, w.types, w.box, w.rc_r, w.rc_a, w.n_max_r, w.n_max_a, w.l_max,
                         w.n_neurons, w.atomic_numbers, w.masses, w.params)
    check_lists(oracle, w2, system, cap_r, cap_a)
    ref2 = oracle.evaluate(h, w.atomic_numbers, w.params, gpos, gvel, w.types, w.box, ocaps[0], ocaps[1])
    compare_outputs(out, ref2, label=label + " final state")


def test_md_c3_pbte_all_1000_steps_final_state(oracle):
    """BASELINE.json configs[3] in full: 1000 NVE steps of the 64,000-atom PbTe cell (the MD legs above follow orc_md for
    20).  A chaotic trajectory cannot be compared step by step that far, and the random-weight PbTe surface heats in the
    oracle too (section 3 of DESIGN.md), so what is checked is the state the GPU arrives at after ~50 in-loop rebuilds
    (permutations composed rebuild after rebuild, velocities carried): lists bit-exact, U, F, W, J at the bars.
    Measured: the seeded random-weight model is not a stable potential at dt = 1 fs -- E/N rises by 12.4 eV over the
    1000 steps (2.6e-4 after 20 steps on the GPU and in orc_md alike, 3.6e-2 after 200), the lists are rebuilt 420
    times -- and the hot, disordered end state still meets every bar: the comparison is about the arithmetic, not the
    physics of a random network."""
    _md_final_state(oracle, inputs.config3(), 1000, 80, 40, 20, "C3 PbTe 64000, 1000 steps", max_drift=None, ocaps=(124, 64))


def test_md_c4_32768_all_1000_steps_final_state(oracle):
    """BASELINE.json configs[4], smallest size, all 1000 steps: energy flat to 2e-5 eV/atom, final state at the bars."""
    _md_final_state(oracle, inputs.config4(32768), 1000, 64, 32, 20, "C4 Si 32768, 1000 steps")


def test_md_c4_262144_gated_rebuild_chain(oracle):
    _md_final_state(oracle, inputs.config4(262144), 60, 64, 32, 2, "C4 Si 262144", oracle_md_steps=20)


def test_md_c4_1048576_benchmarked_configuration(oracle):
    _md_final_state(oracle, inputs.config4(1048576), 60, 64, 32, 2, "C4 Si 1048576")
