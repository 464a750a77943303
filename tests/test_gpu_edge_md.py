"""GPU edge cases and the velocity-Verlet path of libnep_b200.so against the oracle."""
import numpy as np
import pytest

from paper_2107_08119_b200 import inputs
from test_gpu_parity import _gpu, _hyper, compare_outputs, check_lists

pytestmark = pytest.mark.gpu


def _tiny_workload(pts, box, types=None, base=None):
    base = base or inputs.config0()
    pos = np.ascontiguousarray(np.asarray(pts, dtype=np.float64).T)
    n = pos.shape[1]
    w = inputs.Workload("tiny", pos, np.zeros((3, n)), np.zeros(n, dtype=np.int32) if types is None else types,
                        np.asarray(box, dtype=np.float64), base.rc_r, base.rc_a, base.n_max_r, base.n_max_a,
                        base.l_max, base.n_neurons, base.atomic_numbers, base.masses, base.params)
    return w


def test_isolated_atoms_and_dimer(oracle):
    """Empty neighbour lists (reading Q14): q = 0, U_i = sum w2 tanh(-b1) - b2, zero force;
    plus a dimer and a pair between the two cutoffs (radial-only partial force)."""
    torch, api = _gpu()
    pts = [[5, 5, 5], [25, 25, 25], [27.5, 25, 25], [5, 30, 30], [5, 34.5, 30]]     # isolated, dimer, 4.5 A pair
    w = _tiny_workload(pts, [40, 40, 40])
    w.vel = np.ascontiguousarray(inputs.normal(5, 15).reshape(3, 5) * 0.01)
    model, system, pos, vel = api.from_workload(w, 16, 8, 1.0)
    system.neighbors(pos, w.box)
    out = system.compute(pos, vel)
    system.status()
    ref = oracle.evaluate(_hyper(oracle, w), w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box)
    U, F, W, J = [t.cpu().numpy() for t in out]
    assert np.abs(U - ref["U"]).max() < 1e-6
    assert np.abs(F - ref["F"]).max() < 1e-6 and np.all(F[:, 0] == 0)
    assert np.abs(W - ref["W"]).max() < 1e-5 and np.abs(J - ref["J"]).max() < 1e-7
    cnt, idx = system.get_neighbors(0)
    assert cnt.cpu().tolist() == [0, 1, 1, 1, 1]
    cnt, idx = system.get_neighbors(1)
    assert cnt.cpu().tolist() == [0, 1, 1, 0, 0]


def test_single_atom(oracle):
    torch, api = _gpu()
    w = _tiny_workload([[1, 2, 3]], [30, 30, 30])
    model, system, pos, vel = api.from_workload(w, 8, 8, 0.5)
    system.neighbors(pos, w.box)
    U, F, W, J = system.compute(pos, None)
    system.status()
    ref = oracle.evaluate(_hyper(oracle, w), w.atomic_numbers, w.params, w.pos, None, w.types, w.box)
    assert abs(U.item() - ref["U"][0]) < 1e-6 and torch.all(F == 0) and torch.all(W == 0)


def test_error_codes(oracle):
    torch, api = _gpu()
    w = inputs.config0()
    # n_params mismatch / unsupported l_max -> NEP_EINVAL
    with pytest.raises(api.NepError) as e:
        api.Model(w.rc_r, w.rc_a, 7, 7, 4, 30, w.atomic_numbers, w.params[:-1])
    assert e.value.code == -1
    with pytest.raises(api.NepError) as e:
        api.Model(w.rc_r, w.rc_a, 7, 7, 9, 30, w.atomic_numbers, w.params)
    assert e.value.code == -1
    model, system, pos, vel = api.from_workload(w, 64, 32, 1.0)
    with pytest.raises(api.NepError) as e:            # compute before neighbors -> NEP_ESTATE
        system.compute(pos, vel)
    assert e.value.code == -7
    with pytest.raises(api.NepError) as e:            # 10.862 <= 2 (5 + 1) -> NEP_EBOX
        system.neighbors(pos, w.box)
    assert e.value.code == -2
    # capacity overflow is reported, never truncated silently -> NEP_EOVERFLOW
    model, system, pos, vel = api.from_workload(w, 20, 8, 0.4)
    system.neighbors(pos, w.box)
    system.compute(pos, vel)
    with pytest.raises(api.NepError) as e:
        system.status()
    assert e.value.code == -5
    # stale list: move one atom by more than skin/2 -> NEP_ESTALE
    model, system, pos, vel = api.from_workload(w, 64, 32, 0.4)
    system.neighbors(pos, w.box)
    moved = pos.clone(); moved[0, 3] += 0.3
    system.compute(moved, vel)
    with pytest.raises(api.NepError) as e:
        system.status()
    assert e.value.code == -6
    # two atoms at one position: r_ij = 0, the result is not finite -> NEP_ENAN (sticky, reported by nep_status)
    model, system, pos, vel = api.from_workload(w, 64, 32, 0.4)
    twin = pos.clone(); twin[:, 1] = twin[:, 0]
    system.neighbors(twin, w.box)
    system.compute(twin, vel)
    with pytest.raises(api.NepError) as e:
        system.status()
    assert e.value.code == -8


def test_compute_with_moved_positions_within_skin(oracle):
    """Lists built at one set of positions serve positions displaced by < skin/2 (Verlet skin):
    the filtered lists and all outputs must equal the oracle's from-scratch result."""
    torch, api = _gpu()
    w = inputs.config1()
    model, system, pos, vel = api.from_workload(w, 64, 32, 1.0)
    system.neighbors(pos, w.box)
    disp = inputs.normal(123, 3 * w.n_atoms).reshape(3, -1)
    disp = 0.45 * disp / np.maximum(1.0, np.linalg.norm(disp, axis=0))        # |disp| <= 0.45 < skin/2
    w2 = inputs.config1()
    w2.pos = np.ascontiguousarray(w.pos + disp)
    pos2 = torch.from_numpy(w2.pos).cuda()
    out = system.compute(pos2, vel)
    system.status()
    check_lists(oracle, w2, system, 64, 32)
    ref = oracle.evaluate(_hyper(oracle, w2), w2.atomic_numbers, w2.params, w2.pos, w2.vel, w2.types, w2.box)
    compare_outputs(out, ref, label="C1 displaced")


def _md_compare(oracle, w, n_steps, skin, cap_r=64, cap_a=32, path=1):
    torch, api = _gpu()
    model, system, pos, vel = api.from_workload(w, cap_r, cap_a, skin, path=path)
    system.neighbors(pos, w.box)
    heat_sum = torch.zeros((3, w.n_atoms), dtype=torch.float64, device="cuda")
    thermo = torch.zeros((n_steps, 5), dtype=torch.float64, device="cuda")
    out = system.md_step(pos, vel, w.masses, w.dt, n_steps, heat_sum=heat_sum, thermo=thermo)
    system.status()
    ref = oracle.md(_hyper(oracle, w), w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, w.dt, n_steps)
    return system, pos.cpu().numpy(), vel.cpu().numpy(), out, heat_sum.cpu().numpy(), thermo.cpu().numpy(), ref


@pytest.mark.parametrize("path", [1, 2])
def test_md_c0_trajectory_matches_oracle(oracle, path):
    w = inputs.config0()
    n_steps = 50
    system, pos, vel, out, hsum, thermo, ref = _md_compare(oracle, w, n_steps, 0.4, path=path)
    # fp32 forces vs fp64 forces: trajectories stay together over 50 fs
    assert np.abs(pos - ref["pos"]).max() < 2e-6
    assert np.abs(vel - ref["vel"]).max() < 2e-7
    compare_outputs(out, ref, label="C0 after 50 steps")
    E = thermo[:, 0] + thermo[:, 1]
    Eref = ref["thermo"][1:, 0] + ref["thermo"][1:, 1]
    assert np.abs(E - Eref).max() / w.n_atoms < 2e-6
    assert np.abs(E - Eref[0]).max() / w.n_atoms < 2e-5                 # conservation
    jscale = np.abs(ref["thermo"][1:, 2:5]).max()
    assert np.abs(thermo[:, 2:5] - ref["thermo"][1:, 2:5]).max() < 1e-3 * jscale
    assert np.abs(hsum - ref["Jsum"]).max() < 1e-3 * np.abs(ref["Jsum"]).max()


def test_md_c1_nve_with_rebuilds(oracle):
    """C1: 100 NVE steps at dt = 1 fs with per-atom heat current accumulated; the random-weight
    potential heats the crystal, so the Verlet list must rebuild on the device mid-run."""
    w = inputs.config1()
    n_steps = 100
    system, pos, vel, out, hsum, thermo, ref = _md_compare(oracle, w, n_steps, 1.0)
    st = system.stats()
    assert st["rebuilds"] >= 2, st                    # the initial build + at least one in-loop rebuild
    E = thermo[:, 0] + thermo[:, 1]
    Eref = ref["thermo"][1:, 0] + ref["thermo"][1:, 1]
    drift_ref = np.abs(Eref - Eref[0]).max() / w.n_atoms
    drift = np.abs(E - E[0]).max() / w.n_atoms
    print("C1 NVE |E-E0|/N: gpu %.3g  oracle %.3g  rebuilds %d" % (drift, drift_ref, st["rebuilds"]))
    assert drift < max(2 * drift_ref, 2e-5)
    assert np.abs(E - Eref).max() / w.n_atoms < 1e-5
    assert np.abs(pos - ref["pos"]).max() < 1e-4
    compare_outputs(out, ref, tol_u=2e-5, tol_rel=1e-3, label="C1 after 100 steps (trajectory divergence included)")
    assert np.abs(hsum - ref["Jsum"]).max() < 1e-3 * np.abs(ref["Jsum"]).max()


def test_md_c3_pbte_replica_tracks_oracle(oracle):
    """C3 geometry (4x4x4 rock-salt cells, 512 atoms, literal Eq. 19) for 20 NVE steps: the GPU
    trajectory and energies are judged against the oracle's own run at the same dt (the saturating
    network makes the oracle itself drift; SURVEY.md 8(c) 'PbTe conditioning')."""
    w = inputs.config3(cells=(4, 4, 4))
    n_steps = 20
    system, pos, vel, out, hsum, thermo, ref = _md_compare(oracle, w, n_steps, 1.0, cap_r=80, cap_a=40)
    E = thermo[:, 0] + thermo[:, 1]
    Eref = ref["thermo"][1:, 0] + ref["thermo"][1:, 1]
    drift_ref = np.abs(Eref - Eref[0]).max() / w.n_atoms
    drift = np.abs(E - E[0]).max() / w.n_atoms
    print("C3 NVE |E-E0|/N: gpu %.3g  oracle %.3g" % (drift, drift_ref))
    assert drift < 2 * drift_ref + 1e-6
    assert np.abs(E - Eref).max() / w.n_atoms < 1e-5
    assert np.abs(pos - ref["pos"]).max() < 1e-4


def test_md_chunked_calls_continue_trajectory(oracle):
    """nep_md_step(30) + nep_md_step(20) == nep_md_step(50) bit for bit (same launch sequence)."""
    torch, api = _gpu()
    w = inputs.config1()
    res = []
    for chunks in ((50,), (30, 20)):
        model, system, pos, vel = api.from_workload(w, 64, 32, 1.0)
        system.neighbors(pos, w.box)
        for n in chunks:
            out = system.md_step(pos, vel, w.masses, w.dt, n)
        system.status()
        res.append((pos.clone(), vel.clone(), out[1].clone()))
    assert (res[0][0] - res[1][0]).abs().max().item() < 1e-9
    assert (res[0][1] - res[1][1]).abs().max().item() < 1e-10


def test_system_created_and_run_on_a_non_blocking_stream(oracle):
    """nep_system_create clears the workspace and copies the types on the legacy default stream, which
    does not order itself against cudaStreamNonBlocking streams (every PyTorch side stream is one).  With the types
    produced on such a stream right before the call, and nep_neighbors / nep_compute issued on it right after, the
    results must be those of the default-stream run: nep_system_create synchronises the device on both sides."""
    torch, api = _gpu()
    w = inputs.config3((6, 6, 6))                                   # two species: a wrong or late type copy shows
    ref_model, ref_sys, pos, vel = api.from_workload(w, 80, 40, 1.0)
    ref_sys.neighbors(pos, w.box)
    ref = [t.clone() for t in ref_sys.compute(pos, vel)]
    ref_sys.status()
    side = torch.cuda.Stream()
    host_types = torch.from_numpy(w.types).pin_memory()
    filler = torch.empty(1 << 28, dtype=torch.uint8, device="cuda")
    for rep in range(3):
        with torch.cuda.stream(side):
            for _ in range(8):
                filler.fill_(rep)                                   # keeps the side stream busy ahead of the copy
            types = torch.empty(w.n_atoms, dtype=torch.int32, device="cuda")
            types.copy_(host_types, non_blocking=True)
            system = api.System(ref_model, types, 80, 40, 1.0)
            system.neighbors(pos, w.box)
            out = system.compute(pos, vel)
        side.synchronize()
        system.status()
        for a, b in zip(out, ref):
            assert torch.equal(a, b)
        for which in (0, 1):
            ca, ia = system.get_neighbors(which); cb, ib = ref_sys.get_neighbors(which)
            torch.cuda.synchronize()
            assert torch.equal(ca, cb)
