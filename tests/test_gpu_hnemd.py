"""GPU parity of nep_md_step_driven (HNEMD driving force, Eq. 9, and K(t), Eq. 11) against
orc_md_driven on the same seeded inputs."""
import numpy as np
import pytest

from paper_2107_08119_b200 import inputs
from test_gpu_parity import _gpu, _hyper, compare_outputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("which,path", [("c1", 1), ("c1", 2), ("c0", 2)])
def test_driven_trajectory_tracks_oracle(oracle, which, path):
    torch, api = _gpu()
    w = inputs.config1() if which == "c1" else inputs.config0()
    skin = 1.0 if which == "c1" else 0.4
    n_steps = 40
    Fe = np.array([1.0e-2, -5.0e-3, 7.5e-3])
    model, system, pos, vel = api.from_workload(w, 64, 32, skin, path=path)
    system.neighbors(pos, w.box)
    U0, F0, W0, J0 = system.compute(pos, vel)
    w0 = W0.clone()
    thermo = torch.zeros((n_steps, 5), dtype=torch.float64, device="cuda")
    kt = torch.zeros((n_steps, 3), dtype=torch.float64, device="cuda")
    out = system.md_step_driven(pos, vel, w.masses, w.dt, n_steps, Fe, thermo=thermo, w0=w0, kt=kt)
    system.status()
    h = _hyper(oracle, w)
    ref = oracle.md_driven(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, w.dt, n_steps, Fe=Fe)
    nve = oracle.md(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, w.masses, w.dt, n_steps)
    gpos, gvel = pos.cpu().numpy(), vel.cpu().numpy()
    # the driving force matters (the driven and the NVE trajectories separate) and the GPU follows the driven one
    sep = np.abs(ref["pos"] - nve["pos"]).max()
    dpos = np.abs(gpos - ref["pos"]).max()
    print("driven vs NVE separation %.3g A, gpu vs oracle %.3g A" % (sep, dpos))
    assert sep > 1e-4 and dpos < 1e-2 * sep
    th = thermo.cpu().numpy()
    E, Eref = th[:, 0] + th[:, 1], ref["thermo"][1:, 0] + ref["thermo"][1:, 1]
    assert np.abs(E - Eref).max() / w.n_atoms < 1e-5
    jscale = np.abs(ref["thermo"][1:, 2:5]).max()
    assert np.abs(th[:, 2:5] - ref["thermo"][1:, 2:5]).max() < 1e-3 * jscale
    # K(t), Eq. 11, with W_i(0) = the virial nep_compute returned at t = 0
    K, Kref = kt.cpu().numpy(), ref["Kt"][1:]
    assert np.abs(K - Kref).max() < 1e-3 * np.abs(Kref).max()
    # outputs of the last step at the GPU's own final state (force_dev = the potential force of Eq. 4)
    ref2 = oracle.evaluate(h, w.atomic_numbers, w.params, gpos, gvel, w.types, w.box)
    compare_outputs(out, ref2, label="%s driven path %d final state" % (which, path))


def test_null_driving_force_is_nep_md_step():
    torch, api = _gpu()
    w = inputs.config1()
    res = []
    for driven in (False, True):
        model, system, pos, vel = api.from_workload(w, 64, 32, 1.0)
        system.neighbors(pos, w.box)
        if driven:
            system.md_step_driven(pos, vel, w.masses, w.dt, 30, None)
        else:
            system.md_step(pos, vel, w.masses, w.dt, 30)
        system.status()
        res.append((pos.clone(), vel.clone()))
    assert torch.equal(res[0][0], res[1][0]) and torch.equal(res[0][1], res[1][1])
