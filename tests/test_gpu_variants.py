"""GPU parity of the variants of SURVEY.md 8(f) f-4 (nep_create_ex): two or three hidden layers and the
SOAP-like descriptor q_nn'l of Eq. 17-18, against the oracle's variant branches."""
import numpy as np
import pytest

from paper_2107_08119_b200 import inputs
from test_gpu_parity import TOL_REL, _gpu, check_lists, compare_outputs

pytestmark = pytest.mark.gpu


def _setup(oracle, w, layers, kind, caps, skin, seed=41):
    torch, api = _gpu()
    h = oracle.Hyper(w.rc_r, w.rc_a, w.n_max_r, w.n_max_a, w.l_max, layers[0], len(w.atomic_numbers))
    h.nlayers = len(layers); h.nneu2 = layers[1] if len(layers) > 1 else 0; h.nneu3 = layers[2] if len(layers) > 2 else 0
    h.kind = kind
    npar = oracle.num_params(h)
    par = (2.0 * inputs.uniform01(seed, npar) - 1.0) / np.sqrt(30.0)
    model = api.Model(w.rc_r, w.rc_a, w.n_max_r, w.n_max_a, w.l_max, layers[0], w.atomic_numbers, par,
                      hidden_layers=layers if len(layers) > 1 else (layers if kind else None), angular_kind=kind)
    assert model.descriptor_dim == oracle.descriptor_dim(h) and model.num_params == npar
    types = torch.from_numpy(w.types).cuda()
    system = api.System(model, types, caps[0], caps[1], skin)
    assert system.path == 2
    pos = torch.from_numpy(w.pos).cuda().contiguous(); vel = torch.from_numpy(w.vel).cuda().contiguous()
    return h, par, model, system, pos, vel


@pytest.mark.parametrize("which", ["c0", "c2", "c3_replica"])
@pytest.mark.parametrize("layers,kind", [((30, 20), 0), ((24, 16, 9), 0), ((30,), 1), ((20, 12), 1)])
def test_variants_match_oracle(oracle, which, layers, kind):
    w, caps, skin = {"c0": (inputs.config0(), (64, 32), 0.4), "c2": (inputs.config2(), (80, 40), 1.0),
                     "c3_replica": (inputs.config3(cells=(4, 4, 4)), (80, 40), 1.0)}[which]
    h, par, model, system, pos, vel = _setup(oracle, w, layers, kind, caps, skin)
    system.neighbors(pos, w.box)
    out = system.compute(pos, vel)
    system.status()
    ref = oracle.evaluate(h, w.atomic_numbers, par, w.pos, w.vel, w.types, w.box, 96, 64)
    compare_outputs(out, ref, label="%s layers %s kind %d" % (which, layers, kind))


def test_soap_like_intermediate_rows(oracle):
    torch, api = _gpu()
    w = inputs.config0()
    h, par, model, system, pos, vel = _setup(oracle, w, (30,), 1, (64, 32), 0.4)
    system.neighbors(pos, w.box)
    q, fp, p = [t.cpu().numpy().astype(np.float64) for t in system.compute_internals(pos)]
    system.status()
    ocR, oiR, _ = oracle.neighbors(w.pos, w.box, w.rc_r, 96)
    ocA, oiA, _ = oracle.neighbors(w.pos, w.box, w.rc_a, 64)
    ref = oracle.compute(h, w.atomic_numbers, par, w.pos, w.vel, w.types, w.box, ocR, oiR, ocA, oiA, want_internals=True)
    assert q.shape[0] == 8 + 36 * 4
    assert np.abs(q.T - ref["q"]).max() <= 2e-6 * np.abs(ref["q"]).max()
    assert np.abs(fp.T - ref["Fp"]).max() <= 2e-5 * np.abs(ref["Fp"]).max()


def test_md_with_deep_network_conserves_energy_like_the_oracle(oracle):
    torch, api = _gpu()
    w = inputs.config1()
    h, par, model, system, pos, vel = _setup(oracle, w, (30, 20), 0, (64, 32), 1.0)
    system.neighbors(pos, w.box)
    thermo = torch.zeros((40, 5), dtype=torch.float64, device="cuda")
    system.md_step(pos, vel, w.masses, w.dt, 40, thermo=thermo)
    system.status()
    ref = oracle.md(h, w.atomic_numbers, par, w.pos, w.vel, w.types, w.box, w.masses, w.dt, 40)
    th = thermo.cpu().numpy()
    E, Eref = th[:, 0] + th[:, 1], ref["thermo"][1:, 0] + ref["thermo"][1:, 1]
    assert np.abs(E - Eref).max() / w.n_atoms < 1e-5
    assert np.abs(pos.cpu().numpy() - ref["pos"]).max() < 1e-4


def test_create_ex_validation():
    torch, api = _gpu()
    w = inputs.config0()
    with pytest.raises(api.NepError):          # q_nn'l needs n_max <= 7
        api.Model(w.rc_r, w.rc_a, 8, 8, 4, 30, w.atomic_numbers, np.zeros(10), hidden_layers=[30], angular_kind=1)
    with pytest.raises(api.NepError):          # four hidden layers
        api.Model(w.rc_r, w.rc_a, 7, 7, 4, 30, w.atomic_numbers, np.zeros(10), hidden_layers=[30, 20, 10, 5])


@pytest.mark.parametrize("which", ["c0", "c2"])
@pytest.mark.parametrize("l_max,n_max_a", [(5, 7), (6, 5), (8, 3)])
def test_l_max_above_four_matches_oracle(oracle, which, l_max, n_max_a):
    """l_max = 5..8: the general-l kernel (harmonics and gradients by recurrence) against the oracle's
    literal Legendre double sum of Eq. 13 / 25, outputs at the north-star bars, intermediate rows included."""
    torch, api = _gpu()
    w, caps, skin = {"c0": (inputs.config0(), (64, 32), 0.4), "c2": (inputs.config2(), (80, 40), 1.0)}[which]
    h = oracle.Hyper(w.rc_r, w.rc_a, w.n_max_r, n_max_a, l_max, 30, 1)
    dim = oracle.descriptor_dim(h)
    assert dim == (w.n_max_r + 1) + (n_max_a + 1) * l_max
    npar = oracle.num_params(h)
    par = (2.0 * inputs.uniform01(43, npar) - 1.0) / np.sqrt(float(dim))
    model = api.Model(w.rc_r, w.rc_a, w.n_max_r, n_max_a, l_max, 30, w.atomic_numbers, par)
    assert model.descriptor_dim == dim and model.num_params == npar
    system = api.System(model, torch.from_numpy(w.types).cuda(), caps[0], caps[1], skin)
    pos = torch.from_numpy(w.pos).cuda().contiguous(); vel = torch.from_numpy(w.vel).cuda().contiguous()
    system.neighbors(pos, w.box)
    out = system.compute(pos, vel)
    system.status()
    ref = oracle.evaluate(h, w.atomic_numbers, par, w.pos, w.vel, w.types, w.box, 96, 64)
    compare_outputs(out, ref, label="%s l_max %d" % (which, l_max))
    q, fp, p = [t.cpu().numpy().astype(np.float64) for t in system.compute_internals(pos)]
    ocR, oiR, _ = oracle.neighbors(w.pos, w.box, w.rc_r, 96)
    ocA, oiA, _ = oracle.neighbors(w.pos, w.box, w.rc_a, 64)
    refi = oracle.compute(h, w.atomic_numbers, par, w.pos, w.vel, w.types, w.box, ocR, oiR, ocA, oiA, want_internals=True)
    assert np.abs(q.T - refi["q"]).max() <= 2e-6 * np.abs(refi["q"]).max()
    assert np.abs(fp.T - refi["Fp"]).max() <= 2e-5 * np.abs(refi["Fp"]).max()


def _make(api, w, n_max, layers, kind, npar):
    par = (2.0 * inputs.uniform01(47, npar) - 1.0) / np.sqrt(128.0)
    return par, api.Model(w.rc_r, w.rc_a, n_max, n_max, 4, layers[0], w.atomic_numbers, par, hidden_layers=list(layers),
                          angular_kind=kind)


def _npar(dim, layers):
    n, fan = 0, dim
    for wd in layers:
        n += (fan + 1) * wd; fan = wd
    return n + fan + 1


def test_shapes_beyond_the_shared_memory_of_k_gen_are_refused():
    """k_gen stages every layer's weights in shared memory beside its eight per-atom blocks.  Shapes that
    need more than the device's opt-in limit (227 KB per block on B200) used to be accepted by nep_create_ex and then
    failed at every launch; they are NEP_EINVAL now (include/nep_b200.h states the budgets)."""
    torch, api = _gpu()
    si, pbte = inputs.config0(), inputs.config3(cells=(4, 4, 4))
    for w, n_max, layers, kind in ((si, 7, (128, 128, 128), 1),        # 3 x 128 over q_nn'l (D = 152), fp32: ~257 KB
                                   (pbte, 15, (128, 128), 0),          # two species (fp64), 2 x 128 at D = 80: ~328 KB
                                   (pbte, 7, (128,), 1)):              # two species, one layer of 128 over q_nn'l: ~251 KB
        dim = (n_max + 1) + ((n_max + 1) * (n_max + 2) // 2 if kind else (n_max + 1)) * 4
        with pytest.raises(api.NepError) as err:
            _make(api, w, n_max, layers, kind, _npar(dim, layers))
        assert err.value.code == -1


@pytest.mark.parametrize("which,n_max,layers,kind", [("c0", 15, (128, 128, 128), 0), ("c0", 7, (128, 128), 1),
                                                       ("c3_replica", 15, (128,), 0), ("c3_replica", 7, (100,), 1)])
def test_widest_shapes_that_fit_match_oracle(oracle, which, n_max, layers, kind):
    """The widest networks nep_create_ex still accepts per kernel instantiation (fp32 / fp64, n_max <= 7 / > 7): each is
    within a few KB of the shared-memory limit, runs, and meets the north-star bars against the oracle."""
    torch, api = _gpu()
    w, caps, skin = {"c0": (inputs.config0(), (64, 32), 0.4), "c3_replica": (inputs.config3(cells=(4, 4, 4)), (80, 40), 1.0)}[which]
    h = oracle.Hyper(w.rc_r, w.rc_a, n_max, n_max, 4, layers[0], len(w.atomic_numbers))
    h.nlayers = len(layers); h.nneu2 = layers[1] if len(layers) > 1 else 0; h.nneu3 = layers[2] if len(layers) > 2 else 0
    h.kind = kind
    npar = oracle.num_params(h)
    assert npar == _npar(oracle.descriptor_dim(h), layers)
    par, model = _make(api, w, n_max, layers, kind, npar)
    system = api.System(model, torch.from_numpy(w.types).cuda(), caps[0], caps[1], skin)
    assert system.path == 2
    pos = torch.from_numpy(w.pos).cuda().contiguous(); vel = torch.from_numpy(w.vel).cuda().contiguous()
    system.neighbors(pos, w.box)
    out = system.compute(pos, vel)
    system.status()
    ref = oracle.evaluate(h, w.atomic_numbers, par, w.pos, w.vel, w.types, w.box, 96, 64)
    compare_outputs(out, ref, label="%s n_max %d layers %s kind %d" % (which, n_max, layers, kind))
