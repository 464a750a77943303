"""GPU parity of the training side (nep_trainer_*, nep_snes_*) against orc_loss / orc_snes_*."""
import math

import numpy as np
import pytest

from paper_2107_08119_b200 import inputs
from test_gpu_parity import _gpu

pytestmark = pytest.mark.gpu


def _oracle_targets(oracle, h, ts, z, znum=(14,)):
    e, v = [], []
    f = np.zeros((3, ts.n_atoms))
    comp = [0, 4, 8, 1, 5, 6]
    for n in range(ts.n_structures):
        a0, a1 = ts.first[n], ts.first[n + 1]
        out = oracle.evaluate(h, list(znum), z, np.ascontiguousarray(ts.pos[:, a0:a1]), None, ts.types[a0:a1], ts.boxes[n])
        e.append(out["U"].sum() / (a1 - a0)); v.append(out["W"].sum(axis=1)[comp] / (a1 - a0)); f[:, a0:a1] = out["F"]
    return np.array(e), f, np.array(v)


@pytest.mark.parametrize("layers,kind", [((30,), 0), ((16, 8), 1)])
def test_population_losses_match_oracle(oracle, layers, kind):
    torch, api = _gpu()
    ts = inputs.training_set(12, seed=70)
    h = oracle.Hyper(5.0, 4.0, 7, 7, 4, layers[0], 1)
    h.nlayers = len(layers); h.nneu2 = layers[1] if len(layers) > 1 else 0; h.kind = kind
    npar = oracle.num_params(h)
    teacher = (2 * inputs.uniform01(71, npar) - 1) / math.sqrt(30.0)
    e, f, v = _oracle_targets(oracle, h, ts, teacher)
    dev = "cuda"
    pos = torch.from_numpy(ts.pos).to(dev)
    e_t = torch.from_numpy(e.astype(np.float32)).to(dev); f_t = torch.from_numpy(f.astype(np.float32)).to(dev).contiguous()
    v_t = torch.from_numpy(v.astype(np.float32)).to(dev).contiguous()
    tr = api.Trainer(5.0, 4.0, 7, 7, 4, layers, ts.first, ts.boxes, pos, e_t, f_t, v_t, angular_kind=kind)
    assert tr.num_params == npar
    # prediction of the teacher = the targets
    ge, gf, gv = [t.cpu().numpy().astype(np.float64) for t in tr.predict(torch.from_numpy(teacher).to(dev))]
    tr.status()
    frms = math.sqrt((f ** 2).mean())
    assert np.abs(ge - e).max() < 1e-5 and np.abs(gf - f).max() < 1e-4 * frms and np.abs(gv - v).max() < 1e-4 * np.sqrt((v ** 2).mean())
    # a population around the teacher: every loss component against the oracle
    npop = 6
    r = inputs.normal(72, npop * npar).reshape(npop, npar)
    z = teacher[None, :] + 0.05 * r
    z[0] = teacher
    lam = [1.0, 1.0, 1.0, 0.05, 0.05]
    L = tr.losses(torch.from_numpy(z).to(dev).contiguous(), lam).cpu().numpy()
    for k in range(npop):
        ref = oracle.loss(h, [14], z[k], ts.first, ts.pos, ts.types, ts.boxes, e.astype(np.float32), f.astype(np.float32),
                          v.astype(np.float32), lam)
        print(k, L[k], ref)
        assert L[k, 3] == pytest.approx(ref[3], rel=1e-12) and L[k, 4] == pytest.approx(ref[4], rel=1e-12)
        for c in (0, 1, 2):
            assert abs(L[k, c] - ref[c]) < 1e-4 * max(ref[c], 1e-3) + 2e-6, (k, c)
        assert L[k, 5] == pytest.approx(ref[5], rel=2e-4, abs=1e-5)
    assert np.argmin(L[:, 5]) == 0                               # the teacher itself has the smallest loss


def test_snes_generation_matches_oracle(oracle):
    torch, api = _gpu()
    npop, npar = 50, 1261
    m = 0.5 * (2 * inputs.uniform01(80, npar) - 1); s = np.full(npar, 0.1)
    r = inputs.normal(81, npop * npar).reshape(npop, npar)
    loss = inputs.uniform01(82, npop); loss[7] = loss[3]                         # a tie
    dm, ds, dr = [torch.from_numpy(a).cuda() for a in (m, s, r)]
    z = api.snes_sample(dm, ds, dr)
    assert np.allclose(z.cpu().numpy(), oracle.snes_sample(m, s, r), rtol=0, atol=1e-15)      # Eq. 35 (the GPU contracts it into one FMA)
    eta_s = (3 + math.log(npar)) / (5 * math.sqrt(npar))
    api.snes_update(dm, ds, dr, torch.from_numpy(loss).cuda(), 1.0, eta_s)
    m2, s2 = oracle.snes_update(m, s, r, loss, 1.0, eta_s)
    assert np.allclose(dm.cpu().numpy(), m2, rtol=1e-13, atol=1e-15) and np.allclose(ds.cpu().numpy(), s2, rtol=1e-13)


def test_snes_update_ranks_a_nan_member_last(oracle):
    """ADVICE round 2 / reading Q25: one member with a NaN loss and one with +inf; the update equals the oracle's, in
    which both rank last, and stays finite."""
    torch, api = _gpu()
    npop, npar = 12, 300
    m = 0.5 * (2 * inputs.uniform01(83, npar) - 1); s = np.full(npar, 0.1)
    r = inputs.normal(84, npop * npar).reshape(npop, npar)
    loss = inputs.uniform01(85, npop); loss[2] = float("nan"); loss[9] = float("inf")
    dm, ds, dr = [torch.from_numpy(a).cuda() for a in (m, s, r)]
    api.snes_update(dm, ds, dr, torch.from_numpy(loss).cuda(), 1.0, 0.3)
    m2, s2 = oracle.snes_update(m, s, r, loss, 1.0, 0.3)
    assert np.all(np.isfinite(m2)) and np.all(np.isfinite(s2))
    assert np.allclose(dm.cpu().numpy(), m2, rtol=1e-13, atol=1e-15) and np.allclose(ds.cpu().numpy(), s2, rtol=1e-13)


def test_a_broken_member_is_reported_and_ranked_last(oracle):
    """One member of the population has NaN weights: its losses come out non-finite, nep_trainer_status reports
    NEP_ENAN for the generation (sticky bit set in k_assemble), the other members' losses are untouched, and the SNES
    update that follows ranks the broken member last (reading Q25) -- m and s stay finite and equal the oracle's."""
    torch, api = _gpu()
    ts = inputs.training_set(6, seed=93)
    dev = "cuda"
    pos = torch.from_numpy(ts.pos).to(dev)
    probe = api.Trainer(5.0, 4.0, 3, 3, 2, (8,), ts.first, ts.boxes, pos)
    npar = probe.num_params
    teacher = torch.from_numpy((2 * inputs.uniform01(94, npar) - 1) * 0.5).to(dev)
    e_t, f_t, v_t = probe.predict(teacher)
    tr = api.Trainer(5.0, 4.0, 3, 3, 2, (8,), ts.first, ts.boxes, pos, e_t, f_t, v_t)
    npop = 8
    m = 0.5 * (2 * inputs.uniform01(95, npar) - 1); s = np.full(npar, 0.1)
    r = inputs.normal(96, npop * npar).reshape(npop, npar)
    dm, ds, dr = [torch.from_numpy(a).to(dev) for a in (m, s, r)]
    z = api.snes_sample(dm, ds, dr)
    lam = [1.0, 1.0, 1.0, 0.0, 0.0]
    good = tr.losses(z, lam).cpu().numpy()
    tr.status()                                                   # a healthy generation: no error
    z[3] = float("nan")
    L = tr.losses(z, lam)
    with pytest.raises(api.NepError) as err:
        tr.status()
    assert err.value.code == -8                                   # NEP_ENAN
    Lh = L.cpu().numpy()
    # the others as before (to rounding: k_train_reduce adds its per-structure squared errors with fp64 atomics)
    assert not np.isfinite(Lh[3, 5]) and np.allclose(np.delete(Lh, 3, axis=0), np.delete(good, 3, axis=0), rtol=1e-12, atol=0)
    api.snes_update(dm, ds, dr, L, 1.0, 0.3)
    m2, s2 = oracle.snes_update(m, s, r, Lh[:, 5], 1.0, 0.3)
    assert np.all(np.isfinite(m2)) and np.all(np.isfinite(s2))
    assert np.allclose(dm.cpu().numpy(), m2, rtol=1e-13, atol=1e-15) and np.allclose(ds.cpu().numpy(), s2, rtol=1e-13)
    tr.status()                                                   # the sticky bit was cleared by the read above


def test_training_loop_reduces_the_loss():
    """A few SNES generations on synthetic targets (a teacher network evaluated by the library itself): the best loss falls.
    NOT a parity test: the targets are the library's own predictions, so this checks the sample -> losses -> update loop
    only; the comparisons with the oracle are the tests above and below."""
    torch, api = _gpu()
    ts = inputs.training_set(16, seed=90)
    dev = "cuda"
    pos = torch.from_numpy(ts.pos).to(dev)
    probe = api.Trainer(5.0, 4.0, 3, 3, 2, (8,), ts.first, ts.boxes, pos)
    npar = probe.num_params
    teacher = torch.from_numpy((2 * inputs.uniform01(91, npar) - 1) * 0.5).to(dev)
    e_t, f_t, v_t = probe.predict(teacher)
    tr = api.Trainer(5.0, 4.0, 3, 3, 2, (8,), ts.first, ts.boxes, pos, e_t, f_t, v_t)
    npop = 30
    m = torch.from_numpy(0.5 * (2 * inputs.uniform01(92, npar) - 1)).to(dev); s = torch.full((npar,), 0.1, dtype=torch.float64, device=dev)
    eta_s = (3 + math.log(npar)) / (5 * math.sqrt(npar))
    best = []
    for g in range(40):
        r = torch.from_numpy(inputs.normal(100 + g, npop * npar).reshape(npop, npar)).to(dev)
        z = api.snes_sample(m, s, r)
        L = tr.losses(z, [1.0, 1.0, 1.0, 0.0, 0.0])
        api.snes_update(m, s, r, L, 1.0, eta_s)
        best.append(float(L[:, 5].min()))
    tr.status()
    print("best loss first/last:", best[0], best[-1])
    assert best[-1] < 0.6 * best[0]


def test_multispecies_population_losses_match_oracle(oracle):
    """A PbTe training set (Eq. 19 weights, descriptor and network in fp64 on the GPU) against orc_loss."""
    torch, api = _gpu()
    ts = inputs.training_set(8, seed=75, material="pbte")
    znum = (82, 52)
    h = oracle.Hyper(6.0, 4.5, 5, 3, 4, 12, 2)
    npar = oracle.num_params(h)
    teacher = (2 * inputs.uniform01(76, npar) - 1) / math.sqrt(30.0)
    e, f, v = _oracle_targets(oracle, h, ts, teacher, znum)
    dev = "cuda"
    pos = torch.from_numpy(ts.pos).to(dev); types = torch.from_numpy(ts.types).to(dev)
    e_t = torch.from_numpy(e.astype(np.float32)).to(dev); f_t = torch.from_numpy(f.astype(np.float32)).to(dev).contiguous()
    v_t = torch.from_numpy(v.astype(np.float32)).to(dev).contiguous()
    tr = api.Trainer(6.0, 4.5, 5, 3, 4, (12,), ts.first, ts.boxes, pos, e_t, f_t, v_t, cap_radial=80, cap_angular=40,
                     types=types, atomic_numbers=znum)
    npop = 4
    z = teacher[None, :] + 0.02 * inputs.normal(77, npop * npar).reshape(npop, npar)
    z[0] = teacher
    lam = [1.0, 1.0, 1.0, 0.05, 0.05]
    L = tr.losses(torch.from_numpy(z).to(dev).contiguous(), lam).cpu().numpy()
    tr.status()
    for k in range(npop):
        ref = oracle.loss(h, list(znum), z[k], ts.first, ts.pos, ts.types, ts.boxes, e.astype(np.float32), f.astype(np.float32),
                          v.astype(np.float32), lam)
        print(k, L[k], ref)
        for c in (0, 1, 2):
            assert abs(L[k, c] - ref[c]) < 2e-4 * max(ref[c], 1e-3) + 5e-6, (k, c)
    assert np.argmin(L[:, 5]) == 0
