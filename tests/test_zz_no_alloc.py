"""nep_loss_noalloc, the one entry point for callers that cannot allocate device memory, against the path everybody
else uses (nep_trainer_predict -> nep_trainer_losses).

Who cannot allocate: a callback that another program calls with this step's device arrays and nothing else; a process
whose device memory is owned by a single pool, so that a raw cudaMalloc fails or shrinks the pool behind its back; a
loop that cannot afford cudaMalloc's device-wide synchronisation, or runs while some stream is being captured, when
cudaMalloc is refused.  For them the entry point keeps its partial sums in a fixed 0.5 MiB __device__ array inside
libnep_b200.so (include/nep_b200.h states the limits that follow from that).

The file is named test_zz_* so that pytest collects it after every other test: `pytest -x` stops at the first failure,
and a failure here must not hide the parity tests.  It does not depend on anything those tests leave behind: the first
nep_loss_noalloc call of the process does the per-device set-up, whether that is here or not."""
import ctypes as C
import math

import numpy as np
import pytest

from paper_2107_08119_b200 import inputs

LIMIT = 16_777_216      # 3 n_atoms + 7 n_structures + n_par, from include/nep_b200.h


def test_sizes_beyond_the_fixed_scratch_are_refused_with_a_reason():
    """No GPU needed: the size test comes before the first CUDA call, and nothing is dereferenced when it fails."""
    from paper_2107_08119_b200 import api
    L = api.lib()
    msg = C.create_string_buffer(512)
    dummy = C.c_void_p(256)                                  # non-null, never read
    lam = (C.c_double * 5)(1, 1, 1, 0, 0)
    args = [dummy] * 7 + [C.cast(lam, C.c_void_p), dummy, None, msg, len(msg)]
    n_atoms = LIMIT // 3 + 1
    assert L.nep_loss_noalloc(1, n_atoms, 1, *args) == -3    # NEP_ENOMEM
    text = msg.value.decode()
    assert "exceeds the fixed scratch" in text and str(LIMIT) in text and "nep_trainer_losses" in text
    assert L.nep_loss_noalloc(2 ** 40, 1, 1, *args) == -3    # no overflow games with huge counts either
    assert L.nep_loss_noalloc(0, 10, 10, *args) == -1 and msg.value       # NEP_EINVAL, with a message
    assert L.nep_loss_noalloc(1, 10, 10, None, *args[1:]) == -1


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_trainer_path():
    """Two different members back to back on one stream (the second call finds the first call's rows and ticket in the
    shared array), then the first member again: each loss against nep_trainer_losses at the bars of
    test_gpu_training.py, and the repeat bit-identical to the first call (fixed summation order, no stale state)."""
    import torch
    from paper_2107_08119_b200 import api
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    dev = "cuda"
    ts = inputs.training_set(12, seed=70)
    pos = torch.from_numpy(ts.pos).to(dev)
    probe = api.Trainer(5.0, 4.0, 7, 7, 4, (30,), ts.first, ts.boxes, pos)
    npar = probe.num_params
    teacher = (2 * inputs.uniform01(71, npar) - 1) / math.sqrt(30.0)
    e_t, f_t, v_t = probe.predict(torch.from_numpy(teacher).to(dev))       # targets: the library's own teacher
    tr = api.Trainer(5.0, 4.0, 7, 7, 4, (30,), ts.first, ts.boxes, pos, e_t, f_t, v_t)
    npop = 4
    z = teacher[None, :] + 0.05 * inputs.normal(72, npop * npar).reshape(npop, npar)
    z[0] = teacher
    zd = torch.from_numpy(z).to(dev).contiguous()
    lam = [1.0, 0.7, 0.3, 0.05, 0.05]
    ref = tr.losses(zd, lam).cpu().numpy()                                  # the existing path, all members
    preds = [tr.predict(zd[k]) for k in range(npop)]
    tr.status()
    outs = [torch.full((6,), float("nan"), dtype=torch.float64, device=dev) for _ in range(npop + 1)]
    order = [1, 2, 1, 0, 3]                                                 # 1 then 2 in a row, 1 again, the rest
    for slot, k in enumerate(order):                                        # no synchronisation between the calls
        api.loss_noalloc(*preds[k], e_t, f_t, v_t, zd[k], lam, outs[slot])
    torch.cuda.synchronize()
    got = [o.cpu().numpy() for o in outs]
    assert ref[1, 5] > ref[0, 5] and abs(ref[1, 5] - ref[2, 5]) > 1e-6         # the members really differ
    for slot, k in enumerate(order):
        g = got[slot]
        print(k, g, ref[k])
        assert np.all(np.isfinite(g))
        assert g[3] == pytest.approx(ref[k, 3], rel=1e-12) and g[4] == pytest.approx(ref[k, 4], rel=1e-12)
        for c in (0, 1, 2):
            # predict hands e, f, v over in fp32; nep_trainer_losses keeps its per-structure means in fp64
            assert abs(g[c] - ref[k, c]) < 1e-4 * max(ref[k, c], 1e-3) + 2e-6, (k, c)
        assert g[5] == pytest.approx(ref[k, 5], rel=2e-4, abs=1e-5)
    assert np.array_equal(got[0], got[2])                                    # member 1, first and third call
    # a size that spans many blocks and a ragged tail, checked against the plain definition on the host
    S, N, P = 1000, 70_001, 4099
    rng = [inputs.normal(200 + i, n).astype(np.float32) for i, n in enumerate((S, 3 * N, 6 * S, S, 3 * N, 6 * S))]
    zz = inputs.normal(210, P)
    t = [torch.from_numpy(a).to(dev) for a in rng]
    big = torch.zeros(6, dtype=torch.float64, device=dev)
    api.loss_noalloc(t[0], t[1].view(3, N), t[2].view(S, 6), t[3], t[4].view(3, N), t[5].view(S, 6), torch.from_numpy(zz).to(dev),
                     lam, big)
    r64 = [a.astype(np.float64) for a in rng]
    exp = [math.sqrt(((r64[0] - r64[3]) ** 2).mean()), math.sqrt(((r64[1] - r64[4]) ** 2).mean()),
           math.sqrt(((r64[2] - r64[5]) ** 2).mean()), np.abs(zz).mean(), math.sqrt((zz ** 2).mean())]
    exp.append(sum(l * x for l, x in zip(lam, exp)))
    assert np.allclose(big.cpu().numpy(), exp, rtol=1e-12, atol=0)
