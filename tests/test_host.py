"""CPU-side checks of the product: the C-ABI library loads and exports every symbol include/nep_b200.h
declares, argument validation that needs no GPU, the host self-test of the device math, and the
replica logic of bench.py under a world_size-2 gloo group."""
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    from paper_2107_08119_b200 import api, build
    build.build()
    L = api.lib()
    import glob
    header = "".join(open(h).read() for h in sorted(glob.glob(os.path.join(ROOT, "include", "*.h"))))
    declared = set(re.findall(r"\b(nep_[a-z0-9_]+)\s*\(", header))
    declared -= {"nep_error"}
    assert declared == set(api.SYMBOLS), declared ^ set(api.SYMBOLS)
    for sym in declared:
        getattr(L, sym)
    assert b"minimum image" in L.nep_strerror(-2)


def test_argument_validation_without_gpu():
    import ctypes as C
    import numpy as np
    from paper_2107_08119_b200 import api
    L = api.lib()
    h = api.Hyper(5.0, 4.0, 7, 7, 4, 30, 1)
    par = np.zeros(1261)
    out = C.c_void_p()
    # wrong parameter count, unsupported l_max, r_c^A > r_c^R: rejected before any CUDA call
    assert L.nep_create(C.byref(h), None, par.ctypes.data_as(C.c_void_p), 1260, C.byref(out)) == -1
    h3 = api.Hyper(5.0, 4.0, 7, 7, 9, 30, 1)          # l_max 1..8 (5..8: the general-l kernel)
    assert L.nep_create(C.byref(h3), None, par.ctypes.data_as(C.c_void_p), 1261, C.byref(out)) == -1
    h16 = api.Hyper(5.0, 4.0, 16, 7, 4, 30, 1)
    assert L.nep_create(C.byref(h16), None, par.ctypes.data_as(C.c_void_p), 1261, C.byref(out)) == -1
    hb = api.Hyper(4.0, 5.0, 7, 7, 4, 30, 1)
    assert L.nep_create(C.byref(hb), None, par.ctypes.data_as(C.c_void_p), 1261, C.byref(out)) == -1
    assert L.nep_workspace_bytes(None, 100, 64, 32, 1.0) == 0
    import torch
    if not torch.cuda.is_available():       # no CPU fallback: a valid model still needs a device
        assert L.nep_create(C.byref(h), None, par.ctypes.data_as(C.c_void_p), 1261, C.byref(out)) == -4


def test_device_math_selftest_on_host(tmp_path):
    exe = str(tmp_path / "selftest_host")
    src = os.path.join(ROOT, "paper_2107_08119_b200", "csrc", "selftest_host.cpp")
    subprocess.run(["g++", "-O1", "-o", exe, src], check=True)
    r = subprocess.run([exe], capture_output=True, text=True)
    assert r.returncode == 0 and "OK" in r.stdout, r.stdout[-2000:]


def test_flop_model_matches_survey():
    sys.path.insert(0, ROOT)
    import bench
    # M_R = 28, M_A = 16, n = 8, D = 40, H = 30 -> 9.7k + 4.8k + 23.1k ~ 38 kflop
    f = bench.algorithmic_flops_per_atom(8, 8, 40, 30, 28, 16)
    assert 36500 < f + 25 * 28 < 38500      # + the 25 M_R assembly term that k_assemble owns
    assert abs(bench.FP32_PEAK_TFLOPS - 74.45) < 0.01


def test_reference_arm_rank0_only_under_gloo():
    """world_size 2 on CPU: rank 0 prints the reference line, rank 1 exits 0 silently."""
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29517", OMP_NUM_THREADS="2")
    code = (
        "import os, sys, torch.distributed as dist\n"
        "dist.init_process_group('gloo', rank=int(os.environ['RANK']), world_size=2)\n"
        "sys.argv = ['bench.py', '--impl', 'reference', '--gpus', '2', '--steps', '1', '--warmup', '0', '--workload', 'c0']\n"
        "sys.path.insert(0, %r)\n"
        "import bench\n"
        "bench.main()\n"
        "dist.barrier(); dist.destroy_process_group()\n" % ROOT)
    procs = [subprocess.Popen([sys.executable, "-c", code], env=dict(env, RANK=str(r), WORLD_SIZE="2"),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    import json
    line = json.loads(outs[0][0].strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert outs[1][0].strip() == ""
