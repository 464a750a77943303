#!/usr/bin/env python
"""bench.py -- NEP MD atom-steps/s on B200 (BASELINE.json metric), one JSON line on stdout.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4_1048576] [--impl ours|reference]

A "step" is one velocity-Verlet MD step of the whole hot path over the workload: half-kick + drift,
device-side list rebuild when needed, list filter, descriptor + network + partial forces, assembly
of F / W / J, second half-kick, per-step thermo sums.  N > 1 runs N independent replicas
("replicas only"): no data-path collective exists.
`--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "NEP MD atom-steps/s"
UNIT = "atom-steps/s"
# FP32 non-tensor peak: 148 SMs x 128 FP32 lanes x 2 flop (FMA) x 1.965 GHz max SM clock
# (unit counts and clock from /opt/skills/guides/B200_PROFILING.md).
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def algorithmic_flops_per_atom(n_r, n_a, dim, n_neu, m_r, m_a):
    """SURVEY.md 8(d) / DESIGN.md section 7: necessary flops of descriptor + network + partial forces
    per atom-step with the O(M) addition-theorem route (FMA = 2).  k_main covers all but the
    25*M_R assembly term."""
    k_desc = m_r * (17 + 5 * n_r) + m_a * (67 + 52 * n_a) + 48 * n_a
    k_nn = 4 * dim * n_neu
    k_force = 48 * n_a + m_r * (20 + 10 * n_r) + m_a * (370 + 104 * n_a)
    return k_desc + k_nn + k_force


def make_workload(name):
    """c0..c3, c4_<atoms> (BASELINE.json configs) and t1_si / t1_silicene / t1_pbte: the paper's Table I model
    shapes on the 8000 / 6000-atom cells of its own speed test (random weights)."""
    from paper_2107_08119_b200 import inputs
    if name.startswith("c4_"):
        return inputs.config4(int(name[3:]))
    if name.startswith("t1_"):
        return inputs.table1(name[3:])
    return {"c0": inputs.config0, "c1": inputs.config1, "c2": inputs.config2, "c3": inputs.config3}[name]()


def caps_for(name, w):
    """(cap_radial, cap_angular) with head-room for the heated state."""
    if name.startswith("t1_"):
        return {"t1_si": (56, 56), "t1_silicene": (32, 32), "t1_pbte": (86, 24)}[name]
    return (64, 32) if len(w.atomic_numbers) == 1 else (80, 40)


def oracle_sample(w, budget_s, max_reps):
    """Times the oracle as it stands on the workload itself: full fp64 evaluations of U, F, W, J including the
    list build, repeated until `budget_s` seconds of CPU work (at least one)."""
    import oracle
    h = oracle.Hyper(w.rc_r, w.rc_a, w.n_max_r, w.n_max_a, w.l_max, w.n_neurons, len(w.atomic_numbers))
    t0 = time.perf_counter()
    reps = 0
    while reps < 1 or (time.perf_counter() - t0 < budget_s and reps < max_reps):
        oracle.evaluate(h, w.atomic_numbers, w.params, w.pos, w.vel, w.types, w.box, 96, 64)
        reps += 1
    dt = time.perf_counter() - t0
    sample = ("%s itself (%d atoms): %d full fp64 evaluations of U,F,W,J incl. list build (literal O(M^2) Eq. 13/25), %.1f s"
              % (w.name, w.n_atoms, reps, dt))
    return w.n_atoms * reps / dt, oracle.num_threads(), sample, reps, dt


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc = index, [], None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([c.strip() for c in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm, reasons, smax = [], set(), None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); smax = float(r[1])
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def run_reference(args):
    """The oracle as it stands, on the host cores, on a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.workload)
    steps = max(1, min(args.steps, 20))
    value, cores, sample, reps, dt = oracle_sample(w, min(60.0, 8.0 * steps), steps)     # each "step" = one evaluation, bounded
    steps = reps
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": 0, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_train(args):
    """--workload train[_<S>]: the training side.  A "step" is one SNES generation
    over a set of S small periodic structures combined into one system (default 24; the paper's sets hold hundreds to
    thousands): Eq. 35 sample of N_pop = 50 parameter vectors -> nep_trainer_losses (every member evaluates all atoms:
    stage weights, k_gen, k_assemble, per-structure reduction, Eq. 29-34) -> Eq. 36-39 update.  The metric here is
    structure-evaluations/s, NOT BASELINE.json's atom-steps/s: this line measures a "next" row, beside the default."""
    import math
    import torch
    from paper_2107_08119_b200 import api, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    S = int(args.workload.split("_")[1]) if "_" in args.workload else 24
    n_pop, K, Wm = 50, max(1, min(args.steps, 50)), max(min(args.warmup, 10), 3)
    dev = "cuda:0"
    ts = inputs.training_set(S, seed=50)
    pos = torch.from_numpy(ts.pos).to(dev)
    shape = (5.0, 4.0, 7, 7, 4, (30,))
    probe = api.Trainer(*shape, ts.first, ts.boxes, pos)
    npar = probe.num_params
    teacher = torch.from_numpy((2 * inputs.uniform01(51, npar) - 1) / math.sqrt(30.0)).to(dev)
    e_t, f_t, v_t = probe.predict(teacher)                     # synthetic targets: a teacher network (no dataset here)
    tr = api.Trainer(*shape, ts.first, ts.boxes, pos, e_t, f_t, v_t)
    m = torch.from_numpy(0.3 * (2 * inputs.uniform01(52, npar) - 1) / math.sqrt(30.0)).to(dev)
    sd = torch.full((npar,), 0.02, dtype=torch.float64, device=dev)
    r = torch.from_numpy(inputs.normal(53, n_pop * npar).reshape(n_pop, npar)).to(dev)   # the normals are inputs (Eq. 35)
    lam = [1.0, 1.0, 0.1, 0.05, 0.05]
    eta_s = (3 + math.log(npar)) / (5 * math.sqrt(npar))

    def generation():
        z = api.snes_sample(m, sd, r)
        L = tr.losses(z, lam)
        api.snes_update(m, sd, r, L, 1.0, eta_s)
        return L

    for _ in range(Wm):
        generation()
    tr.status()
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(K):
        L = generation()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    tr.status()
    # end to end: the generation's normals come from pinned host memory and its losses go back to the host
    h_r = r.cpu().pin_memory(); h_L = torch.empty((n_pop, 6), dtype=torch.float64).pin_memory()
    ke = min(K, 10)
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for _ in range(ke):
        r.copy_(h_r, non_blocking=True)
        h_L.copy_(generation(), non_blocking=True)
        torch.cuda.current_stream().synchronize()
    t1.record()
    torch.cuda.synchronize()
    e2e_ms = t0.elapsed_time(t1)
    # the oracle's loss for a few members, timed on the host cores
    import oracle
    h = oracle.Hyper(5.0, 4.0, 7, 7, 4, 30, 1)
    z_host = api.snes_sample(m, sd, r).cpu().numpy()
    tgt = [t.cpu().numpy() for t in (e_t, f_t, v_t)]
    c0 = time.perf_counter(); reps = 0
    while reps < 1 or (time.perf_counter() - c0 < 10.0 and reps < n_pop):
        oracle.loss(h, [14], z_host[reps], ts.first, ts.pos, ts.types, ts.boxes, tgt[0], tgt[1], tgt[2], lam)
        reps += 1
    cdt = time.perf_counter() - c0
    flops_atom = algorithmic_flops_per_atom(8, 8, 40, 30, 28.0, 14.0) + 25 * 28.0
    line = {
        "metric": "NEP training structure-evaluations/s", "value": n_pop * S * K / (ms * 1e-3), "unit": "structure-evaluations/s",
        "n_gpus": 1, "steps": K, "warmup": Wm, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "%s: one SNES generation, N_pop = %d members x %d Si structures (%d atoms, 63-64 per structure), "
                               "D=40 NN 40-30-1, targets from a teacher network" % (args.workload, n_pop, S, ts.n_atoms),
                   "n_structures": S, "n_atoms": ts.n_atoms, "n_pop": n_pop, "n_par": npar,
                   "l2": "working set far below L2 by nature of the workload (small structures): L2-resident, stated, not flushed",
                   "best_loss_last_generation": float(L[:, 5].min())},
        "clocks": clocks,
        "e2e": {"value": n_pop * S * ke / (e2e_ms * 1e-3), "unit": "structure-evaluations/s",
                "h2d_bytes_per_step": n_pop * npar * 8, "d2h_bytes_per_step": n_pop * 6 * 8, "steps": ke,
                "what": "per generation: pinned-host normals -> device, sample + losses + update, losses -> pinned host"},
        "gpu_launches": K * (n_pop * 6 + 2),
        "launches_per_generation": n_pop * 6 + 2,
        "roofline": {"bound": "alu", "kernel": "k_gen inside the member loop (whole generation time as the denominator)",
                     "achieved": flops_atom * ts.n_atoms * n_pop / (ms / K * 1e-3) / 1e12, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                     "frac": flops_atom * ts.n_atoms * n_pop / (ms / K * 1e-3) / 1e12 / FP32_PEAK_TFLOPS, "traffic": None,
                     "what": "useful FP32 flops of all members' evaluations / generation time: launch- and latency-bound "
                             "(members run one after another, each a fraction of one wave)"},
        "cpu_baseline": {"value": S * reps / cdt, "unit": "structure-evaluations/s", "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": "orc_loss for %d of the %d members over the same %d structures, %.1f s" % (reps, n_pop, S, cdt)},
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4_1048576")
    ap.add_argument("--skin", type=float, default=None, help="Verlet skin in A (default 1.0; 0.4 for c0, whose box must exceed 2 (r_c^R + skin))")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.workload.startswith("train"):
        if args.impl == "reference":
            raise SystemExit("--impl reference times the MD workloads; the train line carries its own cpu_baseline")
        return run_train(args)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2107_08119_b200 import api

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K, Wm = args.steps, max(args.warmup, 3)
    w = make_workload(args.workload)
    N = w.n_atoms
    cap_r, cap_a = caps_for(args.workload, w)
    if args.skin is None:
        args.skin = 0.4 if args.workload == "c0" else 1.0
    model, system, pos, vel = api.from_workload(w, cap_r, cap_a, args.skin, dev)
    out = system.alloc_outputs()
    heat_sum = torch.zeros((3, N), dtype=torch.float64, device=dev)
    thermo = torch.zeros((max(K, Wm), 5), dtype=torch.float64, device=dev)
    system.neighbors(pos, w.box)
    cnt_r, _ = system.get_neighbors(0)
    cnt_a, _ = system.get_neighbors(1)
    m_r0, m_a0 = cnt_r.float().mean().item(), cnt_a.float().mean().item()

    # ---- warm-up, then the timed region: K steps, device-timed on the launching stream ----
    system.md_step(pos, vel, w.masses, w.dt, Wm, out, heat_sum, thermo)
    system.status()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    l0 = system.launch_count()
    e0.record()
    system.md_step(pos, vel, w.masses, w.dt, K, out, heat_sum, thermo)
    e1.record()
    barrier()
    launches = system.launch_count() - l0
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    system.status()
    st = system.stats()
    th = thermo[:K].cpu().numpy()
    e_tot = th[:, 0] + th[:, 1]
    if world > 1:
        t = torch.tensor([ms], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = t.item()
    value = world * N * K / (ms * 1e-3)

    # ---- per-kernel device timing (same launch sequence, CUDA events inside the library) ----
    kp = min(K, 100)
    system.profile(True)
    system.md_step(pos, vel, w.masses, w.dt, kp, out, heat_sum, thermo)
    prof = system.get_profile()
    system.profile(False)
    cnt_r, _ = system.get_neighbors(0)
    cnt_a, _ = system.get_neighbors(1)
    m_r, m_a = cnt_r.float().mean().item(), cnt_a.float().mean().item()
    main_ms = prof["main"]["ms"] / max(1, prof["main"]["count"])
    flops_atom = algorithmic_flops_per_atom(w.n_max_r + 1, w.n_max_a + 1, w.dim, w.n_neurons, 0.5 * (m_r0 + m_r), 0.5 * (m_a0 + m_a))
    achieved = flops_atom * N / (main_ms * 1e-3) / 1e12
    phase_ms = {k: v["ms"] / kp for k, v in prof.items()}
    tot_phase = sum(phase_ms.values())

    # ---- end to end through the C ABI with HOST buffers: per step H2D(pos, vel) + one MD step + D2H of everything ----
    # The trajectory runs THROUGH the host: step n+1's positions and velocities are the ones step n brought back, so
    # H2D -> step -> D2H(pos, vel) is a true dependency chain.  Only the 67 MB of U, F, W, J are off that chain: they go
    # back on a second stream from one of two output sets while the next step's H2D and compute run, and the host
    # reads them one step late.  Every byte of every step is copied inside the timed region.
    ke = min(K, 50)
    h_pos = pos.cpu().pin_memory(); h_vel = vel.cpu().pin_memory()
    outs = [out, system.alloc_outputs()]
    h_outs = [[torch.empty_like(t, device="cpu").pin_memory() for t in out] for _ in range(2)]
    s_main = torch.cuda.current_stream()
    s_out = torch.cuda.Stream()
    ev_state = [torch.cuda.Event() for _ in range(2)]          # pos, vel of step n are on their way to the host
    ev_out = [torch.cuda.Event() for _ in range(2)]            # output set n % 2 has reached the host
    system.md_step(pos, vel, w.masses, w.dt, 1, out)          # warm the 1-step path
    barrier()
    t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
    t0.record()
    for n in range(ke):
        b = n & 1
        pos.copy_(h_pos, non_blocking=True); vel.copy_(h_vel, non_blocking=True)
        if n >= 2:
            s_main.wait_event(ev_out[b])                       # the step overwrites output set b: its last copy must be done
        system.md_step(pos, vel, w.masses, w.dt, 1, outs[b])
        h_pos.copy_(pos, non_blocking=True); h_vel.copy_(vel, non_blocking=True)
        ev_state[b].record(s_main)
        s_out.wait_event(ev_state[b])                          # after pos, vel: the two D2H transfers do not share the link
        with torch.cuda.stream(s_out):
            for hd, dd in zip(h_outs[b], outs[b]):
                hd.copy_(dd, non_blocking=True)
            ev_out[b].record(s_out)
        s_main.synchronize()                                   # the host has step n's positions and velocities ...
        if n >= 1:
            ev_out[1 - b].synchronize()                        # ... and reads step n-1's U, F, W, J
    s_out.synchronize()
    t1.record()
    barrier()
    e2e_ms = t0.elapsed_time(t1)
    if world > 1:
        t = torch.tensor([e2e_ms], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_ms = t.item()
    h2d = 2 * 3 * N * 8
    d2h = 2 * 3 * N * 8 + sum(t.numel() * 4 for t in out)
    system.status()

    peak_ffma, peak_ffma2 = api.measure_fp32_peak()
    pat_3reg, pat_desc, pat_force = api.measure_fp32_patterns()
    # HBM-bound phases: algorithmic DRAM bytes per atom-step / phase time vs the measured copy peak
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        hbm_src = "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        hbm_peak, hbm_src = 6650.0, "fallback of /opt/skills/guides/B200_PROFILING.md"
    mr, ma = 0.5 * (m_r0 + m_r), 0.5 * (m_a0 + m_a)
    m_md = mr * ((w.rc_r + args.skin) / w.rc_r) ** 3
    bytes_filter = 4 * m_md + 32 + 16 * mr + 32 + 8           # Verlet row, own position, records (with j | rev), masks, counts
    bytes_asm = 16 * mr + 16 * mr + 32 + 16 + 4 + 24 + 64 + 12 + 48   # records, p_ji, masks, Fself, U, v rw, outputs, Fs, kick
    hbm_phases = {}
    for name, nbytes in (("filter", bytes_filter), ("assemble", bytes_asm)):
        gbs = nbytes * N / (prof[name]["ms"] / max(1, prof[name]["count"]) * 1e-3) / 1e9
        hbm_phases[name] = {"bound": "hbm", "bytes_per_atom": nbytes, "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                            "frac": gbs / hbm_peak}
    # Counters of the dominant kernel from the committed ncu --set full capture of this same command
    # (profiles/r3_k_main_counters.json; 1M-atom workload, one thread per atom): DRAM bytes per launch and the
    # EXECUTED FP32 flops per launch (FFMA = 2, FFMA2 = 4, FMUL/FADD = 1, summed over the SASS of one launch).
    traffic = executed = None
    counters_src = None
    try:
        if args.workload == "c4_1048576" and system.path == 1:
            cj = json.load(open(os.path.join(ROOT, "profiles", "r3_k_main_counters.json")))
            traffic = cj["k_main_dram_bytes_per_launch"]
            executed = cj["k_main_executed_fp32_flops_per_launch"]
            counters_src = cj["capture"]
    except Exception:
        traffic = executed = None

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, cores, sample, reps, tt = oracle_sample(w, 12.0, 3)      # the config itself, up to 3 evaluations / ~12-20 s
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": "%s: %d-atom diamond Si (C4), D=%d NN %d-%d-1, rc %.1f/%.1f A, NVE dt=%g fs, W and J every step"
                                   % (args.workload, N, w.dim, w.dim, w.n_neurons, w.rc_r, w.rc_a, w.dt)
                       if args.workload.startswith("c4") else args.workload,
                       "n_atoms": N, "parallelism": "replicas x%d" % world, "skin": args.skin,
                       "l2": "working set %.1f GB per replica >> 126 MB L2, no flush needed" % (system.workspace.numel() / 1e9),
                       "mean_M_R": [m_r0, m_r], "mean_M_A": [m_a0, m_a], "rebuilds_total": st["rebuilds"],
                       "max_M_R": st["max_radial"], "max_M_A": st["max_angular"],
                       "energy_drift_eV_per_atom": float(np.abs(e_tot - e_tot[0]).max() / N)},
            "clocks": clocks,
            "e2e": {"value": world * N * ke / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "steps": ke,
                    "what": "per step: pinned-host pos+vel -> device, nep_md_step(1), pos+vel -> pinned host (the next step's input: a true "
                            "dependency through the host), U+F+W+J -> pinned host on a second stream from double-buffered output "
                            "sets, overlapping the next step; the host reads them one step late"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "kernel": ("k_main, one thread per atom" if system.path == 1 else "k_gen, 16 lanes per atom") +
                                                  " (descriptor + network + partial forces)",
                         "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP32_PEAK_TFLOPS,
                         "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (no FP32 figure in MEASURED_PEAKS.json)",
                         "peak_measured_fma_chain": {"ffma": peak_ffma, "ffma2": peak_ffma2, "unit": "TFLOP/s"},
                         "pattern_ceilings": {"ffma_three_distinct_registers": pat_3reg, "descriptor_contraction_ffma2": pat_desc,
                                              "force_contraction_ffma2": pat_force, "unit": "TFLOP/s",
                                              "what": "register-resident inner-loop patterns of k_main at its residency (8 warps/SM)"},
                         "frac_of_measured_ffma": achieved / peak_ffma,
                         "flops_per_atom": flops_atom, "kernel_ms": main_ms, "kernel_share_of_step": phase_ms["main"] / tot_phase,
                         "traffic": traffic,
                         "executed_frac": (executed / (main_ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS) if executed else None,
                         "counters_source": counters_src},
            "phase_ms_per_step": phase_ms,
            "roofline_hbm_phases": dict(hbm_phases, peak_source=hbm_src),
            "cpu_baseline": cpu,
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
