#!/usr/bin/env python
"""bench.py — mover throughput on BASELINE.json's metric workload (configs[2]: 4,096 cells,
1e8 electrons, 16-mode field, dt = 10, fp32 mover), one JSON line on stdout.

A "step" is one pass of the whole hot path = one pic_move_accumulate call
over every particle.  `value` = particle sub-steps/s with everything resident in HBM (E and jbar
are device arrays); `e2e` = the same through the C-ABI with HOST grid buffers (E^n, E^{n+1} copied
host->device and jbar device->host inside the timed region; the particles are enslaved state that
never leaves the GPU).  `roofline` is the plain-ALU FP32 roofline with the
algorithmic op table of DESIGN.md 6; `cpu_baseline` is the oracle, as it stands, on a bounded
sample.  `--impl reference` times the oracle alone (the reference arm of this tier).

N > 1 (torchrun): independent replicas with different seeds, no data-path collective
("replicas only"); value = total sub-steps of all ranks / max-over-ranks time.
"""
import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1111_5295_b200 import workloads as W  # noqa: E402

METRIC = "mover_particle_substeps_per_s"
UNIT = "sub-steps/s"
# Algorithmic op table (paper's convention: every FP / int / SF thread-operation = 1, FMA = 2;
# P:94-105), SURVEY 8(d) / DESIGN.md 6: per in-cell sub-step and per crossing sub-step.
OPS_INCELL, OPS_CROSS = 43.0, 72.0
# dram__bytes_read.sum + dram__bytes_write.sum of one mover launch from the committed
# `ncu --set full` capture (profiles/r2_mover_ncu.md; re-captured in round 3 with the same
# result, profiles/r3_op_table.md); known only for the default workload.
NCU_TRAFFIC_BYTES = {("cfg2", 100_000_000, "fp32"): 2.365e9, ("cfg2", 100_000_000, "fp64"): 3.970e9}
NCU_TRAFFIC_SOURCE = "profiles/r2_mover_ncu.md (ncu --set full capture of this kernel; not measured in this run)"
# Executed thread-operations per sub-step of the timed kernel, summed over the SASS lines of the
# same ncu capture (source page, predicated-on thread instructions): (a) the paper's convention
# (every instruction 1, FFMA 2, packed FFMA2 4, FMUL2 / FADD2 2), (b) floating-point arithmetic
# only (FADD, FMUL, FFMA, their packed forms; no integer, compare, select, MUFU, memory, control),
# (c) the paper's operation classes only: FP + AL (integer, logic, compare, select,
# min/max, conversions) + SF (MUFU), without control (BRA, BSSY, BSYNC, votes) and data movement
# (MOV, SHFL, LDS/STS, LDG/STG, ATOMS); per-opcode table in profiles/r3_op_table.md (None: not
# split for that kernel).
NCU_EXECUTED_OPS = {("cfg2", 100_000_000, "fp32", "mover2_kernel"): (46.12, 27.45, 38.71),
                    ("cfg2", 100_000_000, "fp64", "mover_kernel"): (81.22, 46.17, None)}


def _workload(name, n, seed):
    if name == "cfg2":
        return W.config2(n=n or 100_000_000, seed=seed)
    if name == "cfg3":
        return W.config3(n=n or 20_000_000, seed=seed)
    if name == "cfg0":
        return W.config0(n=n or 6400, seed=seed)
    if name == "cfg1":
        return W.config1(ppc=(n // 512) if n else 2000, seed=seed)
    if name == "cfg4":
        return W.config4(ppc=(n // 1024) if n else 4000, seed=seed)
    raise SystemExit(f"unknown workload {name}")


class ClockSampler(threading.Thread):
    """SM clock / throttle-reason samples during the timed region (pynvml, 20 ms period)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.samples, self.reasons, self.max_mhz, self.ok = [], set(), None, False
        self._stop_ev = threading.Event()
        try:
            import pynvml as N
            N.nvmlInit()
            self.N = N
            self.h = N.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = N.nvmlDeviceGetMaxClockInfo(self.h, N.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        N = self.N
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                 "sw_thermal_slowdown": 0x20, "hw_power_brake": 0x80}
        while not self._stop_ev.is_set():
            try:
                self.samples.append(N.nvmlDeviceGetClockInfo(self.h, N.NVML_CLOCK_SM))
                try:
                    r = N.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:  # noqa: BLE001
                    r = N.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:  # noqa: BLE001
                pass
            time.sleep(0.02)

    def stop(self):
        self._stop_ev.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def oracle_rate(cfg, sample, threads=1):
    """Time the oracle, as it stands (serial, fp64, Picard), on the first `sample` particles."""
    from oracle import pic_oracle as o
    o.build()
    sp = cfg["species"][0]
    n = min(sample, sp["x"].shape[0])
    c, s = o.bin_particles(cfg["n_cells"], cfg["length"], sp["x"][:n])
    t0 = time.perf_counter()
    r = o.move_accumulate(cfg["n_cells"], cfg["length"], sp["q_over_m"], sp["w_q"], c, s,
                          sp["v"][:n], cfg["E_n"], cfg["E_np1"], cfg["dt"],
                          o.make_params(tol=cfg.get("tol", 1e-10)), want_state=False)
    dt = time.perf_counter() - t0
    return r["stats"].n_sub / dt, r["stats"].n_sub, dt, n


def oracle_rate_parallel(cfg, per_core=1 << 20):
    """The same serial oracle, unchanged, on all host cores: one call per core on disjoint chunks
    of the particle list (orbits are independent given E; each call has its own J), started from
    a thread pool (ctypes releases the GIL during the call).  Labelled separately from the
    one-core baseline."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import pic_oracle as o
    o.build()
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    sp = cfg["species"][0]
    n = min(cores * per_core, sp["x"].shape[0])
    bounds = np.linspace(0, n, cores + 1).astype(np.int64)
    chunks = []
    for a, b in zip(bounds[:-1], bounds[1:]):
        c, s = o.bin_particles(cfg["n_cells"], cfg["length"], sp["x"][a:b])
        chunks.append((c, s, np.ascontiguousarray(sp["v"][a:b])))
    par = o.make_params(tol=cfg.get("tol", 1e-10))

    def one(ch):
        r = o.move_accumulate(cfg["n_cells"], cfg["length"], sp["q_over_m"], sp["w_q"], ch[0], ch[1],
                              ch[2], cfg["E_n"], cfg["E_np1"], cfg["dt"], par, want_state=False)
        return r["stats"].n_sub

    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=cores) as ex:
        subs = list(ex.map(one, chunks))
    dt = time.perf_counter() - t0
    return sum(subs) / dt, int(sum(subs)), dt, int(n), cores


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, bounded sample per step."""
    if rank != 0:
        return
    if args.workload in ("cfg1", "cfg4"):
        return run_reference_iaw(args, world)
    sample = args.ref_sample
    cfg = _workload(args.workload, sample, args.seed)
    for _ in range(args.warmup):
        oracle_rate(cfg, min(sample, 1 << 14))
    tot_sub, tot_t = 0, 0.0
    for _ in range(args.steps):
        _, nsub, dt, n = oracle_rate(cfg, sample)
        tot_sub += nsub
        tot_t += dt
    val = tot_sub / tot_t
    sample_desc = f"first {n} particles of {args.workload} per step, serial fp64 oracle (Picard)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": args.workload, "sample_particles": n},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle",
                             "sample": sample_desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_reference_iaw(args, world):
    """--impl reference on configs[1] / [4]: the implicit step driven by the oracle (the
    harness-side Newton-Krylov of tests/oracle_jfnk.py around oracle.move_accumulate), all host
    cores, on a bounded sample: the same grid and dt with 1/20 of the particles per cell."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from oracle import pic_oracle as o
    from oracle_jfnk import OracleIAW
    o.build()
    full = 2000 if args.workload == "cfg1" else 4000
    ppc = max(full // 20, 10)
    cfg = (W.config1 if args.workload == "cfg1" else W.config4)(ppc=ppc, seed=args.seed)
    S = OracleIAW(o, cfg, o.make_params(cn_mode=o.DIRECT))
    E = S.gauss_field()
    for _ in range(args.warmup):
        E, _ = S.step(E, rtol=1e-8)
    tot_sub, t0 = 0, time.perf_counter()
    for _ in range(args.steps):
        c0 = S.mover_calls
        E, info = S.step(E, rtol=1e-8)
        tot_sub += S.last_n_sub * (S.mover_calls - c0)
    tot_t = time.perf_counter() - t0
    val = tot_sub / tot_t
    desc = (f"{args.workload} grid and dt with {ppc} of {full} particles per cell per species, "
            f"implicit steps (rtol 1e-8) driven by the fp64 oracle on {S.cores} host cores")
    S.close()
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": world,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                      "data": "synthetic", "config": {"workload": args.workload, "sample": desc},
                      "cpu_baseline": {"value": val, "unit": UNIT, "cores": S.cores, "kind": "oracle", "sample": desc},
                      "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                      "gpu_launches": 0}), flush=True)


def run_iaw(args, rank, world, local_rank, explicit_steps):
    """configs[1] / configs[4]: a "step" is one fully implicit time step (pic_jfnk_step: host fp64
    Newton-GMRES, one GPU mover pass per residual, commit + re-binning on convergence; P:111,
    P:321).  value = particle sub-steps of all mover passes of the timed steps / their time; the
    host E in / residual out copies of every pass are inside it (that IS the method's boundary,
    P:31), so e2e = value."""
    import torch
    import torch.distributed as dist
    from paper_1111_5295_b200 import binding as B
    from paper_1111_5295_b200 import replicas
    from paper_1111_5295_b200.iaw import gauss_field
    cfg = _workload(args.workload, args.n, replicas.rank_seed(args.seed, rank))
    ng, L, dt = cfg["n_cells"], cfg["length"], cfg["dt"]
    dx = L / ng
    rtol = args.rtol or (1e-8 if args.precision == "fp64" else 2e-4)     # SURVEY A-14
    stream = torch.cuda.current_stream().cuda_stream
    flags = 0 if args.no_vsort else B.PIC_FLAG_VSORT
    pic = B.Pic(ng, L, cfg["species"], precision=args.precision, cn_mode=args.cn_mode, flags=flags,
                stream=stream)
    jac = None
    if args.defect_correction:
        jac = B.Pic(ng, L, cfg["species"], precision="fp32", cn_mode=args.cn_mode, flags=flags, stream=stream)
    n_p = sum(pic.n)
    E = gauss_field(pic.rho(B.PIC_STATE_N), dx)

    def energy():
        return float(pic.kinetic_energy(B.PIC_STATE_N).sum() + 0.5 * dx * np.sum(E * E))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        info = pic.jfnk_step(E, dt, rtol=rtol, jacobian=jac)
        assert info["converged"], info
    # exact sub-steps / crossings of ONE mover pass from the state the timed steps start at
    # (counting build; the timed passes run the fast build, which counts in groups of 4 rounds)
    pic.set_flags(flags | B.PIC_FLAG_DIAG)
    pic.move_accumulate(E, E, dt)
    exact = pic.get_stats()
    pic.set_flags(flags)
    if not explicit_steps and args.min_seconds > 0:
        t0 = time.perf_counter()
        pic.jfnk_step(E, dt, rtol=rtol, jacobian=jac)
        args.steps = max(args.steps, min(2000, int(math.ceil(args.min_seconds / max(time.perf_counter() - t0, 1e-4)))))
    e_start = energy()
    sampler = ClockSampler(local_rank)
    hist, kms, launches0 = [], [], pic.get_stats()["n_launches"]
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        info = pic.jfnk_step(E, dt, rtol=rtol, jacobian=jac)
        hist.append(info)
    e1.record()
    barrier()
    wall = time.perf_counter() - t0
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    st = pic.get_stats()
    launches = st["n_launches"] - launches0
    assert all(h["converged"] for h in hist), hist
    e_end = energy()
    rho = pic.rho(B.PIC_STATE_N)
    gauss = float(np.linalg.norm((np.roll(E, -1) - E) / dx - rho) / max(np.linalg.norm(rho), 1e-300))
    gauss_abs = float(np.max(np.abs((np.roll(E, -1) - E) / dx - rho)))
    for _ in range(3):                                   # the mover pass alone (library events)
        pic.move_accumulate(E, E, dt)
        kms.append(pic.get_stats()["last_move_ms"])
    k_ms = float(np.mean(kms))
    calls = float(np.sum([h["mover_calls"] for h in hist]))
    calls_resid = float(np.sum([h["mover_calls_resid"] for h in hist]))
    n_sub, n_cross = exact["n_sub"], exact["n_cross"]
    ms, wall, tot_sub, tot_cross = replicas.aggregate(ms, wall, n_sub * calls, n_cross * calls, device="cuda")
    if rank != 0:
        pic.close()
        return
    props = torch.cuda.get_device_properties(local_rank)
    sms = props.multi_processor_count
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:  # noqa: BLE001
        peaks = {}
    sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    lanes = 128 if args.precision == "fp32" else 64
    peak_gops = sms * lanes * 2 * sm_max_mhz * 1e-3
    ops_per_pass = OPS_INCELL * (n_sub - n_cross) + OPS_CROSS * n_cross
    achieved = ops_per_pass / (k_ms * 1e-3) * 1e-9
    value = tot_sub / (ms * 1e-3)
    steps = args.steps
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
        "warmup": args.warmup, "ms_per_step": ms / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if args.precision == "fp32" else "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload}: ion acoustic wave, {ng} cells, "
                               f"{'+'.join(str(n) for n in pic.n)} particles/GPU, dt={dt}, full implicit step",
                   "precision": args.precision + (" residual + fp32 J w (defect correction)" if jac else ""),
                   "cn_mode": args.cn_mode, "jfnk_rtol": rtol,
                   "substeps_per_particle_per_pass": n_sub / max(n_p, 1),
                   "crossing_fraction": n_cross / max(n_sub, 1),
                   "substep_count": "one counting-build pass from the state the timed steps start at, x mover passes",
                   "l2": "particle state %.0f MB/GPU (fits the 126 MB L2 only for cfg1 in fp32); every "
                         "pass rereads all of it" % (n_p * (12 if args.precision == "fp32" else 20) * 1e-6),
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "implicit_step": {
            "ms_per_step": ms / steps, "wall_ms_per_step": 1e3 * wall / steps,
            "newton_its_mean": float(np.mean([h["newton_its"] for h in hist])),
            "gmres_its_mean": float(np.mean([h["gmres_its"] for h in hist])),
            "mover_passes_mean": calls / steps, "mover_passes_fp64_mean": calls_resid / steps if jac else None,
            "mover_ms_per_pass": k_ms,
            "mover_share_of_step": None if jac else k_ms * calls / steps / (ms / steps),
            "energy_rel_change_per_step": abs(e_end - e_start) / e_start / steps,
            "energy_rel_change_total": (e_end - e_start) / e_start,
            "gauss_residual_rel": gauss, "gauss_residual_max_abs": gauss_abs,
            "resid_last": hist[-1]["resid"], "resid0_last": hist[-1]["resid0"]},
        "gop_per_s_model": value * ops_per_pass / max(n_sub, 1) * 1e-9,
        "clocks": clocks,
        "e2e": {"value": value, "unit": UNIT,
                "h2d_bytes_per_step": int(calls / steps * ng * 8 + ng * 8),
                "d2h_bytes_per_step": int(calls / steps * ng * 8),
                "note": "the timed value already passes host E in and the residual out on every mover pass"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_gops, "unit": "GOp/s",
                     "frac": achieved / peak_gops, "traffic": None,
                     "kernel": pic.last_kernel() + " (all species of one pass)", "kernel_ms": k_ms,
                     "ops_per_launch": ops_per_pass,
                     "convention": "paper's op count (P:94-105), algorithmic table of DESIGN.md 6; NOT flops",
                     "peak_source": "derived: SMs x lanes x 2 x sm_max_mhz (DESIGN.md 6)",
                     "note": "passes of 1-4 M particles are latency-bound (two launches of 0.1 ms)"},
    }
    pic.close()
    if jac is not None:
        jac.close()
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def _peak_gops(sms, precision, sm_max_mhz):
    """Derived ALU peak: SMs x lanes x 2 (FMA) x clock, GOp/s."""
    return sms * (128 if precision == "fp32" else 64) * 2 * sm_max_mhz * 1e-3


def extra_iaw_leg(B, torch, workload, precision, steps, warmup, seed, stream, sms, sm_max_mhz):
    """Bounded leg of the default line: `steps` fully implicit time steps (pic_jfnk_step) of
    configs[1] / configs[4] at full size after `warmup` untimed ones, each step timed with CUDA
    events on the library's stream; the numbers `--workload cfg1|cfg4` reports, in short."""
    from paper_1111_5295_b200.iaw import gauss_field
    cfg = _workload(workload, 0, seed)
    ng, L, dt = cfg["n_cells"], cfg["length"], cfg["dt"]
    dx = L / ng
    rtol = 1e-8 if precision == "fp64" else 2e-4                    # SURVEY A-14
    flags = B.PIC_FLAG_VSORT
    pic = B.Pic(ng, L, cfg["species"], precision=precision, cn_mode="direct", flags=flags, stream=stream)
    n_p = sum(pic.n)
    E = gauss_field(pic.rho(B.PIC_STATE_N), dx)

    def energy():   # the diagnostic that allocates nothing: it sits inside the time loop
        return float(pic.kinetic_energy_noalloc(B.PIC_STATE_N).sum() + 0.5 * dx * np.sum(E * E))

    for _ in range(warmup):
        info = pic.jfnk_step(E, dt, rtol=rtol)
        assert info["converged"], info
    pic.set_flags(flags | B.PIC_FLAG_DIAG)          # exact sub-steps / crossings of one pass
    pic.move_accumulate(E, E, dt)
    exact = pic.get_stats()
    pic.set_flags(flags)
    l0 = pic.get_stats()["n_launches"]
    e_start = e_prev = energy()
    ms, hist, drift = [], [], []
    for _ in range(steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        info = pic.jfnk_step(E, dt, rtol=rtol)
        b.record()
        torch.cuda.synchronize()
        assert info["converged"], info
        ms.append(a.elapsed_time(b))
        hist.append(info)
        e_now = energy()
        drift.append(abs(e_now - e_prev) / e_start)
        e_prev = e_now
    launches = pic.get_stats()["n_launches"] - l0
    kms = []
    for _ in range(3):
        pic.move_accumulate(E, E, dt)
        kms.append(pic.get_stats()["last_move_ms"])
    k_ms = float(np.mean(kms))
    kernel = pic.last_kernel()
    pic.close()
    n_sub, n_cross = exact["n_sub"], exact["n_cross"]
    passes = float(np.mean([h["mover_calls"] for h in hist]))
    ops = OPS_INCELL * (n_sub - n_cross) + OPS_CROSS * n_cross
    peak = _peak_gops(sms, precision, sm_max_mhz)
    mean_ms = float(np.mean(ms))
    return {"workload": f"{workload}: ion acoustic wave, {ng} cells, "
                        f"{'+'.join(str(n) for n in pic.n)} particles, dt={dt}, full implicit step",
            "precision": precision, "jfnk_rtol": rtol, "steps": steps, "warmup": warmup,
            "ms_per_step": mean_ms, "ms_per_step_min": float(np.min(ms)),
            "ms_per_step_median": float(np.median(ms)), "ms_per_step_max": float(np.max(ms)),
            "value": n_sub * passes / (mean_ms * 1e-3), "unit": UNIT,
            "newton_its_mean": float(np.mean([h["newton_its"] for h in hist])),
            "gmres_its_mean": float(np.mean([h["gmres_its"] for h in hist])),
            "mover_passes_mean": passes, "mover_ms_per_pass": k_ms,
            "mover_share_of_step": k_ms * passes / mean_ms,
            "substeps_per_particle_per_pass": n_sub / max(n_p, 1),
            "crossing_fraction": n_cross / max(n_sub, 1),
            "energy_rel_change_per_step_max": float(np.max(drift)),
            "energy_rel_change_total": (e_prev - e_start) / e_start,
            "gpu_launches": int(launches), "kernel": kernel,
            "roofline_frac_pass": ops / (k_ms * 1e-3) * 1e-9 / peak}


def extra_cfg3_leg(B, torch, seed, stream, sms, sm_max_mhz, timed=5, warmup=3):
    """Bounded leg of the default line: configs[3] (2e7 two-stream particles, dt = 50, the
    divergence stress case) in fp32: one counting step for the exact sub-step counts and their
    percentiles, then `timed` launches of the fast build timed by the library's events."""
    cfg = _workload("cfg3", 0, seed)
    sp = cfg["species"][0]
    n_p = sp["x"].shape[0]
    flags = B.PIC_FLAG_VSORT
    pic = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision="fp32", cn_mode="direct",
                flags=flags | B.PIC_FLAG_COUNTS, stream=stream)
    dEn = torch.from_numpy(cfg["E_n"]).cuda()
    dEp = torch.from_numpy(cfg["E_np1"]).cuda()
    dj = torch.empty(cfg["n_cells"], dtype=torch.float64, device="cuda")
    dt, tol = cfg["dt"], cfg.get("tol", 1e-10)
    pic.set_flags(flags | B.PIC_FLAG_COUNTS | B.PIC_FLAG_DIAG)
    pic.move_accumulate(dEn, dEp, dt, tol, jbar_out=dj)
    exact = pic.get_stats()
    mean = exact["n_sub"] / max(n_p, 1)
    width = max(1, int(math.ceil(2.0 * mean / 64)))
    hs, _ = pic.count_histogram(0, width, 65)
    cum = np.cumsum(hs) / max(int(hs.sum()), 1)
    pct = {str(q): int((np.searchsorted(cum, q / 100.0) + 1) * width) for q in (50, 90, 99)}
    pic.set_flags(flags)
    kms = []
    for i in range(warmup + timed):
        pic.move_accumulate(dEn, dEp, dt, tol, jbar_out=dj)
        if i >= warmup:
            kms.append(pic.get_stats()["last_move_ms"])
    kernel = pic.last_kernel()
    pic.close()
    k_ms = float(np.mean(kms))
    n_sub, n_cross = exact["n_sub"], exact["n_cross"]
    ops = OPS_INCELL * (n_sub - n_cross) + OPS_CROSS * n_cross
    return {"workload": f"cfg3: {cfg['n_cells']} cells, {n_p} two-stream particles, dt={dt}",
            "precision": "fp32", "steps": timed, "warmup": warmup, "kernel": kernel,
            "kernel_ms": k_ms, "kernel_ms_min": float(np.min(kms)), "kernel_ms_max": float(np.max(kms)),
            "value": n_sub / (k_ms * 1e-3), "unit": UNIT,
            "substeps_per_particle": mean, "crossing_fraction": n_cross / max(n_sub, 1),
            "n_sub_percentile_upper_bounds": pct, "histogram_bin_width": width,
            "roofline_frac": ops / (k_ms * 1e-3) * 1e-9 / _peak_gops(sms, "fp32", sm_max_mhz)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0,
                    help="timed steps; 0 = 10, raised until the timed region lasts --min-seconds")
    ap.add_argument("--min-seconds", type=float, default=2.0,
                    help="without --steps: time enough steps for a region this long (clock samples)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"],
                    help="BASELINE.json configs[k]; cfg1 / cfg4 time the full implicit step (JFNK)")
    ap.add_argument("--rtol", type=float, default=0.0, help="cfg1/cfg4: nonlinear tolerance (0 = per precision)")
    ap.add_argument("--defect-correction", action="store_true",
                    help="cfg1/cfg4 with --precision fp64: fp32 Jacobian-vector products (P:325-331)")
    ap.add_argument("--n", type=int, default=0, help="override the particle count (debug)")
    ap.add_argument("--precision", default=None, choices=["fp32", "fp64"],
                    help="default: fp32 (cfg1: fp64, BASELINE.json configs[1])")
    ap.add_argument("--cn-mode", default="direct", choices=["direct", "picard"])
    ap.add_argument("--seed", type=int, default=W.DEFAULT_SEED)
    ap.add_argument("--cpu-sample", type=int, default=1 << 22)
    ap.add_argument("--ref-sample", type=int, default=1 << 19)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-vsort", action="store_true", help="bin by cell only (default: phase-space cell)")
    ap.add_argument("--fp64-n", type=int, default=-1,
                    help="with --precision fp32: also time the fp64 mover on the first N particles of "
                         "the same workload and report it under 'fp64' (-1 = all of them, 0 = skip)")
    ap.add_argument("--microbench", action="store_true",
                    help="only run the P:86 instruction micro-benchmarks (pic_microbench) and print them")
    ap.add_argument("--histogram", action="store_true",
                    help="report the per-particle sub-step / crossing histograms of a step "
                         "(BASELINE.json configs[3]); keeps 8 B per particle of counters")
    ap.add_argument("--one-per-lane", action="store_true",
                    help="fp32: the one-particle-per-lane kernel instead of the packed two-per-lane one")
    ap.add_argument("--strided", action="store_true",
                    help="the paper's particle order (Eq. 15): consecutive particles in consecutive cells")
    ap.add_argument("--per-visit", action="store_true",
                    help="deposit per cell visit with shared fp64 atomics (P:222) instead of the end-point form")
    ap.add_argument("--no-extra-legs", action="store_true",
                    help="default cfg2 line only: skip the bounded configs[4] / [1] / [3] legs "
                         "('implicit_step', 'cfg1', 'cfg3' in the JSON line)")
    ap.add_argument("--vp", action="store_true",
                    help="Vlasov-Poisson variant of the mover: orbits without the current deposit (P:281)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.precision is None:
        args.precision = "fp64" if args.workload == "cfg1" else "fp32"
    explicit_steps = args.steps > 0
    if not explicit_steps:
        args.steps = 10

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # --gpus N outside torchrun: launch the N replicas ourselves (one rank per GPU)
        import subprocess
        port = 29500 + os.getpid() % 2000
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
               f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1", "--master-port",
               str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.gpus != world and "WORLD_SIZE" in os.environ and rank == 0:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; using the launcher's {world}",
              file=sys.stderr)
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_1111_5295_b200 import binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    B.load()
    if args.microbench:
        if rank == 0:
            try:
                mhz = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("sm_max_mhz") or 1965.0)
            except Exception:  # noqa: BLE001
                mhz = 1965.0
            sampler = ClockSampler(local_rank)
            sampler.start()
            mb = B.microbench(iters=200000, sm_mhz=mhz)
            print(json.dumps({"microbench": mb, "sm_mhz_for_per_clk": mhz, "clocks": sampler.stop(),
                              "fp32_gflops_measured_ffma": 2 * mb["ffma"]["thread_gops"],
                              "fp64_gflops_measured_dfma": 2 * mb["dfma"]["thread_gops"]}), flush=True)
        return

    if args.workload in ("cfg1", "cfg4"):
        run_iaw(args, rank, world, local_rank, explicit_steps)
        return

    # replicas only: every rank runs its own copy of the workload with its own seed
    from paper_1111_5295_b200 import replicas as _rep
    cfg = _workload(args.workload, args.n, _rep.rank_seed(args.seed, rank))
    sp = cfg["species"][0]
    n_p = sp["x"].shape[0]
    stream = torch.cuda.current_stream().cuda_stream
    flags = 0 if args.no_vsort else B.PIC_FLAG_VSORT
    if args.vp:
        flags |= B.PIC_FLAG_NO_DEPOSIT
    if args.one_per_lane:
        flags |= B.PIC_FLAG_ONE_PER_LANE
    if args.strided:
        flags |= B.PIC_FLAG_STRIDED
    if args.per_visit:
        flags |= B.PIC_FLAG_DEPOSIT_PER_VISIT
    init_flags = flags | (B.PIC_FLAG_COUNTS if args.histogram else 0)   # allocates the counters
    pic = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision=args.precision,
                cn_mode=args.cn_mode, flags=init_flags, stream=stream)
    ng = cfg["n_cells"]
    dEn = torch.from_numpy(cfg["E_n"]).cuda()
    dEp = torch.from_numpy(cfg["E_np1"]).cuda()
    dj = torch.empty(ng, dtype=torch.float64, device="cuda")
    hEn = torch.from_numpy(cfg["E_n"]).pin_memory()
    hEp = torch.from_numpy(cfg["E_np1"]).pin_memory()
    hj = torch.empty(ng, dtype=torch.float64).pin_memory()
    dt, tol = cfg["dt"], cfg.get("tol", 1e-10)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- one step of the counting build (PIC_FLAG_DIAG) for the exact sub-step / crossing
    # counts of a step (state n is constant, so every step does the same work); the timed steps
    # run the fast build, which does not count per sub-step
    pic.set_flags(init_flags | B.PIC_FLAG_DIAG)
    pic.move_accumulate(dEn, dEp, dt, tol, jbar_out=dj)
    exact = pic.get_stats()
    hist = None
    if args.histogram:
        # 64 bins over [0, 2 x mean) for sub-steps and crossings, last bin = everything above
        mean = exact["n_sub"] / max(n_p, 1)
        width = max(1, int(math.ceil(2.0 * mean / 64)))
        hs, hc = pic.count_histogram(0, width, 65)
        cum = np.cumsum(hs) / max(int(hs.sum()), 1)
        pct = {q: int((np.searchsorted(cum, q / 100.0) + 1) * width) for q in (50, 90, 99)}
        hist = {"bin_width": width, "n_sub": [int(x) for x in hs], "n_cross": [int(x) for x in hc],
                "n_sub_percentile_upper_bounds": pct}
    pic.set_flags(flags)

    # ---- device-resident timing
    for _ in range(args.warmup):
        pic.move_accumulate(dEn, dEp, dt, tol, jbar_out=dj)
    torch.cuda.synchronize()
    if not explicit_steps and args.min_seconds > 0:
        # enough steps for a timed region of --min-seconds (the clock record needs samples under
        # load); every rank takes the same count
        w_ms = max(pic.get_stats()["last_move_ms"], 1e-3)
        want = int(math.ceil(args.min_seconds * 1e3 / w_ms))
        if world > 1:
            t = torch.tensor([want], device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            want = int(t.item())
        args.steps = max(args.steps, min(want, 100000))
    st0 = pic.get_stats()
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        pic.move_accumulate(dEn, dEp, dt, tol, jbar_out=dj)
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    st1 = pic.get_stats()
    n_sub, n_cross = exact["n_sub"], exact["n_cross"]    # per step, exact
    assert n_sub <= st1["n_sub"] < n_sub + 4 * n_p
    launches = st1["n_launches"] - st0["n_launches"]

    # ---- end to end: host E^n, E^{n+1} in, host jbar out, every step
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        pic.move_accumulate(hEn.numpy(), hEp.numpy(), dt, tol, jbar_out=hj.numpy())
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0

    # ---- dominant kernel alone: CUDA events around the mover launches (library-side events)
    kms = []
    for _ in range(min(args.steps, 20)):
        pic.move_accumulate(dEn, dEp, dt, tol, jbar_out=dj)
        kms.append(pic.get_stats()["last_move_ms"])
    k_ms = float(np.mean(kms))
    # ---- pic_commit (accept state n+1, re-bin by phase-space cell): once per time step, never per
    # residual; timed last because it replaces state n
    c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    c0.record()
    pic.commit()
    c1.record()
    torch.cuda.synchronize()
    commit_ms = c0.elapsed_time(c1)

    from paper_1111_5295_b200 import replicas
    ms, e2e_s, tot_sub, tot_cross = replicas.aggregate(ms, e2e_s, n_sub, n_cross, device="cuda")
    if rank != 0:
        pic.close()
        if world > 1:
            dist.destroy_process_group()
        return

    value = tot_sub * args.steps / (ms * 1e-3)
    e2e = tot_sub * args.steps / e2e_s
    props = torch.cuda.get_device_properties(local_rank)
    sms = props.multi_processor_count
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:  # noqa: BLE001
        pass
    sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    if args.precision == "fp32":
        peak_gops = sms * 128 * 2 * sm_max_mhz * 1e-3      # Eq. 1: lanes x 2 (FMA) x clock
    else:
        peak_gops = sms * 64 * 2 * sm_max_mhz * 1e-3       # FP64: 64 DFMA lanes per SM
    ops_per_launch = OPS_INCELL * (n_sub - n_cross) + OPS_CROSS * n_cross
    kernel_name = pic.last_kernel()        # the kernel the timed launches ran (library's word)
    achieved = ops_per_launch / (k_ms * 1e-3) * 1e-9
    executed = NCU_EXECUTED_OPS.get((args.workload, n_p, args.precision, kernel_name))
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if args.precision == "fp32" else "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload}: {ng} cells, {n_p} particles/GPU, dt={dt}",
                   "precision": args.precision, "cn_mode": args.cn_mode,
                   "variant": "VP (no current deposit, P:281)" if args.vp else "VA (orbit-averaged current)",
                   "binning": "cell" if args.no_vsort else
                              ("strided (P:244-250, Eq. 15): velocity class + offset class + cell" if args.strided
                               else "phase-space cell: cell + offset class + velocity class (P:242-250)"),
                   "deposit": "per cell visit, shared fp64 atomics (P:222)" if args.per_visit else "end-point form",
                   "substeps_per_particle": n_sub / max(n_p, 1),
                   "crossing_fraction": n_cross / max(n_sub, 1),
                   "l2": "inputs larger than L2 (particle state %.0f MB/GPU)" % (n_p * 12e-6),
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "gop_per_s_model": value * ops_per_launch / max(n_sub, 1) * 1e-9,
        "commit": {"ms": commit_ms, "note": "pic_commit after one step: swap + re-binning of all particles, "
                                            "once per time step (P:250); a time step is 13-33 mover passes"},
        "clocks": clocks,
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": 2 * ng * 8,
                "d2h_bytes_per_step": ng * 8},
        "gpu_launches": int(launches),
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_gops, "unit": "GOp/s",
                     "frac": achieved / peak_gops,
                     "traffic": NCU_TRAFFIC_BYTES.get((args.workload, n_p, args.precision)),
                     "traffic_unit": "bytes per launch (ncu dram read+write); algorithmic %d"
                                     % (n_p * (24 if args.precision == "fp32" else 40)),
                     "traffic_source": NCU_TRAFFIC_SOURCE,
                     "convention": "paper's op count (P:94-105): every FP/int/SF thread-operation 1, "
                                   "FMA 2, from the algorithmic table of DESIGN.md 6; NOT flops",
                     "frac_executed": (executed[0] * n_sub / (k_ms * 1e-3) * 1e-9 / peak_gops
                                       if executed else None),
                     "frac_fp_only": (executed[1] * n_sub / (k_ms * 1e-3) * 1e-9 / peak_gops
                                      if executed else None),
                     "frac_executed_paper_classes": (executed[2] * n_sub / (k_ms * 1e-3) * 1e-9 / peak_gops
                                                     if executed and executed[2] else None),
                     "executed_source": "thread-operations per sub-step from the SASS counters of "
                                        + NCU_TRAFFIC_SOURCE + ": all instructions by the paper's "
                                        "convention / floating-point arithmetic only / executed FP + AL + SF "
                                        "operations without control and data movement "
                                        "(profiles/r3_op_table.md)",
                     "kernel": kernel_name, "kernel_ms": k_ms,
                     "kernel_ms_launches": {"n": len(kms), "min": float(np.min(kms)),
                                            "median": float(np.median(kms)), "max": float(np.max(kms))},
                     "ops_per_launch": ops_per_launch,
                     "peak_source": "derived: SMs x lanes x 2 x sm_max_mhz (DESIGN.md 6)",
                     "hbm_gbs_algorithmic": n_p * (24 if args.precision == "fp32" else 40) / (k_ms * 1e-3) * 1e-9},
    }
    if hist is not None:
        line["substep_histogram"] = hist
    pic.close()
    pic = None
    # ---- BASELINE.json's metric names both precisions: the fp64 instantiation of the mover on
    # the first fp64_n particles of the same workload (same fields, same dt), kernel-timed
    if args.precision == "fp32" and args.fp64_n != 0 and not args.vp and args.workload in ("cfg2", "cfg3"):
        n64 = n_p if args.fp64_n < 0 else min(args.fp64_n, n_p)
        sp64 = dict(sp, x=sp["x"][:n64], v=sp["v"][:n64], w_q=sp["w_q"] * n_p / n64)
        p64 = B.Pic(cfg["n_cells"], cfg["length"], [sp64], precision="fp64", cn_mode=args.cn_mode,
                    flags=(0 if args.no_vsort else B.PIC_FLAG_VSORT) | B.PIC_FLAG_DIAG, stream=stream)
        p64.move_accumulate(dEn, dEp, dt, tol, jbar_out=dj)
        ex64 = p64.get_stats()
        p64.set_flags(0 if args.no_vsort else B.PIC_FLAG_VSORT)
        for _ in range(3):
            p64.move_accumulate(dEn, dEp, dt, tol, jbar_out=dj)
        k64 = []
        for _ in range(5):
            p64.move_accumulate(dEn, dEp, dt, tol, jbar_out=dj)
            k64.append(p64.get_stats()["last_move_ms"])
        k64 = float(np.mean(k64))
        ops64 = OPS_INCELL * (ex64["n_sub"] - ex64["n_cross"]) + OPS_CROSS * ex64["n_cross"]
        peak64 = sms * 64 * 2 * sm_max_mhz * 1e-3
        line["fp64"] = {"value": ex64["n_sub"] / (k64 * 1e-3), "unit": UNIT, "n_particles": n64,
                        "kernel": p64.last_kernel(), "kernel_ms": k64,
                        "roofline": {"bound": "alu", "achieved": ops64 / (k64 * 1e-3) * 1e-9,
                                     "peak": peak64, "unit": "GOp/s",
                                     "frac": ops64 / (k64 * 1e-3) * 1e-9 / peak64}}
        p64.close()
    # ---- the other configs of BASELINE.json in the same record (bounded: ~10 s in all): the
    # implicit step of configs[4] (fp32) and configs[1] (fp64), the mover on configs[3]
    default_line = (args.workload == "cfg2" and args.precision == "fp32" and world == 1 and not args.n
                    and not (args.vp or args.strided or args.per_visit or args.one_per_lane or args.no_vsort))
    if default_line and not args.no_extra_legs:
        del dEn, dEp, dj
        line["implicit_step"] = extra_iaw_leg(B, torch, "cfg4", "fp32", 20, 3, args.seed, stream, sms, sm_max_mhz)
        line["cfg1"] = extra_iaw_leg(B, torch, "cfg1", "fp64", 10, 3, args.seed, stream, sms, sm_max_mhz)
        line["cfg3"] = extra_cfg3_leg(B, torch, args.seed, stream, sms, sm_max_mhz)
    if not args.no_cpu_baseline:
        rate, nsub_s, dts, ns = oracle_rate(cfg, args.cpu_sample)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"first {ns} particles of {args.workload} "
                                          f"({nsub_s} sub-steps, {dts:.1f} s), serial fp64 oracle"}
        ratep, nsubp, dtp, npar, cores = oracle_rate_parallel(cfg)
        line["cpu_baseline_all_cores"] = {
            "value": ratep, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {npar} particles of {args.workload} in {cores} chunks, one serial "
                      f"oracle call per core ({nsubp} sub-steps, {dtp:.1f} s)"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
