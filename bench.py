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
# `ncu --set full` capture (profiles/r1_mover_ncu.md); known only for the default workload.
NCU_TRAFFIC_BYTES = {("cfg2", 100_000_000, "fp32"): 2.366e9}


def _workload(name, n, seed):
    if name == "cfg2":
        return W.config2(n=n or 100_000_000, seed=seed)
    if name == "cfg3":
        return W.config3(n=n or 20_000_000, seed=seed)
    if name == "cfg0":
        return W.config0(n=n or 6400, seed=seed)
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg0", "cfg2", "cfg3"])
    ap.add_argument("--n", type=int, default=0, help="override the particle count (debug)")
    ap.add_argument("--precision", default="fp32", choices=["fp32", "fp64"])
    ap.add_argument("--cn-mode", default="direct", choices=["direct", "picard"])
    ap.add_argument("--seed", type=int, default=W.DEFAULT_SEED)
    ap.add_argument("--cpu-sample", type=int, default=1 << 22)
    ap.add_argument("--ref-sample", type=int, default=1 << 19)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-vsort", action="store_true", help="bin by cell only (default: phase-space cell)")
    ap.add_argument("--fp64-n", type=int, default=20_000_000,
                    help="with --precision fp32: also time the fp64 mover on the first N particles of "
                         "the same workload and report it under 'fp64' (0 = skip)")
    ap.add_argument("--microbench", action="store_true",
                    help="only run the P:86 instruction micro-benchmarks (pic_microbench) and print them")
    ap.add_argument("--histogram", action="store_true",
                    help="report the per-particle sub-step / crossing histograms of a step "
                         "(BASELINE.json configs[3]); keeps 8 B per particle of counters")
    ap.add_argument("--one-per-lane", action="store_true",
                    help="fp32: the one-particle-per-lane kernel instead of the packed two-per-lane one")
    ap.add_argument("--vp", action="store_true",
                    help="Vlasov-Poisson variant of the mover: orbits without the current deposit (P:281)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
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
    for _ in range(min(args.steps, 5)):
        pic.move_accumulate(dEn, dEp, dt, tol, jbar_out=dj)
        kms.append(pic.get_stats()["last_move_ms"])
    k_ms = float(np.mean(kms))

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
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if args.precision == "fp32" else "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload}: {ng} cells, {n_p} particles/GPU, dt={dt}",
                   "precision": args.precision, "cn_mode": args.cn_mode,
                   "variant": "VP (no current deposit, P:281)" if args.vp else "VA (orbit-averaged current)",
                   "binning": "cell" if args.no_vsort else "phase-space cell: cell + offset class + velocity class (P:242-250)",
                   "substeps_per_particle": n_sub / max(n_p, 1),
                   "crossing_fraction": n_cross / max(n_sub, 1),
                   "l2": "inputs larger than L2 (particle state %.0f MB/GPU)" % (n_p * 12e-6),
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "gop_per_s_model": value * ops_per_launch / max(n_sub, 1) * 1e-9,
        "clocks": clocks,
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": 2 * ng * 8,
                "d2h_bytes_per_step": ng * 8},
        "gpu_launches": int(launches),
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_gops, "unit": "GOp/s",
                     "frac": achieved / peak_gops,
                     "traffic": NCU_TRAFFIC_BYTES.get((args.workload, n_p, args.precision)),
                     "traffic_unit": "bytes per launch (ncu dram read+write); algorithmic %d"
                                     % (n_p * (24 if args.precision == "fp32" else 40)),
                     "kernel": kernel_name, "kernel_ms": k_ms,
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
    if args.precision == "fp32" and args.fp64_n > 0 and not args.vp:
        n64 = min(args.fp64_n, n_p)
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
