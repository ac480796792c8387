"""GPU-side test utilities: run a workload dict through the C-ABI (via the ctypes binding) and
compare with the oracle using the parity metrics of SURVEY.md 8(c).  Used only by `-m gpu` tests
and __graft_entry__.smoke()."""
import numpy as np

from paper_1111_5295_b200 import binding as B
from paper_1111_5295_b200 import workloads as W
from helpers import (continuity_residual, oracle_run, periodic_dist, rel_l2,
                     round_to_fp32_state)

# north_star tolerances
TOL = {"fp64": dict(x=1e-10, v=1e-10, j=1e-10, cont=1e-10),
       "fp32": dict(x=1e-5, v=1e-5, j=1e-4, cont=1e-5)}
# max-norm gates beside the L2 ones: per non-flipped particle, |d xi| in cell units
# and |d v| / v_rms.  A single orbit's error is the L2 figure times a tail factor (errors are
# rounding random walks amplified by the orbit's own sensitivity); 100 x the L2 bar still
# catches one bad particle in 1e5, which the L2 norm alone would let through 300-fold.
TOL_MAX = {"fp64": dict(xi=1e-8, v=1e-8), "fp32": dict(xi=1e-3, v=1e-3)}


def gpu_run(cfg, precision, cn_mode="direct", flags=B.PIC_FLAG_COUNTS | B.PIC_FLAG_DIAG,
            subset=None, **kw):
    """pic_init + pic_move_accumulate on cfg (optionally on a per-species index subset)."""
    species = []
    for j, sp in enumerate(cfg["species"]):
        idx = slice(None) if subset is None else subset[j]
        species.append(dict(q_over_m=sp["q_over_m"], w_q=sp["w_q"],
                            x=np.ascontiguousarray(sp["x"][idx]),
                            v=np.ascontiguousarray(sp["v"][idx])))
    pic = B.Pic(cfg["n_cells"], cfg["length"], species, precision=precision, cn_mode=cn_mode,
                flags=flags, **kw)
    jbar = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"], cfg.get("tol", 1e-10))
    out = dict(pic=pic, jbar=jbar, stats=pic.get_stats(), species=[])
    for j in range(len(species)):
        r = pic.get_particles(j, B.PIC_STATE_NP1)
        r0 = pic.get_particles(j, B.PIC_STATE_N)
        r.update(cell0=r0["cell"], xi0=r0["xi"], v0=r0["v"])
        if flags & B.PIC_FLAG_COUNTS:
            r["n_sub"], r["n_cross"] = pic.get_counts(j)
        out["species"].append(r)
    return out


def oracle_state_for(cfg, precision, subset=None):
    """The start state the oracle must be given so that input rounding is not charged to the
    kernel: fp64 -> oracle's own binning of x; fp32 -> the fp32-rounded (cell, xi, v)."""
    if precision == "fp64" and subset is None:
        return None
    dx = cfg["length"] / cfg["n_cells"]
    st = []
    if precision == "fp32":
        for j, r in enumerate(round_to_fp32_state(cfg)):
            idx = slice(None) if subset is None else subset[j]
            st.append((r["cell"][idx], r["xi"][idx].astype(np.float64) * dx,
                       r["v"][idx].astype(np.float64)))
    else:
        from oracle import pic_oracle as o
        for j, sp in enumerate(cfg["species"]):
            idx = subset[j]
            c, s = o.bin_particles(cfg["n_cells"], cfg["length"], sp["x"][idx])
            st.append((c, s, sp["v"][idx]))
    return st


def sub_cfg(cfg, subset):
    out = dict(cfg)
    out["species"] = [dict(sp, x=sp["x"][idx], v=sp["v"][idx])
                      for sp, idx in zip(cfg["species"], subset)]
    return out


def parity(o, cfg, precision, cn_mode="direct", oracle_params=None, extra_flags=0, fast=False,
           pic_kw=None):
    """Run both sides; return metrics (SURVEY 8(c) 'Parity metrics').  Particles whose
    (n_sub, n_cross, cell) differ are branch flips (A-12): excluded from x/v, counted, and
    jbar is then recomputed on both sides on the non-flipped subset.

    fast=True: x, v, jbar and continuity are those of the FAST build (no per-particle counters;
    fp32 on power-of-two grids: mover2_kernel, two particles per lane).  The per-particle
    counts that identify flips still come from a counting-build run, whose orbits must be
    bit-identical to the fast build's (asserted here)."""
    dx = cfg["length"] / cfg["n_cells"]
    pic_kw = pic_kw or {}
    flags = B.PIC_FLAG_COUNTS | B.PIC_FLAG_DIAG | extra_flags
    g = gpu_run(cfg, precision, cn_mode, flags=flags, **pic_kw)
    if fast:
        flags = extra_flags
        gf = gpu_run(cfg, precision, cn_mode, flags=flags, **pic_kw)
        gf["kernel"] = gf["pic"].last_kernel()
        for a, b in zip(gf["species"], g["species"]):
            for k in ("x", "v", "cell", "xi"):
                assert np.array_equal(a[k], b[k]), f"fast build differs from counting build in {k}"
            a["n_sub"], a["n_cross"] = b["n_sub"], b["n_cross"]
        gf["stats"] = dict(gf["stats"], n_substep_cap=g["stats"]["n_substep_cap"])
        g["pic"].close()
        g = gf
    oc = sub_cfg(cfg, [slice(None)] * len(cfg["species"]))
    ref = oracle_run(o, oc, oracle_params, state=oracle_state_for(cfg, precision))
    m = dict(flips=0, n=0, x=[], v=[], xi_max=[], v_max=[], stats=g["stats"],
             ostats=ref["stats"].as_dict())
    keep = []
    for gs, rs in zip(g["species"], ref["species"]):
        same = (gs["n_sub"] == rs["n_sub"]) & (gs["n_cross"] == rs["n_cross"]) & \
               (gs["cell"] == rs["cell"])
        keep.append(same)
        m["flips"] += int((~same).sum())
        m["n"] += same.size
        xr = rs["cell"] * dx + rs["s"]
        d = periodic_dist(gs["x"][same], xr[same], cfg["length"])
        m["x"].append(float(np.linalg.norm(d) / max(np.linalg.norm(xr[same]), 1e-300)))
        m["v"].append(rel_l2(gs["v"][same], rs["v"][same]))
        # max norms over the non-flipped particles: position error in CELL units, velocity error
        # relative to the species' rms speed (one bad orbit cannot hide inside an L2 norm)
        m["xi_max"].append(float(d.max() / dx) if d.size else 0.0)
        vrms = float(np.sqrt(np.mean(rs["v"] ** 2))) if rs["v"].size else 1.0
        m["v_max"].append(float(np.max(np.abs(gs["v"][same] - rs["v"][same])) / max(vrms, 1e-300))
                          if d.size else 0.0)
    if m["flips"] == 0:
        gj, rj = g["jbar"], ref["jbar"]
    else:
        sub = [np.nonzero(k)[0] for k in keep]
        g2 = gpu_run(cfg, precision, cn_mode, flags=flags, subset=sub, **pic_kw)
        r2 = oracle_run(o, sub_cfg(cfg, sub), oracle_params,
                        state=oracle_state_for(cfg, precision, sub))
        gj, rj = g2["jbar"], r2["jbar"]
        g2["pic"].close()
    m["j"] = rel_l2(gj, rj)
    # continuity with the GPU's OWN (cell, xi) output and its own jbar (all particles)
    start = [(gs["cell0"], gs["xi0"] * dx) for gs in g["species"]]
    end = [(gs["cell"], gs["xi"] * dx) for gs in g["species"]]
    res, div = continuity_residual(o, cfg, start, end, g["jbar"])
    m["cont"] = float(np.linalg.norm(res) / max(np.linalg.norm(div), 1e-300))
    m["cont_max"] = float(np.max(np.abs(res)))
    m["gpu"], m["ref"] = g, ref
    return m


def assert_parity(m, precision, max_flip_frac=1e-3, max_norms=True):
    t = TOL[precision]
    if max_norms:
        tm = TOL_MAX[precision]
        assert max(m["xi_max"]) <= tm["xi"], f"max |d xi| {max(m['xi_max'])} cells > {tm['xi']}"
        assert max(m["v_max"]) <= tm["v"], f"max |d v|/v_rms {max(m['v_max'])} > {tm['v']}"
    assert m["flips"] <= max_flip_frac * m["n"], f"too many branch flips: {m['flips']}/{m['n']}"
    for x in m["x"]:
        assert x <= t["x"], f"x rel L2 {x} > {t['x']}"
    for v in m["v"]:
        assert v <= t["v"], f"v rel L2 {v} > {t['v']}"
    assert m["j"] <= t["j"], f"jbar rel L2 {m['j']} > {t['j']}"
    assert m["cont"] <= t["cont"], f"continuity {m['cont']} > {t['cont']}"
    assert m["stats"]["n_substep_cap"] == 0
