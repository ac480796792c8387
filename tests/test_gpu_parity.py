"""`-m gpu` parity tests: the CUDA path (through the C-ABI) against the oracle, element by
element on the same seeded inputs, with the tolerances of BASELINE.json's north_star:
fp64 rel L2 1e-10 on jbar, x, v; fp32 1e-4 on jbar, 1e-5 on x, v, continuity 1e-5 relative.
Branch-flipped particles (SURVEY A-12) are excluded, counted and reported."""
import math

import numpy as np
import pytest

from paper_1111_5295_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    import gpu_helpers
    from paper_1111_5295_b200 import binding
    binding.load()
    return gpu_helpers


def _report(name, m):
    print(f"[parity] {name}: x={max(m['x']):.2e} v={max(m['v']):.2e} j={m['j']:.2e} "
          f"max|dxi|={max(m['xi_max']):.2e} cells max|dv|/vrms={max(m['v_max']):.2e} "
          f"cont={m['cont']:.2e} flips={m['flips']}/{m['n']} "
          f"sub={m['stats']['n_sub']} cross={m['stats']['n_cross']}")


# ---- configs[0]: 6,400 electrons, 64 cells, dt = 0.5 ------------------------------------------
@pytest.mark.parametrize("precision,cn_mode", [("fp64", "picard"), ("fp64", "direct"),
                                               ("fp32", "direct"), ("fp32", "picard")])
def test_cfg0_parity(G, oracle, precision, cn_mode):
    cfg = W.config0()
    m = G.parity(oracle, cfg, precision, cn_mode)
    _report(f"cfg0 {precision} {cn_mode}", m)
    G.assert_parity(m, precision)
    if precision == "fp64":
        assert m["flips"] == 0
        assert m["stats"]["n_sub"] == m["ostats"]["n_sub"]
        assert m["stats"]["n_cross"] == m["ostats"]["n_cross"]
    m["gpu"]["pic"].close()


# ---- configs[2] / [3] shapes at sizes the oracle finishes in seconds (several tiles + a
# ragged tail: 200,003 is not a multiple of 32) --------------------------------------------------
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_cfg2_small_parity(G, oracle, precision):
    cfg = W.config2(n=200_003)
    m = G.parity(oracle, cfg, precision)
    _report(f"cfg2/200k {precision}", m)
    G.assert_parity(m, precision)
    assert m["stats"]["n_sub"] > 20 * 200_003   # paper-shaped: tens of sub-steps per particle
    m["gpu"]["pic"].close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_cfg3_small_invariants(G, oracle, precision):
    """configs[3] orbits are sensitive.  fp64: north_star's bars.  fp32: the
    invariants at north_star's bar, and per-particle parity at the tolerance the arithmetic
    allows here (DESIGN.md 2 "cfg3 in fp32", tests/test_sensitivity.py): the oracle's own
    response to ONE fp32 ulp of input error, times sqrt(n_sub) for a kernel that rounds at every
    sub-step, times 3 for the spread of that estimate.  The remaining-time bookkeeping is not
    the cause: PIC_FLAG_EXACT_TIME (exact accounting) leaves the figures unchanged."""
    from paper_1111_5295_b200 import binding as B
    from helpers import ulp_response
    cfg = W.config3(n=20_011)
    m = G.parity(oracle, cfg, precision)
    _report(f"cfg3/20k {precision}", m)
    if precision == "fp64":
        # L2 bars: north_star's.  Max norms: the generic 1e-8 gates assume a 100-fold tail over
        # the L2 figure; on these orbits the tail is the orbits' own (a few of them amplify an
        # error a hundred times more than the average one), so the bar is derived from the
        # oracle's MAX-norm response to one fp64 ulp: an fp64 kernel rounds about ten times per
        # sub-step on the way to (x, v) (Eq. 11's denominator and quotient, the two updates, the
        # remaining time; discriminant, root and quotient on a crossing), a random walk of
        # 10 n_sub such errors, times 3 for the spread of the estimate.
        G.assert_parity(m, "fp64", max_flip_frac=5e-3, max_norms=False)
        r = ulp_response(oracle, cfg, fp64=True)
        k = 3.0 * math.sqrt(10.0 * r["n_sub_mean"])
        print(f"[parity] cfg3 fp64 derived max-norm bars: xi {k * r['xi_max']:.2e} cells "
              f"(got {max(m['xi_max']):.2e}), v {k * r['v_max']:.2e} (got {max(m['v_max']):.2e}); "
              f"L2 estimates x {k * r['x']:.1e} v {k * r['v']:.1e}")
        assert max(m["xi_max"]) <= k * r["xi_max"] and max(m["v_max"]) <= k * r["v_max"]
    else:
        r = ulp_response(oracle, cfg)
        k = 3.0 * math.sqrt(r["n_sub_mean"])
        print(f"[parity] cfg3 fp32 derived bars: x {k * r['x']:.2e} v {k * r['v']:.2e} j {k * r['j']:.2e}")
        assert max(m["x"]) <= k * r["x"] and max(m["v"]) <= k * r["v"] and m["j"] <= k * r["j"]
        assert m["j"] <= G.TOL["fp32"]["j"]                    # jbar does meet north_star's 1e-4
        assert m["cont"] <= G.TOL["fp32"]["cont"]
        assert m["flips"] <= 0.05 * m["n"]
        m["gpu"]["pic"].close()
        # exact time accounting: same orbits to within the same tolerance (so far it has not
        # come out better either -- reported, not required: a better kernel must not fail here)
        m2 = G.parity(oracle, cfg, precision, extra_flags=B.PIC_FLAG_EXACT_TIME)
        _report("cfg3/20k fp32 exact-time", m2)
        print(f"[parity] cfg3 fp32 exact-time / plain: v {max(m2['v']) / max(m['v']):.2f} "
              f"x {max(m2['x']) / max(m['x']):.2f}")
        assert max(m2["v"]) <= k * r["v"] and max(m2["x"]) <= k * r["x"]
        m = m2
    assert m["stats"]["n_substep_cap"] == 0
    m["gpu"]["pic"].close()


# ---- the paper's per-cell-visit register accumulation as the deposit mode ------------
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("which", ["cfg0", "cfg2"])
def test_per_visit_deposit_parity(G, oracle, precision, which):
    from paper_1111_5295_b200 import binding as B
    cfg = W.config0() if which == "cfg0" else W.config2(n=100_001)
    m = G.parity(oracle, cfg, precision, extra_flags=B.PIC_FLAG_DEPOSIT_PER_VISIT)
    _report(f"{which} {precision} per-visit", m)
    G.assert_parity(m, precision)
    # and the two deposit modes agree with each other to rounding
    g2 = G.gpu_run(cfg, precision)
    assert G.rel_l2(m["gpu"]["jbar"], g2["jbar"]) < (1e-12 if precision == "fp64" else 1e-6)
    m["gpu"]["pic"].close()
    g2["pic"].close()


# ---- (cell, velocity class) binning: same results, original order kept ---------------
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_vsort_parity_and_commit(G, oracle, precision):
    from paper_1111_5295_b200 import binding as B
    cfg = W.config2(n=150_001)
    m = G.parity(oracle, cfg, precision, extra_flags=B.PIC_FLAG_VSORT)
    _report(f"cfg2/150k {precision} vsort", m)
    G.assert_parity(m, precision)
    pic = m["gpu"]["pic"]
    # commit re-bins by (cell, velocity class); getters still answer in the caller's order
    before = pic.get_particles(0, B.PIC_STATE_NP1)
    pic.commit()
    after = pic.get_particles(0, B.PIC_STATE_N)
    for k in ("x", "v", "cell", "xi"):
        assert np.array_equal(before[k], after[k]), k
    pic.close()


# ---- the paper's own particle order (Eq. 15): consecutive particles in consecutive cells ----------
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("per_visit", [False, True])
def test_strided_layout_parity(G, oracle, precision, per_visit):
    from paper_1111_5295_b200 import binding as B
    cfg = W.config2(n=150_001)
    extra = B.PIC_FLAG_VSORT | B.PIC_FLAG_STRIDED | (B.PIC_FLAG_DEPOSIT_PER_VISIT if per_visit else 0)
    m = G.parity(oracle, cfg, precision, extra_flags=extra, fast=not per_visit)
    _report(f"cfg2/150k {precision} strided per_visit={per_visit}", m)
    G.assert_parity(m, precision)
    pic = m["gpu"]["pic"]
    before = pic.get_particles(0, B.PIC_STATE_NP1)
    pic.commit()
    after = pic.get_particles(0, B.PIC_STATE_N)
    for k in ("x", "v", "cell", "xi"):
        assert np.array_equal(before[k], after[k]), k
    pic.close()


# ---- the fast build (no per-sub-step counting) computes the same orbits as the counting build --
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_fast_build_matches_counting_build(G, precision):
    from paper_1111_5295_b200 import binding as B
    cfg = W.config2(n=120_007)
    sp = cfg["species"][0]
    out = {}
    for name, flags in (("fast", B.PIC_FLAG_VSORT), ("count", B.PIC_FLAG_VSORT | B.PIC_FLAG_DIAG)):
        pic = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision=precision, flags=flags)
        j = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
        out[name] = (pic.get_particles(0, B.PIC_STATE_NP1), j, pic.get_stats())
        pic.close()
    (pf, jf, sf), (pc, jc, sc) = out["fast"], out["count"]
    for k in ("x", "v", "cell", "xi"):
        assert np.array_equal(pf[k], pc[k]), k            # bit-identical orbits
    assert G.rel_l2(jf, jc) < 1e-13                       # same deposits, atomics in any order
    assert sf["n_cross"] in (0, sc["n_cross"])            # not counted on power-of-two grids
    assert sc["n_sub"] <= sf["n_sub"] < sc["n_sub"] + 4 * 120_007   # grouped upper bound


def _tiny_ring(n_cells, n=10_007):
    """2- or 4-cell ring, dt = 4: every orbit wraps the ring several times (whole-turn deposits)."""
    length = 0.7 * n_cells
    xf = W.face_positions(n_cells, length)
    x = W.uniform01(31, 1, n) * length * (1 - 1e-12)
    v = 1.5 * W.normal01(31, 2, n)
    return dict(n_cells=n_cells, length=length, dt=4.0, tol=1e-12,
                E_n=0.2 * np.sin(2 * math.pi * xf / length),
                E_np1=0.2 * np.sin(2 * math.pi * xf / length + 0.4),
                species=[dict(name="e", q_over_m=-1.0, w_q=-length / n, x=x, v=v)])



# ---- the fast build straight against the oracle: fp32 on power-of-two grids this is
# mover2_kernel (two particles per lane, packed FP32), fp64 the fast build of mover_kernel
@pytest.mark.parametrize("case", ["cfg0", "cfg2", "cfg2-vsort", "iaw-2species", "ring-2-cells"])
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_fast_build_parity_with_oracle(G, oracle, precision, case):
    from paper_1111_5295_b200 import binding as B
    cfg = {"cfg0": lambda: W.config0(), "cfg2": lambda: W.config2(n=100_003),
           "cfg2-vsort": lambda: W.config2(n=200_003), "iaw-2species": lambda: W.config1(ppc=40),
           "ring-2-cells": lambda: _tiny_ring(2)}[case]()
    extra = B.PIC_FLAG_VSORT if case in ("cfg2-vsort", "iaw-2species") else 0
    m = G.parity(oracle, cfg, precision, extra_flags=extra, fast=True)
    _report(f"fast build {case} {precision} [{m['gpu']['kernel']}]", m)
    assert m["gpu"]["kernel"] == ("mover2_kernel" if precision == "fp32" else "mover_kernel")
    G.assert_parity(m, precision)
    m["gpu"]["pic"].close()


# ---- the production fp32 kernel (two particles per lane, packed FFMA2/FMUL2/FADD2, mover2.cuh)
# against the one-particle-per-lane kernel: same arithmetic in the same order => identical orbits
@pytest.mark.parametrize("case", ["cfg0", "cfg2-vsort", "cfg2-cell", "cfg3-vsort", "cfg2-odd-tail",
                                  "ring-2-cells", "ring-4-cells-vsort"])
def test_two_per_lane_matches_one_per_lane(G, case):
    from paper_1111_5295_b200 import binding as B
    cfg = {"cfg0": lambda: W.config0(), "cfg2-vsort": lambda: W.config2(n=150_001),
           "cfg2-cell": lambda: W.config2(n=90_001), "cfg3-vsort": lambda: W.config3(n=20_011),
           "cfg2-odd-tail": lambda: W.config2(n=65), "ring-2-cells": lambda: _tiny_ring(2),
           "ring-4-cells-vsort": lambda: _tiny_ring(4)}[case]()
    base = 0 if case in ("cfg0", "cfg2-cell", "ring-2-cells") else B.PIC_FLAG_VSORT
    sp = cfg["species"][0]
    out = {}
    for name, flags in (("two", base), ("one", base | B.PIC_FLAG_ONE_PER_LANE)):
        pic = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision="fp32", flags=flags)
        j = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
        j2 = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])      # repeatable
        assert G.rel_l2(j2, j) < 1e-13
        assert pic.last_kernel() == ("mover2_kernel" if name == "two" else "mover_kernel")
        out[name] = (pic.get_particles(0, B.PIC_STATE_NP1), j, pic.get_stats())
        pic.close()
    (p2, j2, s2), (p1, j1, s1) = out["two"], out["one"]
    for k in ("x", "v", "cell", "xi"):
        assert np.array_equal(p2[k], p1[k]), k            # bit-identical orbits
    assert np.any(j1 != 0.0) and G.rel_l2(j2, j1) < 1e-13  # same deposits, atomics in any order
    assert s2["n_sub"] == s1["n_sub"]                      # same grouped sub-step count


# ---- grids whose cell count is not a power of two take the generic wrap path --------------------
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("n_cells", [3, 48, 100])
def test_non_power_of_two_grid(G, oracle, precision, n_cells):
    from paper_1111_5295_b200 import binding as B
    length = 0.7 * n_cells
    xf = W.face_positions(n_cells, length)
    n = 30_011
    x = W.uniform01(21, 1, n) * length * (1 - 1e-12)
    v = 1.5 * W.normal01(21, 2, n)
    cfg = dict(n_cells=n_cells, length=length, dt=4.0, tol=1e-12,
               E_n=0.2 * np.sin(2 * math.pi * xf / length),
               E_np1=0.2 * np.sin(2 * math.pi * xf / length + 0.4),
               species=[dict(name="e", q_over_m=-1.0, w_q=-length / n, x=x, v=v)])
    for extra in (0, B.PIC_FLAG_VSORT, B.PIC_FLAG_DEPOSIT_PER_VISIT):
        m = G.parity(oracle, cfg, precision, extra_flags=extra)
        _report(f"n_cells={n_cells} {precision} flags+{extra}", m)
        G.assert_parity(m, precision, max_flip_frac=2e-3)
        r = m["ref"]["species"][0]
        unwrapped = r["cell0"].astype(np.int64) + r["k"]
        assert np.any(unwrapped < 0) and np.any(unwrapped >= n_cells)     # orbits cross the seam
        m["gpu"]["pic"].close()


# ---- grids too large for a block's shared memory: the global-memory grid fallback (S7 hard part 6)
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("n_cells", [20_000, 100_003])
def test_large_grid_global_memory_fallback(G, oracle, precision, n_cells):
    from paper_1111_5295_b200 import binding as B
    length = 0.7 * n_cells
    xf = W.face_positions(n_cells, length)
    n = 60_013
    x = W.uniform01(41, 1, n) * length * (1 - 1e-12)
    v = 1.5 * W.normal01(41, 2, n)
    k = 2 * math.pi * round(n_cells / 150) / length            # ~150 cells per wavelength
    cfg = dict(n_cells=n_cells, length=length, dt=4.0, tol=1e-12, E_n=0.2 * np.sin(k * xf),
               E_np1=0.2 * np.sin(k * xf + 0.4),
               species=[dict(name="e", q_over_m=-1.0, w_q=-length / n, x=x, v=v)])
    for extra in (0, B.PIC_FLAG_VSORT):
        m = G.parity(oracle, cfg, precision, extra_flags=extra, fast=True)
        _report(f"n_cells={n_cells} {precision} flags+{extra} [{m['gpu']['kernel']}]", m)
        assert m["gpu"]["kernel"] == "mover_kernel (global-memory grid)"
        G.assert_parity(m, precision, max_flip_frac=2e-3)
        pic = m["gpu"]["pic"]
        # the diagnostics and the commit work on such grids too
        dx = length / n_cells
        end = pic.get_particles(0, B.PIC_STATE_NP1)
        ref = oracle.rho(n_cells, length, cfg["species"][0]["w_q"], end["cell"], end["xi"] * dx)
        assert G.rel_l2(pic.rho(B.PIC_STATE_NP1), ref) < 1e-12
        pic.commit()
        after = pic.get_particles(0, B.PIC_STATE_N)
        assert np.array_equal(end["x"], after["x"]) and np.array_equal(end["v"], after["v"])
        pic.close()
    with pytest.raises(B.PicError):      # the per-visit deposit needs the grid in shared memory
        B.Pic(n_cells, length, cfg["species"], precision=precision, flags=B.PIC_FLAG_DEPOSIT_PER_VISIT)
    # what the global-memory-grid kernels do not implement is refused, at pic_init and at
    # pic_set_flags alike, never silently dropped; the refused call leaves the flags as they were
    if precision == "fp32":
        with pytest.raises(B.PicError):
            B.Pic(n_cells, length, cfg["species"], precision=precision, flags=B.PIC_FLAG_EXACT_TIME)
    pic = B.Pic(n_cells, length, cfg["species"], precision=precision)
    j0 = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
    bad = [B.PIC_FLAG_DEPOSIT_PER_VISIT] + ([B.PIC_FLAG_EXACT_TIME] if precision == "fp32" else [])
    for flag in bad:
        with pytest.raises(B.PicError) as ei:
            pic.set_flags(flag)
        assert ei.value.code == B.PIC_ERR_UNSUPPORTED and "too large" in str(ei.value)
    pic.set_flags(B.PIC_FLAG_NO_STORE)                 # a supported one still goes through
    j1 = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
    assert G.rel_l2(j1, j0) < 1e-12
    pic.close()


# ---- Vlasov-Poisson variant: orbits without the current deposit, rho at the end
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_vp_variant_no_deposit(G, oracle, precision):
    from paper_1111_5295_b200 import binding as B
    cfg = W.config2(n=60_013)
    sp = cfg["species"][0]
    dx = cfg["length"] / cfg["n_cells"]
    va = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision=precision, flags=B.PIC_FLAG_VSORT)
    vp = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision=precision,
               flags=B.PIC_FLAG_VSORT | B.PIC_FLAG_NO_DEPOSIT)
    ja = va.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
    jp = vp.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
    assert np.all(jp == 0.0) and np.any(ja != 0.0)
    a, b = va.get_particles(0, B.PIC_STATE_NP1), vp.get_particles(0, B.PIC_STATE_NP1)
    for k in ("x", "v", "cell", "xi"):
        assert np.array_equal(a[k], b[k]), k                      # same orbits
    # charge density of state n+1 (quadratic spline, A-10) against the oracle's O11 on the
    # kernel's own end state, and continuity ties it to the VA run's jbar
    rho1 = vp.rho(B.PIC_STATE_NP1)
    ref = oracle.rho(cfg["n_cells"], cfg["length"], sp["w_q"], b["cell"], b["xi"] * dx)
    assert G.rel_l2(rho1, ref) < 1e-12
    rho0 = vp.rho(B.PIC_STATE_N)
    div = cfg["dt"] * (np.roll(ja, -1) - ja) / dx
    assert np.linalg.norm(rho1 - rho0 + div) <= 1e-10 * np.linalg.norm(div)
    va.close()
    vp.close()


# ---- device-side sub-step / crossing histograms (BJ configs[3]) against numpy on the counts ----
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_count_histogram(G, precision):
    from paper_1111_5295_b200 import binding as B
    cfg = W.config3(n=30_011)
    sp = cfg["species"][0]
    pic = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision=precision,
                flags=B.PIC_FLAG_COUNTS | B.PIC_FLAG_VSORT)
    pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
    ns, nc = pic.get_counts(0)
    for width, nb in ((1, 4096), (16, 64), (100, 7)):
        hs, hc = pic.count_histogram(0, width, nb)
        for h, v in ((hs, ns), (hc, nc)):
            ref = np.bincount(np.minimum(v // width, nb - 1), minlength=nb)
            assert np.array_equal(h.astype(np.int64), ref)
        assert int(hs.sum()) == 30_011
    st = pic.get_stats()
    assert int(ns.sum()) == st["n_sub"] and int(nc.sum()) == st["n_cross"]
    with pytest.raises(B.PicError):
        pic.count_histogram(0, 0, 16)
    pic.close()
    nocount = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision=precision)
    nocount.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
    with pytest.raises(B.PicError):
        nocount.count_histogram(0, 1, 16)
    nocount.close()


# ---- long orbits: many wraps of the periodic ring (end-point deposit: whole turns) -----------
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_ring_wraps(G, oracle, precision):
    n_cells, length = 8, 4.0
    xf = W.face_positions(n_cells, length)
    E = 0.05 * np.sin(2 * math.pi * xf / length)
    n = 257
    x = W.uniform01(5, 1, n) * length * (1 - 1e-12)
    v = 6.0 * W.normal01(5, 2, n)          # |v| dt / L up to ~10 turns either way
    cfg = dict(n_cells=n_cells, length=length, dt=3.0, tol=1e-12, E_n=E, E_np1=E,
               species=[dict(name="e", q_over_m=-1.0, w_q=-length / n, x=x, v=v)])
    m = G.parity(oracle, cfg, precision)
    _report(f"ring-wraps {precision}", m)
    G.assert_parity(m, precision, max_flip_frac=0.02)
    assert np.max(np.abs(m["ref"]["species"][0]["k"])) > 3 * n_cells   # really wrapped
    m["gpu"]["pic"].close()


# ---- two species (IAW shape, small), multi-species sum of jbar ---------------------------------
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_two_species_parity(G, oracle, precision):
    cfg = W.config1(ppc=40)
    xf = W.face_positions(cfg["n_cells"], cfg["length"])
    cfg["E_n"] = 0.02 * np.sin(2 * math.pi * xf / cfg["length"])
    cfg["E_np1"] = 0.02 * np.sin(2 * math.pi * xf / cfg["length"] + 0.2)
    m = G.parity(oracle, cfg, precision)
    _report(f"iaw-small {precision}", m)
    G.assert_parity(m, precision)
    m["gpu"]["pic"].close()


# ---- closed forms on the GPU (the oracle's pins P-1, P-2 applied to the kernel) ----------------
@pytest.mark.parametrize("precision,tol", [("fp64", 1e-12), ("fp32", 2e-5)])
def test_free_streaming_and_uniform_field(G, precision, tol):
    n_cells, length, dt = 32, 10.0, 2.5
    n = 1000
    x = W.uniform01(11, 1, n) * length * (1 - 1e-12)
    v = W.normal01(11, 2, n)
    dx = length / n_cells
    for E0 in (0.0, 0.3):
        E = np.full(n_cells, E0)
        cfg = dict(n_cells=n_cells, length=length, dt=dt, tol=1e-12, E_n=E, E_np1=E,
                   species=[dict(name="e", q_over_m=-1.0, w_q=-length / n, x=x, v=v)])
        g = G.gpu_run(cfg, precision)
        s = g["species"][0]
        a = -E0
        X0 = (s["cell0"] + s["xi0"]) * dx          # the (possibly fp32-rounded) start
        X1 = X0 + s["v0"] * dt + 0.5 * a * dt * dt
        d = np.abs(((s["x"] - X1 + length / 2) % length) - length / 2)
        assert d.max() < tol * 10, (E0, d.max())
        assert np.max(np.abs(s["v"] - (s["v0"] + a * dt))) < tol * 10
        # P-8: sum_f J_f = w_q sum_p (X1 - X0)  <=>  sum_f jbar_f = w_q sum (X1-X0)/(dt dx)
        lhs = g["jbar"].sum()
        rhs = (-length / n) * np.sum(s["v0"] * dt + 0.5 * a * dt * dt) / (dt * dx)
        assert abs(lhs - rhs) <= (1e-11 if precision == "fp64" else 2e-5) * max(abs(rhs), 1.0)
        g["pic"].close()


# ---- edge cases --------------------------------------------------------------------------------
def test_edge_cases(G, oracle):
    n_cells, length = 8, 4.0
    dx = length / n_cells
    xf = W.face_positions(n_cells, length)
    E = 0.5 * np.sin(2 * math.pi * xf / length)
    # particles exactly on faces (A-5), at 0, just below L, zero velocity, and a single particle
    x = np.array([0.0, dx, 3 * dx, np.nextafter(length, 0.0), 1.3, 2.0, 0.25])
    v = np.array([1.0, -1.0, 0.0, 2.0, 0.0, -3.0, 1e-9])
    cfg = dict(n_cells=n_cells, length=length, dt=1.7, tol=1e-12, E_n=E, E_np1=0.9 * E,
               species=[dict(name="e", q_over_m=-1.0, w_q=-0.5, x=x, v=v)])
    for cn in ("picard", "direct"):
        m = G.parity(oracle, cfg, "fp64", cn)
        _report(f"edge fp64 {cn}", m)
        G.assert_parity(m, "fp64", max_flip_frac=0.0)
        m["gpu"]["pic"].close()
    # fp32: the same orbits at north_star's fp32 bars.  Seven particles: one branch flip (a
    # particle that starts ON a face may round to the other side of a decision) is 14 % of them,
    # so flips are reported and bounded by one, and the bars are asserted on the others
    for cn in ("picard", "direct"):
        m = G.parity(oracle, cfg, "fp32", cn)
        _report(f"edge fp32 {cn}", m)
        assert m["flips"] <= 1, m["flips"]
        G.assert_parity(m, "fp32", max_flip_frac=1.0)
        m["gpu"]["pic"].close()
    # one cell only: both faces are face 0
    cfg1 = dict(n_cells=1, length=1.0, dt=0.9, tol=1e-12, E_n=np.array([0.3]),
                E_np1=np.array([0.1]),
                species=[dict(name="e", q_over_m=1.0, w_q=1.0, x=np.array([0.2, 0.7]),
                              v=np.array([1.5, -2.5]))])
    m = G.parity(oracle, cfg1, "fp64")
    # one cell: jbar_{c+1} - jbar_c = 0 identically, so the relative continuity metric has no
    # denominator; check the absolute residual (rho is constant) and the rest as usual
    assert m["cont_max"] < 1e-12 and m["flips"] == 0
    assert max(m["x"]) < 1e-10 and max(m["v"]) < 1e-10 and m["j"] < 1e-10
    m["gpu"]["pic"].close()


def test_empty_species_and_bad_input(G):
    from paper_1111_5295_b200 import binding as B
    n_cells, length = 16, 8.0
    E = np.zeros(n_cells)
    e = np.empty(0)
    pic = B.Pic(n_cells, length, [dict(q_over_m=-1.0, w_q=-1.0, x=e, v=e)], precision="fp32")
    j = pic.move_accumulate(E, E, 1.0)
    assert np.all(j == 0.0) and pic.get_stats()["n_sub"] == 0
    pic.close()
    with pytest.raises(B.PicError):   # x outside [0, L)
        B.Pic(n_cells, length, [dict(q_over_m=-1.0, w_q=-1.0, x=np.array([8.5]), v=np.array([0.0]))])
    with pytest.raises(B.PicError):   # non-finite v
        B.Pic(n_cells, length, [dict(q_over_m=-1.0, w_q=-1.0, x=np.array([1.0]), v=np.array([np.nan]))])


def test_substep_cap_is_reported(G):
    from paper_1111_5295_b200 import binding as B
    # the kernel tests the cap once per 64 sub-steps (A-9), so take orbits that need
    # many more than that: configs[3] shape, ~590 sub-steps per particle
    cfg = W.config3(n=2000)
    sp = cfg["species"][0]
    pic = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision="fp64", max_substeps=16)
    # the binding raises on the cap like on any other error ...
    with pytest.raises(B.PicError) as ei:
        pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
    assert ei.value.code == B.PIC_ERR_SUBSTEP_CAP
    assert pic.get_stats()["n_substep_cap"] > 0
    pic.set_step(cfg["E_n"], cfg["dt"])
    with pytest.raises(B.PicError) as ei:
        pic.residual(cfg["E_np1"])
    assert ei.value.code == B.PIC_ERR_SUBSTEP_CAP
    # ... unless the truncated result is asked for: jbar of the cut-off orbits, as written by the call
    j = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"], allow_cap=True)
    R = pic.residual(cfg["E_np1"], allow_cap=True)
    assert np.all(np.isfinite(j)) and np.any(j != 0.0)
    ref = (cfg["E_np1"] - cfg["E_n"]) / cfg["dt"] + j - j.mean()
    assert np.max(np.abs(R - ref)) <= 1e-12 * np.max(np.abs(ref))
    pic.close()


# ---- boundary: residual, repeatability, device pointers, commit ---------------------------------
def test_residual_repeat_commit(G, oracle):
    import torch
    from paper_1111_5295_b200 import binding as B
    cfg = W.config0()
    sp = cfg["species"][0]
    pic = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision="fp64", cn_mode="picard",
                flags=B.PIC_FLAG_COUNTS, stream=torch.cuda.current_stream().cuda_stream)
    dt = cfg["dt"]
    j1 = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], dt)
    j2 = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], dt)     # state n untouched: repeatable
    assert np.max(np.abs(j1 - j2)) <= 1e-13 * np.max(np.abs(j1))
    # device pointers in, device pointer out (no host copies inside the call)
    dEn = torch.from_numpy(cfg["E_n"]).cuda()
    dEp = torch.from_numpy(cfg["E_np1"]).cuda()
    dj = torch.empty(cfg["n_cells"], dtype=torch.float64, device="cuda")
    pic.move_accumulate(dEn, dEp, dt, jbar_out=dj)
    torch.cuda.synchronize()
    assert np.max(np.abs(dj.cpu().numpy() - j1)) <= 1e-13 * np.max(np.abs(j1))
    # a9 against the oracle's residual of the oracle's jbar
    pic.set_step(cfg["E_n"], dt)
    R = pic.residual(cfg["E_np1"])
    ref = G.oracle_run(oracle, cfg)
    Rref = oracle.residual(cfg["E_n"], cfg["E_np1"], dt, ref["jbar"])
    assert G.rel_l2(R, Rref) < 1e-10
    # P-12: sum_f R_f = sum_f (E^{n+1} - E^n)/dt
    assert abs(R.sum() - (cfg["E_np1"] - cfg["E_n"]).sum() / dt) < 1e-12
    # commit: state n+1 becomes state n (re-binned); a second move must match the oracle
    # continuing from its own n+1 state
    r1 = ref["species"][0]
    pic.commit()
    got = pic.get_particles(0, B.PIC_STATE_N)
    assert np.array_equal(got["cell"], r1["cell"])
    j3 = pic.move_accumulate(cfg["E_np1"], cfg["E_np1"], dt)
    cfgb = dict(cfg, E_n=cfg["E_np1"])
    ref2 = G.oracle_run(oracle, cfgb, state=[(r1["cell"], r1["s"], r1["v"])])
    assert G.rel_l2(j3, ref2["jbar"]) < 1e-9
    after = pic.get_particles(0, B.PIC_STATE_NP1)
    assert G.rel_l2(after["v"], ref2["species"][0]["v"]) < 1e-9
    pic.close()


def test_energy_identity_on_gpu(G):
    """P-9 on the kernel: sum_p w_m (v1^2 - v0^2)/2 = dt dx sum_f jbar_f E^{n+1/2}_f."""
    from paper_1111_5295_b200 import binding as B
    cfg = W.config2(n=100_000)
    sp = cfg["species"][0]
    dx = cfg["length"] / cfg["n_cells"]
    for precision, tol in (("fp64", 1e-11), ("fp32", 1e-4)):
        pic = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision=precision)
        jbar = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
        dK = pic.kinetic_energy(B.PIC_STATE_NP1)[0] - pic.kinetic_energy(B.PIC_STATE_N)[0]
        work = cfg["dt"] * dx * np.sum(jbar * 0.5 * (cfg["E_n"] + cfg["E_np1"]))
        print(f"[energy] {precision}: dK={dK:.6e} work={work:.6e} rel={(dK - work) / abs(work):.2e}")
        assert abs(dK - work) <= tol * abs(work)
        pic.close()


def test_residual_host_in_device_out_back_to_back(G):
    """pic_residual with a HOST field and a DEVICE residual returns without synchronising, and its
    field goes to the device through the handle's one pinned staging buffer.  Two such calls in a
    row, issued while the stream is still busy with earlier work, must each see their OWN field:
    the second call has to wait for the first call's copy before it rewrites the buffer
    (pic_api.cu: pin_wait)."""
    import torch
    from paper_1111_5295_b200 import binding as B
    cfg = W.config2(n=400_000)
    ng, dt = cfg["n_cells"], cfg["dt"]
    pic = B.Pic(ng, cfg["length"], cfg["species"], precision="fp32",
                stream=torch.cuda.current_stream().cuda_stream)
    pic.set_step(cfg["E_n"], dt)
    E1 = np.ascontiguousarray(cfg["E_np1"])
    E2 = np.ascontiguousarray(1.5 * cfg["E_np1"] + 0.01 * np.cos(2 * np.pi * np.arange(ng) / ng))
    R1, R2 = pic.residual(E1).copy(), pic.residual(E2).copy()      # host in, host out
    assert G.rel_l2(R1, R2) > 1e-3                                 # the two fields tell apart
    busy = torch.empty(1 << 28, dtype=torch.float32, device="cuda")   # 1 GiB
    d1 = torch.empty(ng, dtype=torch.float64, device="cuda")
    d2 = torch.empty(ng, dtype=torch.float64, device="cuda")
    for rep in range(3):
        for _ in range(12):
            busy.fill_(float(rep))              # a few ms of queued work ahead of the copies
        pic.residual(E1, resid_out=d1)          # host in, device out: no synchronisation
        pic.residual(E2, resid_out=d2)
        torch.cuda.synchronize()
        assert G.rel_l2(d1.cpu().numpy(), R1) < 1e-9, rep
        assert G.rel_l2(d2.cpu().numpy(), R2) < 1e-9, rep
    # and the host/host path right after a device-out call (same staging buffer, graph replay)
    for _ in range(12):
        busy.fill_(7.0)
    pic.residual(E1, resid_out=d1)
    assert G.rel_l2(pic.residual(E2), R2) < 1e-9
    torch.cuda.synchronize()
    assert G.rel_l2(d1.cpu().numpy(), R1) < 1e-9
    pic.close()


def test_residual_graph_not_stale_after_copy_state(G, oracle):
    """The host/host pic_residual is a CUDA graph replayed per (flags, dt, tol).  pic_copy_state
    gives the handle another state AND another sort key (here: the paper's strided order instead
    of the cell-major one), which changes launch arguments the graph holds by value: the next
    pic_residual must be captured afresh (handle epoch) and agree with the oracle from the new
    state and with the plain-launch path (device pointers) of the same handle."""
    import torch
    from paper_1111_5295_b200 import binding as B
    cfg = W.config0()
    sp, dt = cfg["species"][0], cfg["dt"]
    En, Ep = cfg["E_n"], cfg["E_np1"]
    ref = G.oracle_run(oracle, cfg)
    r1 = ref["species"][0]
    src = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision="fp64",
                flags=B.PIC_FLAG_VSORT | B.PIC_FLAG_STRIDED)
    src.move_accumulate(En, Ep, dt)
    src.commit()                                   # src's state n = the oracle's state n+1
    dst = B.Pic(cfg["n_cells"], cfg["length"], [sp], precision="fp64", flags=B.PIC_FLAG_VSORT)
    dst.set_step(Ep, dt)
    Ra = dst.residual(Ep).copy()                   # captured from the initial state
    refa = G.oracle_run(oracle, dict(cfg, E_n=Ep))
    assert G.rel_l2(Ra, oracle.residual(Ep, Ep, dt, refa["jbar"])) < 1e-10
    n0 = dst.get_stats()["n_launches"]
    dst.copy_state_from(src)
    Rb = dst.residual(Ep).copy()
    refb = G.oracle_run(oracle, dict(cfg, E_n=Ep), state=[(r1["cell"], r1["s"], r1["v"])])
    Rb_ref = oracle.residual(Ep, Ep, dt, refb["jbar"])
    assert G.rel_l2(Rb, Rb_ref) < 1e-9
    assert G.rel_l2(Ra, Rb) > 1e-6                 # the two states tell apart
    assert dst.get_stats()["n_launches"] > n0
    dE = torch.from_numpy(Ep).cuda()
    dR = torch.empty(cfg["n_cells"], dtype=torch.float64, device="cuda")
    dst.residual(dE, resid_out=dR)                 # plain launches, arguments packed now
    torch.cuda.synchronize()
    assert G.rel_l2(dR.cpu().numpy(), Rb) < 1e-12
    assert G.rel_l2(dst.residual(Ep), Rb) < 1e-12  # replay of the new graph
    src.close()
    dst.close()
