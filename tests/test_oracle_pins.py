"""Pins of the ORACLE against what the paper and the mathematics fix.
CPU only.  Each pin is chosen so that a plausible mistake in oracle/pic_oracle.cpp (a dropped
term, a wrong sign or face index, a transposed operand) fails at least one of them."""
import math

import numpy as np
import pytest

from paper_1111_5295_b200 import workloads as W
from helpers import (LOOSE, continuity_residual, kappa_cap_cfg, landing_cfg, oracle_run,
                     unwrapped)


def _cfg(n_cells, length, x, v, E_n, E_np1, dt, q_over_m=-1.0, w_q=None):
    x, v = np.asarray(x, float), np.asarray(v, float)
    w_q = -length / x.size if w_q is None else w_q
    return dict(n_cells=n_cells, length=length, dt=dt, tol=1e-12,
                species=[dict(name="e", q_over_m=q_over_m, w_q=w_q, x=x, v=v)],
                E_n=np.asarray(E_n, float), E_np1=np.asarray(E_np1, float))


def _random_particles(n, length, seed=7, vth=1.0):
    return (W.uniform01(seed, 1, n) * length * (1 - 1e-12), vth * W.normal01(seed, 2, n))


# P-1 (north_star): with E = 0 free streaming is exact: X^{n+1} = X^n + v dt, v unchanged.
@pytest.mark.parametrize("mode", ["picard", "direct"])
def test_p1_free_streaming(oracle, mode):
    n_cells, length, dt = 16, 8.0, 3.7
    x, v = _random_particles(500, length)
    z = np.zeros(n_cells)
    cfg = _cfg(n_cells, length, x, v, z, z, dt)
    p = oracle.make_params(cn_mode=oracle.PICARD if mode == "picard" else oracle.DIRECT)
    r = oracle_run(oracle, cfg, p)["species"][0]
    X0, X1 = unwrapped(cfg, r)
    assert np.max(np.abs(X1 - (X0 + v * dt))) < 5e-14
    assert np.array_equal(r["v"], v)
    # E = 0: alpha = 0, so dtau = r (A-1): every sub-step but the last one is a crossing
    assert np.all(r["n_sub"] == r["n_cross"] + 1)
    # every crossing was counted: k = floor(X1/dx) - cell0 up to face landings
    assert np.all(np.abs(r["k"] - (np.floor(X1 / (length / n_cells)) - r["cell0"])) <= 1)


# P-2 (north_star): uniform E: x = x0 + v0 t + (q/m) E t^2/2, v = v0 + (q/m) E t, to rounding
# for any sub-step sequence (CN is exact for constant acceleration; Eq. 12 is its energy form).
@pytest.mark.parametrize("E0,qm", [(0.3, -1.0), (-0.7, 2.0), (0.05, 1.0 / 2000.0)])
def test_p2_uniform_field(oracle, E0, qm):
    n_cells, length, dt = 32, 10.0, 2.5
    x, v = _random_particles(800, length, seed=11)
    E = np.full(n_cells, E0)
    cfg = _cfg(n_cells, length, x, v, E, E, dt, q_over_m=qm)
    out = oracle_run(oracle, cfg)
    r = out["species"][0]
    X0, X1 = unwrapped(cfg, r)
    a = qm * E0
    assert np.max(np.abs(X1 - (X0 + v * dt + 0.5 * a * dt * dt))) < 2e-13
    assert np.max(np.abs(r["v"] - (v + a * dt))) < 2e-13
    assert out["stats"].n_sub > 3 * x.size  # adaptivity really sub-stepped


def test_p2_uses_time_centred_field(oracle):
    """A-11: the mover sees (E^n + E^{n+1})/2: (0, 2E) must act like (E, E)."""
    n_cells, length, dt = 8, 4.0, 1.0
    x, v = _random_particles(100, length, seed=3)
    E = np.full(n_cells, 0.2)
    a = oracle_run(oracle, _cfg(n_cells, length, x, v, 0 * E, 2 * E, dt))["species"][0]
    b = oracle_run(oracle, _cfg(n_cells, length, x, v, E, E, dt))["species"][0]
    assert np.array_equal(a["v"], b["v"]) and np.array_equal(a["s"], b["s"])


# P-3: Eq. 11 is the fixed point of the Picard iteration of Eq. 9-10.
def test_p3_direct_equals_picard(oracle):
    cfg = W.config0()
    pic = oracle_run(oracle, cfg, oracle.make_params(tol=1e-14, cn_mode=oracle.PICARD))
    dire = oracle_run(oracle, cfg, oracle.make_params(cn_mode=oracle.DIRECT))
    a, b = pic["species"][0], dire["species"][0]
    same = (a["n_sub"] == b["n_sub"]) & (a["n_cross"] == b["n_cross"])
    assert same.mean() > 0.999
    assert np.max(np.abs(a["v"][same] - b["v"][same])) < 1e-12
    assert np.max(np.abs(a["s"][same] - b["s"][same])) < 1e-12
    assert pic["stats"].n_picard_cap == 0
    # and directly on one sub-step: plug Eq. 11's v' back into Eq. 9-10
    recs, _ = oracle.trace_particle(64, cfg["length"], -1.0, 1.0, 5, 0.03, 0.8, cfg["E_n"],
                                    cfg["E_np1"], 0.5, oracle.make_params(cn_mode=oracle.DIRECT))
    for q in recs:
        if q.crossed == 0:
            a_mid = q.a + q.aprime * (q.dtau * (q.v0 + q.v1) / 4.0)
            assert abs((q.v1 - q.v0) - q.dtau * a_mid) < 1e-15
            assert abs((q.s1 - q.s0) - q.dtau * (q.v0 + q.v1) / 2.0) < 1e-15


# P-4: the max() of Eq. 7-8 brackets the positive root of the quadratic Eq. 6:
#   dtau_est <= root <= 2 dtau_est.
def test_p4_estimator_brackets_quadratic_root(oracle):
    rng = np.random.default_rng(5)
    for _ in range(2000):
        a, ap, v = rng.normal() * 10 ** rng.uniform(-3, 1), rng.normal(), rng.normal() * 3
        eps_a, eps_r = 10 ** rng.uniform(-10, -4), 10 ** rng.uniform(-3, -1)
        alpha = 0.5 * (abs(a) + abs(ap * v))
        beta = eps_r * (abs(a) + abs(v))
        root = (beta + math.sqrt(beta * beta + 4 * alpha * eps_a)) / (2 * alpha)
        est = oracle.estimate_dtau(a, ap, v, eps_a, eps_r)
        assert est <= root * (1 + 1e-12) and root <= 2 * est * (1 + 1e-12)
    # the two regimes separately: eps_r = 0 -> sqrt(eps_a/alpha); eps_a = 0 -> beta/alpha
    assert oracle.estimate_dtau(2.0, 0.0, 0.0, 1e-8, 0.0) == pytest.approx(1e-4, rel=1e-14)
    assert oracle.estimate_dtau(1.0, 3.0, 1.0, 0.0, 0.02) == pytest.approx(0.02, rel=1e-14)
    # A-1: a = a' = 0 gives "no limit"
    assert oracle.estimate_dtau(0.0, 0.0, 1.0, 1e-8, 0.02) > 1e100


def _multi_mode_cfg(n=3000, n_cells=32, dt=4.0, amp=0.3, seed=21):
    length = n_cells * 0.8
    x, v = _random_particles(n, length, seed=seed)
    ph = W.uniform01(seed, 3, 4) * 2 * math.pi
    E0 = W.fourier_field(n_cells, length, range(1, 5), amp, ph)
    E1 = W.fourier_field(n_cells, length, range(1, 5), amp, ph + 0.2)
    return _cfg(n_cells, length, x, v, E0, E1, dt)


# P-5: after a crossing the particle sits exactly on the face, Eq. 12 holds,
# F(dtau_c) = (a_m/2) dtau^2 + v dtau - d = 0, and dtau_c is the root bisection finds.
def test_p5_crossing_invariants(oracle):
    cfg = _multi_mode_cfg()
    n_cells, length = cfg["n_cells"], cfg["length"]
    dx = length / n_cells
    sp = cfg["species"][0]
    cell, s = oracle.bin_particles(n_cells, length, sp["x"])
    ncheck = 0
    for p in range(0, 300):
        recs, fin = oracle.trace_particle(n_cells, length, sp["q_over_m"], sp["w_q"], cell[p],
                                          s[p], sp["v"][p], cfg["E_n"], cfg["E_np1"], cfg["dt"])
        assert sum(q.dtau for q in recs) == pytest.approx(cfg["dt"], rel=1e-12)
        for i, q in enumerate(recs):
            assert 0.0 <= q.dtau <= q.dtau_est * (1 + 1e-15) + 1e-300
            if q.crossed == 0:
                assert 0.0 <= q.s1 <= dx
                continue
            ncheck += 1
            assert q.s1 == (dx if q.crossed > 0 else 0.0)
            d = q.s1 - q.s0
            assert q.v1 * q.crossed >= 0.0
            assert q.v1 ** 2 - q.v0 ** 2 == pytest.approx(2 * q.a_mid * d, abs=1e-13)
            F = lambda t: 0.5 * q.a_mid * t * t + q.v0 * t - d
            assert abs(F(q.dtau)) < 1e-13
            # bisection for the FIRST root of F in (0, tentative dtau]
            if d != 0.0:
                lo, hi = 0.0, q.dtau * (1 + 1e-9) + 1e-15
                if F(lo) * F(hi) < 0:
                    for _ in range(200):
                        mid = 0.5 * (lo + hi)
                        lo, hi = (mid, hi) if F(lo) * F(mid) > 0 else (lo, mid)
                    assert q.dtau == pytest.approx(0.5 * (lo + hi), abs=1e-11)
            # the next sub-step starts on the near face of the neighbouring cell
            if i + 1 < len(recs):
                nxt = recs[i + 1]
                assert nxt.cell == (q.cell + q.crossed) % n_cells
                assert nxt.s0 == (0.0 if q.crossed > 0 else dx) and nxt.v0 == q.v1
    assert ncheck > 500


# P-6 (north_star): discrete continuity per cell,
#   rho^{n+1}_c - rho^n_c + dt (jbar_{c+1} - jbar_c)/dx = 0, for ANY E, dt, tolerances.
@pytest.mark.parametrize("eps_r,tol", [(0.02, 1e-10), (0.3, 1e-2)])
def test_p6_continuity_per_cell(oracle, eps_r, tol):
    cfg = _multi_mode_cfg(dt=6.0)
    out = oracle_run(oracle, cfg, oracle.make_params(eps_r=eps_r, tol=tol))
    r = out["species"][0]
    res, div = continuity_residual(oracle, cfg, [(r["cell0"], r["s0"])], [(r["cell"], r["s"])],
                                   out["jbar"])
    assert np.linalg.norm(div) > 1e-3
    assert np.linalg.norm(res) / np.linalg.norm(div) < 1e-12
    assert out["stats"].n_cross > r["v"].size


# P-7: jbar depends only on the unwrapped end points: J_f = w_q sum_images
#   [G(X1 - x_f) - G(X0 - x_f)],  G(y) = int_{-inf}^{y} S1  (S1 = hat of half-width dx).
def _G(y, dx):
    y = np.clip(y, -dx, dx)
    return np.where(y <= 0, (dx + y) ** 2 / (2 * dx), dx - (dx - y) ** 2 / (2 * dx))


def test_p7_endpoint_formula_and_p8_mean_current(oracle):
    cfg = _multi_mode_cfg(n=400, n_cells=12, dt=9.0)
    out = oracle_run(oracle, cfg)
    r = out["species"][0]
    X0, X1 = unwrapped(cfg, r)
    n_cells, length = cfg["n_cells"], cfg["length"]
    dx = length / n_cells
    w_q = cfg["species"][0]["w_q"]
    J = np.zeros(n_cells)
    m_lo = int(math.floor(min(X0.min(), X1.min()) / length)) - 1
    m_hi = int(math.ceil(max(X0.max(), X1.max()) / length)) + 1
    for f in range(n_cells):
        for m in range(m_lo, m_hi + 1):
            xf = f * dx + m * length
            J[f] += w_q * np.sum(_G(X1 - xf, dx) - _G(X0 - xf, dx))
    assert np.max(np.abs(J - out["J"])) < 1e-12 * max(1.0, np.abs(J).max())
    assert np.abs(r["k"]).max() >= 3
    # P-8: sum_f J_f = w_q sum_p (X1 - X0)
    assert out["J"].sum() == pytest.approx(w_q * np.sum(X1 - X0), abs=1e-12)


# P-9: per-call energy identity, for any given E:
#   sum_p w_m (v1^2 - v0^2)/2 = dt dx sum_f jbar_f E^{n+1/2}_f.
@pytest.mark.parametrize("mode", ["picard", "direct"])
def test_p9_energy_identity(oracle, mode):
    cfg = _multi_mode_cfg(dt=5.0, amp=0.5)
    p = oracle.make_params(tol=1e-13, cn_mode=oracle.PICARD if mode == "picard" else oracle.DIRECT)
    out = oracle_run(oracle, cfg, p)
    sp, r = cfg["species"][0], out["species"][0]
    w_m = sp["w_q"] / sp["q_over_m"]
    dK = 0.5 * w_m * np.sum(r["v"] ** 2 - r["v0"] ** 2)
    dx = cfg["length"] / cfg["n_cells"]
    work = cfg["dt"] * dx * np.sum(out["jbar"] * 0.5 * (cfg["E_n"] + cfg["E_np1"]))
    assert abs(dK) > 1e-4
    assert abs(dK - work) < 1e-12 * max(abs(dK), 1.0)


# P-10: refinement.  Two cells, E = (+e, -e) on the faces, q/m = +1: inside cell 0 the
# acceleration is a(s) = e - 2 e s/dx, a harmonic oscillator about s = dx/2 with
# omega^2 = 2e/dx (textbook special case of the piecewise-linear field); CN is 2nd order, so
# (eps_r, eps_a) -> (eps_r/2, eps_a/4) must cut the error ~4x.
def test_p10_refinement_to_harmonic_oscillator(oracle):
    e, dx, dt = 0.4, 1.0, 7.0
    om = math.sqrt(2 * e / dx)
    s0, v0 = 0.5 + 0.2, 0.1
    exact_s = 0.5 + 0.2 * math.cos(om * dt) + v0 / om * math.sin(om * dt)
    exact_v = -0.2 * om * math.sin(om * dt) + v0 * math.cos(om * dt)
    errs = []
    for lvl in range(4):
        p = oracle.make_params(eps_r=0.02 / 2 ** lvl, eps_a=1e-8 / 4 ** lvl, tol=1e-14)
        recs, fin = oracle.trace_particle(2, 2 * dx, 1.0, 1.0, 0, s0, v0, [e, -e], [e, -e], dt, p)
        assert fin["cell"] == 0 and all(q.crossed == 0 for q in recs)
        errs.append(math.hypot(fin["s"] - exact_s, fin["v"] - exact_v))
    assert errs[0] < 1e-2
    for a, b in zip(errs, errs[1:]):
        assert 3.0 < a / b < 5.5, errs


def test_p10_refinement_multi_cell_vs_ode(oracle):
    """Many cells, crossings included: converge to a high-accuracy ODE solution of
    x' = v, v' = (q/m) E_half(x), E_half piecewise linear (scipy DOP853, rtol 1e-12)."""
    from scipy.integrate import solve_ivp
    n_cells, length, dt, qm = 16, 8.0, 3.0, -1.0
    dx = length / n_cells
    xf = np.arange(n_cells + 1) * dx
    E = 0.3 * np.sin(2 * math.pi * xf[:-1] / length) + 0.1 * np.cos(4 * math.pi * xf[:-1] / length)
    Ew = np.append(E, E[0])
    rhs = lambda t, y: [y[1], qm * np.interp(y[0] % length, xf, Ew)]
    starts = [(1.3, 0.9), (6.1, -1.4), (3.9, 0.2)]
    errs = []
    for lvl in (0, 2):
        p = oracle.make_params(eps_r=0.02 / 2 ** lvl, eps_a=1e-8 / 4 ** lvl, tol=1e-14)
        err = 0.0
        for x0, v0 in starts:
            ref = solve_ivp(rhs, (0, dt), [x0, v0], method="DOP853", rtol=1e-12, atol=1e-13,
                            max_step=0.01).y[:, -1]
            c0 = int(x0 // dx)
            _, fin = oracle.trace_particle(n_cells, length, qm, 1.0, c0, x0 - c0 * dx, v0, E, E,
                                           dt, p)
            X1 = (c0 + fin["k"]) * dx + fin["s"]
            err = max(err, abs(X1 - ref[0]), abs(fin["v"] - ref[1]))
        errs.append(err)
    assert errs[0] < 5e-3 and 8.0 < errs[0] / errs[1] < 24.0, errs


# P-11: hand-stepped tiny cases (tests/golden/p11_hand_cases.txt).
def test_p11_hand_cases(oracle):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "p11_hand_cases.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(rows) == 2
    for name, x0, v0, E0, dt, x1, v1, *J in rows:
        x0, v0, E0, dt, x1, v1 = map(float, (x0, v0, E0, dt, x1, v1))
        J = np.array(list(map(float, J)))
        E = np.full(4, E0)
        for mode in (oracle.PICARD, oracle.DIRECT):
            recs, fin = oracle.trace_particle(4, 4.0, 1.0, 1.0, 0, x0, v0, E, E, dt,
                                              oracle.make_params(tol=1e-15, cn_mode=mode))
            assert fin["k"] + fin["s"] == pytest.approx(x1, abs=1e-14)
            assert fin["v"] == pytest.approx(v1, abs=1e-14)
            assert np.max(np.abs(fin["J"] - J)) < 1e-14
            if name == "free":
                assert [q.crossed for q in recs] == [1, 1, 0]
                assert [q.dtau for q in recs] == pytest.approx([0.5, 2 / 3, 1 / 3], abs=1e-15)
                assert [q.cell for q in recs] == [0, 1, 2]
            else:
                first = next(q for q in recs if q.crossed)
                assert sum(q.dtau for q in recs[:recs.index(first) + 1]) == pytest.approx(1.0, abs=1e-13)
                assert first.v1 == pytest.approx(1.0, abs=1e-13)


def test_p11_leftward_and_wraparound(oracle):
    """Mirror image: moving left through face 0 wraps to cell n_cells-1, deposits on the
    mirrored faces, k goes negative."""
    z = np.zeros(4)
    recs, fin = oracle.trace_particle(4, 4.0, 1.0, 1.0, 0, 0.75, -1.5, z, z, 1.5)
    assert fin["cell"] == 2 and fin["k"] == -2 and fin["s"] == pytest.approx(0.5)
    # by hand: cell 0, delta=-0.75, w_R=0.375: J1 -= 0.28125, J0 -= 0.46875; cell 3, delta=-1:
    # J0 -= 0.5, J3 -= 0.5; cell 2, delta=-0.5, w_R=0.75: J3 -= 0.375, J2 -= 0.125.
    assert np.max(np.abs(fin["J"] + np.array([0.96875, 0.28125, 0.125, 0.875]))) < 1e-15
    assert [q.cell for q in recs] == [0, 3, 2]


def test_a5_particle_on_face(oracle):
    """A-5: a particle sitting on its cell's right face moving right makes a zero-length
    crossing first; total displacement is unaffected."""
    z = np.zeros(4)
    recs, fin = oracle.trace_particle(4, 4.0, 1.0, 1.0, 1, 1.0, 0.5, z, z, 1.0)
    assert recs[0].crossed == 1 and recs[0].dtau == 0.0
    assert fin["cell"] == 2 and fin["s"] == pytest.approx(0.5) and fin["J"].sum() == pytest.approx(0.5)


# P-12: sum_f R_f = sum_f (E^{n+1}_f - E^n_f)/dt exactly (the mean of jbar is removed), and R
# is the Ampere residual of the north_star for a hand-made jbar.
def test_p12_residual(oracle):
    rng = np.random.default_rng(2)
    E0, E1, jb = rng.normal(size=16), rng.normal(size=16), rng.normal(size=16) + 3.0
    R = oracle.residual(E0, E1, 0.25, jb)
    assert R.sum() == pytest.approx(np.sum(E1 - E0) / 0.25, abs=1e-12)
    assert R[3] == pytest.approx((E1[3] - E0[3]) / 0.25 + jb[3] - jb.mean(), abs=1e-14)
    assert np.allclose(oracle.residual(E0, E0, 1.0, np.full(16, 7.0)), 0.0, atol=1e-14)


def test_rho_quadratic_spline_partition_of_unity(oracle):
    """O11/A-10: S2 sums to 1 over cells (total charge), and is the exact hand values at
    s = 0, dx/2: (1/2, 1/2, 0) and (1/8, 3/4, 1/8)."""
    dx = 0.5
    rho = oracle.rho(8, 4.0, 2.0, np.array([3, 5]), np.array([0.0, dx / 2]))
    assert rho.sum() * dx == pytest.approx(4.0)
    assert rho[2] * dx == pytest.approx(1.0) and rho[3] * dx == pytest.approx(1.0)
    assert rho[4] * dx == pytest.approx(0.25) and rho[5] * dx == pytest.approx(1.5)
    assert rho[6] * dx == pytest.approx(0.25)


def test_workload_shape_cfg0(oracle):
    """cfg0 statistics the survey's probe found: ~6.1 sub-steps/particle, ~66 % crossings."""
    out = oracle_run(oracle, W.config0())
    st = out["stats"]
    assert 5.5 < st.n_sub / 6400 < 6.8 and 0.55 < st.n_cross / st.n_sub < 0.75
    assert st.n_kappa_cap == st.n_substep_cap == st.n_neg_disc == st.n_picard_cap == 0


# ---- oracle_bin (x -> cell, s): the start state of every other pin ------------------------------
def test_oracle_bin(oracle):
    """cell*dx + s == x to rounding, 0 <= s <= dx, cell in range; exact hand values on a grid
    whose dx is a power of two; the edges x = 0, a face, nextafter(L, 0)."""
    n_cells, length = 8, 4.0                       # dx = 0.5: everything below is exact
    x = np.array([0.0, 0.5, 1.25, 3.5, np.nextafter(4.0, 0.0), 0.4999999999999999, 2.0])
    cell, s = oracle.bin_particles(n_cells, length, x)
    assert cell.tolist() == [0, 1, 2, 7, 7, 0, 4]
    assert s.tolist() == [0.0, 0.0, 0.25, 0.0, np.nextafter(4.0, 0.0) - 3.5, 0.4999999999999999, 0.0]
    # a grid whose dx is not representable: the identity and the bounds, to rounding
    n_cells, length = 4096, 4096 * (100.0 * math.pi / 256.0)
    dx = length / n_cells
    rng = np.random.default_rng(4)
    x = np.concatenate([rng.uniform(0, length, 20000), np.arange(n_cells) * dx,
                        np.nextafter(np.arange(1, n_cells + 1) * dx, 0.0), [0.0]])
    x = np.minimum(x, np.nextafter(length, 0.0))
    cell, s = oracle.bin_particles(n_cells, length, x)
    assert cell.min() >= 0 and cell.max() <= n_cells - 1
    assert s.min() >= 0.0 and s.max() <= dx
    assert np.max(np.abs(cell * dx + s - x)) <= 2 * np.spacing(length)
    # a plausible slip (cell = round or ceil, s measured from the wrong face) moves s by ~dx
    frac = x / dx - np.floor(x / dx)
    assert np.max(np.abs(s / dx - frac)) < 1e-9
    # x on a face may bin into either neighbour (A-5: s = 0 or s = dx), never elsewhere
    faces = np.arange(n_cells) * dx
    c2, s2 = oracle.bin_particles(n_cells, length, faces)
    ok = ((c2 == np.arange(n_cells)) & (s2 < 1e-9)) | ((c2 == np.arange(n_cells) - 1) & (dx - s2 < 1e-9))
    assert ok.all()


# ---- guard branches (SURVEY A-2, A-3, O7): workloads on which they EXECUTE, checked against
# what the mathematics still fixes when they do -------------------------------------------------
def test_guard_kappa_cap_binds(oracle):
    """A-2: dtau <= sqrt(4 kappa_max/|a'|).  With loose estimator tolerances the cap binds on
    most sub-steps; then 1 - kappa stays in [0.5, 1.5] (Eq. 11's denominator), every
    orbit still uses up exactly dt, the crossing solve keeps a real root in (0, dtau] (no
    discriminant or crossing-time clamp), and continuity (P-6) and the energy identity (P-9)
    hold to rounding -- they do not depend on the step sizes."""
    cfg = kappa_cap_cfg()
    for mode in (oracle.PICARD, oracle.DIRECT):
        p = oracle.make_params(cn_mode=mode, tol=1e-14, **LOOSE)
        out = oracle_run(oracle, cfg, p)
        st, r, sp = out["stats"], out["species"][0], cfg["species"][0]
        assert st.n_kappa_cap > 0.5 * st.n_sub and st.n_neg_disc == 0 and st.n_clamped_tau == 0
        assert st.n_picard_cap == 0 and st.n_substep_cap == 0
        res, div = continuity_residual(oracle, cfg, [(r["cell0"], r["s0"])],
                                       [(r["cell"], r["s"])], out["jbar"])
        assert np.linalg.norm(res) < 1e-12 * np.linalg.norm(div)
        w_m = sp["w_q"] / sp["q_over_m"]
        dK = 0.5 * w_m * np.sum(r["v"] ** 2 - r["v0"] ** 2)
        dx = cfg["length"] / cfg["n_cells"]
        work = cfg["dt"] * dx * np.sum(out["jbar"] * 0.5 * (cfg["E_n"] + cfg["E_np1"]))
        assert abs(dK) > 1e-3 and abs(dK - work) < 1e-11 * abs(dK)
        # per sub-step, on traced orbits
        capped = binding = 0
        for i in range(60):
            recs, _ = oracle.trace_particle(cfg["n_cells"], cfg["length"], sp["q_over_m"],
                                            sp["w_q"], r["cell0"][i], r["s0"][i], r["v0"][i],
                                            cfg["E_n"], cfg["E_np1"], cfg["dt"], p)
            assert sum(q.dtau for q in recs) == pytest.approx(cfg["dt"], rel=1e-13)
            for q in recs:
                assert abs(q.aprime) * q.dtau ** 2 / 4.0 <= 0.5 * (1 + 1e-15)
                if q.aprime != 0.0:
                    cap = math.sqrt(4.0 * 0.5 / abs(q.aprime))
                    binding += q.dtau_est > cap
                    if q.crossed == 0 and q.dtau_est > cap and q.dtau == cap:
                        capped += 1            # an accepted step of exactly the cap's length
                    assert q.dtau <= cap
                if q.crossed:           # the truncated step satisfies Eq. 12 and F(dtau_c) = 0
                    d = q.s1 - q.s0
                    assert q.v1 ** 2 - q.v0 ** 2 == pytest.approx(2 * q.a_mid * d, abs=1e-12)
                    assert abs(0.5 * q.a_mid * q.dtau ** 2 + q.v0 * q.dtau - d) < 1e-12
        assert capped > 50 and binding > 300
    # the cap is what keeps Eq. 11 finite: without it (kappa_max -> 1) 1 - kappa reaches ~0
    # for a' > 0 and the same workload trips the crossing guards
    wild = oracle_run(oracle, cfg, oracle.make_params(cn_mode=oracle.DIRECT, kappa_max=0.999999,
                                                      **LOOSE))
    assert wild["stats"].n_kappa_cap < out["stats"].n_kappa_cap


@pytest.mark.parametrize("kind", ["land", "turn"])
def test_guard_crossing_clamps(oracle, kind):
    """O7 guards: D = v^2 + 2 a_m d clamped at 0 and dtau_c clamped to [0, dtau].  In exact
    arithmetic neither can bind (SURVEY A-2: F(dtau) has the sign of the overshoot), so they
    are reached only through rounding: particles that in exact arithmetic END the step exactly
    on a face (helpers.landing_cfg).  Whichever branch rounding picks -- in-cell landing on the
    face, crossing, crossing with a clamp -- the uniform-field closed form (P-2) fixes the
    result: X1 = the face, v1 = v0 + a dt; and continuity / energy hold to rounding."""
    tot = dict(n_neg_disc=0, n_clamped_tau=0, n_cross=0)
    for seed in range(6):
        for dt in (1.0, 0.7, 1.9):
            cfg, state, (X1, v1) = landing_cfg(kind, dt=dt, seed=seed)
            for mode in (oracle.PICARD, oracle.DIRECT):
                out = oracle_run(oracle, cfg, oracle.make_params(cn_mode=mode, eps_a=1.0, eps_r=1.0),
                                 state=state)
                st, r = out["stats"], out["species"][0]
                for k in tot:
                    tot[k] += getattr(st, k)
                _, X = unwrapped(cfg, r)
                assert np.max(np.abs(X - X1)) < 4e-15
                # 'turn': v1 = 0 is a square root of a rounding error (sensitivity of Eq. 12 at
                # the apex), so |v1| ~ 1e-8; 'land': v1 to rounding
                assert np.max(np.abs(r["v"] - v1)) < (2e-7 if kind == "turn" else 4e-15)
                assert st.n_sub < 2.01 * X1.size and st.n_substep_cap == 0
                res, div = continuity_residual(oracle, cfg, [(r["cell0"], r["s0"])],
                                               [(r["cell"], r["s"])], out["jbar"])
                assert np.max(np.abs(res)) < 1e-13
                sp = cfg["species"][0]
                dK = 0.5 * sp["w_q"] / sp["q_over_m"] * np.sum(r["v"] ** 2 - r["v0"] ** 2)
                work = cfg["dt"] * np.sum(out["jbar"] * cfg["E_n"])
                assert abs(dK - work) < 1e-12 * max(abs(dK), 1.0)
    assert tot["n_cross"] > 1000                      # about half overshoot the face
    # per sub-step: no step is longer than the time that was left (the dtau_c clamp), the
    # discriminant's root is real (v1 finite), and the time adds up
    cfg, state, _ = landing_cfg(kind, dt=0.7, seed=1)
    sp, (cells, s0, v0) = cfg["species"][0], state[0]
    p = oracle.make_params(cn_mode=oracle.DIRECT, eps_a=1.0, eps_r=1.0)
    for i in range(cells.size):
        recs, _ = oracle.trace_particle(cfg["n_cells"], cfg["length"], sp["q_over_m"], sp["w_q"],
                                        cells[i], s0[i], v0[i], cfg["E_n"], cfg["E_np1"], 0.7, p)
        left = 0.7
        for q in recs:
            assert 0.0 <= q.dtau <= left and math.isfinite(q.v1) and math.isfinite(q.s1)
            left = 0.0 if q.dtau == left else left - q.dtau
        assert left == 0.0
    if kind == "land":
        assert tot["n_clamped_tau"] > 50, tot         # the dtau_c clamp executed
    else:
        assert tot["n_neg_disc"] > 0, tot             # the D < 0 clamp executed


def test_guard_picard_cap(oracle):
    """A-3: the Picard loop stops after picard_max iterations.  With picard_max = 1 and tol = 0
    every sub-step is cut off after its first iterate, which is the explicit midpoint rule
    v' = v + dtau a(s + dtau v/2): checked by hand per sub-step.  With picard_max = k the error
    against the converged step shrinks like |kappa|^k (contraction factor of Eq. 9-10).
    Continuity (P-6) is exact whatever the iteration does."""
    cfg = kappa_cap_cfg(n=600)
    sp = cfg["species"][0]
    p1 = oracle.make_params(cn_mode=oracle.PICARD, tol=0.0, picard_max=1)
    out = oracle_run(oracle, cfg, p1)
    st, r = out["stats"], out["species"][0]
    assert st.n_picard_cap == st.n_sub == st.n_picard_it
    res, div = continuity_residual(oracle, cfg, [(r["cell0"], r["s0"])], [(r["cell"], r["s"])],
                                   out["jbar"])
    assert np.linalg.norm(res) < 1e-12 * np.linalg.norm(div)
    n = 0
    for i in range(20):
        recs, _ = oracle.trace_particle(cfg["n_cells"], cfg["length"], sp["q_over_m"], sp["w_q"],
                                        r["cell0"][i], r["s0"][i], r["v0"][i], cfg["E_n"],
                                        cfg["E_np1"], cfg["dt"], p1)
        for q in recs:
            if q.crossed == 0:
                v1 = q.v0 + q.dtau * (q.a + q.aprime * (q.dtau * q.v0 / 2.0))
                assert q.v1 == pytest.approx(v1, abs=1e-15 * max(1.0, abs(v1)))
                assert q.s1 - q.s0 == pytest.approx(q.dtau * (q.v0 + v1) / 2.0, abs=1e-15)
                n += 1
    assert n > 1000
    # convergence with the cap: one orbit segment, same dtau sequence forced by one sub-step
    recs = {}
    for k in (1, 2, 3, 50):
        p = oracle.make_params(cn_mode=oracle.PICARD, tol=0.0 if k < 50 else 1e-15, picard_max=k,
                               eps_a=1.0, eps_r=0.9)
        rec, _ = oracle.trace_particle(2, 2.0, 1.0, 1.0, 0, 0.5, 0.1, [0.2, -0.2], [0.2, -0.2],
                                       0.5, p)
        assert len(rec) == 1 and rec[0].crossed == 0 and rec[0].dtau == 0.5
        recs[k] = rec[0].v1
    kappa = abs(-0.4 * 0.5 ** 2 / 4.0)
    e = [abs(recs[k] - recs[50]) for k in (1, 2, 3)]
    assert e[0] > 1e-6 and e[1] == pytest.approx(kappa * e[0], rel=1e-6)
    assert e[2] == pytest.approx(kappa * e[1], rel=1e-4)


def test_guard_substep_cap(oracle):
    """A-9: an orbit that has taken max_substeps sub-steps with time left is aborted and counted.
    The aborted orbit is exactly the first max_substeps sub-steps of the uncapped one (prefix
    property, from the trace), the count is the number of particles that needed more, and
    continuity (P-6) still holds to rounding: the deposit matches the distance actually
    travelled, whether or not dt was used up."""
    cfg = _multi_mode_cfg(n=800, dt=6.0)
    sp = cfg["species"][0]
    free = oracle_run(oracle, cfg)
    need = free["species"][0]["n_sub"]
    cap = int(np.median(need))
    assert need.min() < cap < need.max()
    out = oracle_run(oracle, cfg, oracle.make_params(tol=cfg["tol"], max_substeps=cap))
    r, st = out["species"][0], out["stats"]
    assert st.n_substep_cap == int((need > cap).sum()) > 100
    assert np.all(r["n_sub"] == np.minimum(need, cap))
    # untouched by the cap where it does not bind
    ok = need <= cap
    f = free["species"][0]
    assert np.array_equal(r["v"][ok], f["v"][ok]) and np.array_equal(r["s"][ok], f["s"][ok])
    # prefix property on the aborted ones
    for i in np.nonzero(~ok)[0][:40]:
        recs, _ = oracle.trace_particle(cfg["n_cells"], cfg["length"], sp["q_over_m"], sp["w_q"],
                                        r["cell0"][i], r["s0"][i], r["v0"][i], cfg["E_n"],
                                        cfg["E_np1"], cfg["dt"], oracle.make_params(tol=cfg["tol"]))
        q = recs[cap - 1]
        assert sum(t.dtau for t in recs[:cap]) < cfg["dt"]
        assert r["v"][i] == q.v1
        n_cells = cfg["n_cells"]
        dx = cfg["length"] / n_cells
        if q.crossed:       # the record ends on the face; the state has entered the neighbour
            assert r["cell"][i] == (q.cell + q.crossed) % n_cells
            assert r["s"][i] == (0.0 if q.crossed > 0 else dx)
        else:
            assert r["cell"][i] == q.cell and r["s"][i] == q.s1
    res, div = continuity_residual(oracle, cfg, [(r["cell0"], r["s0"])], [(r["cell"], r["s"])],
                                   out["jbar"])
    assert np.linalg.norm(res) < 1e-12 * np.linalg.norm(div)
