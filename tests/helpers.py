"""Shared test utilities: run the ORACLE on a workload dict and the parity metrics of
SURVEY.md 8(c).  Nothing here is used by the product path."""
import numpy as np


def oracle_run(o, cfg, params=None, state=None):
    """All species of `cfg` through the oracle.  `state` optionally overrides the per-species
    (cell, s, v) start state (fp32-rounded inputs).  Returns per-species results + jbar."""
    n_cells, length, dt = cfg["n_cells"], cfg["length"], cfg["dt"]
    params = params or o.make_params(tol=cfg.get("tol", 1e-10))
    J = np.zeros(n_cells)
    stats = o.Stats()
    res = []
    for j, sp in enumerate(cfg["species"]):
        if state is None:
            cell0, s0 = o.bin_particles(n_cells, length, sp["x"])
            v0 = sp["v"]
        else:
            cell0, s0, v0 = state[j]
        r = o.move_accumulate(n_cells, length, sp["q_over_m"], sp["w_q"], cell0, s0, v0,
                              cfg["E_n"], cfg["E_np1"], dt, params, J=J, stats=stats)
        r.update(cell0=np.asarray(cell0), s0=np.asarray(s0), v0=np.asarray(v0))
        res.append(r)
    return dict(species=res, J=J, jbar=o.jbar_from_J(n_cells, length, dt, J), stats=stats)


def unwrapped(cfg, r):
    """(X0, X1) unwrapped positions from (cell0, s0) and (k, s1)."""
    dx = cfg["length"] / cfg["n_cells"]
    X0 = r["cell0"] * dx + r["s0"]
    X1 = (r["cell0"].astype(np.int64) + r["k"]) * dx + r["s"]
    return X0, X1


def rel_l2(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    den = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (den if den > 0 else 1.0)


def periodic_dist(xa, xb, length):
    d = np.abs(np.asarray(xa, np.float64) - np.asarray(xb, np.float64))
    return np.minimum(d, length - d)


def continuity_residual(o, cfg, start, end, jbar):
    """rho^{n+1}_c - rho^n_c + dt (jbar_{c+1} - jbar_c)/dx per cell (north_star), rho by
    the oracle's O11 in fp64.  start/end: per-species lists of (cell, s)."""
    n_cells, length, dt = cfg["n_cells"], cfg["length"], cfg["dt"]
    dx = length / n_cells
    rho0, rho1 = np.zeros(n_cells), np.zeros(n_cells)
    for sp, (c0, s0), (c1, s1) in zip(cfg["species"], start, end):
        o.rho(n_cells, length, sp["w_q"], c0, s0, rho0)
        o.rho(n_cells, length, sp["w_q"], c1, s1, rho1)
    div = dt * (np.roll(jbar, -1) - jbar) / dx
    return rho1 - rho0 + div, div


def round_to_fp32_state(cfg):
    """For fp32 parity runs both sides get fp32-representable inputs: returns,
    per species, cell = floor(x/dx), xi = fp32(x/dx - cell) (in-cell offset in cell units) and
    v = fp32(v).  Pure representation change; no method arithmetic."""
    dx = cfg["length"] / cfg["n_cells"]
    out = []
    for sp in cfg["species"]:
        u = sp["x"] / dx
        cell = np.clip(np.floor(u), 0, cfg["n_cells"] - 1).astype(np.int32)
        xi = np.clip(u - cell, 0.0, 1.0).astype(np.float32)
        out.append(dict(cell=cell, xi=xi, v=sp["v"].astype(np.float32)))
    return out


# ---- workloads that EXECUTE the guard branches of the mover ----------
# Input design only (kinematics of a uniformly accelerated particle); no arithmetic of the method.
def kappa_cap_cfg(n=4000, seed=9):
    """Strong, short-wavelength field and slow particles: with loose estimator tolerances the
    A-2 cap dtau <= sqrt(4 kappa_max/|a'|) binds on most sub-steps (a' of both signs)."""
    import math
    from paper_1111_5295_b200 import workloads as W
    n_cells, length = 16, 8.0
    xf = W.face_positions(n_cells, length)
    E = 3.0 * np.sin(2 * math.pi * xf / length) + 2.0 * np.cos(6 * math.pi * xf / length)
    x = W.uniform01(seed, 1, n) * length * (1 - 1e-12)
    v = 0.3 * W.normal01(seed, 2, n)
    return dict(n_cells=n_cells, length=length, dt=6.0, tol=1e-12, E_n=E, E_np1=0.8 * E,
                species=[dict(name="e", q_over_m=-1.0, w_q=-length / n, x=x, v=v)])


LOOSE = dict(eps_a=1.0, eps_r=0.9)      # estimator tolerances under which the cap binds


def landing_cfg(kind, n_cells=4096, dt=1.0, seed=3, q_over_m=-1.0):
    """Rounding-coincidence workload for the crossing guards (O7: D < 0 clamp, dtau_c clamp).
    dx = 1.  Every even cell c carries a UNIFORM field (faces c and c+1 equal) and one particle
    that moves towards its right (c % 4 == 0) or left (c % 4 == 2) face at distance `dist`, with
    the field chosen so that in exact arithmetic it is exactly ON that face at t = dt:
      kind 'land': arrives with a random non-zero velocity (a = 2 (dist - v0 dt)/dt^2);
      kind 'turn': arrives with v = 0, the apex of its parabola (v0 = 2 dist/dt, a = -v0/dt).
    With estimator tolerances eps_a = eps_r = 1 the whole dt is ONE tentative sub-step, which
    lands within an ulp or two of the face: about half the particles overshoot it and take the
    crossing branch with a discriminant / crossing time within rounding of its bound.
    `dist` is a multiple of 2^-30 so that x = cell + s is exact in fp64 (and xi in the kernel).
    Returns (cfg, state, closed_form) with closed_form = (X1 unwrapped, v1)."""
    rng = np.random.default_rng(seed)
    m = n_cells // 2
    sgn = np.where(np.arange(m) % 2 == 0, 1.0, -1.0)
    dist = np.round(rng.uniform(0.1, 0.9, m) * 2.0 ** 30) / 2.0 ** 30
    if kind == "turn":
        v0 = 2.0 * dist / dt
        a = -v0 / dt
    else:
        v0 = rng.uniform(0.2, 1.5, m) * dist / dt
        a = 2.0 * (dist - v0 * dt) / dt ** 2
    v0, a = sgn * v0, sgn * a
    E = np.zeros(n_cells)
    E[0::2] = a / q_over_m
    E[1::2] = a / q_over_m
    cells = np.arange(0, n_cells, 2).astype(np.int32)
    s0 = np.where(sgn > 0, 1.0 - dist, dist)
    x = cells + s0
    assert np.array_equal(x - cells, s0)
    cfg = dict(n_cells=n_cells, length=float(n_cells), dt=dt, tol=1e-12, E_n=E, E_np1=E.copy(),
               species=[dict(name="e", q_over_m=q_over_m, w_q=-float(n_cells) / m, x=x, v=v0)])
    X1 = cells + np.where(sgn > 0, 1.0, 0.0)
    return cfg, [(cells, s0, v0)], (X1, v0 + a * dt)


def ulp_response(o, cfg, seed=1, fp64=False):
    """How much the METHOD amplifies one rounding error (cfg3): run the oracle
    (fp64) twice from inputs that differ by one ulp in every particle's velocity (random sign) --
    one fp32 ulp from fp32-representable inputs, or with fp64=True one fp64 ulp from the fp64
    inputs -- and return the relative L2 response of x, v (over the particles that took the same
    branches) and jbar, the max-norm responses in the units of the parity metrics (xi_max: cells,
    v_max: relative to the rms speed), plus the mean sub-steps per particle.  A kernel of that
    precision makes such an error at every one of its n_sub sub-steps, so its distance from the
    oracle is about response x sqrt(n_sub) (random walk) whatever its arithmetic."""
    dx = cfg["length"] / cfg["n_cells"]
    rng = np.random.default_rng(seed)
    st0, st1 = [], []
    if fp64:
        for sp in cfg["species"]:
            c, s = o.bin_particles(cfg["n_cells"], cfg["length"], sp["x"])
            v0 = np.asarray(sp["v"], np.float64)
            toward = np.where(rng.random(v0.size) < 0.5, -np.inf, np.inf)
            st0.append((c, s, v0))
            st1.append((c, s, np.nextafter(v0, toward)))
    else:
        for r in round_to_fp32_state(cfg):
            s = r["xi"].astype(np.float64) * dx
            toward = np.where(rng.random(r["v"].size) < 0.5, -np.inf, np.inf).astype(np.float32)
            v1 = np.nextafter(r["v"], toward)
            st0.append((r["cell"], s, r["v"].astype(np.float64)))
            st1.append((r["cell"], s, v1.astype(np.float64)))
    p = o.make_params(cn_mode=o.DIRECT)
    a, b = oracle_run(o, cfg, p, state=st0), oracle_run(o, cfg, p, state=st1)
    out = dict(x=0.0, v=0.0, flips=0, xi_max=0.0, v_max=0.0)
    for ra, rb in zip(a["species"], b["species"]):
        same = (ra["n_sub"] == rb["n_sub"]) & (ra["n_cross"] == rb["n_cross"]) & \
               (ra["cell"] == rb["cell"])
        out["flips"] += int((~same).sum())
        xa = ra["cell"] * dx + ra["s"]
        d = periodic_dist(xa[same], (rb["cell"] * dx + rb["s"])[same], cfg["length"])
        out["x"] = max(out["x"], float(np.linalg.norm(d) / np.linalg.norm(xa[same])))
        out["v"] = max(out["v"], rel_l2(rb["v"][same], ra["v"][same]))
        vrms = float(np.sqrt(np.mean(ra["v"] ** 2)))
        out["xi_max"] = max(out["xi_max"], float(d.max() / dx))
        out["v_max"] = max(out["v_max"], float(np.max(np.abs(rb["v"][same] - ra["v"][same])) / vrms))
    out["j"] = rel_l2(b["jbar"], a["jbar"])
    n = sum(r["n_sub"].size for r in a["species"])
    out["n_sub_mean"] = a["stats"].n_sub / n
    return out
