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
