"""`-m gpu`: the guard branches of the mover on the CUDA path (SURVEY 8(c) A-2 kappa cap, A-3
Picard cap, O7 discriminant / crossing-time clamps).  The kernels implement them with different
mechanisms than the oracle (a precomputed c rsqrt|dA| table, NaN-dropping min/max, compare-select
in fp64), so they are run here on workloads on which the guards EXECUTE (tests/helpers.py, the
same ones that pin the oracle's branches in test_oracle_pins.py), in fp64 and fp32, counting and
fast builds, against the oracle and against what the mathematics fixes; in fp64 the DIAG
counters must equal the oracle's."""
import numpy as np
import pytest

from helpers import LOOSE, kappa_cap_cfg, landing_cfg

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    import gpu_helpers
    from paper_1111_5295_b200 import binding
    binding.load()
    return gpu_helpers


def _report(name, m):
    s, o = m["stats"], m["ostats"]
    print(f"[guards] {name}: x={max(m['x']):.2e} v={max(m['v']):.2e} j={m['j']:.2e} "
          f"max|dxi|={max(m['xi_max']):.2e} max|dv|/vrms={max(m['v_max']):.2e} cont={m['cont']:.2e} "
          f"flips={m['flips']}/{m['n']} | kernel/oracle kappa_cap {s['n_kappa_cap']}/{o['n_kappa_cap']} "
          f"picard_cap {s['n_picard_cap']}/{o['n_picard_cap']} neg_disc {s['n_neg_disc']}/{o['n_neg_disc']} "
          f"clamped {s['n_clamped_tau']}/{o['n_clamped_tau']} sub {s['n_sub']}/{o['n_sub']}")


@pytest.mark.parametrize("cn_mode", ["direct", "picard"])
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_kappa_cap_parity(G, oracle, precision, cn_mode):
    """A-2 binding on most sub-steps (1 - kappa down to 0.5, both signs of a')."""
    cfg = kappa_cap_cfg()
    op = oracle.make_params(cn_mode=oracle.DIRECT if cn_mode == "direct" else oracle.PICARD,
                            tol=cfg["tol"], **LOOSE)
    m = G.parity(oracle, cfg, precision, cn_mode, oracle_params=op, pic_kw=LOOSE)
    _report(f"kappa-cap {precision} {cn_mode}", m)
    assert m["ostats"]["n_kappa_cap"] > 0.5 * m["ostats"]["n_sub"]
    assert m["stats"]["n_kappa_cap"] > 0.5 * m["stats"]["n_sub"]
    G.assert_parity(m, precision, max_flip_frac=5e-3)
    if precision == "fp64":
        # same branches => same counters, particle for particle; a flipped orbit may differ by
        # its own sub-steps
        slack = 0 if m["flips"] == 0 else 200 * m["flips"]
        for k in ("n_sub", "n_cross", "n_kappa_cap", "n_neg_disc", "n_clamped_tau", "n_picard_cap"):
            assert abs(m["stats"][k] - m["ostats"][k]) <= slack, k
    m["gpu"]["pic"].close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_kappa_cap_fast_build(G, oracle, precision):
    """The production builds (fp32: mover2_kernel with its per-cell cap TABLE) on the same
    workload: bit-identical to the counting build (asserted inside parity) and to the oracle."""
    cfg = kappa_cap_cfg()
    op = oracle.make_params(cn_mode=oracle.DIRECT, **LOOSE)
    m = G.parity(oracle, cfg, precision, "direct", oracle_params=op, pic_kw=LOOSE, fast=True)
    _report(f"kappa-cap fast {precision} [{m['gpu']['kernel']}]", m)
    assert m["gpu"]["kernel"] == ("mover2_kernel" if precision == "fp32" else "mover_kernel")
    G.assert_parity(m, precision, max_flip_frac=5e-3)
    m["gpu"]["pic"].close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_picard_cap_parity(G, oracle, precision):
    """A-3: picard_max = 2 with a tolerance (almost) no second iterate can meet: the sub-steps
    are cut off.  The kernel floors the tolerance at 4 ulp of its precision (A-3);
    both sides get that value, so that they stop at the same iterate."""
    tol = 1e-15 if precision == "fp64" else 4.0 * 2.0 ** -23
    from paper_1111_5295_b200 import workloads as W
    cfg = dict(W.config2(n=50_003), tol=tol)
    op = oracle.make_params(cn_mode=oracle.PICARD, tol=tol, picard_max=2)
    m = G.parity(oracle, cfg, precision, "picard", oracle_params=op, pic_kw=dict(picard_max=2))
    _report(f"picard-cap {precision}", m)
    assert m["ostats"]["n_picard_cap"] > (0.9 if precision == "fp64" else 0.3) * m["ostats"]["n_sub"]
    G.assert_parity(m, precision, max_flip_frac=5e-3)
    if precision == "fp64":
        slack = 0 if m["flips"] == 0 else 200 * m["flips"]
        # a sub-step whose second iterate happens to meet 1e-15 (fp64 kernel: floored at 4 ulp)
        # may be counted differently: allow 1e-3 of the sub-steps
        assert abs(m["stats"]["n_picard_cap"] - m["ostats"]["n_picard_cap"]) <= \
            slack + 1e-3 * m["ostats"]["n_sub"]
        assert abs(m["stats"]["n_picard_it"] - m["ostats"]["n_picard_it"]) <= \
            slack + 1e-3 * m["ostats"]["n_sub"]
    else:
        assert abs(m["stats"]["n_picard_cap"] - m["ostats"]["n_picard_cap"]) <= 0.01 * m["ostats"]["n_sub"]
    m["gpu"]["pic"].close()


def test_picard_cap_fp32_at_the_callers_tolerance(G, oracle):
    """The same workload with the tolerance left where a caller would put it (1e-10): the oracle
    iterates against 1e-10, the fp32 kernel against its floor of 4 ulp = 4.8e-7 (a tolerance
    below a few ulp can never be met in fp32, A-3).  What the floor changes: with
    picard_max = 2 the oracle now hits the cap on (nearly) every sub-step, the kernel only where
    its two iterates differ by more than 4.8e-7 relative -- fewer -- and both still end on the
    SECOND iterate or closer than 4.8e-7 to it, so the orbits agree at the fp32 bars all the same."""
    from paper_1111_5295_b200 import workloads as W
    cfg = dict(W.config2(n=50_003), tol=1e-10)
    op = oracle.make_params(cn_mode=oracle.PICARD, tol=1e-10, picard_max=2)
    m = G.parity(oracle, cfg, "fp32", "picard", oracle_params=op, pic_kw=dict(picard_max=2))
    _report("picard-cap fp32, oracle at the caller's tol", m)
    assert m["ostats"]["n_picard_cap"] > 0.9 * m["ostats"]["n_sub"]
    assert m["stats"]["n_picard_cap"] <= m["ostats"]["n_picard_cap"]
    G.assert_parity(m, "fp32", max_flip_frac=5e-3)
    m["gpu"]["pic"].close()


@pytest.mark.parametrize("kind", ["land", "turn"])
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_crossing_clamps(G, oracle, precision, kind):
    """O7 guards through rounding coincidences: particles that, in exact arithmetic, end their
    single sub-step exactly on a face.  Which branch rounding picks differs between kernel and
    oracle (different arithmetic: cell units, FMA), so most particles count as branch flips;
    what is checked is the closed form (uniform field: X1 = the face, v1 = v0 + a dt) on EVERY
    particle of the kernel's own output, its continuity, and that the kernel's guards ran."""
    from paper_1111_5295_b200 import binding as B
    eps = dict(eps_a=1.0, eps_r=1.0)
    fp64 = precision == "fp64"
    tot = dict(n_neg_disc=0, n_clamped_tau=0, n_cross=0)
    for seed in range(4):
        for dt in (1.0, 0.7, 1.9):
            cfg, _, (X1, v1) = landing_cfg(kind, dt=dt, seed=seed)
            for cn in ("direct", "picard"):
                g = G.gpu_run(cfg, precision, cn, **eps)
                s = g["species"][0]
                for k in tot:
                    tot[k] += g["stats"][k]
                assert g["stats"]["n_substep_cap"] == 0
                # unwrapped end position from the kernel's own (cell, xi): the face, from either
                # side (cell c with xi = 1, or cell c+1 with xi = 0)
                L = cfg["length"]
                d = np.abs(((s["cell"] + s["xi"]) - X1 + L / 2) % L - L / 2)
                assert np.all(np.isfinite(s["v"])) and np.all(np.isfinite(s["xi"]))
                assert d.max() < (4e-15 if fp64 else 1e-6), d.max()
                vtol = (2e-7 if fp64 else 2e-3) if kind == "turn" else (4e-15 if fp64 else 1e-6)
                assert np.max(np.abs(s["v"] - v1)) < vtol, np.max(np.abs(s["v"] - v1))
                # continuity with the kernel's own output
                res, div = G.continuity_residual(oracle, cfg, [(s["cell0"], s["xi0"])],
                                                 [(s["cell"], s["xi"])], g["jbar"])
                assert np.max(np.abs(res)) < 1e-12
                g["pic"].close()
    print(f"[guards] clamps {kind} {precision}: {tot}")
    assert tot["n_cross"] > 200
    assert tot["n_neg_disc"] + tot["n_clamped_tau"] > 0, tot
    # and against the oracle on the particles that took the same branches
    cfg, _, _ = landing_cfg(kind, dt=0.7, seed=1)
    op = oracle.make_params(cn_mode=oracle.DIRECT, **eps)
    m = G.parity(oracle, cfg, precision, "direct", oracle_params=op, pic_kw=eps)
    _report(f"clamps {kind} {precision}", m)
    if kind == "land":
        G.assert_parity(m, precision, max_flip_frac=1.0)
    else:
        # 'turn': the end velocity is the square root of a rounding error (exact value 0), so a
        # relative velocity norm means nothing; positions, jbar and continuity still must agree
        t = G.TOL[precision]
        assert max(m["x"]) <= t["x"] and m["j"] <= t["j"] and m["cont"] <= t["cont"]
    m["gpu"]["pic"].close()


def _raw_jfnk(pic, E, dt, **kw):
    """pic_jfnk_step through the bare C call: (rc, info) without the binding's exception."""
    from paper_1111_5295_b200 import binding as B
    o = dict(rtol=1e-8, atol=0.0, fd_eps=0.0, gmres_rtol=1e-2, max_newton=20, gmres_restart=30,
             max_gmres=200)
    o.update(kw)
    opts = B.PicJfnkOpts(o["rtol"], o["atol"], o["fd_eps"], o["gmres_rtol"], o["max_newton"],
                         o["gmres_restart"], o["max_gmres"], 0)
    info = B.PicJfnkInfo()
    rc = pic._L.pic_jfnk_step(pic._h, B._ptr(E), B.C.c_double(dt), B.C.c_double(1e-10),
                              B.C.byref(opts), B.C.byref(info))
    return rc, info.as_dict()


def test_jfnk_rejected_step_changes_nothing():
    """include/pic.h, pic_jfnk_step: E^{n+1} is delivered only together with the committed state.
    A step that is rejected -- Newton short of rtol (PIC_ERR_STATE), or converged on orbits that
    were cut off at max_substeps (PIC_ERR_SUBSTEP_CAP, A-9) -- leaves E at E^n and the particles
    at state n; the same handle then still takes an acceptable step."""
    from paper_1111_5295_b200 import binding as B
    from paper_1111_5295_b200 import workloads as W
    cfg = W.config1(ppc=40)                      # IAW, 256 cells, 2 x 10,240 particles
    dt = cfg["dt"]
    E0 = np.ascontiguousarray(cfg["E_n"])

    def state(pic):
        return [pic.get_particles(s, B.PIC_STATE_N) for s in range(pic.n_species)]

    def same(a, b):
        return all(np.array_equal(p["cell"], q["cell"]) and np.array_equal(p["xi"], q["xi"]) and
                   np.array_equal(p["v"], q["v"]) for p, q in zip(a, b))

    # (1) not converged: one Newton step cannot reach 1e-13
    pic = B.Pic(cfg["n_cells"], cfg["length"], cfg["species"], precision="fp64")
    s0 = state(pic)
    E = E0.copy()
    rc, info = _raw_jfnk(pic, E, dt, rtol=1e-13, max_newton=1)
    assert rc == -5 and info["converged"] == 0 and info["newton_its"] == 1, (rc, info)
    assert info["resid"] < info["resid0"]        # the iterate did move ...
    assert np.array_equal(E, E0)                 # ... but the caller's field did not
    assert same(state(pic), s0)
    # the same handle, acceptable settings: accepted, E and the state change together
    rc, info = _raw_jfnk(pic, E, dt, rtol=1e-8)
    assert rc == 0 and info["converged"] == 1, (rc, info)
    assert not np.array_equal(E, E0) and not same(state(pic), s0)
    pic.close()

    # (2) converged on truncated orbits: dt = 100 needs a hundred and more sub-steps per electron,
    # the cap is 16 (the kernel tests it every 64 sub-steps); a loose rtol is met after >= 1 update
    pic = B.Pic(cfg["n_cells"], cfg["length"], cfg["species"], precision="fp64", max_substeps=16)
    s0 = state(pic)
    E = E0.copy()
    rc, info = _raw_jfnk(pic, E, 100.0, rtol=0.5, max_newton=10)
    print(f"[guards] jfnk on capped orbits: rc={rc} {info}")
    assert rc == B.PIC_ERR_SUBSTEP_CAP and info["converged"] == 1 and info["newton_its"] >= 1, (rc, info)
    assert b"not committed" in pic._L.pic_last_error(pic._h)
    assert pic.get_stats()["n_substep_cap"] > 0
    assert np.array_equal(E, E0)
    assert same(state(pic), s0)
    pic.close()
