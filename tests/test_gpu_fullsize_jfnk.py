"""`-m gpu`: (1) parity at BASELINE.json's full size (configs[2], 1e8 particles) in the launch
configuration bench.py times: sampled orbits against the oracle one by one, plus the invariants
that hold at any size (continuity, energy identity); (2) the host JFNK driver around the GPU
mover (configs[1] shape, reduced particle count) checked with the oracle's residual."""
import ctypes as C
import math

import numpy as np
import pytest

from paper_1111_5295_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _device_state(pic, B, torch, which):
    n = pic.n[0]
    cell = torch.empty(n, dtype=torch.int32, device="cuda")
    xi = torch.empty(n, dtype=torch.float64, device="cuda")
    v = torch.empty(n, dtype=torch.float64, device="cuda")
    pic._chk(pic._L.pic_get_particles(pic._h, C.c_int(0), C.c_int(which), None, B._ptr(v),
                                      B._ptr(cell), B._ptr(xi)))
    return cell, xi, v


def test_cfg2_full_size_sampled(oracle):
    import torch
    from paper_1111_5295_b200 import binding as B
    import gpu_helpers as G
    cfg = W.config2()                      # 4,096 cells, 1e8 electrons, dt = 10
    sp = cfg["species"][0]
    n, ng, dt = sp["x"].shape[0], cfg["n_cells"], cfg["dt"]
    dx = cfg["length"] / ng
    pic = B.Pic(ng, cfg["length"], [sp], precision="fp32", cn_mode="direct",
                flags=B.PIC_FLAG_VSORT | B.PIC_FLAG_COUNTS,
                stream=torch.cuda.current_stream().cuda_stream)
    # (a) the counting build: exact per-particle sub-step / crossing counts (flip detection)
    jbar_c = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], dt)
    st = pic.get_stats()
    assert st["n_substep_cap"] == 0 and st["n_sub"] > 40 * n
    c0, x0, v0 = _device_state(pic, B, torch, B.PIC_STATE_N)
    cc, xc, vc = _device_state(pic, B, torch, B.PIC_STATE_NP1)
    nsub = torch.empty(n, dtype=torch.int32, device="cuda")
    ncross = torch.empty(n, dtype=torch.int32, device="cuda")
    pic._chk(pic._L.pic_get_counts(pic._h, C.c_int(0), B._ptr(nsub), B._ptr(ncross)))
    # (b) the launch configuration bench.py times: the fast build = mover2_kernel (two particles
    # per lane, packed FP32).  All 1e8 orbits must be bit-identical to the counting build's;
    # everything below is checked on ITS output.
    pic.set_flags(B.PIC_FLAG_VSORT)
    jbar = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], dt)
    assert pic.last_kernel() == "mover2_kernel"
    c1, x1, v1 = _device_state(pic, B, torch, B.PIC_STATE_NP1)
    assert torch.equal(c1, cc) and torch.equal(x1, xc) and torch.equal(v1, vc)
    assert G.rel_l2(jbar, jbar_c) < 1e-12
    del cc, xc, vc
    # ---- sampled orbits, one by one through the oracle (particles are independent given E)
    idx = torch.from_numpy(np.sort(np.random.default_rng(3).choice(n, 1 << 16, replace=False))).cuda()
    h = lambda t: t[idx].cpu().numpy()
    r = oracle.move_accumulate(ng, cfg["length"], sp["q_over_m"], sp["w_q"], h(c0), h(x0) * dx,
                               h(v0), cfg["E_n"], cfg["E_np1"], dt, oracle.make_params())
    same = (r["n_sub"] == h(nsub).astype(np.uint32)) & (r["n_cross"] == h(ncross).astype(np.uint32)) \
        & (r["cell"] == h(c1))
    flips = int((~same).sum())
    xg = (h(c1) + h(x1)) * dx
    xr = r["cell"] * dx + r["s"]
    ex = np.linalg.norm(G.periodic_dist(xg[same], xr[same], cfg["length"])) / np.linalg.norm(xr[same])
    ev = G.rel_l2(h(v1)[same], r["v"][same])
    print(f"[full] sampled 65536 of {n}: x={ex:.2e} v={ev:.2e} flips={flips}")
    assert flips <= 1e-3 * idx.numel() and ex <= 1e-5 and ev <= 1e-5
    # ---- energy identity (P-9) at full size
    dK = pic.kinetic_energy(B.PIC_STATE_NP1)[0] - pic.kinetic_energy(B.PIC_STATE_N)[0]
    work = dt * dx * np.sum(jbar * 0.5 * (cfg["E_n"] + cfg["E_np1"]))
    print(f"[full] energy identity rel={(dK - work) / abs(work):.2e}")
    assert abs(dK - work) <= 1e-4 * abs(work)
    # ---- per-cell continuity (P-6) at full size, rho by the oracle in fp64 from the kernel's
    # own (cell, xi)
    rho0 = oracle.rho(ng, cfg["length"], sp["w_q"], c0.cpu().numpy(), x0.cpu().numpy() * dx)
    rho1 = oracle.rho(ng, cfg["length"], sp["w_q"], c1.cpu().numpy(), x1.cpu().numpy() * dx)
    div = dt * (np.roll(jbar, -1) - jbar) / dx
    cont = np.linalg.norm(rho1 - rho0 + div) / np.linalg.norm(div)
    print(f"[full] continuity rel={cont:.2e}")
    assert cont <= 1e-5
    # the device rho diagnostic agrees with the oracle's
    assert G.rel_l2(pic.rho(B.PIC_STATE_NP1), rho1) < 1e-10
    del rho0, rho1
    # ---- jbar of the WHOLE launch against the oracle: all 1e8 orbits through the serial oracle,
    # one call per chunk on every host core (orbits are independent given E; each call has its
    # own raw J, summed afterwards).  Continuity fixes jbar only up to a constant and the energy
    # identity barely constrains that constant; this pins the mean current (P-8) as well.
    # Orbits that took another branch than the kernel's (flips, by the exact per-particle counts
    # of the counting build) are taken out of BOTH sums: the deposit is linear in the particles,
    # so each side's jbar of the flipped orbits alone is subtracted from its total.
    import os
    from concurrent.futures import ThreadPoolExecutor
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    c0h, s0h, v0h = c0.cpu().numpy(), x0.cpu().numpy() * dx, v0.cpu().numpy()
    nsh, nch, c1h = nsub.cpu().numpy().astype(np.uint32), ncross.cpu().numpy().astype(np.uint32), c1.cpu().numpy()
    bounds = np.linspace(0, n, 8 * cores + 1).astype(np.int64)
    par = oracle.make_params()

    def one(k):
        a, b = int(bounds[k]), int(bounds[k + 1])
        r = oracle.move_accumulate(ng, cfg["length"], sp["q_over_m"], sp["w_q"], c0h[a:b], s0h[a:b],
                                   v0h[a:b], cfg["E_n"], cfg["E_np1"], dt, par)
        flip = (r["n_sub"] != nsh[a:b]) | (r["n_cross"] != nch[a:b]) | (r["cell"] != c1h[a:b])
        return r["J"], a + np.nonzero(flip)[0]

    with ThreadPoolExecutor(max_workers=cores) as ex:
        parts = list(ex.map(one, range(8 * cores)))
    J_all = np.sum([q[0] for q in parts], axis=0)
    F = np.concatenate([q[1] for q in parts])
    print(f"[full] oracle on all {n} orbits ({cores} cores): flips={F.size}")
    assert F.size <= 1e-3 * n
    j_o = oracle.jbar_from_J(ng, cfg["length"], dt, J_all)
    j_g = jbar.copy()
    if F.size:
        rF = oracle.move_accumulate(ng, cfg["length"], sp["q_over_m"], sp["w_q"], c0h[F], s0h[F],
                                    v0h[F], cfg["E_n"], cfg["E_np1"], dt, par, want_state=False)
        j_o = j_o - oracle.jbar_from_J(ng, cfg["length"], dt, rF["J"])
        gF = G.gpu_run(cfg, "fp32", flags=B.PIC_FLAG_VSORT, subset=[F])   # same inputs, same rounding
        j_g = j_g - gF["jbar"]
        gF["pic"].close()
    ej = G.rel_l2(j_g, j_o)
    mean_err = abs(j_g.sum() - j_o.sum()) / np.abs(j_o).sum()
    print(f"[full] jbar of the whole launch vs the oracle: rel L2 {ej:.2e}, |sum_f dj| / sum_f |j| {mean_err:.2e}")
    assert ej <= G.TOL["fp32"]["j"] and mean_err <= 1e-6
    pic.close()


def test_jfnk_steps_iaw(oracle):
    from paper_1111_5295_b200 import binding as B
    import gpu_helpers as G
    cfg = W._iaw("iaw-test", 64, 500, 1.0, W.DEFAULT_SEED)     # configs[1] shape, 2 x 32,000
    ng, L, dt = cfg["n_cells"], cfg["length"], cfg["dt"]
    dx = L / ng
    pic = B.Pic(ng, L, cfg["species"], precision="fp64", cn_mode="direct")
    # A-13: E0 from the discrete Gauss law (E_{c+1} - E_c)/dx = rho_c, zero mean
    rho = pic.rho(B.PIC_STATE_N)
    E = np.concatenate(([0.0], np.cumsum(rho[:-1] * dx)))
    E -= E.mean()

    def energy():
        return float(pic.kinetic_energy(B.PIC_STATE_N).sum() + 0.5 * dx * np.sum(E * E))

    e0 = energy()
    for step in range(3):
        En = E.copy()
        before = [pic.get_particles(j, B.PIC_STATE_N) for j in range(2)]
        info = pic.jfnk_step(E, dt, rtol=1e-9)
        assert info["rc"] == 0 and info["converged"] == 1, info
        assert info["resid"] <= 1e-9 * info["resid0"] * 1.0001
        # the oracle's residual at the converged field, from the same state n, is as small
        state = [(b["cell"], b["xi"] * dx, b["v"]) for b in before]
        c2 = dict(cfg, E_n=En, E_np1=E)
        ref = G.oracle_run(oracle, c2, oracle.make_params(cn_mode=oracle.DIRECT), state=state)
        R = oracle.residual(En, E, dt, ref["jbar"])
        print(f"[jfnk] step {step}: newton={info['newton_its']} gmres={info['gmres_its']} "
              f"|R0|={info['resid0']:.2e} |R|={info['resid']:.2e} oracle |R|={np.linalg.norm(R):.2e} "
              f"dE/E={(energy() - e0) / e0:.2e}")
        assert np.linalg.norm(R) <= 1e-7 * info["resid0"]
    # energy conserved to the nonlinear tolerance level
    assert abs(energy() - e0) / e0 < 1e-8
    pic.close()


def test_defect_correction_matches_fp64(oracle):
    """S8(f) #2 / P:325-331: residual from the fp64 mover, Jacobian-vector products from the fp32
    mover: the converged fields must equal the all-fp64 solve to the nonlinear tolerance, with
    most mover calls in fp32."""
    from paper_1111_5295_b200 import binding as B
    from paper_1111_5295_b200.iaw import gauss_field
    cfg = W._iaw("iaw-dc", 64, 500, 1.0, W.DEFAULT_SEED)
    ng, L, dt = cfg["n_cells"], cfg["length"], cfg["dt"]
    dx = L / ng
    ref = B.Pic(ng, L, cfg["species"], precision="fp64", flags=B.PIC_FLAG_VSORT)
    h64 = B.Pic(ng, L, cfg["species"], precision="fp64", flags=B.PIC_FLAG_VSORT)
    h32 = B.Pic(ng, L, cfg["species"], precision="fp32", flags=B.PIC_FLAG_VSORT)
    E_ref = gauss_field(ref.rho(B.PIC_STATE_N), dx)
    E_dc = E_ref.copy()
    e0 = float(h64.kinetic_energy(B.PIC_STATE_N).sum() + 0.5 * dx * np.sum(E_dc * E_dc))
    import gpu_helpers as G
    for step in range(3):
        En = E_dc.copy()
        before = [h64.get_particles(j, B.PIC_STATE_N) for j in range(2)]
        ia = ref.jfnk_step(E_ref, dt, rtol=1e-9)
        ib = h64.jfnk_step(E_dc, dt, rtol=1e-9, jacobian=h32)
        assert ia["converged"] == 1 and ib["converged"] == 1, (ia, ib)
        # the ORACLE's residual at the field the defect-correction solve converged to, from the
        # same state n: as small as the solver's own (DP accuracy with SP products)
        state = [(b["cell"], b["xi"] * dx, b["v"]) for b in before]
        oref = G.oracle_run(oracle, dict(cfg, E_n=En, E_np1=E_dc),
                            oracle.make_params(cn_mode=oracle.DIRECT), state=state)
        Ro = np.linalg.norm(oracle.residual(En, E_dc, dt, oref["jbar"]))
        print(f"[dc] step {step}: oracle |R| at the dc solution = {Ro:.2e} (|R0| {ib['resid0']:.2e})")
        assert Ro <= 1e-7 * ib["resid0"]
        err = np.linalg.norm(E_dc - E_ref) / np.linalg.norm(E_ref)
        print(f"[dc] step {step}: fp64 newton={ia['newton_its']} calls={ia['mover_calls']} | "
              f"dc newton={ib['newton_its']} calls={ib['mover_calls']} of which fp64 "
              f"{ib['mover_calls_resid']} |R|={ib['resid']:.2e} |E_dc-E_64|/|E|={err:.2e}")
        assert err < 1e-7
        assert ib["mover_calls_resid"] <= 0.5 * ib["mover_calls"]      # most calls are fp32
        # the fp32 handle follows the committed fp64 state (converted), in the same order
        a, b = h64.get_particles(0, B.PIC_STATE_N), h32.get_particles(0, B.PIC_STATE_N)
        assert np.array_equal(a["cell"], b["cell"])
        assert np.max(np.abs(a["v"] - b["v"])) <= 1e-6 * np.max(np.abs(a["v"]))
    e1 = float(h64.kinetic_energy(B.PIC_STATE_N).sum() + 0.5 * dx * np.sum(E_dc * E_dc))
    assert abs(e1 - e0) / e0 < 1e-8
    for p in (ref, h64, h32):
        p.close()


def test_cfg1_full_size_ten_steps(oracle):
    """BASELINE.json configs[1] as stated: 256 cells, 2 x 512,000 particles, dt = 1, host fp64
    JFNK at nonlinear relative tolerance 1e-8 around the fp64 GPU mover, 10 steps.  At every step
    the ORACLE's residual at the converged field, from the same state n, must be as small as the
    solver's; total energy is conserved to the nonlinear tolerance."""
    from paper_1111_5295_b200 import binding as B
    from paper_1111_5295_b200.iaw import gauss_field
    import gpu_helpers as G
    cfg = W.config1()
    ng, L, dt = cfg["n_cells"], cfg["length"], cfg["dt"]
    dx = L / ng
    pic = B.Pic(ng, L, cfg["species"], precision="fp64", cn_mode="direct", flags=B.PIC_FLAG_VSORT)
    E = gauss_field(pic.rho(B.PIC_STATE_N), dx)

    def energy():
        return float(pic.kinetic_energy(B.PIC_STATE_N).sum() + 0.5 * dx * np.sum(E * E))

    e0 = energy()
    for step in range(10):
        En = E.copy()
        before = [pic.get_particles(j, B.PIC_STATE_N) for j in range(2)]
        info = pic.jfnk_step(E, dt, rtol=1e-8)
        assert info["rc"] == 0 and info["converged"] == 1, info
        state = [(b["cell"], b["xi"] * dx, b["v"]) for b in before]
        ref = G.oracle_run(oracle, dict(cfg, E_n=En, E_np1=E),
                           oracle.make_params(cn_mode=oracle.DIRECT), state=state)
        Ro = float(np.linalg.norm(oracle.residual(En, E, dt, ref["jbar"])))
        print(f"[cfg1] step {step + 1}: newton={info['newton_its']} gmres={info['gmres_its']} "
              f"passes={info['mover_calls']} |R0|={info['resid0']:.2e} |R|={info['resid']:.2e} "
              f"oracle |R|={Ro:.2e} dE/E={(energy() - e0) / e0:+.2e}")
        assert Ro <= 2e-8 * info["resid0"]
        rho = pic.rho(B.PIC_STATE_N)
        assert np.linalg.norm((np.roll(E, -1) - E) / dx - rho) <= 1e-6 * np.linalg.norm(rho)
    assert abs(energy() - e0) / e0 < 1e-9
    pic.close()


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_cfg3_full_size_invariants(oracle, precision):
    """BASELINE.json configs[3] at full size (2e7 particles) in the launch configuration the bench
    times: properties that hold at any size -- per-cell continuity with rho by the oracle from the
    kernel's own (cell, xi), the energy identity, no sub-step cap -- plus sampled orbits against
    the oracle one by one (fp64: north_star's bars; fp32: the derived bars of DESIGN.md 2)."""
    import torch
    from paper_1111_5295_b200 import binding as B
    import gpu_helpers as G
    from helpers import ulp_response
    cfg = W.config3()
    sp = cfg["species"][0]
    n, ng, dt = sp["x"].shape[0], cfg["n_cells"], cfg["dt"]
    dx = cfg["length"] / ng
    pic = B.Pic(ng, cfg["length"], [sp], precision=precision, flags=B.PIC_FLAG_VSORT | B.PIC_FLAG_COUNTS,
                stream=torch.cuda.current_stream().cuda_stream)
    pic.move_accumulate(cfg["E_n"], cfg["E_np1"], dt)                 # counting build
    st = pic.get_stats()
    assert st["n_substep_cap"] == 0 and st["n_sub"] > 500 * n
    nsub = torch.empty(n, dtype=torch.int32, device="cuda")
    ncross = torch.empty(n, dtype=torch.int32, device="cuda")
    pic._chk(pic._L.pic_get_counts(pic._h, C.c_int(0), B._ptr(nsub), B._ptr(ncross)))
    pic.set_flags(B.PIC_FLAG_VSORT)                                   # the timed (fast) build
    jbar = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], dt)
    assert pic.last_kernel() == ("mover2_kernel" if precision == "fp32" else "mover_kernel")
    c0, x0, v0 = _device_state(pic, B, torch, B.PIC_STATE_N)
    c1, x1, v1 = _device_state(pic, B, torch, B.PIC_STATE_NP1)
    rho0 = oracle.rho(ng, cfg["length"], sp["w_q"], c0.cpu().numpy(), x0.cpu().numpy() * dx)
    rho1 = oracle.rho(ng, cfg["length"], sp["w_q"], c1.cpu().numpy(), x1.cpu().numpy() * dx)
    div = dt * (np.roll(jbar, -1) - jbar) / dx
    cont = np.linalg.norm(rho1 - rho0 + div) / np.linalg.norm(div)
    dK = pic.kinetic_energy(B.PIC_STATE_NP1)[0] - pic.kinetic_energy(B.PIC_STATE_N)[0]
    work = dt * dx * np.sum(jbar * 0.5 * (cfg["E_n"] + cfg["E_np1"]))
    print(f"[cfg3 full] {precision}: continuity {cont:.2e} energy identity {(dK - work) / abs(work):.2e}")
    assert cont <= (1e-10 if precision == "fp64" else 1e-5)
    assert abs(dK - work) <= (1e-9 if precision == "fp64" else 1e-3) * abs(work)
    idx = torch.from_numpy(np.sort(np.random.default_rng(4).choice(n, 1 << 13, replace=False))).cuda()
    h = lambda t: t[idx].cpu().numpy()
    r = oracle.move_accumulate(ng, cfg["length"], sp["q_over_m"], sp["w_q"], h(c0), h(x0) * dx, h(v0),
                               cfg["E_n"], cfg["E_np1"], dt, oracle.make_params(cn_mode=oracle.DIRECT))
    same = (r["n_sub"] == h(nsub).astype(np.uint32)) & (r["n_cross"] == h(ncross).astype(np.uint32)) \
        & (r["cell"] == h(c1))
    xg, xr = (h(c1) + h(x1)) * dx, r["cell"] * dx + r["s"]
    ex = np.linalg.norm(G.periodic_dist(xg[same], xr[same], cfg["length"])) / np.linalg.norm(xr[same])
    ev = G.rel_l2(h(v1)[same], r["v"][same])
    print(f"[cfg3 full] {precision}: sampled 8192 of {n}: x={ex:.2e} v={ev:.2e} flips={int((~same).sum())}")
    if precision == "fp64":
        assert ex <= 1e-10 and ev <= 1e-10 and (~same).sum() <= 8
    else:
        u = ulp_response(oracle, W.config3(n=20_011))
        k = 3.0 * math.sqrt(u["n_sub_mean"])
        assert ex <= k * u["x"] and ev <= k * u["v"] and (~same).sum() <= 0.05 * same.size
    pic.close()
