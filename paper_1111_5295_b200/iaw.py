"""Ion acoustic wave runs (BASELINE.json configs[1] and [4]): the full implicit step
(pic_jfnk_step: host fp64 Newton-GMRES around the GPU mover) over several time
steps, with the conservation diagnostics the paper reports: total-energy change per
step, total momentum, and the Gauss-law residual (local charge conservation).

    python -m paper_1111_5295_b200.iaw --config 1 --steps 10
    python -m paper_1111_5295_b200.iaw --config 4 --steps 50 --precision fp32 --rtol 2e-4

Everything on the device goes through the C-ABI binding; this module only drives it and does
O(n_cells) host arithmetic on the fields it gets back."""
import argparse
import json
import time

import numpy as np

from . import binding as B
from . import workloads as W


def gauss_field(rho, dx):
    """A-13: E on faces from the discrete Gauss law (E_{c+1} - E_c)/dx = rho_c, zero mean."""
    E = np.concatenate(([0.0], np.cumsum(rho[:-1] * dx)))
    return E - E.mean()


def run(config=1, steps=10, precision=None, rtol=None, ppc=None, flags=B.PIC_FLAG_VSORT,
        verbose=True, defect_correction=False):
    cfg = (W.config1(ppc or 2000) if config == 1 else W.config4(ppc or 4000))
    precision = precision or ("fp64" if config == 1 else "fp32")
    # A-14: 1e-8 needs the fp64 mover; the fp32 mover stalls below ~2e-4
    rtol = rtol or (1e-8 if precision == "fp64" else 2e-4)
    ng, L, dt = cfg["n_cells"], cfg["length"], cfg["dt"]
    dx = L / ng
    pic = B.Pic(ng, L, cfg["species"], precision=precision, cn_mode="direct", flags=flags)
    # defect correction: residual from `pic` (fp64), J w from an fp32 twin
    jac = (B.Pic(ng, L, cfg["species"], precision="fp32", cn_mode="direct", flags=flags)
           if defect_correction else None)
    E = gauss_field(pic.rho(B.PIC_STATE_N), dx)
    w_m = [sp["w_q"] / sp["q_over_m"] for sp in cfg["species"]]

    def diagnostics():
        ke = pic.kinetic_energy(B.PIC_STATE_N)
        rho = pic.rho(B.PIC_STATE_N)
        gauss = (np.roll(E, -1) - E) / dx - rho
        mom = 0.0
        for j, wm in enumerate(w_m):
            mom += wm * float(pic.get_particles(j, B.PIC_STATE_N)["v"].sum())
        return dict(ke=[float(k) for k in ke], field=float(0.5 * dx * np.sum(E * E)),
                    gauss=float(np.linalg.norm(gauss) / max(np.linalg.norm(rho), 1e-300)),
                    momentum=mom)

    d0 = diagnostics()
    e0 = sum(d0["ke"]) + d0["field"]
    hist = []
    for n in range(steps):
        t0 = time.perf_counter()
        info = pic.jfnk_step(E, dt, rtol=rtol, jacobian=jac)
        wall = time.perf_counter() - t0
        if not info["converged"]:
            raise RuntimeError(f"step {n}: Newton did not converge: {info}")
        d = diagnostics()
        etot = sum(d["ke"]) + d["field"]
        rec = dict(step=n + 1, newton=info["newton_its"], gmres=info["gmres_its"],
                   mover_calls=info["mover_calls"], mover_calls_resid=info["mover_calls_resid"],
                   resid0=info["resid0"], resid=info["resid"],
                   dE_rel=(etot - e0) / e0, gauss=d["gauss"], momentum=d["momentum"],
                   ke=d["ke"], field=d["field"], wall_s=wall)
        hist.append(rec)
        if verbose:
            print(f"step {n + 1:4d}: newton {rec['newton']} gmres {rec['gmres']:3d} "
                  f"calls {rec['mover_calls']:3d} |R| {rec['resid']:.2e} dE/E {rec['dE_rel']:+.2e} "
                  f"gauss {rec['gauss']:.2e} P {rec['momentum']:+.3e} wall {wall * 1e3:.1f} ms",
                  flush=True)
    pic.close()
    if jac is not None:
        jac.close()
    return dict(config=config, precision=precision + ("+fp32 J" if defect_correction else ""), rtol=rtol, n_cells=ng,
                particles=[int(sp["x"].shape[0]) for sp in cfg["species"]], dt=dt, e0=e0,
                history=hist)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=1, choices=[1, 4])
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--precision", default=None, choices=["fp32", "fp64"])
    ap.add_argument("--rtol", type=float, default=None)
    ap.add_argument("--ppc", type=int, default=None, help="particles per cell per species")
    ap.add_argument("--defect-correction", action="store_true",
                    help="fp64 residual, fp32 Jacobian-vector products (needs --precision fp64)")
    ap.add_argument("--json", default=None, help="write the history to this file")
    a = ap.parse_args()
    out = run(a.config, a.steps, a.precision, a.rtol, a.ppc, defect_correction=a.defect_correction)
    h = out["history"]
    print(json.dumps(dict(config=out["config"], precision=out["precision"], rtol=out["rtol"],
                          steps=len(h), newton_mean=float(np.mean([r["newton"] for r in h])),
                          gmres_mean=float(np.mean([r["gmres"] for r in h])),
                          mover_calls_mean=float(np.mean([r["mover_calls"] for r in h])),
                          mover_calls_resid_mean=float(np.mean([r["mover_calls_resid"] for r in h])),
                          max_abs_dE_rel=float(np.max(np.abs([r["dE_rel"] for r in h]))),
                          max_gauss=float(np.max([r["gauss"] for r in h])),
                          wall_ms_per_step=float(1e3 * np.mean([r["wall_s"] for r in h])))))
    if a.json:
        with open(a.json, "w") as f:
            json.dump(out, f)


if __name__ == "__main__":
    main()
