"""Run under PIC_B200_CHECK=1 (the bounds-checked debug build, csrc/pic_check.cuh): a tour of the
library's kernels on ragged sizes, odd grids, long orbits, every deposit / ordering / precision
mode, commit and the diagnostics; prints BOUNDS_VIOLATIONS=<n> at the end.  Started by
tests/test_gpu_bounds_check.py in a process of its own (the library is chosen at load time)."""
import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

from paper_1111_5295_b200 import binding as B  # noqa: E402
from paper_1111_5295_b200 import workloads as W  # noqa: E402
from helpers import LOOSE, kappa_cap_cfg, landing_cfg  # noqa: E402


def ring(n_cells, n=10_007, vth=1.5, dt=4.0, seed=31):
    length = 0.7 * n_cells
    xf = W.face_positions(n_cells, length)
    x = W.uniform01(seed, 1, n) * length * (1 - 1e-12)
    v = vth * W.normal01(seed, 2, n)
    return dict(n_cells=n_cells, length=length, dt=dt, tol=1e-12,
                E_n=0.2 * np.sin(2 * math.pi * xf / length),
                E_np1=0.2 * np.sin(2 * math.pi * xf / length + 0.4),
                species=[dict(name="e", q_over_m=-1.0, w_q=-length / n, x=x, v=v)])


def tour(cfg, big=False, **kw):
    n_moves = 0
    for precision in ("fp32", "fp64"):
        for cn in ("direct", "picard"):
            for flags in (0, B.PIC_FLAG_VSORT, B.PIC_FLAG_COUNTS | B.PIC_FLAG_DIAG) if big else (0, B.PIC_FLAG_VSORT, B.PIC_FLAG_VSORT | B.PIC_FLAG_STRIDED,
                          B.PIC_FLAG_DEPOSIT_PER_VISIT, B.PIC_FLAG_COUNTS | B.PIC_FLAG_DIAG,
                          B.PIC_FLAG_VSORT | B.PIC_FLAG_ONE_PER_LANE, B.PIC_FLAG_EXACT_TIME):
                pic = B.Pic(cfg["n_cells"], cfg["length"], cfg["species"], precision=precision,
                            cn_mode=cn, flags=flags, **kw)
                for _ in range(2):
                    j = pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"], cfg.get("tol", 1e-10))
                    assert np.all(np.isfinite(j))
                    pic.commit()
                    n_moves += 1
                pic.rho(B.PIC_STATE_N)
                pic.kinetic_energy(B.PIC_STATE_N)
                for s in range(len(cfg["species"])):
                    pic.get_particles(s, B.PIC_STATE_N)
                if flags & B.PIC_FLAG_COUNTS:
                    pic.move_accumulate(cfg["E_n"], cfg["E_np1"], cfg["dt"])
                    pic.get_counts(0)
                    pic.count_histogram(0, 3, 64)
                pic.close()
    return n_moves


def main():
    assert os.environ.get("PIC_B200_CHECK") == "1"
    B.load()
    assert B.debug_bounds() == 0, "not the check build, or violations at load"
    assert B.debug_bounds(self_test=True) == 1          # the counter counts
    moves = 0
    moves += tour(W.config0())
    moves += tour(W.config2(n=100_003))
    moves += tour(W.config2(n=65))
    moves += tour(W.config3(n=5_003))
    moves += tour(W.config1(ppc=40))
    for ng in (1, 2, 3, 4, 48, 100):
        moves += tour(ring(ng))
    moves += tour(ring(8, n=257, vth=6.0, dt=3.0, seed=5))         # ~10 turns of the ring
    moves += tour(ring(20_001, n=30_011), big=True)                # global-memory grid fallback
    moves += tour(kappa_cap_cfg(n=1500), **LOOSE)
    for kind in ("land", "turn"):
        moves += tour(landing_cfg(kind, dt=0.7, seed=1)[0], eps_a=1.0, eps_r=1.0)
    # the implicit step incl. defect correction (pic_copy_state, re-binning of both handles)
    cfg = W._iaw("iaw-check", 64, 200, 1.0, W.DEFAULT_SEED)
    from paper_1111_5295_b200.iaw import gauss_field
    dx = cfg["length"] / cfg["n_cells"]
    h64 = B.Pic(64, cfg["length"], cfg["species"], precision="fp64", flags=B.PIC_FLAG_VSORT)
    h32 = B.Pic(64, cfg["length"], cfg["species"], precision="fp32", flags=B.PIC_FLAG_VSORT)
    E = gauss_field(h64.rho(B.PIC_STATE_N), dx)
    for _ in range(2):
        assert h64.jfnk_step(E, 1.0, rtol=1e-8, jacobian=h32)["converged"]
    h64.close()
    h32.close()
    v = B.debug_bounds()
    print(f"MOVES={moves}")
    print(f"BOUNDS_VIOLATIONS={v - 1}")                  # minus the self-test's one


if __name__ == "__main__":
    main()
