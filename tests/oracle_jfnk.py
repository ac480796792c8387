"""TEST INFRASTRUCTURE: the fully implicit time step driven by the ORACLE (BASELINE.json
configs[4]: "... reported against the fp64 oracle run for the first 20 steps"; the paper's Fig. 6
compares the hybrid run with the CPU-only double-precision run).

A plain Newton-Krylov loop (numpy, fp64) around oracle.move_accumulate + oracle.residual:
unknown = E^{n+1} on the faces, particles enslaved (every residual restarts from state n),
J w by finite differences of the residual, unpreconditioned GMRES.  The serial oracle is called
unchanged, once per host core on disjoint chunks of the particle list (orbits are independent
given E; ctypes releases the GIL).  Shares no code with the CUDA path or its JFNK driver
(csrc/pic_jfnk.cu) and is imported by tests only."""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np


def n_cores():
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


class OracleIAW:
    """State n of every species as the oracle holds it: (cell, s, v) in fp64."""

    def __init__(self, o, cfg, params=None, cores=None):
        self.o, self.cfg = o, cfg
        self.ng, self.L, self.dt = cfg["n_cells"], cfg["length"], cfg["dt"]
        self.dx = self.L / self.ng
        self.params = params or o.make_params(cn_mode=o.DIRECT)
        self.cores = cores or n_cores()
        self.pool = ThreadPoolExecutor(max_workers=self.cores)
        self.state = []
        for sp in cfg["species"]:
            c, s = o.bin_particles(self.ng, self.L, sp["x"])
            self.state.append([c, s, np.ascontiguousarray(sp["v"], dtype=np.float64)])
        self.mover_calls = 0

    def close(self):
        self.pool.shutdown()

    # -- one mover pass over all species from state n (O1-O10); optionally returns state n+1
    def move(self, E_n, E_np1, want_state=False):
        o, jobs = self.o, []
        for j, (sp, (c, s, v)) in enumerate(zip(self.cfg["species"], self.state)):
            b = np.linspace(0, c.size, self.cores + 1).astype(np.int64)
            for a0, a1 in zip(b[:-1], b[1:]):
                if a1 > a0:
                    jobs.append((j, a0, a1))

        def one(job):
            j, a0, a1 = job
            sp = self.cfg["species"][j]
            c, s, v = self.state[j]
            return job, o.move_accumulate(self.ng, self.L, sp["q_over_m"], sp["w_q"], c[a0:a1],
                                          s[a0:a1], v[a0:a1], E_n, E_np1, self.dt, self.params,
                                          want_state=want_state)

        J = np.zeros(self.ng)
        new = [[np.empty_like(c), np.empty_like(s), np.empty_like(v)] for c, s, v in self.state] \
            if want_state else None
        n_sub = 0
        for (j, a0, a1), r in self.pool.map(one, jobs):
            J += r["J"]
            n_sub += r["stats"].n_sub
            if want_state:
                new[j][0][a0:a1], new[j][1][a0:a1], new[j][2][a0:a1] = r["cell"], r["s"], r["v"]
        self.mover_calls += 1
        self.last_n_sub = n_sub
        return o.jbar_from_J(self.ng, self.L, self.dt, J), new

    def residual(self, E_n, E_np1):
        jbar, _ = self.move(E_n, E_np1)
        return self.o.residual(E_n, E_np1, self.dt, jbar)

    # -- diagnostics of state n
    def rho(self):
        rho = np.zeros(self.ng)
        for sp, (c, s, v) in zip(self.cfg["species"], self.state):
            self.o.rho(self.ng, self.L, sp["w_q"], c, s, rho)
        return rho

    def kinetic(self):
        return [0.5 * sp["w_q"] / sp["q_over_m"] * float(np.sum(v * v))
                for sp, (c, s, v) in zip(self.cfg["species"], self.state)]

    def gauss_field(self):
        """SURVEY A-13: (E_{c+1} - E_c)/dx = rho_c, zero mean."""
        rho = self.rho()
        E = np.concatenate(([0.0], np.cumsum(rho[:-1] * self.dx)))
        return E - E.mean()

    # -- one implicit step: Newton + GMRES(restart) on R(E^{n+1}) = 0, then accept state n+1
    def step(self, E, rtol=1e-8, fd_eps=1e-6, gmres_rtol=1e-2, max_newton=20, restart=30):
        En = E.copy()
        Ek = E.copy()
        R = self.residual(En, Ek)
        r0 = rn = float(np.linalg.norm(R))
        newton = gm_total = 0
        calls0 = self.mover_calls - 1
        while rn > rtol * r0 and newton < max_newton:
            scale = fd_eps * (1.0 + float(np.linalg.norm(Ek)))
            V = [(-R) / rn]
            H = np.zeros((restart + 1, restart))
            g = np.zeros(restart + 1)
            g[0] = rn
            k_used = 0
            for k in range(restart):
                w = (self.residual(En, Ek + scale * V[k]) - R) / scale
                for i in range(k + 1):                      # modified Gram-Schmidt
                    H[i, k] = float(w @ V[i])
                    w = w - H[i, k] * V[i]
                H[k + 1, k] = float(np.linalg.norm(w))
                k_used = k + 1
                y, res, *_ = np.linalg.lstsq(H[:k + 2, :k + 1], g[:k + 2], rcond=None)
                lin = float(np.linalg.norm(H[:k + 2, :k + 1] @ y - g[:k + 2]))
                if lin <= gmres_rtol * rn or H[k + 1, k] == 0.0:
                    break
                V.append(w / H[k + 1, k])
            gm_total += k_used
            Ek = Ek + sum(yi * Vi for yi, Vi in zip(y, V))
            R = self.residual(En, Ek)
            rn = float(np.linalg.norm(R))
            newton += 1
        # accept: state n+1 of the converged field becomes state n
        _, new = self.move(En, Ek, want_state=True)
        self.state = new
        return Ek, dict(newton_its=newton, gmres_its=gm_total, resid0=r0, resid=rn,
                        converged=int(rn <= rtol * r0), mover_calls=self.mover_calls - calls0)
