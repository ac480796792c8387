"""Seeded synthetic workloads shaped like BASELINE.json's configs.

This module serves BOTH the oracle-side tests and the CUDA path, so it holds none of the
method's arithmetic: only counter-based random numbers, particle placement and the field
formulas the configs state.  It imports neither `oracle/` nor the CUDA binding.

Every array is generated in fp64 on the host from Philox keyed by (seed, stream, chunk), in
chunks of 2**20 particles, so any chunk-aligned subsample is reproducible on its own.
The paper measures on its own synthetic plasma set-ups (Maxwellian particles, an ion acoustic
wave), not on a public dataset; these inputs stand in for them.
"""
import math

import numpy as np

DEFAULT_SEED = 12345
CHUNK = 1 << 20
# streams
_S_X, _S_V, _S_PHASE, _S_DPHASE, _S_COIN = 1, 2, 3, 4, 5
# Proposed cell size for cfg2/cfg3: the IAW grid's dx = 100*pi/256.
DX_THROUGHPUT = 100.0 * math.pi / 256.0


def _gen(seed, stream, chunk):
    return np.random.Generator(np.random.Philox(key=[int(seed), (int(stream) << 32) | int(chunk)]))


def _chunks(n, start):
    """(chunk index, offset in chunk, count) covering particles [start, start+n)."""
    p, end = start, start + n
    while p < end:
        ch, off = divmod(p, CHUNK)
        cnt = min(CHUNK - off, end - p)
        yield ch, off, cnt
        p += cnt


def uniform01(seed, stream, n, start=0):
    out = np.empty(n, np.float64)
    w = 0
    for ch, off, cnt in _chunks(n, start):
        out[w:w + cnt] = _gen(seed, stream, ch).random(CHUNK)[off:off + cnt]
        w += cnt
    return out


def normal01(seed, stream, n, start=0):
    out = np.empty(n, np.float64)
    w = 0
    for ch, off, cnt in _chunks(n, start):
        out[w:w + cnt] = _gen(seed, stream, ch).standard_normal(CHUNK)[off:off + cnt]
        w += cnt
    return out


def _wrap(x, length):
    """Keep x in [0, L) after rounding (u*L can round to L)."""
    x = np.where(x >= length, np.nextafter(length, 0.0), x)
    return np.where(x < 0.0, 0.0, x)


def face_positions(n_cells, length):
    return np.arange(n_cells, dtype=np.float64) * (length / n_cells)


def fourier_field(n_cells, length, modes, amplitude, phases):
    """E_f = sum_m amplitude * cos(2 pi m x_f / L + phase_m), m in `modes`."""
    xf = face_positions(n_cells, length)
    E = np.zeros(n_cells)
    for m, ph in zip(modes, phases):
        E += amplitude * np.cos(2.0 * math.pi * m * xf / length + ph)
    return E


def default_params(precision="fp64", cn_mode="picard", tol=1e-10):
    """eps_a, eps_r from P:277; kappa_max, max_substeps from SURVEY A-2, A-9."""
    return dict(eps_a=1e-8, eps_r=0.02, kappa_max=0.5, max_substeps=1 << 20, tol=tol,
                precision=precision, cn_mode=cn_mode)


def _species(name, q_over_m, w_q, x, v):
    return dict(name=name, q_over_m=float(q_over_m), w_q=float(w_q), x=x, v=v)


def config0(n=6400, seed=DEFAULT_SEED):
    """BASELINE.json configs[0]: L=2pi, 64 cells, electrons, dt=0.5."""
    n_cells, length = 64, 2.0 * math.pi
    xf = face_positions(n_cells, length)
    x = _wrap(uniform01(seed, _S_X, n) * length, length)
    v = normal01(seed, _S_V, n)
    return dict(name="cfg0", n_cells=n_cells, length=length, dt=0.5, tol=1e-10,
                species=[_species("e", -1.0, -length / n, x, v)],
                E_n=0.1 * np.sin(xf), E_np1=0.1 * np.sin(xf + 0.3))


def _throughput_cfg(name, n_cells, n, seed, modes, amplitude, dt, v):
    length = n_cells * DX_THROUGHPUT
    x = _wrap(uniform01(seed, _S_X, n) * length, length)
    nm = len(modes)
    ph = uniform01(seed, _S_PHASE, nm) * 2.0 * math.pi
    dph = (uniform01(seed, _S_DPHASE, nm) * 2.0 - 1.0) * 0.3
    return dict(name=name, n_cells=n_cells, length=length, dt=dt, tol=1e-10,
                species=[_species("e", -1.0, -length / n, x, v)],
                E_n=fourier_field(n_cells, length, modes, amplitude, ph),
                E_np1=fourier_field(n_cells, length, modes, amplitude, ph + dph))


def config2(n=100_000_000, seed=DEFAULT_SEED):
    """configs[2]: 4096 cells, 1e8 electrons, 16 Fourier modes of amplitude 0.05, dt=10."""
    v = normal01(seed, _S_V, n)
    return _throughput_cfg("cfg2", 4096, n, seed, range(1, 17), 0.05, 10.0, v)


def config3(n=20_000_000, seed=DEFAULT_SEED):
    """configs[3]: 1024 cells, 2e7 two-stream particles N(+-3, 0.5), |E|=1 on modes 1-8, dt=50."""
    coin = np.where(uniform01(seed, _S_COIN, n) < 0.5, -3.0, 3.0)
    v = coin + 0.5 * normal01(seed, _S_V, n)
    return _throughput_cfg("cfg3", 1024, n, seed, range(1, 9), 1.0, 50.0, v)


def _perturbed_positions(n, length, amp):
    """Inverse CDF of n0(1 + amp cos(2 pi x/L)) on quantiles (k+1/2)/n (SURVEY A-13)."""
    q = (np.arange(n, dtype=np.float64) + 0.5) / n
    k = 2.0 * math.pi / length
    x = q * length
    for _ in range(50):  # Newton on F(x) = x + amp sin(kx)/k - q L
        f = x + amp * np.sin(k * x) / k - q * length
        x = x - f / (1.0 + amp * np.cos(k * x))
    return _wrap(x, length)


def _iaw(name, n_cells, ppc, dt, seed, amp=0.1, mass_ratio=2000.0, te_over_ti=10.0):
    length = 100.0 * math.pi
    n = n_cells * ppc
    sp = []
    for j, (nm, q, m, temp) in enumerate((("e", -1.0, 1.0, 1.0),
                                           ("i", +1.0, mass_ratio, 1.0 / te_over_ti))):
        x = _perturbed_positions(n, length, amp)
        v = math.sqrt(temp / m) * normal01(seed, _S_V + 16 * (j + 1), n)
        sp.append(_species(nm, q / m, q * length / n, x, v))
    z = np.zeros(n_cells)
    return dict(name=name, n_cells=n_cells, length=length, dt=dt, tol=1e-10, species=sp,
                E_n=z, E_np1=z.copy())


def config1(ppc=2000, seed=DEFAULT_SEED):
    """configs[1]: IAW, 256 cells, 2000 particles/cell/species, dt=1 (E from Gauss's law is
    the JFNK driver's job; E_n here is a zero placeholder)."""
    return _iaw("cfg1", 256, ppc, 1.0, seed)


def config4(ppc=4000, seed=DEFAULT_SEED):
    """configs[4]: IAW, 512 cells, 4000 particles/cell/species, dt=5."""
    return _iaw("cfg4", 512, ppc, 5.0, seed)
