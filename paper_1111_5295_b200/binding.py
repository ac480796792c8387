"""Thin ctypes binding of the C-ABI in include/pic.h (same names, argument marshalling only:
every step of the path runs in the CUDA kernels of csrc/).  PyTorch is used by callers for
device memory and streams; this module accepts numpy arrays (host) or torch tensors (host or
CUDA) and passes their raw pointers.

There is NO CPU fallback: if libpic_b200.so is missing or no CUDA device is present, the
calls raise.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))

PIC_FP32, PIC_FP64 = 0, 1
PIC_CN_PICARD, PIC_CN_DIRECT = 0, 1
PIC_STATE_N, PIC_STATE_NP1 = 0, 1
PIC_FLAG_COUNTS, PIC_FLAG_DIAG, PIC_FLAG_NO_STORE, PIC_FLAG_VSORT = 1, 2, 4, 8
PIC_FLAG_DEPOSIT_PER_VISIT = 16
PIC_FLAG_NO_DEPOSIT = 32
PIC_FLAG_ONE_PER_LANE = 64
PIC_FLAG_EXACT_TIME = 128
PIC_FLAG_STRIDED = 256
PIC_ERR_SUBSTEP_CAP = -4
PIC_ERR_UNSUPPORTED = -6
PIC_KE_NOALLOC_MAX_SPECIES = 8

EXPORTS = ["pic_init", "pic_move_accumulate", "pic_set_step", "pic_residual", "pic_commit",
           "pic_get_particles", "pic_get_counts", "pic_get_stats", "pic_set_flags",
           "pic_kinetic_energy", "pic_rho", "pic_jfnk_step", "pic_jfnk_step_dc",
           "pic_copy_state", "pic_destroy", "pic_last_error", "pic_last_kernel", "pic_version", "pic_count_histogram", "pic_microbench",
           "pic_debug_bounds", "pic_kinetic_energy_noalloc"]


class PicGrid(C.Structure):
    _fields_ = [("n_cells", C.c_int32), ("pad_", C.c_int32), ("length", C.c_double)]


class PicSpecies(C.Structure):
    _fields_ = [("q_over_m", C.c_double), ("macro_charge", C.c_double), ("n", C.c_int64)]


class PicParams(C.Structure):
    _fields_ = [("eps_a", C.c_double), ("eps_r", C.c_double), ("kappa_max", C.c_double),
                ("max_substeps", C.c_int32), ("picard_max", C.c_int32),
                ("precision", C.c_int32), ("cn_mode", C.c_int32), ("flags", C.c_uint32),
                ("pad_", C.c_int32)]


class PicStats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in
                ("n_sub", "n_cross", "n_picard_it", "n_picard_cap", "n_kappa_cap",
                 "n_substep_cap", "n_neg_disc", "n_clamped_tau", "n_launches")] + \
               [("last_move_ms", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class PicJfnkOpts(C.Structure):
    _fields_ = [("rtol", C.c_double), ("atol", C.c_double), ("fd_eps", C.c_double),
                ("gmres_rtol", C.c_double), ("max_newton", C.c_int32),
                ("gmres_restart", C.c_int32), ("max_gmres", C.c_int32), ("pad_", C.c_int32)]


class PicJfnkInfo(C.Structure):
    _fields_ = [("newton_its", C.c_int32), ("gmres_its", C.c_int32),
                ("mover_calls", C.c_int32), ("converged", C.c_int32),
                ("resid0", C.c_double), ("resid", C.c_double),
                ("mover_calls_resid", C.c_int32), ("pad_", C.c_int32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class PicError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"pic error {code}: {msg}")
        self.code = code


_lib = None


def lib_path():
    return _build.LIB


def load():
    """dlopen libpic_b200.so (building it first if the sources are newer).  Raises if absent.
    PIC_B200_CHECK=1 in the environment selects the bounds-checked debug build
    (libpic_b200_check.so, see pic_debug_bounds)."""
    global _lib
    if _lib is None:
        path = _build.build(check=os.environ.get("PIC_B200_CHECK", "0") == "1")
        if not os.path.exists(path):
            raise RuntimeError(f"CUDA extension missing: {path} (run __graft_entry__.build())")
        L = C.CDLL(path)
        L.pic_last_error.restype = C.c_char_p
        L.pic_last_error.argtypes = [C.c_void_p]
        L.pic_last_kernel.restype = C.c_char_p
        L.pic_last_kernel.argtypes = [C.c_void_p]
        for name in EXPORTS:
            getattr(L, name)  # fail loudly on a missing symbol
        _lib = L
    return _lib


def _ptr(a):
    """Raw address of a numpy array / torch tensor (contiguous), or None."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return C.c_void_p(a.ctypes.data)
    # torch tensor
    assert a.is_contiguous()
    return C.c_void_p(a.data_ptr())


def _check_f64(a, n, name):
    if isinstance(a, np.ndarray):
        ok, size = a.dtype == np.float64, a.size
    else:
        import torch
        ok, size = a.dtype == torch.float64, a.numel()
    if not ok or size != n:
        raise ValueError(f"{name}: need float64[{n}]")


MICROBENCH = {0: "ffma", 1: "ffma2", 2: "fmnmx", 3: "mufu_rsq", 4: "dfma", 5: "ffma2+fmnmx",
              6: "8ffma+4fmnmx", 7: "4ffma+4fmnmx", 8: "2ffma2+4ffma+4fmnmx", 9: "4ffma2+2mufu"}


def microbench(iters=20000, sm_mhz=1965.0):
    """P:86 micro-benchmarks: 1e9 thread-operations per second per instruction class, and the
    same per clock and SM at `sm_mhz`."""
    L = load()
    out = {}
    for which, name in MICROBENCH.items():
        gops, sms = C.c_double(0.0), C.c_int(0)
        rc = L.pic_microbench(C.c_int(which), C.c_int(iters), C.byref(gops), C.byref(sms))
        if rc != 0:
            raise PicError(rc, "pic_microbench")
        out[name] = {"thread_gops": gops.value,
                     "per_clk_per_sm": gops.value * 1e3 / (sms.value * sm_mhz)}
    return out


def debug_bounds(self_test=False):
    """pic_debug_bounds: index violations counted by the check build (-1: production build)."""
    v = C.c_int64(0)
    rc = load().pic_debug_bounds(C.byref(v), C.c_int(1 if self_test else 0))
    if rc != 0:
        raise PicError(rc, "pic_debug_bounds")
    return v.value


def version():
    buf = C.create_string_buffer(256)
    load().pic_version(buf, 256)
    return buf.value.decode()


class Pic:
    """Owner of one pic_handle.  Method names mirror the C-ABI entry points."""

    def __init__(self, n_cells, length, species, precision="fp32", cn_mode="direct",
                 eps_a=1e-8, eps_r=0.02, kappa_max=0.5, max_substeps=1 << 20, picard_max=100,
                 flags=0, stream=None):
        """pic_init.  species: list of dicts(q_over_m, w_q, x, v) with x, v float64 numpy
        arrays or torch tensors (host or CUDA).  stream: a cudaStream_t integer, e.g.
        torch.cuda.current_stream().cuda_stream (None = default stream)."""
        L = load()
        self._L = L
        self.n_cells, self.length = int(n_cells), float(length)
        self.n_species = len(species)
        self.n = [int(sp["x"].shape[0]) for sp in species]
        self.precision = precision
        grid = PicGrid(self.n_cells, 0, self.length)
        spec = (PicSpecies * self.n_species)(*[
            PicSpecies(float(sp["q_over_m"]), float(sp["w_q"]), n) for sp, n in zip(species, self.n)])
        for sp, n in zip(species, self.n):
            _check_f64(sp["x"], n, "x")
            _check_f64(sp["v"], n, "v")
        xs = (C.c_void_p * self.n_species)(*[_ptr(sp["x"]) for sp in species])
        vs = (C.c_void_p * self.n_species)(*[_ptr(sp["v"]) for sp in species])
        par = PicParams(eps_a, eps_r, kappa_max, max_substeps, picard_max,
                        PIC_FP32 if precision == "fp32" else PIC_FP64,
                        PIC_CN_DIRECT if cn_mode == "direct" else PIC_CN_PICARD, flags, 0)
        h = C.c_void_p()
        rc = L.pic_init(C.byref(h), C.byref(grid), spec, C.c_int(self.n_species), xs, vs,
                        C.byref(par), C.c_void_p(stream or 0))
        if rc != 0:
            raise PicError(rc, "pic_init failed (no CUDA device, bad particles or arguments)")
        self._h = h

    # -- helpers
    def _chk(self, rc, allow=()):
        if rc != 0 and rc not in allow:
            raise PicError(rc, self._L.pic_last_error(self._h).decode())
        return rc

    def close(self):
        if getattr(self, "_h", None):
            self._L.pic_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- C-ABI mirrors
    def move_accumulate(self, E_n, E_np1, dt, tol=1e-10, jbar_out=None, allow_cap=False):
        """pic_move_accumulate -> jbar (numpy float64[n_cells] unless jbar_out is given).
        PIC_ERR_SUBSTEP_CAP (orbits cut off at max_substeps: jbar is that of the truncated orbits)
        raises like every other error; allow_cap=True returns the truncated jbar instead."""
        out = np.empty(self.n_cells) if jbar_out is None else jbar_out
        self._chk(self._L.pic_move_accumulate(self._h, _ptr(E_n), _ptr(E_np1), C.c_double(dt),
                                              C.c_double(tol), _ptr(out)),
                  allow=(PIC_ERR_SUBSTEP_CAP,) if allow_cap else ())
        return out

    def set_step(self, E_n, dt, tol=1e-10):
        self._chk(self._L.pic_set_step(self._h, _ptr(E_n), C.c_double(dt), C.c_double(tol)))

    def residual(self, E_np1, resid_out=None, allow_cap=False):
        """pic_residual -> R (numpy float64[n_cells] unless resid_out is given); allow_cap as in
        move_accumulate."""
        out = np.empty(self.n_cells) if resid_out is None else resid_out
        self._chk(self._L.pic_residual(self._h, _ptr(E_np1), _ptr(out)),
                  allow=(PIC_ERR_SUBSTEP_CAP,) if allow_cap else ())
        return out

    def commit(self):
        self._chk(self._L.pic_commit(self._h))

    def get_particles(self, species=0, which=PIC_STATE_NP1):
        n = self.n[species]
        x, v, xi = np.empty(n), np.empty(n), np.empty(n)
        cell = np.empty(n, np.int32)
        self._chk(self._L.pic_get_particles(self._h, C.c_int(species), C.c_int(which), _ptr(x),
                                            _ptr(v), _ptr(cell), _ptr(xi)))
        return dict(x=x, v=v, cell=cell, xi=xi)

    def get_counts(self, species=0):
        n = self.n[species]
        a, b = np.empty(n, np.uint32), np.empty(n, np.uint32)
        self._chk(self._L.pic_get_counts(self._h, C.c_int(species), _ptr(a), _ptr(b)))
        return a, b

    def count_histogram(self, species=0, bin_width=1, n_bins=256):
        a, b = np.zeros(n_bins, np.uint64), np.zeros(n_bins, np.uint64)
        self._chk(self._L.pic_count_histogram(self._h, C.c_int(species), C.c_uint32(bin_width),
                                              C.c_int32(n_bins), _ptr(a), _ptr(b)))
        return a, b

    def get_stats(self):
        st = PicStats()
        self._chk(self._L.pic_get_stats(self._h, C.byref(st)))
        return st.as_dict()

    def last_kernel(self):
        return self._L.pic_last_kernel(self._h).decode()

    def set_flags(self, flags):
        self._chk(self._L.pic_set_flags(self._h, C.c_uint32(flags)))

    def kinetic_energy(self, which=PIC_STATE_N):
        out = np.empty(self.n_species)
        self._chk(self._L.pic_kinetic_energy(self._h, C.c_int(which), _ptr(out)))
        return out

    def kinetic_energy_noalloc(self, which=PIC_STATE_N, ke_out=None):
        """pic_kinetic_energy_noalloc: kinetic_energy() without any device allocation (block sums
        in the library's static 64 KiB device array), for programs that may not allocate in their
        time loop.  At most PIC_KE_NOALLOC_MAX_SPECIES species.  ke_out: float64[n_species] numpy
        array or CUDA tensor to fill (default: a new numpy array).  Calls that can overlap on
        the GPU share the array and race; make the first call on a device before any capture."""
        out = np.empty(self.n_species) if ke_out is None else ke_out
        _check_f64(out, self.n_species, "ke_out")
        self._chk(self._L.pic_kinetic_energy_noalloc(self._h, C.c_int(which), _ptr(out)))
        return out

    def rho(self, which=PIC_STATE_N, rho_out=None):
        out = np.empty(self.n_cells) if rho_out is None else rho_out
        self._chk(self._L.pic_rho(self._h, C.c_int(which), _ptr(out)))
        return out

    def copy_state_from(self, other):
        """pic_copy_state(self, other): state n of `other` becomes state n of this handle."""
        self._chk(self._L.pic_copy_state(self._h, other._h))

    def jfnk_step(self, E, dt, tol=1e-10, rtol=1e-8, atol=0.0, fd_eps=0.0, gmres_rtol=1e-2,
                  max_newton=20, gmres_restart=30, max_gmres=200, jacobian=None):
        """pic_jfnk_step: E (numpy float64[n_cells]) is E^n on entry, E^{n+1} on return.
        jacobian: another Pic built from the same particles (the fp32 mover) -> pic_jfnk_step_dc
        (defect correction: residual from this handle, Jacobian-vector products from that one)."""
        assert isinstance(E, np.ndarray) and E.dtype == np.float64
        opts = PicJfnkOpts(rtol, atol, fd_eps, gmres_rtol, max_newton, gmres_restart, max_gmres, 0)
        info = PicJfnkInfo()
        if jacobian is None:
            rc = self._L.pic_jfnk_step(self._h, _ptr(E), C.c_double(dt), C.c_double(tol),
                                       C.byref(opts), C.byref(info))
        else:
            rc = self._L.pic_jfnk_step_dc(self._h, jacobian._h, _ptr(E), C.c_double(dt),
                                          C.c_double(tol), C.byref(opts), C.byref(info))
        d = info.as_dict()
        d["rc"] = rc
        if rc != 0 and not (rc == -5 and not d["converged"]):
            self._chk(rc)
        return d
