"""CPU oracle for the GANDALF KRMHD hot path -- TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It wraps ``gandalf_oracle.cpp`` (plain
C++17 written from PAPER.md, see that file's header for the passage each function follows)
through ctypes.  It shares nothing with ``paper_2511_21891_b200``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gandalf_oracle.cpp")
_LIB = os.path.join(_HERE, "libgandalf_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 -fopenmp (it is never tuned beyond that)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c++17", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class OracleParams(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("M", C.c_int),
        ("Lx", C.c_double), ("Ly", C.c_double), ("Lz", C.c_double), ("vA", C.c_double),
        ("eta", C.c_double), ("r", C.c_int), ("eta_normalized", C.c_int),
        ("eta_z", C.c_double), ("r_z", C.c_int),
        ("eta_g", C.c_double),
        ("nu_coll", C.c_double), ("p", C.c_double),
        ("closure", C.c_int), ("if_variant", C.c_int), ("g_sign", C.c_int), ("nonlinear", C.c_int),
        ("hermite_coeff", C.c_int),
        ("force_eps", C.c_double), ("force_nperp_min", C.c_int), ("force_nperp_max", C.c_int),
        ("force_nz_max", C.c_int),
        ("seed", C.c_ulonglong),
        ("cfl", C.c_double),
        ("force_g_amp", C.c_double), ("force_g_nz", C.c_int),
        ("nspecies", C.c_int),
        ("dt_max", C.c_double),
        ("hermite_exact", C.c_int),
        ("m_offset", C.c_int), ("M_global", C.c_int),
    ]


_DEFAULTS = dict(M=0, Lx=2 * np.pi, Ly=2 * np.pi, Lz=2 * np.pi, vA=1.0, eta=0.0, r=1, eta_normalized=0,
                 eta_z=0.0, r_z=1, eta_g=0.0, nu_coll=0.0, p=1.0, closure=0, if_variant=0, g_sign=1,
                 nonlinear=1, hermite_coeff=0, force_eps=0.0, force_nperp_min=1, force_nperp_max=2,
                 force_nz_max=1, seed=0, cfl=0.3, force_g_amp=0.0, force_g_nz=1, nspecies=1, dt_max=0.0, hermite_exact=0,
                 m_offset=0, M_global=0)

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        P = C.POINTER(C.c_double)
        lib.oracle_create.argtypes = [C.POINTER(OracleParams), C.POINTER(C.c_void_p)]
        lib.oracle_destroy.argtypes = [C.c_void_p]
        lib.oracle_set_state.argtypes = [C.c_void_p, P, P]
        lib.oracle_get_state.argtypes = [C.c_void_p, P, P]
        lib.oracle_rhs.argtypes = [C.c_void_p, P, P]
        lib.oracle_step.argtypes = [C.c_void_p, C.c_double, C.c_int]
        lib.oracle_energy.argtypes = [C.c_void_p, P]
        lib.oracle_kperp_spectrum.argtypes = [C.c_void_p, C.c_int, C.c_int, P]
        lib.oracle_hermite_spectrum.argtypes = [C.c_void_p, P]
        lib.oracle_kpar_spectrum.argtypes = [C.c_void_p, C.c_int, P]
        lib.oracle_truncation_ratio.argtypes = [C.c_void_p, P]
        lib.oracle_energy_history.argtypes = [C.c_void_p, C.c_int, P, C.POINTER(C.c_int)]
        lib.oracle_get_time.argtypes = [C.c_void_p, P, C.POINTER(C.c_longlong), P]
        lib.oracle_set_time.argtypes = [C.c_void_p, C.c_double, C.c_longlong]
        lib.oracle_last_error.argtypes = [C.c_void_p]
        lib.oracle_last_error.restype = C.c_char_p
        lib.oracle_fft1d.argtypes = [C.c_int, C.c_int, P, P]
        lib.oracle_dft1d.argtypes = [C.c_int, C.c_int, P, P]
        lib.oracle_fft1d.restype = None
        lib.oracle_dft1d.restype = None
        lib.oracle_bracket_full.argtypes = [C.c_void_p, P, P, P, P]
        lib.oracle_get_full.argtypes = [C.c_void_p, C.c_int, P]
        lib.oracle_set_full.argtypes = [C.c_void_p, C.c_int, P]
        lib.oracle_step_stage.argtypes = [C.c_void_p, C.c_double, C.c_int]
        lib.oracle_get_stage_full.argtypes = [C.c_void_p, C.c_int, P]
        lib.oracle_set_stage_full.argtypes = [C.c_void_p, C.c_int, P]
        lib.oracle_num_threads.restype = C.c_int
        lib.oracle_set_num_threads.argtypes = [C.c_int]
        lib.oracle_set_num_threads.restype = None
        _lib = lib
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _as_pairs(a) -> np.ndarray:
    """complex128 array -> contiguous float64 view with a trailing (re, im) axis."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a.view(np.float64)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def fft1d(x, sign: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    _load().oracle_fft1d(x.size, sign, _dp(x.view(np.float64)), _dp(out.view(np.float64)))
    return out


def dft1d(x, sign: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    _load().oracle_dft1d(x.size, sign, _dp(x.view(np.float64)), _dp(out.view(np.float64)))
    return out


class Oracle:
    """One oracle context.  Arrays at the boundary are complex128 numpy arrays of shape
    (fields, nz, ny, nx//2+1): the potentials zeta = xi^+- (2 fields) and g_m (M fields)."""

    def __init__(self, nx, ny, nz, **kw):
        lib = _load()
        vals = dict(_DEFAULTS)
        for k in kw:
            if k not in vals:
                raise TypeError(f"unknown oracle parameter {k!r}")
        vals.update(kw)
        self.params = OracleParams(nx=nx, ny=ny, nz=nz, **vals)
        self.nx, self.ny, self.nz, self.M = nx, ny, nz, int(vals["M"]) * int(vals["nspecies"])   # M = moment FIELDS
        self.hx = nx // 2 + 1
        h = C.c_void_p()
        rc = lib.oracle_create(C.byref(self.params), C.byref(h))
        if rc != 0:
            raise ValueError(f"oracle_create failed: {rc}")
        self._h = h
        self._lib = lib

    def close(self):
        if getattr(self, "_h", None):
            self._lib.oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, what):
        if rc != 0:
            raise RuntimeError(f"{what} failed ({rc}): {self._lib.oracle_last_error(self._h).decode()}")

    def _half(self, nf):
        return np.zeros((nf, self.nz, self.ny, self.hx), dtype=np.complex128)

    def set_state(self, zeta_hat, g_hat=None):
        z = np.ascontiguousarray(zeta_hat, dtype=np.complex128)
        assert z.shape == (2, self.nz, self.ny, self.hx), z.shape
        if self.M > 0:
            g = np.ascontiguousarray(g_hat, dtype=np.complex128)
            assert g.shape == (self.M, self.nz, self.ny, self.hx), g.shape
        else:
            g = np.zeros(1, dtype=np.complex128)
        self._check(self._lib.oracle_set_state(self._h, _dp(z.view(np.float64)), _dp(g.view(np.float64))), "set_state")

    def get_state(self):
        z = self._half(2)
        g = self._half(max(self.M, 1))
        self._check(self._lib.oracle_get_state(self._h, _dp(z.view(np.float64)), _dp(g.view(np.float64))), "get_state")
        return z, g[: self.M]

    def rhs(self):
        dw = self._half(2)
        dg = self._half(max(self.M, 1))
        self._check(self._lib.oracle_rhs(self._h, _dp(dw.view(np.float64)), _dp(dg.view(np.float64))), "rhs")
        return dw, dg[: self.M]

    def step(self, dt, nsteps=1):
        self._check(self._lib.oracle_step(self._h, float(dt), int(nsteps)), "step")

    def energy(self):
        out = np.zeros(6)
        self._check(self._lib.oracle_energy(self._h, _dp(out)), "energy")
        return out

    def kperp_spectrum(self, nbins, literal_eq26=False):
        out = np.zeros(nbins)
        self._check(self._lib.oracle_kperp_spectrum(self._h, nbins, int(literal_eq26), _dp(out)), "spectrum")
        return out

    def hermite_spectrum(self):
        out = np.zeros(max(self.M, 1))
        self._check(self._lib.oracle_hermite_spectrum(self._h, _dp(out)), "hermite spectrum")
        return out[: self.M]

    def truncation_ratio(self):
        out = np.zeros(1)
        self._check(self._lib.oracle_truncation_ratio(self._h, _dp(out)), "truncation ratio")
        return float(out[0])

    def kpar_spectrum(self, nbins):
        out = np.zeros(nbins)
        self._check(self._lib.oracle_kpar_spectrum(self._h, nbins, _dp(out)), "kpar spectrum")
        return out

    def energy_history(self, max_records=1 << 20):
        n = C.c_int(0)
        self._check(self._lib.oracle_energy_history(self._h, 0, None, C.byref(n)), "history")
        # first call with max 0 returns 0 records; ask for the real count with a large buffer
        buf = np.zeros((max_records, 7))
        self._check(self._lib.oracle_energy_history(self._h, max_records, _dp(buf), C.byref(n)), "history")
        return buf[: n.value].copy()

    def time(self):
        t = C.c_double(0)
        s = C.c_longlong(0)
        d = C.c_double(0)
        self._lib.oracle_get_time(self._h, C.byref(t), C.byref(s), C.byref(d))
        return t.value, s.value, d.value

    def set_time(self, t, step):
        self._check(self._lib.oracle_set_time(self._h, float(t), int(step)), "set_time")

    # full-spectrum helpers used by the pins
    def bracket_full(self, f_hat, g_hat):
        f = np.ascontiguousarray(f_hat, dtype=np.complex128)
        g = np.ascontiguousarray(g_hat, dtype=np.complex128)
        assert f.shape == (self.nz, self.ny, self.nx) and g.shape == f.shape
        out = np.empty_like(f)
        mi = C.c_double(0)
        self._check(self._lib.oracle_bracket_full(self._h, _dp(f.view(np.float64)), _dp(g.view(np.float64)),
                                                  _dp(out.view(np.float64)), C.byref(mi)), "bracket")
        return out, mi.value

    def step_stage(self, dt, stage):
        """One stage of a step (0: RHS + predictor, 1: midpoint RHS + corrector + ...); a moment-sharded run refreshes its
        halo moments in between (Q31)."""
        self._check(self._lib.oracle_step_stage(self._h, float(dt), int(stage)), "step_stage")

    def get_stage_full(self, field):
        out = np.empty((self.nz, self.ny, self.nx), dtype=np.complex128)
        self._check(self._lib.oracle_get_stage_full(self._h, field, _dp(out.view(np.float64))), "get_stage_full")
        return out

    def set_stage_full(self, field, a):
        a = np.ascontiguousarray(a, dtype=np.complex128)
        assert a.shape == (self.nz, self.ny, self.nx)
        self._check(self._lib.oracle_set_stage_full(self._h, field, _dp(a.view(np.float64))), "set_stage_full")

    def get_full(self, field):
        out = np.empty((self.nz, self.ny, self.nx), dtype=np.complex128)
        self._check(self._lib.oracle_get_full(self._h, field, _dp(out.view(np.float64))), "get_full")
        return out

    def set_full(self, field, a):
        a = np.ascontiguousarray(a, dtype=np.complex128)
        assert a.shape == (self.nz, self.ny, self.nx)
        self._check(self._lib.oracle_set_full(self._h, field, _dp(a.view(np.float64))), "set_full")
