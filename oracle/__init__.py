"""CPU test oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT) — ctypes wrapper around oracle/liboracle.so.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It does not import, and is not imported by, paper_1810_12707_b200's CUDA binding.
"""
from __future__ import annotations

import ctypes as C
import math

import numpy as np

from . import build_oracle

_lib = None


class OrcDiag(C.Structure):
    _fields_ = [("t", C.c_double), ("step", C.c_longlong), ("ke", C.c_double), ("me", C.c_double),
                ("ie", C.c_double), ("mass", C.c_double), ("mom", C.c_double * 3), ("etot", C.c_double),
                ("max_divb", C.c_double), ("rho_min", C.c_double), ("p_min", C.c_double)]


def lib():
    global _lib
    if _lib is None:
        path = build_oracle.build()
        L = C.CDLL(path)
        PP = C.POINTER(C.c_void_p)
        L.orc_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_double, C.c_double, C.c_double,
                                 C.c_double, C.c_double, C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_last_error.restype = C.c_char_p
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_get_threads.restype = C.c_int
        L.orc_use_direct_dft.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_variant.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int]
        L.orc_set_integrator.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_stress.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_fields.argtypes = [C.c_void_p, C.c_int, PP]
        L.orc_get_fields.argtypes = [C.c_void_p, C.c_int, PP]
        L.orc_rhs.argtypes = [C.c_void_p, PP]
        L.orc_rhs_scales.argtypes = [C.c_void_p, PP, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_step.argtypes = [C.c_void_p, C.c_int]
        L.orc_nspec.argtypes = [C.c_void_p]
        L.orc_diagnostics.argtypes = [C.c_void_p, C.POINTER(OrcDiag), C.c_void_p, C.c_void_p, C.c_int]
        L.orc_apply.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_fft3.argtypes = [C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_dft3_direct.argtypes = [C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_cic.argtypes = [C.c_int, C.c_double, C.c_int, PP, C.c_longlong, PP, PP]
        L.orc_tracers_push.argtypes = [C.c_int, C.c_double, C.c_double, PP, C.c_longlong, PP, PP, C.c_int]
        L.orc_tracers_set.argtypes = [C.c_void_p, C.c_longlong, PP, PP]
        L.orc_tracers_get.argtypes = [C.c_void_p, PP, PP]
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise RuntimeError("oracle: " + lib().orc_last_error().decode())


def _ptrs(arrs):
    a = (C.c_void_p * 8)()
    for i, x in enumerate(arrs):
        a[i] = x.ctypes.data
    return a


def set_threads(n: int):
    lib().orc_set_threads(int(n))


def get_threads() -> int:
    return int(lib().orc_get_threads())


def _c_in(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def fft3(a: np.ndarray, sign: int = -1, long_double: bool = False, direct: bool = False) -> np.ndarray:
    """3-D DFT of a complex [N][N][N] array with the oracle's own FFT (or the O(N^6) definition)."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    N = a.shape[0]
    assert a.shape == (N, N, N)
    out = np.empty_like(a)
    fn = lib().orc_dft3_direct if direct else lib().orc_fft3
    _check(fn(N, int(sign), int(long_double), a.ctypes.data, out.ctypes.data))
    return out


def _ptrn(arrs):
    a = (C.c_void_p * len(arrs))()
    for i, x in enumerate(arrs):
        a[i] = x.ctypes.data
    return a


def cic(fields, pos, L=2 * math.pi):
    """Eq. 20: cloud-in-cell interpolation of the [N][N][N] grid fields to the positions pos (3 arrays of np)."""
    g = [_c_in(x) for x in fields]
    N = g[0].shape[0]
    p = [_c_in(x) for x in pos]
    n = p[0].size
    out = [np.empty(n) for _ in g]
    _check(lib().orc_cic(N, L, len(g), _ptrn(g), n, _ptrn(p), _ptrn(out)))
    return out


def tracers_push(B, pos, vel, dt, nsteps=1, L=2 * math.pi):
    """nsteps Boris pushes (Eq. 21-22) in the frozen grid field B; returns new (pos, vel)."""
    g = [_c_in(x) for x in B]
    N = g[0].shape[0]
    p = [np.array(x, dtype=np.float64) for x in pos]
    v = [np.array(x, dtype=np.float64) for x in vel]
    _check(lib().orc_tracers_push(N, L, dt, _ptrn(g), p[0].size, _ptrn(p), _ptrn(v), int(nsteps)))
    return p, v


class Oracle:
    """One solver instance.  Fields are lists of 8 float64 [N][N][N] arrays (z,y,x)."""

    def __init__(self, N, L=2 * math.pi, gamma=5.0 / 3.0, mu=0.0, eta=0.0, dt=1e-3, long_double=False):
        self.N = int(N)
        self._h = C.c_void_p()
        _check(lib().orc_create(C.byref(self._h), self.N, L, gamma, mu, eta, dt, int(long_double)))

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _new(self):
        return [np.empty((self.N,) * 3, dtype=np.float64) for _ in range(8)]

    def use_direct_dft(self, on=True):
        _check(lib().orc_use_direct_dft(self._h, int(on)))

    def set_stress(self, on=True):
        """Viscous terms of PAPER.md Eq. 11-12 (div(2 nu rho S), energy flux -2 nu rho u.S) instead of mu lap u."""
        _check(lib().orc_set_stress(self._h, int(bool(on))))

    def set_integrator(self, which):
        """'ab2' (default), 'rk4' or 'pc' (predictor-corrector / Heun)."""
        _check(lib().orc_set_integrator(self._h, {"ab2": 0, "rk4": 1, "pc": 2}[which]))

    def set_variant(self, cs2=0.0, f0=0.0, kf=1, evolve=3):
        """Equation-set variants: barotropic closure (cs2 > 0), ABC forcing (f0, kf), switched-off equations."""
        _check(lib().orc_set_variant(self._h, float(cs2), float(f0), int(kf), int(evolve)))

    def set_fields(self, fields, kind="primitive"):
        f = [_c_in(x) for x in fields]
        assert len(f) == 8 and all(x.shape == (self.N,) * 3 for x in f)
        _check(lib().orc_set_fields(self._h, 1 if kind == "primitive" else 0, _ptrs(f)))

    def get_fields(self, kind="conservative"):
        out = self._new()
        _check(lib().orc_get_fields(self._h, 1 if kind == "primitive" else 0, _ptrs(out)))
        return out

    def rhs(self):
        out = self._new()
        _check(lib().orc_rhs(self._h, _ptrs(out)))
        return out

    def rhs_scales(self):
        """(R, phi, dsc): RHS plus per-field stacked-flux norm and diffusion scale."""
        out = self._new()
        phi = (C.c_double * 8)()
        dsc = (C.c_double * 8)()
        _check(lib().orc_rhs_scales(self._h, _ptrs(out), phi, dsc))
        return out, np.array(phi[:]), np.array(dsc[:])

    def step(self, n=1):
        _check(lib().orc_step(self._h, int(n)))

    def nspec(self):
        return int(lib().orc_nspec(self._h))

    def diagnostics(self, spectra=False):
        d = OrcDiag()
        if spectra:
            ns = self.nspec()
            sk = np.zeros(ns)
            sm = np.zeros(ns)
            _check(lib().orc_diagnostics(self._h, C.byref(d), sk.ctypes.data, sm.ctypes.data, ns))
        else:
            sk = sm = None
            _check(lib().orc_diagnostics(self._h, C.byref(d), None, None, 0))
        out = {k: getattr(d, k) for k in ("t", "step", "ke", "me", "ie", "mass", "etot", "max_divb",
                                            "rho_min", "p_min")}
        out["mom"] = [d.mom[0], d.mom[1], d.mom[2]]
        if spectra:
            out["spec_kin"], out["spec_mag"] = sk, sm
        return out

    def tracers_set(self, pos, vel=None):
        p = [_c_in(x) for x in pos]
        self._np = p[0].size
        v = [_c_in(x) for x in vel] if vel is not None else None
        _check(lib().orc_tracers_set(self._h, self._np, _ptrn(p), _ptrn(v) if v is not None else None))

    def tracers_get(self):
        p = [np.empty(self._np) for _ in range(3)]
        v = [np.empty(self._np) for _ in range(3)]
        _check(lib().orc_tracers_get(self._h, _ptrn(p), _ptrn(v)))
        return p, v

    def apply(self, op, f):
        names = {"dx": 0, "dy": 1, "dz": 2, "lap": 3, "project": 4}
        f = _c_in(f)
        out = np.empty_like(f)
        _check(lib().orc_apply(self._h, names[op], f.ctypes.data, out.ctypes.data))
        return out
