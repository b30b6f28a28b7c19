"""ctypes wrapper around the CPU oracle `libgkref.so` (oracle/gkref.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libgkref.so")
_SRC = [os.path.join(_HERE, "gkref.cpp"), os.path.join(_HERE, "gkref.h")]

T_I, T_II, T_IV, T_V, T_VII, T_VIII, T_DISS_S, T_DISS_V, T_HYP, T_III = (1 << k for k in range(10))
T_ALL = 1023


def build(force: bool = False) -> str:
    """Compile the oracle with g++ if the shared object is missing or older than its source."""
    stale = force or not os.path.exists(_SO) or any(
        os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if stale:
        tmp = _SO + f".{os.getpid()}.tmp"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC",
                               _SRC[0], "-o", tmp])
        os.replace(tmp, _SO)
    return _SO


class _Grid(C.Structure):
    _fields_ = [("nkx", C.c_int), ("nky", C.c_int), ("ns", C.c_int), ("nvpar", C.c_int),
                ("nmu", C.c_int), ("ky0", C.c_double), ("ikxspace", C.c_int),
                ("vpar_max", C.c_double), ("mu_grid", C.c_int), ("vperp_max", C.c_double)]


class _Species(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("Z", "mass", "temp", "dens", "rlt", "rln")]


class _Geom(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("q", "shat", "eps")]


class _Opts(C.Structure):
    _fields_ = [("nspecies", C.c_int), ("adiabatic_electrons", C.c_int), ("te", C.c_double),
                ("ne", C.c_double), ("nonlinear", C.c_int), ("disp_par", C.c_double),
                ("disp_vp", C.c_double), ("disp_x", C.c_double), ("disp_y", C.c_double),
                ("s_closure", C.c_int), ("term_mask", C.c_int), ("bracket_method", C.c_int),
                ("pad_mx", C.c_int), ("pad_my", C.c_int), ("geometry", C.c_int)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        lib.gkref_create.restype = C.c_void_p
        lib.gkref_create.argtypes = [C.POINTER(_Grid), C.POINTER(_Species), C.POINTER(_Geom),
                                     C.POINTER(_Opts)]
        lib.gkref_destroy.argtypes = [C.c_void_p]
        lib.gkref_set_threads.restype = C.c_int
        lib.gkref_set_threads.argtypes = [C.c_int]
        lib.gkref_field_solve.argtypes = [C.c_void_p, dp, dp]
        lib.gkref_rhs.argtypes = [C.c_void_p, dp, dp, dp]
        lib.gkref_rhs_slab.argtypes = [C.c_void_p, dp, dp, C.c_int, C.c_int, C.c_int, C.c_int, dp]
        lib.gkref_rk4_step.argtypes = [C.c_void_p, dp, C.c_double]
        lib.gkref_fluxes.argtypes = [C.c_void_p, dp, dp, dp]
        lib.gkref_spectra.argtypes = [C.c_void_p, dp, dp, dp]
        lib.gkref_estimate_dt.argtypes = [C.c_void_p, dp, dp]
        lib.gkref_bracket_slab.argtypes = [C.c_void_p, dp, dp, C.c_int, C.c_int, C.c_int, dp]
        lib.gkref_table.restype = C.c_size_t
        lib.gkref_table.argtypes = [C.c_void_p, C.c_char_p, dp]
        _lib = lib
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def set_threads(n: int = 0) -> int:
    return _load().gkref_set_threads(n)


class GkRef:
    """Oracle context for one configuration dictionary (see gkinputs.CONFIGS)."""

    def __init__(self, cfg: dict, term_mask: int = 0, bracket_method: int = 0, pad=(0, 0)):
        lib = _load()
        g, o = cfg["grid"], cfg["opts"]
        self.cfg = cfg
        self.nsp = len(cfg["species"])
        self.shape = (self.nsp, g["nvpar"], g["nmu"], g["ns"], g["nkx"], g["nky"])
        self.phi_shape = (g["ns"], g["nkx"], g["nky"])
        grid = _Grid(g["nkx"], g["nky"], g["ns"], g["nvpar"], g["nmu"], g["ky0"], g["ikxspace"],
                     g["vpar_max"], g["mu_grid"], g["vperp_max"])
        sp = (_Species * self.nsp)(*[_Species(s["Z"], s["mass"], s["temp"], s["dens"], s["rlt"],
                                              s["rln"]) for s in cfg["species"]])
        geo = _Geom(cfg["geom"]["q"], cfg["geom"]["shat"], cfg["geom"]["eps"])
        opts = _Opts(self.nsp, o["adiabatic_electrons"], o["te"], o["ne"], o["nonlinear"],
                     o["disp_par"], o["disp_vp"], o["disp_x"], o["disp_y"], o["s_closure"],
                     term_mask, bracket_method, pad[0], pad[1], int(o.get("geometry", 0)))
        self._h = lib.gkref_create(C.byref(grid), sp, C.byref(geo), C.byref(opts))
        if not self._h:
            raise ValueError("gkref_create rejected the configuration")

    def __del__(self):
        if getattr(self, "_h", None):
            _load().gkref_destroy(self._h)
            self._h = None

    @staticmethod
    def _c128(a, shape):
        a = np.ascontiguousarray(a, dtype=np.complex128)
        assert a.shape == tuple(shape), (a.shape, shape)
        return a

    def field_solve(self, f):
        f = self._c128(f, self.shape)
        phi = np.empty(self.phi_shape, np.complex128)
        _load().gkref_field_solve(self._h, _dp(f), _dp(phi))
        return phi

    def rhs(self, f):
        f = self._c128(f, self.shape)
        phi = np.empty(self.phi_shape, np.complex128)
        out = np.empty(self.shape, np.complex128)
        _load().gkref_rhs(self._h, _dp(f), _dp(phi), _dp(out))
        return out, phi

    def rhs_slab(self, f, phi, a, j, l, i):
        f = self._c128(f, self.shape)
        phi = self._c128(phi, self.phi_shape)
        out = np.empty(self.shape[4:], np.complex128)
        _load().gkref_rhs_slab(self._h, _dp(f), _dp(phi), a, j, l, i, _dp(out))
        return out

    def rk4_step(self, f, dt, steps: int = 1):
        f = self._c128(f, self.shape).copy()
        for _ in range(steps):
            _load().gkref_rk4_step(self._h, _dp(f), float(dt))
        return f

    def fluxes(self, f, phi):
        f = self._c128(f, self.shape)
        phi = self._c128(phi, self.phi_shape)
        out = np.empty((self.nsp, 3), np.float64)
        _load().gkref_fluxes(self._h, _dp(f), _dp(phi), _dp(out))
        return out

    def spectra(self, phi):
        """(kx_spec[nkx], ky_spec[nky]) of |phi|^2."""
        phi = self._c128(phi, self.phi_shape)
        kxs, kys = np.empty(self.shape[4], np.float64), np.empty(self.shape[5], np.float64)
        _load().gkref_spectra(self._h, _dp(phi), _dp(kxs), _dp(kys))
        return kxs, kys

    def estimate_dt(self, phi):
        """(dt, dt_nl, dt_lin, dt_field): largest RK4-stable steps (R21-R23), no safety factor."""
        phi = self._c128(phi, self.phi_shape)
        out = np.empty(4, np.float64)
        _load().gkref_estimate_dt(self._h, _dp(phi), _dp(out))
        return out

    def bracket_slab(self, chi, fs, method=0, mx=0, my=0):
        chi = self._c128(chi, self.shape[4:])
        fs = self._c128(fs, self.shape[4:])
        out = np.empty(self.shape[4:], np.complex128)
        _load().gkref_bracket_slab(self._h, _dp(chi), _dp(fs), method, mx, my, _dp(out))
        return out

    def table(self, which: str) -> np.ndarray:
        n = _load().gkref_table(self._h, which.encode(), None)
        if n == 0:
            raise KeyError(which)
        out = np.empty(n, np.float64)
        _load().gkref_table(self._h, which.encode(), _dp(out))
        g = self.cfg["grid"]
        shapes = {"J0": (self.nsp, g["nmu"], g["ns"], g["nkx"], g["nky"]),
                  "Gamma0": (self.nsp, g["ns"], g["nkx"], g["nky"]),
                  "FM": (g["nvpar"], g["nmu"], g["ns"]),
                  "Apol": self.phi_shape, "kperp2": self.phi_shape, "kappa": self.phi_shape,
                  "sclass": self.phi_shape, "dcoef": (5, 2, 5)}
        # further names: "ef" (ExB factor relative to ky/2), "gpz", "gzz" (normalised metric), "kthnorm", "dkx"
        return out.reshape(shapes.get(which, (n,)))
