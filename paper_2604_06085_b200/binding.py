"""Thin ctypes binding of libgk.so with the same names as include/gk.h.  Argument marshalling only:
every step of the path runs in the CUDA kernels.  Tensors are torch CUDA tensors used as device
buffers (complex64, or complex-half viewed as (..., 2) float16/bfloat16)."""
from __future__ import annotations

import ctypes as C
import os
import re

from . import build as _build

T_I, T_II, T_IV, T_V, T_VII, T_VIII, T_DISS_S, T_DISS_V, T_HYP, T_III = (1 << k for k in range(10))
T_ALL = 1023

GK_OK, GK_EINVAL, GK_ENOMEM, GK_ECUDA, GK_EUNSUPPORTED = 0, -1, -2, -3, -4
_ERRNAMES = {GK_EINVAL: "GK_EINVAL", GK_ENOMEM: "GK_ENOMEM", GK_ECUDA: "GK_ECUDA",
             GK_EUNSUPPORTED: "GK_EUNSUPPORTED"}


class GkError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_ERRNAMES.get(code, code)}: {msg}")
        self.code = code


class _Grid(C.Structure):
    _fields_ = [("nkx", C.c_int), ("nky", C.c_int), ("ns", C.c_int), ("nvpar", C.c_int),
                ("nmu", C.c_int), ("ky0", C.c_double), ("ikxspace", C.c_int),
                ("vpar_max", C.c_double), ("mu_grid", C.c_int), ("vperp_max", C.c_double)]


class _Species(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("Z", "mass", "temp", "dens", "rlt", "rln")]


class _Salpha(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("q", "shat", "eps")]


class _Opts(C.Structure):
    _fields_ = [("nspecies", C.c_int), ("adiabatic_electrons", C.c_int), ("te", C.c_double),
                ("ne", C.c_double), ("nonlinear", C.c_int), ("disp_par", C.c_double),
                ("disp_vp", C.c_double), ("disp_x", C.c_double), ("disp_y", C.c_double),
                ("s_closure", C.c_int), ("storage", C.c_int), ("term_mask", C.c_int),
                ("pad_mx", C.c_int), ("pad_my", C.c_int), ("geometry", C.c_int)]


def lib_path() -> str:
    return _build.LIB


def exported_symbols() -> list[str]:
    """Names declared in include/*.h (functions)."""
    src = ""
    for name in sorted(os.listdir(_build.INCLUDE)):
        if name.endswith(".h"):
            with open(os.path.join(_build.INCLUDE, name)) as fh:
                src += fh.read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gk_[a-z0-9_]+)\s*\(", src)))


_lib = None


def load_library(build_if_missing: bool = True):
    """dlopen libgk.so (building it with nvcc first if it is missing or stale).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        _build.build()
    if not os.path.exists(_build.LIB):
        raise ImportError(f"{_build.LIB} is missing: run `python -m paper_2604_06085_b200.build`")
    lib = C.CDLL(_build.LIB)
    vp, dp = C.c_void_p, C.POINTER(C.c_double)
    lib.gk_create.argtypes = [C.POINTER(_Grid), C.POINTER(_Species), C.POINTER(_Salpha),
                              C.POINTER(_Opts), vp, C.POINTER(vp)]
    lib.gk_destroy.argtypes = [vp]
    lib.gk_workspace_bytes.restype = C.c_size_t
    lib.gk_workspace_bytes.argtypes = [vp]
    lib.gk_workspace_bytes_rhs.restype = C.c_size_t
    lib.gk_workspace_bytes_rhs.argtypes = [vp]
    lib.gk_set_workspace.argtypes = [vp, vp, C.c_size_t]
    lib.gk_field_solve.argtypes = [vp, vp, vp]
    lib.gk_rhs.argtypes = [vp, vp, vp, vp]
    lib.gk_rk4_step.argtypes = [vp, vp, C.c_double]
    lib.gk_rk4_steps.argtypes = [vp, vp, C.c_double, C.c_int]
    lib.gk_fluxes.argtypes = [vp, vp, vp, dp]
    lib.gk_rk4_step_host.argtypes = [vp, vp, vp, vp, C.c_double]
    lib.gk_rk4_batch_host.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.c_int, vp, vp, C.c_double]
    lib.gk_spectra.argtypes = [vp, vp, dp, dp]
    lib.gk_spectra_static.argtypes = [vp, C.c_int, C.c_int, C.c_int, dp, dp, vp]
    lib.gk_spectra_static_max.restype = C.c_size_t
    lib.gk_spectra_static_max.argtypes = []
    lib.gk_spectra_static_error.restype = C.c_char_p
    lib.gk_spectra_static_error.argtypes = []
    lib.gk_set_diagnostics.argtypes = [vp, C.c_int]
    lib.gk_fluxes_last.argtypes = [vp, dp]
    lib.gk_estimate_dt.argtypes = [vp, dp]
    lib.gk_reset_cfl.argtypes = [vp]
    lib.gk_rk4_steps_cfl.argtypes = [vp, vp, C.c_int, C.c_double, C.c_double, dp, dp]
    lib.gk_export_table.restype = C.c_size_t
    lib.gk_export_table.argtypes = [vp, C.c_char_p, dp, C.c_size_t]
    lib.gk_launch_count.restype = C.c_longlong
    lib.gk_launch_count.argtypes = [vp]
    lib.gk_set_profiling.argtypes = [vp, C.c_int]
    lib.gk_stage_kernel_time.argtypes = [vp, dp, C.POINTER(C.c_longlong), C.c_int]
    lib.gk_last_error.restype = C.c_char_p
    lib.gk_last_error.argtypes = [vp]
    lib.gk_version.restype = C.c_char_p
    _lib = lib
    return lib


def gk_spectra_static(phi, stream=None):
    """(kx_spec[nkx], ky_spec[nky]) of |phi|^2 without a context and without any device allocation: for hosts of
    this library whose device memory is already fully claimed by another allocator, or capped, so that gk_create's
    cudaMalloc calls cannot succeed.  `phi`: contiguous CUDA complex64 tensor [ns, nkx, nky] on the current device;
    nkx + nky <= gk_spectra_static_max().  The device-side staging array is shared by every call: do not overlap
    calls.  Same numbers as GkContext.gk_spectra."""
    import numpy as np
    import torch
    lib = load_library()
    if not (phi.is_cuda and phi.dtype == torch.complex64 and phi.is_contiguous() and phi.dim() == 3):
        raise ValueError("phi: expected a contiguous CUDA complex64 tensor [ns, nkx, nky]")
    ns, nkx, nky = (int(n) for n in phi.shape)
    kxs, kys = np.zeros(nkx, np.float64), np.zeros(nky, np.float64)
    st = stream if stream is not None else torch.cuda.current_stream(phi.device)
    with torch.cuda.device(phi.device):
        rc = lib.gk_spectra_static(C.c_void_p(phi.data_ptr()), ns, nkx, nky, kxs.ctypes.data_as(C.POINTER(C.c_double)),
                                   kys.ctypes.data_as(C.POINTER(C.c_double)), C.c_void_p(st.cuda_stream))
    if rc != GK_OK:
        raise GkError(rc, lib.gk_spectra_static_error().decode())
    return kxs, kys


def gk_spectra_static_max() -> int:
    return int(load_library().gk_spectra_static_max())


_STORAGE = {"complex64": 0, "fp16": 1, "bf16": 2, 0: 0, 1: 1, 2: 2}


class GkContext:
    """One gk_ctx.  `cfg` is a configuration dictionary as in gkinputs.CONFIGS."""

    def __init__(self, cfg: dict, device="cuda:0", term_mask: int = 0, pad=(0, 0), stream=None,
                 full_workspace: bool = True):
        import torch
        if not torch.cuda.is_available():
            raise GkError(GK_ECUDA, "no CUDA device: libgk has no CPU fallback")
        self._torch = torch
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        g, o = cfg["grid"], cfg["opts"]
        self.cfg = cfg
        self.nsp = len(cfg["species"])
        self.shape = (self.nsp, g["nvpar"], g["nmu"], g["ns"], g["nkx"], g["nky"])
        self.phi_shape = (g["ns"], g["nkx"], g["nky"])
        self.storage = _STORAGE[o.get("storage", 0)]
        grid = _Grid(g["nkx"], g["nky"], g["ns"], g["nvpar"], g["nmu"], g["ky0"], g["ikxspace"],
                     g["vpar_max"], g["mu_grid"], g["vperp_max"])
        sp = (_Species * self.nsp)(*[_Species(s["Z"], s["mass"], s["temp"], s["dens"], s["rlt"],
                                              s["rln"]) for s in cfg["species"]])
        geo = _Salpha(cfg["geom"]["q"], cfg["geom"]["shat"], cfg["geom"]["eps"])
        opts = _Opts(self.nsp, o["adiabatic_electrons"], o["te"], o["ne"], o["nonlinear"],
                     o["disp_par"], o["disp_vp"], o["disp_x"], o["disp_y"], o["s_closure"],
                     self.storage, term_mask, pad[0], pad[1], int(o.get("geometry", 0)))
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = self.lib.gk_create(C.byref(grid), sp, C.byref(geo), C.byref(opts),
                                C.c_void_p(self._stream.cuda_stream), C.byref(h))
        self._h = h
        if rc != GK_OK:
            msg = self.lib.gk_last_error(h).decode() if h else "gk_create failed"
            if h:
                self.lib.gk_destroy(h)
            self._h = None
            raise GkError(rc, msg)
        nbytes = self.lib.gk_workspace_bytes(h) if full_workspace else self.lib.gk_workspace_bytes_rhs(h)
        self._ws = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=self.device)
        self._check(self.lib.gk_set_workspace(h, C.c_void_p(self._ws.data_ptr()), C.c_size_t(self._ws.numel())))

    # ---- helpers ----
    def _check(self, rc):
        if rc != GK_OK:
            raise GkError(rc, self.lib.gk_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self.lib.gk_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def state_dtype(self):
        t = self._torch
        return {0: t.complex64, 1: t.float16, 2: t.bfloat16}[self.storage]

    def empty_state(self):
        """Uninitialised device buffer with the layout/storage of f."""
        t = self._torch
        if self.storage == 0:
            return t.empty(self.shape, dtype=t.complex64, device=self.device)
        return t.empty(self.shape + (2,), dtype=self.state_dtype(), device=self.device)

    def to_state(self, f_host):
        """numpy complex array -> device buffer in this context's storage type."""
        t = self._torch
        x = t.from_numpy(f_host).to(self.device)
        if self.storage == 0:
            return x.to(t.complex64).contiguous()
        return t.view_as_real(x.to(t.complex64)).to(self.state_dtype()).contiguous()

    def from_state(self, f_dev):
        """device buffer -> numpy complex64."""
        t = self._torch
        if self.storage == 0:
            return f_dev.cpu().numpy()
        return t.view_as_complex(f_dev.float().contiguous()).cpu().numpy()

    def _chk_state(self, x, name):
        want = self.shape if self.storage == 0 else self.shape + (2,)
        if tuple(x.shape) != want or x.dtype != self.state_dtype() or not x.is_contiguous() or not x.is_cuda:
            raise ValueError(f"{name}: expected contiguous CUDA tensor {want} {self.state_dtype()}")

    # ---- the C-ABI calls ----
    def gk_field_solve(self, f, phi=None):
        t = self._torch
        self._chk_state(f, "f")
        if phi is None:
            phi = t.empty(self.phi_shape, dtype=t.complex64, device=self.device)
        self._check(self.lib.gk_field_solve(self._h, C.c_void_p(f.data_ptr()), C.c_void_p(phi.data_ptr())))
        return phi

    def gk_rhs(self, f, phi=None, rhs=None):
        t = self._torch
        self._chk_state(f, "f")
        if phi is None:
            phi = t.empty(self.phi_shape, dtype=t.complex64, device=self.device)
        if rhs is None:
            rhs = self.empty_state()
        self._check(self.lib.gk_rhs(self._h, C.c_void_p(f.data_ptr()), C.c_void_p(phi.data_ptr()),
                                    C.c_void_p(rhs.data_ptr())))
        return rhs, phi

    def gk_rk4_step(self, f, dt):
        self._chk_state(f, "f")
        self._check(self.lib.gk_rk4_step(self._h, C.c_void_p(f.data_ptr()), C.c_double(dt)))
        return f

    def gk_rk4_steps(self, f, dt, nsteps):
        self._chk_state(f, "f")
        self._check(self.lib.gk_rk4_steps(self._h, C.c_void_p(f.data_ptr()), C.c_double(dt), int(nsteps)))
        return f

    def gk_rk4_step_host(self, f_host_in, f_host_out, f_dev, dt: float):
        """One RK4 step on host buffers (torch CPU tensors, pinned for asynchronous copies) through the
        device scratch f_dev; asynchronous on the context stream."""
        self._chk_state(f_dev, "f_dev")
        for t in (f_host_in, f_host_out):
            if t.device.type != "cpu" or not t.is_contiguous() or t.numel() != f_dev.numel() or t.dtype != f_dev.dtype:
                raise ValueError("host buffers must be contiguous CPU tensors of the shape and dtype of f")
        self._check(self.lib.gk_rk4_step_host(self._h, C.c_void_p(f_host_in.data_ptr()), C.c_void_p(f_host_out.data_ptr()),
                                              C.c_void_p(f_dev.data_ptr()), float(dt)))

    def gk_rk4_batch_host(self, f_host_in, f_host_out, f_dev0, f_dev1, dt: float):
        """Independent RK4 steps on lists of pinned host tensors, pipelined over two device buffers
        (upload, compute and download overlap).  Synchronises."""
        self._chk_state(f_dev0, "f_dev0")
        self._chk_state(f_dev1, "f_dev1")
        n = len(f_host_in)
        if len(f_host_out) != n:
            raise ValueError("as many outputs as inputs")
        for t in list(f_host_in) + list(f_host_out):
            if t.device.type != "cpu" or not t.is_contiguous() or t.numel() != f_dev0.numel() or t.dtype != f_dev0.dtype:
                raise ValueError("host buffers must be contiguous CPU tensors of the shape and dtype of f")
        ins = (C.c_void_p * max(n, 1))(*[t.data_ptr() for t in f_host_in])
        outs = (C.c_void_p * max(n, 1))(*[t.data_ptr() for t in f_host_out])
        self._check(self.lib.gk_rk4_batch_host(self._h, ins, outs, n, C.c_void_p(f_dev0.data_ptr()),
                                               C.c_void_p(f_dev1.data_ptr()), float(dt)))

    def gk_fluxes(self, f, phi):
        import numpy as np
        self._chk_state(f, "f")
        out = np.zeros((self.nsp, 3), np.float64)
        self._check(self.lib.gk_fluxes(self._h, C.c_void_p(f.data_ptr()), C.c_void_p(phi.data_ptr()),
                                       out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def gk_set_diagnostics(self, on: bool):
        self._check(self.lib.gk_set_diagnostics(self._h, int(bool(on))))

    def gk_fluxes_last(self):
        """Fluxes of the state at the start of the most recent step (diagnostics on)."""
        import numpy as np
        out = np.zeros((self.nsp, 3), np.float64)
        self._check(self.lib.gk_fluxes_last(self._h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def gk_estimate_dt(self):
        """(dt, dt_nl, dt_lin, dt_field); the nonlinear bound is that of the most recent stage launch."""
        import numpy as np
        out = np.zeros(4, np.float64)
        self._check(self.lib.gk_estimate_dt(self._h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def gk_reset_cfl(self):
        """Forget the nonlinear CFL bound of the last stage launch (context reused for another state)."""
        self._check(self.lib.gk_reset_cfl(self._h))

    def gk_rk4_steps_cfl(self, f, nsteps, safety, dt_max=0.0):
        """CFL-adaptive steps; returns (dt of every step, time advanced)."""
        import numpy as np
        self._chk_state(f, "f")
        dts = np.zeros(max(int(nsteps), 1), np.float64)
        t = C.c_double()
        self._check(self.lib.gk_rk4_steps_cfl(self._h, C.c_void_p(f.data_ptr()), int(nsteps), float(safety), float(dt_max),
                                              dts.ctypes.data_as(C.POINTER(C.c_double)), C.byref(t)))
        return dts[:int(nsteps)], t.value

    def gk_spectra(self, phi):
        """(kx_spec[nkx], ky_spec[nky]) of |phi|^2."""
        import numpy as np
        kxs, kys = np.zeros(self.shape[4], np.float64), np.zeros(self.shape[5], np.float64)
        self._check(self.lib.gk_spectra(self._h, C.c_void_p(phi.data_ptr()),
                                        kxs.ctypes.data_as(C.POINTER(C.c_double)),
                                        kys.ctypes.data_as(C.POINTER(C.c_double))))
        return kxs, kys

    def gk_export_table(self, which: str):
        import numpy as np
        n = self.lib.gk_export_table(self._h, which.encode(), None, 0)
        if n == 0:
            raise KeyError(which)
        out = np.empty(n, np.float64)
        self.lib.gk_export_table(self._h, which.encode(), out.ctypes.data_as(C.POINTER(C.c_double)), n)
        return out

    def gk_launch_count(self) -> int:
        return int(self.lib.gk_launch_count(self._h))

    def gk_set_profiling(self, on: bool):
        self._check(self.lib.gk_set_profiling(self._h, int(bool(on))))

    def gk_stage_kernel_time(self, reset=True):
        ms = C.c_double()
        n = C.c_longlong()
        self._check(self.lib.gk_stage_kernel_time(self._h, C.byref(ms), C.byref(n), int(reset)))
        return ms.value, n.value

    def workspace_bytes(self):
        return int(self.lib.gk_workspace_bytes(self._h)), int(self.lib.gk_workspace_bytes_rhs(self._h))

    def plan(self) -> dict:
        p = self.gk_export_table("pad")
        return dict(mx=int(p[0]), my=int(p[1]), rc=int(p[2]), gchi_in_smem=int(p[3]), jchunk=int(p[4]),
                    nchunk=int(p[5]), stage_grid=int(p[6]), stage_smem=int(p[7]), threads=int(p[8]), cluster=int(p[9]),
                    nsh=int(p[10]), kind=int(p[11]))
