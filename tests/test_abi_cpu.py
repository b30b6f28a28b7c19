"""CPU-side checks of the boundary: the C-ABI library builds/loads, exports every symbol that
include/*.h declare, and refuses to work without a CUDA device (no CPU fallback)."""
import ctypes as C
import os
import subprocess

import pytest

import gkinputs
from paper_2604_06085_b200 import binding


def test_library_loads_and_exports_every_declared_symbol():
    lib = binding.load_library()
    names = binding.exported_symbols()
    assert {"gk_create", "gk_destroy", "gk_field_solve", "gk_rhs", "gk_rk4_step", "gk_rk4_steps",
            "gk_fluxes", "gk_workspace_bytes", "gk_set_workspace", "gk_export_table",
            "gk_last_error", "gk_estimate_dt", "gk_rk4_steps_cfl", "gk_set_diagnostics", "gk_fluxes_last",
            "gk_spectra", "gk_launch_count", "gk_stage_kernel_time"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert b"sm_100a" in lib.gk_version()


def test_extern_c_symbols_are_unmangled_and_sm100a_code_is_embedded():
    out = subprocess.run(["nm", "-D", "--defined-only", binding.lib_path()], capture_output=True, text=True).stdout
    for n in binding.exported_symbols():
        assert f" T {n}\n" in out, n
    res = subprocess.run(["cuobjdump", "-lelf", binding.lib_path()], capture_output=True, text=True)
    if res.returncode == 0:
        assert "sm_100a" in res.stdout


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(binding.GkError) as ei:
        binding.GkContext(gkinputs.config(1))
    assert ei.value.code == binding.GK_ECUDA
    # and straight through the C ABI: gk_create must return GK_ECUDA, not succeed
    lib = binding.load_library()
    g = binding._Grid(9, 4, 8, 8, 2, 0.1, 1, 4.0, 0, 3.0)
    sp = (binding._Species * 1)(binding._Species(1, 1, 1, 1, 7, 2))
    geo = binding._Salpha(1.5, 0.8, 0.18)
    o = binding._Opts(1, 1, 1.0, 1.0, 1, 1.0, 0.2, 0.1, 0.1, 0, 0, 0, 0, 0, 0)
    h = C.c_void_p()
    rc = lib.gk_create(C.byref(g), sp, C.byref(geo), C.byref(o), None, C.byref(h))
    assert rc == binding.GK_ECUDA
    if h:
        lib.gk_destroy(h)


def test_gk_create_rejects_bad_arguments_before_touching_the_device():
    lib = binding.load_library()
    sp = (binding._Species * 1)(binding._Species(1, 1, 1, 1, 7, 2))
    geo = binding._Salpha(1.5, 0.8, 0.18)
    o = binding._Opts(1, 1, 1.0, 1.0, 1, 1.0, 0.2, 0.1, 0.1, 0, 0, 0, 0, 0, 0)
    h = C.c_void_p()
    for bad in [dict(nkx=8), dict(ns=3), dict(nvpar=3), dict(nky=0), dict(nmu=0), dict(ikxspace=0)]:
        kw = dict(nkx=9, nky=4, ns=8, nvpar=8, nmu=2, ky0=0.1, ikxspace=1, vpar_max=4.0, mu_grid=0, vperp_max=3.0)
        kw.update(bad)
        g = binding._Grid(*[kw[k] for k in ("nkx", "nky", "ns", "nvpar", "nmu", "ky0", "ikxspace", "vpar_max", "mu_grid", "vperp_max")])
        assert lib.gk_create(C.byref(g), sp, C.byref(geo), C.byref(o), None, C.byref(h)) == binding.GK_EINVAL, bad
    assert lib.gk_create(None, sp, C.byref(geo), C.byref(o), None, C.byref(h)) == binding.GK_EINVAL
    assert lib.gk_workspace_bytes(None) == 0
    assert lib.gk_destroy(None) == binding.GK_EINVAL


def test_product_package_does_not_import_the_oracle():
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    pkg = os.path.join(root, "paper_2604_06085_b200")
    for dp, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dp, fn)).read()
                assert "gkref" not in src and "import oracle" not in src and "from oracle" not in src, fn
