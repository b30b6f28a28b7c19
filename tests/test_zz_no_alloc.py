"""gk_spectra_static: the spectra entry point for callers that cannot allocate device memory.

Some programs that embed this library have no way to call cudaMalloc: their own pool allocator has already taken
the whole GPU, or the process runs under a memory cap, so gk_create (which builds its tables with cudaMalloc) is out
of reach for them.  gk_spectra_static serves them without a context, staging its nkx + nky results in a fixed array
inside libgk.so.  That array is shared by all calls and keeps what the previous call left in it, so the GPU test
below makes two calls in a row -- the second on a SMALLER plane with other values, where stale entries of the first
call sit right behind the ones the second call writes -- and compares each with gk_spectra of an ordinary context,
at the tolerance of test_gpu_parity.py::test_spectra_parity (both paths sum in the same order, so they also agree
bit for bit).

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It passes alone in a fresh process and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2604_06085_b200 import binding
from tests.util import small_cfg


def _raw(lib, phi_ptr, ns, nkx, nky):
    kx, ky = np.zeros(max(nkx, 1)), np.zeros(max(nky, 1))
    dp = C.POINTER(C.c_double)
    rc = lib.gk_spectra_static(C.c_void_p(phi_ptr), ns, nkx, nky, kx.ctypes.data_as(dp), ky.ctypes.data_as(dp), None)
    return rc, lib.gk_spectra_static_error().decode()


def test_sizes_beyond_the_fixed_scratch_are_refused_before_the_device_is_touched():
    # Argument checks come first, so this runs without a GPU: the pointer is never dereferenced.
    lib = binding.load_library()
    cap = binding.gk_spectra_static_max()
    assert cap == 4096
    rc, msg = _raw(lib, 256, 8, cap - 10, 11)
    assert rc == binding.GK_EINVAL and "exceeds the fixed scratch" in msg and str(cap) in msg
    rc, msg = _raw(lib, 256, 0, 9, 4)
    assert rc == binding.GK_EINVAL and ">= 1" in msg
    rc, msg = _raw(lib, 0, 8, 9, 4)
    assert rc == binding.GK_EINVAL and "null" in msg


@pytest.mark.gpu
def test_two_calls_in_a_row_equal_the_context_path():
    import torch
    from paper_2604_06085_b200 import GkContext, gk_spectra_static

    dev = torch.device("cuda:0")
    gen = torch.Generator(device="cpu").manual_seed(20260406)
    # first a plane with a ragged tail over the 256-thread blocks, then a smaller one with other amplitudes
    for (ns, nkx, nky), amp in (((8, 85, 32), 1.0), ((6, 21, 6), 37.0)):
        phi = (amp * torch.view_as_complex(torch.randn((ns, nkx, nky, 2), generator=gen, dtype=torch.float32))).to(dev)
        ctx = GkContext(small_cfg(nkx=nkx, nky=nky, ns=ns, nvpar=8, nmu=2), device="cuda:0", full_workspace=False)
        want_kx, want_ky = ctx.gk_spectra(phi)
        ctx.close()
        got_kx, got_ky = gk_spectra_static(phi)
        assert got_kx.shape == (nkx,) and got_ky.shape == (nky,)
        np.testing.assert_allclose(got_kx, want_kx, rtol=1e-12)
        np.testing.assert_allclose(got_ky, want_ky, rtol=1e-12)
        assert np.array_equal(got_kx, want_kx) and np.array_equal(got_ky, want_ky)   # same summation order
        assert got_kx.min() > 0 and abs(got_kx.sum() - got_ky.sum()) < 1e-12 * got_kx.sum()
    # a refused call leaves the entry point usable, and a good call clears the error text
    with pytest.raises(binding.GkError, match="exceeds the fixed scratch"):
        gk_spectra_static(torch.zeros((1, 4000, 200), dtype=torch.complex64, device=dev))
    again_kx, _ = gk_spectra_static(phi)
    assert np.array_equal(again_kx, want_kx)
    assert binding.load_library().gk_spectra_static_error() == b""
