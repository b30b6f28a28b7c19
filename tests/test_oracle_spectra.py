"""Pins for the oracle's spectra diagnostics (ky_spec = sum_{s,kx} |phi|^2,
kx_spec = sum_{s,ky} |phi|^2; Parseval factor P_ky and Delta s applied; reading R20)."""
import numpy as np

from oracle.gkref import GkRef
from tests.util import small_cfg, rand_c


def _herm_phi(rng, shape):
    """phi(s,kx,ky) whose ky=0 column is Hermitian in kx: a real field in (x,y)."""
    phi = rand_c(rng, shape)
    K = (shape[1] - 1) // 2
    for p in range(1, K + 1):
        phi[:, K - p, 0] = np.conj(phi[:, K + p, 0])
    phi[:, K, 0] = phi[:, K, 0].real
    return phi


def test_spectra_equal_the_real_space_mean_square():
    # Parseval through an independent route (numpy irfft2 on a grid fine enough to hold every mode):
    # sum_p kx_spec = sum_m ky_spec = (1/ns) sum_s <phi(x,y)^2>_{x,y}.  Pins the factor P_m
    # (1 at ky=0, 2 otherwise), the Delta s weight and both index orders.
    cfg = small_cfg(nkx=9, nky=4, ns=8, nvpar=8, nmu=2)
    o = GkRef(cfg)
    ns, nkx, nky = o.phi_shape
    K = (nkx - 1) // 2
    phi = _herm_phi(np.random.default_rng(5), o.phi_shape)
    kxs, kys = o.spectra(phi)
    nx, ny = 16, 8
    ms = 0.0
    for i in range(ns):
        full = np.zeros((nx, ny // 2 + 1), complex)
        for p in range(-K, K + 1):
            full[p % nx, :nky] = phi[i, p + K, :]
        real = np.fft.irfft2(full, s=(nx, ny)) * (nx * ny)
        ms += np.mean(real ** 2) / ns
    assert abs(kxs.sum() - ms) < 1e-12 * ms
    assert abs(kys.sum() - ms) < 1e-12 * ms


def test_single_mode_closed_form_and_index_order():
    # one mode (i0, p0, m0) of amplitude A: kx_spec = ds P A^2 at p0 only, ky_spec = ds P A^2 at m0 only
    cfg = small_cfg(nkx=9, nky=4, ns=8, nvpar=8, nmu=2)
    o = GkRef(cfg)
    ns, nkx, nky = o.phi_shape
    for (i0, p0, m0, P) in [(3, 6, 2, 2.0), (0, 1, 0, 1.0)]:
        phi = np.zeros(o.phi_shape, complex)
        phi[i0, p0, m0] = 0.3 - 0.4j
        kxs, kys = o.spectra(phi)
        want = P * 0.25 / ns
        ex, ey = np.zeros(nkx), np.zeros(nky)
        ex[p0], ey[m0] = want, want
        assert np.allclose(kxs, ex, rtol=0, atol=1e-16)
        assert np.allclose(kys, ey, rtol=0, atol=1e-16)


def test_spectra_from_numpy_definition():
    cfg = small_cfg(nkx=9, nky=4, ns=8, nvpar=8, nmu=2)
    o = GkRef(cfg)
    phi = rand_c(np.random.default_rng(9), o.phi_shape)
    kxs, kys = o.spectra(phi)
    P = np.array([1.0, 2.0, 2.0, 2.0])
    a2 = np.abs(phi) ** 2 * P[None, None, :] / o.phi_shape[0]
    assert np.allclose(kxs, a2.sum(axis=(0, 2)), rtol=1e-14)
    assert np.allclose(kys, a2.sum(axis=(0, 1)), rtol=1e-14)
