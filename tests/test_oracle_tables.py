"""Pins for the oracle's create-time tables: quadrature, Maxwellian, Bessel kernels, geometry,
connectivity.  Everything here is checked against closed forms, library routines
(numpy / scipy.special) or invariants -- never against the oracle's own formulas."""
import numpy as np
import pytest
import scipy.special as sc

from oracle.gkref import GkRef
from tests.util import small_cfg


def test_gauss_laguerre_n2_closed_form():
    # 2-point Gauss-Laguerre: x = 2 -+ sqrt2, w = (2 +- sqrt2)/4  (textbook)
    o = GkRef(small_cfg(nmu=2, mu_grid=0))
    x = np.array([2 - np.sqrt(2), 2 + np.sqrt(2)])
    w = np.array([(2 + np.sqrt(2)) / 4, (2 - np.sqrt(2)) / 4])
    np.testing.assert_allclose(o.table("mu"), x / 2, rtol=1e-13)
    np.testing.assert_allclose(o.table("wmu"), w * np.exp(x) / 2, rtol=1e-12)


@pytest.mark.parametrize("n", [3, 8, 16])
def test_gauss_laguerre_vs_numpy(n):
    o = GkRef(small_cfg(nmu=n, mu_grid=0))
    x, w = np.polynomial.laguerre.laggauss(n)
    np.testing.assert_allclose(o.table("mu"), x / 2, rtol=1e-11)
    np.testing.assert_allclose(o.table("wmu"), w * np.exp(x) / 2, rtol=1e-9)


def test_uniform_vperp_grid_weights():
    # mu = v_perp^2/2 uniform in v_perp, weight 2 pi v_perp dv_perp (the 2 pi B
    # is applied in the velocity sum): sum of weights = int_0^vmax v dv = vmax^2/2 exactly.
    o = GkRef(small_cfg(nmu=8, mu_grid=1))
    vp = np.sqrt(2 * o.table("mu"))
    np.testing.assert_allclose(np.diff(vp), 3.0 / 8, rtol=1e-13)
    np.testing.assert_allclose(o.table("wmu").sum(), 4.5, rtol=1e-13)


@pytest.mark.parametrize("mu_grid,nmu,tol", [(0, 16, 1e-7), (1, 64, 2e-3)])
def test_maxwellian_normalised(mu_grid, nmu, tol):
    # int F_M d^3v = 1 with d^3v = 2 pi B dvpar dmu at every s
    o = GkRef(small_cfg(nvpar=64, nmu=nmu, mu_grid=mu_grid, vperp_max=4.0))
    FM, B = o.table("FM"), o.table("B")
    wv, wmu = o.table("wv")[0], o.table("wmu")
    tot = 2 * np.pi * B * np.einsum("jli,l->i", FM, wmu) * wv
    np.testing.assert_allclose(tot, 1.0, atol=tol)


@pytest.mark.parametrize("nsp", [1, 2])
def test_weber_identity_pins_J0_and_Gamma0(nsp):
    # int J0(k_perp rho v_perp/B)^2 F_M d^3v = I0(b) e^-b, b = (m vR k_perp / Z B)^2 / 2
    # (Weber's second exponential integral).  Checks the mu weights, the J0 argument and the
    # Gamma0 argument against each other; Gamma0 itself against scipy.special.ive.
    o = GkRef(small_cfg(nkx=9, nky=4, ns=8, nvpar=64, nmu=24, mu_grid=0, nspecies=nsp, adiabatic=2 - nsp))
    FM, B, J0, G0 = o.table("FM"), o.table("B"), o.table("J0"), o.table("Gamma0")
    wv, wmu = o.table("wv")[0], o.table("wmu")
    quad = 2 * np.pi * np.einsum("i,jli,l,alipm->aipm", B, FM, wmu, J0 ** 2) * wv
    np.testing.assert_allclose(quad, G0, atol=2e-6)
    # Gamma0 against the library routine, b from k_perp^2 table and the species parameters
    kp2 = o.table("kperp2")
    for a, s in enumerate(o.cfg["species"]):
        vR = np.sqrt(s["temp"] / s["mass"])
        b = 0.5 * (s["mass"] * vR / s["Z"]) ** 2 * kp2 / B[:, None, None] ** 2
        np.testing.assert_allclose(G0[a], sc.ive(0, b), rtol=1e-12)
    assert np.all(G0 <= 1.0 + 1e-15) and np.all(G0 > 0)


def test_j0_table_is_library_bessel():
    o = GkRef(small_cfg(nmu=4, mu_grid=1))
    kp = np.sqrt(o.table("kperp2"))
    B, mu = o.table("B"), o.table("mu")
    lam = kp[None] * np.sqrt(2 * mu[:, None, None, None] / B[None, :, None, None])
    np.testing.assert_allclose(o.table("J0")[0], sc.j0(lam), atol=1e-14)


def test_salpha_geometry_invariants():
    cfg = small_cfg(ns=64)
    o = GkRef(cfg)
    q, eps = cfg["geom"]["q"], cfg["geom"]["eps"]
    s, B, F, BG, R = (o.table(k) for k in ("s", "B", "F", "BG", "R"))
    np.testing.assert_allclose(s, -0.5 + (np.arange(64) + 0.5) / 64, rtol=1e-14)
    np.testing.assert_allclose(B * R, 1.0, rtol=1e-14)            # B = 1/(1+eps cos theta)
    np.testing.assert_allclose(F, 1 / (2 * np.pi * q), rtol=1e-14)
    # G = F d_s B / B: differentiate B(s) numerically (complex step on the closed form)
    h = 1e-30
    dB = np.imag(1.0 / (1.0 + eps * np.cos(2 * np.pi * (s + 1j * h)))) / h
    np.testing.assert_allclose(BG, F * dB, rtol=1e-12, atol=1e-15)
    # mirror force is odd in s, field is even, minimum of B at the outboard midplane
    np.testing.assert_allclose(BG, -BG[::-1], atol=1e-15)
    np.testing.assert_allclose(B, B[::-1], rtol=1e-14)
    assert np.argmin(B) in (31, 32)


def test_kperp_is_textbook_salpha_and_continuous_along_chains():
    cfg = small_cfg(nkx=21, nky=4, ns=8, ikxspace=2)
    o = GkRef(cfg)
    shat = cfg["geom"]["shat"]
    kx, ky, th, kp2 = o.table("kx"), o.table("ky"), o.table("theta"), o.table("kperp2")
    # spacing of kx: dkx = 2 pi shat ky0 / ikxspace
    np.testing.assert_allclose(np.diff(kx), 2 * np.pi * shat * 0.1 / 2, rtol=1e-13)
    np.testing.assert_allclose(kx[10], 0, atol=1e-15)
    # on the extended ballooning angle theta_ext the local radial wavenumber kx + shat*theta*ky is
    # ONE linear function along a connected chain: walking i -> i+1 through the seam to
    # (p + m*ikxspace) must keep kperp^2 - ky^2 a perfect square of a linear function, i.e. its
    # third difference along the chain vanishes (wrong seam direction or spacing breaks this).
    ns, nkx = 8, 21
    for m in (1, 2, 3):
        p = 0
        while p - m * 2 >= 0:
            p -= m * 2  # start of the chain
        vals = []
        while p < nkx:
            vals.extend(kp2[:, p, m] - ky[m] ** 2)
            p += m * 2
        vals = np.array(vals)
        assert len(vals) >= 2 * ns
        np.testing.assert_allclose(np.diff(vals, 3), 0, atol=1e-12 * vals.max())
        lin = np.sqrt(vals)
        # also a direct textbook check at the first segment
    np.testing.assert_allclose(kp2[:, 3, 2], (kx[3] + shat * th * ky[2]) ** 2 + ky[2] ** 2, rtol=1e-13)


def test_stencil_class_marks_open_chain_ends_only():
    cfg = small_cfg(nkx=9, nky=4, ns=8, ikxspace=1)
    o = GkRef(cfg)
    cls = o.table("sclass").astype(int)
    assert np.all(cls[:, :, 0] == 0)                      # zonal mode: periodic
    for m in (1, 2, 3):
        for p in range(9):
            open_minus = p - m < 0
            open_plus = p + m > 8
            exp = np.zeros(8, int)
            if open_minus:
                exp[0], exp[1] = -2, -1
            if open_plus:
                exp[6], exp[7] = 1, 2
            np.testing.assert_array_equal(cls[:, p, m], exp)


def test_padded_size_rule():
    # 3/2 rule minimum, small primes <= 7: cfg3-like sizes
    o = GkRef(small_cfg(nkx=85, nky=32, ns=4, nvpar=4, nmu=1))
    assert list(o.table("pad")) == [128, 96]
    o = GkRef(small_cfg(nkx=9, nky=4))
    assert list(o.table("pad")) == [14, 10]
