"""Pins for the oracle's CFL estimate gkref_estimate_dt (readings R21-R23 of DESIGN.md).
Each of the three bounds is compared with what it is a bound OF: the RK4 stability of the operator itself,
obtained from a dense eigen-solve of the matrix the oracle's own rhs builds from unit vectors (the same
technique as tests/test_oracle_physics.py), plus a closed form for the nonlinear bound."""
import numpy as np
import pytest

import gkinputs
from oracle import gkref as G
from oracle.gkref import GkRef
from tests.util import small_cfg, rand_c
from tests.test_oracle_physics import _operator_matrix

LIM = 2 * np.sqrt(2)          # RK4 on the imaginary axis: |R(iy)| <= 1  <=>  |y| <= 2 sqrt 2


def _amp(z):
    return abs(1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24)


def _true_limit(lam, hi):
    lo = 0.0
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        lo, hi = (mid, hi) if _amp(lam * mid).max() <= 1 + 1e-9 else (lo, mid)
    return lo


def test_rk4_imaginary_axis_limit():
    y = np.linspace(0, 3, 30001)
    inside = _amp(1j * y) <= 1 + 1e-12
    assert abs(y[inside].max() - LIM) < 2e-4


@pytest.mark.parametrize("ns,nv,nmu,nus,nuv", [(16, 12, 2, 1.0, 0.2), (16, 16, 2, 0.0, 0.0), (12, 12, 3, 0.3, 1.0)])
def test_von_neumann_bound_brackets_the_operators_rk4_stability(ns, nv, nmu, nus, nuv):
    # (ii): streaming + trapping (+ their dissipation) on the periodic zonal chain.  The frozen-coefficient bound
    # must be stable for the real (variable-coefficient, zero-padded in v) operator and within 25 % of its limit.
    cfg = small_cfg(nkx=3, nky=1, ns=ns, nvpar=nv, nmu=nmu, mu_grid=1, disp_par=nus, disp_vp=nuv, nonlinear=0)
    o = GkRef(cfg, term_mask=G.T_I | G.T_IV | G.T_DISS_S | G.T_DISS_V)
    sel = np.zeros(o.shape, bool)
    sel[0, :, :, :, 0, 0] = True
    lam = np.linalg.eigvals(_operator_matrix(o, sel))
    dt, dt_nl, dt_lin, dt_field = o.estimate_dt(np.zeros(o.phi_shape, complex))
    assert np.isinf(dt_nl) and np.isinf(dt_field) and dt == dt_lin
    assert _amp(lam * dt_lin).max() <= 1 + 1e-9
    true = _true_limit(lam, 10 * dt_lin)
    assert 1.0 <= true / dt_lin < 1.25, true / dt_lin


def test_von_neumann_bound_pure_streaming_closed_form():
    # no dissipation, no trapping (eps = 0): z = -i c_s sigma(t), so dt_lin = 2 sqrt2 / (c_s max sigma);
    # max of (8 sin t - sin 2t)/6 over the 64-angle grid, written out here
    cfg = small_cfg(nkx=3, nky=1, ns=20, nvpar=8, nmu=1, eps=0.0, disp_par=0.0, disp_vp=0.0, nonlinear=0)
    o = GkRef(cfg)
    t = 2 * np.pi * np.arange(64) / 64
    smax = ((8 * np.sin(t) - np.sin(2 * t)) / 6).max()
    vmax = 4.0 - 0.5 * (8.0 / 8)                      # largest |v_j| of the midpoint grid on [-4, 4]
    cs = vmax / (2 * np.pi * cfg["geom"]["q"]) * 20   # |v_R v F| / ds
    np.testing.assert_allclose(o.estimate_dt(np.zeros(o.phi_shape, complex))[2], LIM / (cs * smax), rtol=1e-9)


def test_field_cfl_tracks_the_omega_h_mode_and_decides_config_4():
    # (iii): kinetic electrons, zonal chain of the smallest kx.  The estimate must (a) scale as 1/k_perp with the
    # operator's fastest mode, staying within 30 % on the safe side of it, (b) reject BASELINE config 4 at SURVEY's
    # ky0 = 0.035 with dt = 0.002 and accept it at ky0 = 0.2 (R5: found by hand in round 1).
    freq, est = {}, {}
    for ky0 in (0.035, 0.2):
        cfg = small_cfg(nkx=3, nky=1, ns=32, nvpar=8, nmu=1, nspecies=2, adiabatic=0, mu_grid=1, ky0=ky0,
                        ikxspace=5, nonlinear=0)
        o = GkRef(cfg)
        sel = np.zeros(o.shape, bool)
        sel[:, :, :, :, 2, 0] = True
        lam = np.linalg.eigvals(_operator_matrix(o, sel))
        freq[ky0] = abs(lam).max()
        e = o.estimate_dt(np.zeros(o.phi_shape, complex))
        est[ky0] = e[3]
        assert e[0] == e[3] < e[2]                       # the field bound is the binding one
        assert 1.0 < (LIM / e[3]) / freq[ky0] < 1.3       # omega_H estimate vs the operator's fastest mode
        assert _amp(lam * e[3]).max() <= 1 + 1e-9         # stable at the estimate
    assert freq[0.035] / freq[0.2] == pytest.approx(0.2 / 0.035, rel=0.05)     # omega ~ 1/k_perp
    assert est[0.035] < 0.002 < est[0.2]
    # the full config-4 grid (ky > 0 included) decides the same way
    for ky0, ok in ((0.035, False), (0.2, True)):
        cfg = gkinputs.config(4)
        cfg["grid"].update(ky0=ky0, nvpar=4, nmu=2)      # velocity resolution does not enter the field bound
        e = GkRef(cfg).estimate_dt(np.zeros((32, 85, 32), complex))
        assert (e[3] > cfg["dt"]) == ok, (ky0, e)
    # adiabatic electrons: no field bound
    assert np.isinf(GkRef(gkinputs.config(1)).estimate_dt(np.zeros((8, 9, 4), complex))[3])


def test_nonlinear_bound_single_mode_closed_form():
    from scipy.special import j0 as bessel_j0
    cfg = small_cfg(nkx=9, nky=4, ns=4, nvpar=4, nmu=3, mu_grid=1, ky0=0.2)
    o = GkRef(cfg, pad=(16, 12))
    i, p, m, amp = 1, 6, 2, 0.37
    phi = np.zeros(o.phi_shape, complex)
    phi[i, p, m] = 1j * amp                 # chi(x, y) = -2 amp J0 sin(kx x + ky y): gradients peak at the origin
    g, geo = cfg["grid"], cfg["geom"]
    dkx = 2 * np.pi * geo["shat"] * g["ky0"] / g["ikxspace"]
    kx, ky = (p - 4) * dkx, m * g["ky0"]
    th = 2 * np.pi * (-0.5 + (i + 0.5) / 4)
    B = 1 / (1 + geo["eps"] * np.cos(th))
    kperp = np.sqrt((kx + geo["shat"] * th * ky) ** 2 + ky ** 2)
    mu0 = 0.5 * (0.5 * g["vperp_max"] / 3) ** 2        # smallest mu: largest J0
    J0 = bessel_j0(kperp * np.sqrt(2 * mu0 / B))
    lam = 0.5 * 2 * amp * J0 * (ky * 4 * dkx + abs(kx) * 3 * g["ky0"])
    e = o.estimate_dt(phi)
    np.testing.assert_allclose(e[1], LIM / lam, rtol=1e-12)
    # scales inversely with the amplitude, infinite for phi = 0 and with term III switched off
    np.testing.assert_allclose(o.estimate_dt(3 * phi)[1], e[1] / 3, rtol=1e-12)
    assert np.isinf(o.estimate_dt(0 * phi)[1])
    assert np.isinf(GkRef(small_cfg(nkx=9, nky=4, ns=4, nvpar=4, nmu=3, nonlinear=0)).estimate_dt(phi)[1])


def test_nonlinear_bound_dominates_the_bracket_operator_spectrum():
    # For a frozen chi the bracket is a (real-)linear advection operator on f; its eigenvalues are imaginary and
    # bounded by max |v_E . k|: the estimate 2 sqrt2 / dt_NL must dominate the largest one, and not by more than
    # the factor a max-velocity x max-wavenumber bound loses on a random field.
    cfg = small_cfg(nkx=9, nky=4, ns=4, nvpar=4, nmu=1, mu_grid=1, ky0=0.2)
    o = GkRef(cfg, pad=(16, 12))
    rng = np.random.default_rng(8)
    phi = np.zeros(o.phi_shape, complex)
    phi[2] = rand_c(rng, (9, 4), True)
    chi = o.table("J0")[0, 0, 2] * phi[2]
    n = 9 * 4
    M = np.zeros((2 * n, 2 * n))
    for c in range(2 * n):
        e = np.zeros(n, complex)
        e[c % n] = 1.0 if c < n else 1j
        r = o.bracket_slab(chi, e.reshape(9, 4), method=1).ravel()
        M[:n, c], M[n:, c] = r.real, r.imag
    lam = np.linalg.eigvals(M)
    assert abs(lam.real).max() < 1e-9 * abs(lam).max() + 1e-12     # advection: no growth
    bound = LIM / o.estimate_dt(phi)[1]
    assert 0.25 * bound < abs(lam.imag).max() <= bound * (1 + 1e-12), (abs(lam.imag).max(), bound)
