"""Pins for the oracle's field solve, fluxes invariant and RK4
(PAPER.md:356)."""
import numpy as np
import pytest

from oracle.gkref import GkRef
from tests.util import small_cfg, rand_c, rel_l2


def _numerator(o, f):
    """N(i,p,m) = sum_a Z n 2 pi B sum_jl w_v w_mu J0 f, re-assembled with numpy from the tables."""
    J0, B = o.table("J0"), o.table("B")
    wv, wmu = o.table("wv")[0], o.table("wmu")
    N = 0
    for a, s in enumerate(o.cfg["species"]):
        N = N + s["Z"] * s["dens"] * 2 * np.pi * np.einsum("i,l,lipm,jlipm->ipm", B, wmu, J0[a], f[a]) * wv
    return N


def test_adiabatic_quasineutrality_residual_incl_zonal_branch():
    # Substitute phi back into quasineutrality (reading R10):
    #   N - A phi - (ne/Te) (phi - delta_{m0} <phi>_s) = 0,  A = Z^2 n (1-Gamma0)/T
    cfg = small_cfg(nkx=9, nky=3, ns=8, nvpar=8, nmu=3)
    o = GkRef(cfg)
    f = rand_c(np.random.default_rng(11), o.shape)
    phi = o.field_solve(f)
    N = _numerator(o, f)
    G0 = o.table("Gamma0")[0]
    A = (1 - G0)            # Z = n = T = 1
    ae = 1.0
    fsa = phi.mean(axis=0, keepdims=True) * np.array([1.0, 0, 0])[None, None, :]
    res = N - A * phi - ae * (phi - fsa)
    res[:, 4, 0] = 0        # (kx,ky)=(0,0) is gauged to zero instead
    assert abs(res).max() < 1e-13 * abs(N).max()
    assert np.all(phi[:, 4, 0] == 0)
    # the zonal correction matters: it is not the plain division
    assert abs(phi[:, 5, 0] - N[:, 5, 0] / (A[:, 5, 0] + ae)).max() > 1e-3 * abs(phi).max()


def test_adiabatic_response_to_maxwellian_perturbation():
    # f = c(i,p,m) J0 F_M  =>  N = c Gamma0 (Weber)  =>  phi = c Gamma0 / (1 - Gamma0 + 1) for ky > 0
    cfg = small_cfg(nkx=5, nky=3, ns=8, nvpar=64, nmu=24)
    o = GkRef(cfg)
    rng = np.random.default_rng(12)
    c = rng.standard_normal(o.phi_shape) + 1j * rng.standard_normal(o.phi_shape)
    f = (c[None, None] * o.table("J0")[0][None] * o.table("FM")[:, :, :, None, None])[None]
    phi = o.field_solve(f)
    G0 = o.table("Gamma0")[0]
    np.testing.assert_allclose(phi[:, :, 1:], (c * G0 / (2 - G0))[:, :, 1:], rtol=2e-6)


def test_kinetic_electron_field_solve():
    # numerator and denominator sum over species; no zonal correction; (0,0) -> 0.
    cfg = small_cfg(nkx=5, nky=3, ns=8, nvpar=8, nmu=3, nspecies=2, adiabatic=0)
    o = GkRef(cfg)
    f = rand_c(np.random.default_rng(13), o.shape)
    phi = o.field_solve(f)
    N = _numerator(o, f)
    G0 = o.table("Gamma0")
    den = sum(s["Z"] ** 2 * s["dens"] * (1 - G0[a]) / s["temp"] for a, s in enumerate(cfg["species"]))
    den[:, 2, 0] = 1.0
    exp = N / den
    exp[:, 2, 0] = 0
    np.testing.assert_allclose(phi, exp, rtol=1e-12, atol=1e-14)
    # electron FLR retained but tiny: Gamma0_e in (0.99, 1]
    assert G0[1].min() > 0.99 and G0[1].max() <= 1.0
    # equal and opposite charge perturbations with the same gyro-averaged shape cancel: phi = 0
    g = rand_c(np.random.default_rng(14), o.shape[1:])
    J0 = o.table("J0")
    f2 = np.stack([g, g * (J0[0] / J0[1])[None]])
    assert abs(o.field_solve(f2)).max() < 1e-10 * abs(g).max()


def test_particle_flux_vanishes_for_adiabatic_electrons():
    # "particle flux vanishes identically" with adiabatic electrons.
    cfg = small_cfg(nkx=9, nky=4, ns=8, nvpar=8, nmu=2)
    o = GkRef(cfg)
    f = rand_c(np.random.default_rng(15), o.shape)
    phi = o.field_solve(f)
    fl = o.fluxes(f, phi)
    assert abs(fl[0, 0]) < 1e-13 * abs(fl[0, 1])
    assert abs(fl[0, 1]) > 0


def test_rk4_is_the_classical_tableau_taylor_identity():
    # For a linear autonomous system one classical RK4 step equals sum_{n<=4} (dt L)^n / n! f
    # (four evaluations of the full RHS, phi re-solved at each).
    cfg = small_cfg(nkx=9, nky=3, ns=8, nvpar=8, nmu=2, nonlinear=0)
    o = GkRef(cfg)
    f = rand_c(np.random.default_rng(16), o.shape)
    dt = 0.013
    acc, term = f.copy(), f.copy()
    for n in range(1, 5):
        term = o.rhs(term)[0] * dt / n
        acc = acc + term
    assert rel_l2(o.rk4_step(f, dt), acc) < 1e-14


def test_rk4_fourth_order_convergence_nonlinear():
    cfg = small_cfg(nkx=9, nky=4, ns=8, nvpar=8, nmu=2)
    o = GkRef(cfg, bracket_method=1)
    f = 1.0 * rand_c(np.random.default_rng(17), o.shape)      # O(1) amplitude: bracket matters
    T = 0.02
    ref = o.rk4_step(f, T / 16, 16)
    e1 = rel_l2(o.rk4_step(f, T, 1), ref)
    e2 = rel_l2(o.rk4_step(f, T / 2, 2), ref)
    assert 10 < e1 / e2 < 22, (e1, e2)
    # the nonlinear term really contributed
    lin = GkRef(small_cfg(nkx=9, nky=4, ns=8, nvpar=8, nmu=2, nonlinear=0))
    assert rel_l2(lin.rk4_step(f, T, 1), ref) > 100 * e1
