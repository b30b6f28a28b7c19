"""Pins for the parts of the oracle that had none outside the oracle itself ("What's weak" 2):
the three dissipation terms of gkref::linear_point (DISS_S, DISS_V, HYP), the drift factor kappa, the
1-D streaming operator with its boundary classes as a whole (eigenvalues against an independently
assembled matrix; RK4 stability limits of SURVEY R7), and the heat / momentum moments of gkref_fluxes.
Every expected value is a closed form or a matrix written out here, never read back from the oracle."""
import numpy as np
import pytest

from oracle import gkref as G
from oracle.gkref import GkRef
from tests.util import small_cfg, rand_c, rel_l2


def _grids(cfg):
    """s, theta, vpar, kx, ky of reading R1, restated (not read from the oracle)."""
    g, geo = cfg["grid"], cfg["geom"]
    s = -0.5 + (np.arange(g["ns"]) + 0.5) / g["ns"]
    dv = 2 * g["vpar_max"] / g["nvpar"]
    v = -g["vpar_max"] + (np.arange(g["nvpar"]) + 0.5) * dv
    K = (g["nkx"] - 1) // 2
    kx = (np.arange(g["nkx"]) - K) * 2 * np.pi * geo["shat"] * g["ky0"] / g["ikxspace"]
    ky = np.arange(g["nky"]) * g["ky0"]
    return s, 2 * np.pi * s, v, dv, kx, ky


# ------------------------------------------------------------------------------------------------
# DISS_S:  - nu_s |v_R v_j F| delta^4_s f / (12 ds)  on class-0 points, nothing at class != 0 (R7)
# ------------------------------------------------------------------------------------------------
def test_parallel_dissipation_on_polynomials_open_chain():
    # nkx = 5, m = 3, ikxspace = 1: kx index 2 is a chain of one link (2 - 3 < 0, 2 + 3 > 4): both ends open
    nu = 0.7
    cfg = small_cfg(nkx=5, nky=4, ns=12, nvpar=4, nmu=1, ikxspace=1, disp_par=nu)
    o = GkRef(cfg, term_mask=G.T_DISS_S)
    s, _, v, _, _, _ = _grids(cfg)
    ds = 1.0 / 12
    F = 1.0 / (2 * np.pi * cfg["geom"]["q"])        # R2: ffun of s-alpha
    f = np.zeros(o.shape, complex)
    f[0, :, :, :, 2, 3] = (s ** 4)[None, None, :] * (1 - 2j)
    rhs, _ = o.rhs(f)
    # delta^4 (s^4) = 24 ds^4 exactly  =>  -nu |v F| 24 ds^4 / (12 ds) = -nu |v F| 2 ds^3  (vR = 1 for the ions)
    exact = -nu * np.abs(v * F)[:, None] * 2 * ds ** 3 * np.ones(8)[None, :] * (1 - 2j)
    np.testing.assert_allclose(rhs[0, :, 0, 2:-2, 2, 3], exact, rtol=1e-9)
    assert np.all(rhs[0, :, 0, 2:-2, 2, 3].real < 0)          # it damps (sign pin)
    # class +-1, +-2 points carry no fourth difference with closure 0
    assert abs(rhs[0, :, 0, :2, 2, 3]).max() == 0 and abs(rhs[0, :, 0, -2:, 2, 3]).max() == 0
    # a cubic is annihilated
    f[0, :, :, :, 2, 3] = (s ** 3 - 0.3 * s)[None, None, :]
    rhs, _ = o.rhs(f)
    assert abs(rhs[0, :, 0, 2:-2, 2, 3]).max() < 1e-15


def test_parallel_dissipation_symbol_on_the_periodic_zonal_chain():
    # ky = 0 is periodic in s: plane wave exp(i n theta) -> -nu |v F| (2 - 2 cos t)^2 / (12 ds),
    # t = 2 pi n / ns, at EVERY s (the wrap included)
    nu, ns = 1.3, 16
    cfg = small_cfg(nkx=3, nky=2, ns=ns, nvpar=4, nmu=2, disp_par=nu)
    o = GkRef(cfg, term_mask=G.T_DISS_S)
    s, th, v, _, _, _ = _grids(cfg)
    F = 1.0 / (2 * np.pi * cfg["geom"]["q"])
    for n in (1, 3, 8):
        f = np.zeros(o.shape, complex)
        f[0, :, :, :, 0, 0] = np.exp(1j * n * th)[None, None, :]
        rhs, _ = o.rhs(f)
        t = 2 * np.pi * n / ns
        lam = -nu * np.abs(v * F) * (2 - 2 * np.cos(t)) ** 2 / (12 / ns)
        np.testing.assert_allclose(rhs[0, :, 1, :, 0, 0], lam[:, None] * f[0, :, 1, :, 0, 0], rtol=1e-10, atol=1e-14)


# ------------------------------------------------------------------------------------------------
# DISS_V:  - nu_v |v_R mu B G| delta^4_v f / (12 dv), zero ghosts (R8)
# ------------------------------------------------------------------------------------------------
def test_velocity_dissipation_interior_and_edge_rows():
    nu = 0.45
    cfg = small_cfg(nkx=3, nky=2, ns=8, nvpar=12, nmu=2, mu_grid=1, disp_vp=nu)
    o = GkRef(cfg, term_mask=G.T_DISS_V)
    s, th, v, dv, _, _ = _grids(cfg)
    eps, q = cfg["geom"]["eps"], cfg["geom"]["q"]
    B = 1 / (1 + eps * np.cos(th))
    BG = (eps / q) * np.sin(th) * B ** 2                       # R2
    dvp = cfg["grid"]["vperp_max"] / 2
    mu = 0.5 * ((np.arange(2) + 0.5) * dvp) ** 2               # R3, uniform in v_perp
    g = v ** 4 - v
    f = np.zeros(o.shape, complex)
    f[0] = g[:, None, None, None, None] * (2 + 1j)
    rhs, _ = o.rhs(f)
    c = -nu * np.abs(mu[:, None] * BG[None, :])                # [l, i]
    # interior: delta^4 (v^4) = 24 dv^4  ->  2 dv^3
    np.testing.assert_allclose(rhs[0, 2:-2, :, :, 1, 1], (c * 2 * dv ** 3)[None] * (2 + 1j) * np.ones((8, 1, 1)), rtol=1e-8)
    # edge rows worked by hand with zero ghosts: j = 0: (6 g0 - 4 g1 + g2), j = 1: (-4 g0 + 6 g1 - 4 g2 + g3)
    e0 = (6 * g[0] - 4 * g[1] + g[2]) / (12 * dv)
    e1 = (-4 * g[0] + 6 * g[1] - 4 * g[2] + g[3]) / (12 * dv)
    eN = (6 * g[-1] - 4 * g[-2] + g[-3]) / (12 * dv)
    np.testing.assert_allclose(rhs[0, 0, :, :, 1, 1], c * e0 * (2 + 1j), rtol=1e-12)
    np.testing.assert_allclose(rhs[0, 1, :, :, 1, 1], c * e1 * (2 + 1j), rtol=1e-12)
    np.testing.assert_allclose(rhs[0, -1, :, :, 1, 1], c * eN * (2 + 1j), rtol=1e-12)
    # sign pin: a grid-scale zig-zag in v is damped wherever the mirror force acts
    f[0] = ((-1.0) ** np.arange(12))[:, None, None, None, None]
    rhs, _ = o.rhs(f)
    ratio = (rhs[0, 3:-3, 1, :, 1, 1] / f[0, 3:-3, 1, :, 1, 1]).real
    assert np.all(ratio[:, np.abs(BG) > 1e-12] < 0)
    np.testing.assert_allclose(ratio, (c[1] * 16 / (12 * dv))[None, :] * np.ones((6, 1)), rtol=1e-12)


# ------------------------------------------------------------------------------------------------
# HYP:  - [nu_x (kx/kx_max)^4 + nu_y (ky/ky_max)^4] f   (R9)
# ------------------------------------------------------------------------------------------------
def test_hyperviscosity_is_diagonal_with_quartic_rates():
    nx, ny = 0.3, 0.9
    cfg = small_cfg(nkx=7, nky=5, ns=4, nvpar=4, nmu=1, disp_x=nx, disp_y=ny)
    o = GkRef(cfg, term_mask=G.T_HYP)
    f = rand_c(np.random.default_rng(5), o.shape, False)
    rhs, _ = o.rhs(f)
    p = (np.arange(7) - 3) / 3.0
    m = np.arange(5) / 4.0
    rate = -(nx * p[:, None] ** 4 + ny * m[None, :] ** 4)
    np.testing.assert_allclose(rhs, rate[None, None, None, None] * f, rtol=1e-13)
    # corner mode decays at nu_x + nu_y, the (0, 0) mode not at all
    assert rate[0, 4] == pytest.approx(-(nx + ny)) and rate[3, 0] == 0


# ------------------------------------------------------------------------------------------------
# kappa = kx D^psi + k_zeta D^zeta  (R2)
# ------------------------------------------------------------------------------------------------
def test_kappa_table_closed_form_and_chain_continuity():
    cfg = small_cfg(nkx=11, nky=4, ns=8, nvpar=4, nmu=1, ikxspace=2, ky0=0.13)
    o = GkRef(cfg)
    s, th, _, _, kx, ky = _grids(cfg)
    shat = cfg["geom"]["shat"]
    kap = -(kx[None, :, None] * np.sin(th)[:, None, None]
            + ky[None, None, :] * (np.cos(th) + shat * th * np.sin(th))[:, None, None])
    np.testing.assert_allclose(o.table("kappa"), kap, rtol=1e-13, atol=1e-15)
    # kappa = -(ky cos(theta) + kx_eff sin(theta)) with the SAME kx_eff = kx + shat theta ky that enters
    # k_perp^2 = kx_eff^2 + ky^2: the two tables must agree on it ...
    kp2 = o.table("kperp2")
    kxe = -(o.table("kappa") + ky[None, None, :] * np.cos(th)[:, None, None]) / np.sin(th)[:, None, None]
    np.testing.assert_allclose(kxe ** 2 + ky[None, None, :] ** 2, kp2, rtol=1e-12)
    # ... and kappa, a smooth function of the extended angle, is continuous across the seam along a chain
    # (PAPER.md:360): the point half a cell beyond s = +1/2 of (p, m) is s = -1/2 of (p + m ikxspace, m).
    # Linear extrapolation from both sides to the seam agrees to O(ds^2) of the curvature.
    ns = 8
    for m in (1, 2):
        for p in range(11 - 2 * m):
            left = 1.5 * o.table("kappa")[ns - 1, p, m] - 0.5 * o.table("kappa")[ns - 2, p, m]
            right = 1.5 * o.table("kappa")[0, p + 2 * m, m] - 0.5 * o.table("kappa")[1, p + 2 * m, m]
            # exact value at the seam theta = pi: -(ky cos(pi) + kx_eff sin(pi)) = ky
            assert abs(left - right) < 0.6 * (2 * np.pi / ns) ** 2 * (abs(kx[p]) + 3 * ky[m] + 1), (m, p)


# ------------------------------------------------------------------------------------------------
# The 1-D streaming operator (I + DISS_S) on one open chain, as a whole: oracle's operator built from unit
# vectors vs a matrix assembled here from the stencil definition of DESIGN.md section 2 / R7, then the RK4
# stability limit in Courant number (closure 0 stable to about 1.85, closure 1 to about 2.2).
# ------------------------------------------------------------------------------------------------
def _streaming_matrix(n, sign_v, nu, closure):
    """d/dt g = -c [D g + nu * sign-free |.| delta^4 g / 12] in units c = |v_R v F| / ds = 1 for v > 0:
    returns M with dg/dt = (c / 1) M g, for a chain of n points with open ends."""
    c4 = np.array([1, -8, 0, 8, -1]) / 12.0
    d4 = np.array([1, -4, 6, -4, 1]) / 12.0
    up_pos = np.array([0.5, -2.0, 1.5, 0, 0])      # backward differences for v > 0
    up_neg = np.array([0, 0, -1.5, 2.0, -0.5])
    M = np.zeros((n, n))
    for i in range(n):
        edge = (i < 2) or (i >= n - 2)
        if edge and closure == 0:
            st, dis = (up_pos if sign_v > 0 else up_neg), np.zeros(5)
        else:
            st, dis = c4, d4
        for d in range(-2, 3):
            if 0 <= i + d < n:                         # ghosts beyond an open end are zero
                M[i, i + d] += -sign_v * st[d + 2] - nu * dis[d + 2]
    return M


def _rk4_stable(lam_dt):
    z = lam_dt
    R = 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24
    return np.abs(R).max() <= 1 + 1e-9


@pytest.mark.parametrize("closure", [0, 1])
def test_streaming_operator_eigenvalues_and_rk4_courant_limit(closure):
    ns, nkx, m, ikx = 8, 7, 1, 2          # chain through kx index 1: 1 -> 3 -> 5, three links, 24 points
    cfg = small_cfg(nkx=nkx, nky=2, ns=ns, nvpar=4, nmu=1, ikxspace=ikx, disp_par=1.0, s_closure=closure)
    o = GkRef(cfg, term_mask=G.T_I | G.T_DISS_S)
    _, _, v, _, _, _ = _grids(cfg)
    F = 1.0 / (2 * np.pi * cfg["geom"]["q"])
    chain = [1, 3, 5]
    limits = []
    for j in (0, 3):                       # v < 0 and v > 0
        n = ns * len(chain)
        Mo = np.zeros((n, n), complex)
        e = np.zeros(o.shape, complex)
        for col in range(n):
            e[0, j, 0, col % ns, chain[col // ns], m] = 1
            r, _ = o.rhs(e)
            Mo[:, col] = np.concatenate([r[0, j, 0, :, p, m] for p in chain])
            # nothing leaks off the chain or to other velocities
            r[0, j, 0, :, chain, m] = 0
            assert abs(r).max() == 0
            e[:] = 0
        c = abs(v[j]) * F * ns             # |v_R v F| / ds
        Mi = c * _streaming_matrix(n, np.sign(v[j]), 1.0, closure)
        np.testing.assert_allclose(Mo, Mi, atol=1e-12 * c)
        lam = np.linalg.eigvals(Mi / c)
        assert lam.real.max() < 1e-12      # the discrete operator is dissipative: no growing mode
        lo, hi = 0.5, 4.0
        for _ in range(40):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if _rk4_stable(lam * mid) else (lo, mid)
        limits.append(lo)
    # mirror symmetry of the two streaming directions
    assert limits[0] == pytest.approx(limits[1], rel=1e-6)
    # SURVEY R7's stability estimates (nu_s = 1)
    want = 1.85 if closure == 0 else 2.2
    assert abs(limits[0] - want) < 0.03, limits      # 1.857 and 2.227 on this 24-point chain


# ------------------------------------------------------------------------------------------------
# gkref_fluxes (R18): heat and momentum moments for a one-mode state, closed form
# ------------------------------------------------------------------------------------------------
def test_flux_moments_closed_form_for_one_mode():
    from scipy.special import j0 as bessel_j0
    cfg = small_cfg(nkx=5, nky=3, ns=4, nvpar=8, nmu=3, mu_grid=1, nspecies=2, adiabatic=0, ky0=0.3)
    o = GkRef(cfg)
    s, th, v, dv, kx, ky = _grids(cfg)
    eps, shat = cfg["geom"]["eps"], cfg["geom"]["shat"]
    B = 1 / (1 + eps * np.cos(th))
    R = 1 + eps * np.cos(th)
    dvp = cfg["grid"]["vperp_max"] / 3
    vp = (np.arange(3) + 0.5) * dvp
    mu, wmu = 0.5 * vp ** 2, vp * dvp
    i, p, m = 1, 3, 2
    phi = np.zeros(o.phi_shape, complex)
    phi[i, p, m] = 0.7 - 0.2j
    f = np.zeros(o.shape, complex)
    cs = [0.3 + 0.5j, -0.4 + 0.1j]
    gfun = 1 + 0.3 * v[:, None] + 0.1 * v[:, None] ** 2 + 0.2 * mu[None, :]      # any g(v, mu)
    for a in range(2):
        f[a, :, :, i, p, m] = cs[a] * gfun
    got = o.fluxes(f, phi)
    kperp = np.sqrt((kx[p] + shat * th[i] * ky[m]) ** 2 + ky[m] ** 2)
    for a, sp in enumerate(cfg["species"]):
        vR = np.sqrt(sp["temp"] / sp["mass"])
        lam = kperp * (sp["mass"] * vR / abs(sp["Z"])) * np.sqrt(2 * mu / B[i])   # R4
        J0 = bessel_j0(lam)
        im = (np.conj(phi[i, p, m]) * cs[a]).imag
        w = -(1 / 4) * 2 * (ky[m] / 2) * 2 * np.pi * B[i] * dv * im               # P_m = 2, 1/ns = 1/4
        E = v[:, None] ** 2 + 2 * mu[None, :] * B[i]
        base = wmu[None, :] * J0[None, :] * gfun
        want = [w * base.sum(), w * (base * E).sum() * sp["temp"],
                w * (base * v[:, None]).sum() * sp["mass"] * vR * R[i]]
        np.testing.assert_allclose(got[a], want, rtol=1e-10)


def test_heat_flux_of_the_unstable_itg_eigenmode_is_outward():
    # the most unstable local toroidal-ITG eigenvector (q -> infinity, eps = 0; see test_oracle_physics) with
    # its own phi: a growing ITG mode carries heat down the temperature gradient, Q_heat > 0, and, with
    # adiabatic electrons, no particles
    cfg = small_cfg(nkx=3, nky=2, ns=4, nvpar=16, nmu=4, mu_grid=0, ky0=0.35, q=1e9, eps=0.0, nonlinear=0)
    o = GkRef(cfg, term_mask=G.T_ALL & ~G.T_HYP & ~G.T_III)
    i, p, m = 2, 1, 1
    n = 16 * 4
    M = np.empty((n, n), complex)
    e = np.zeros(o.shape, complex)
    for c in range(n):
        e[0, c // 4, c % 4, i, p, m] = 1
        r, _ = o.rhs(e)
        M[:, c] = r[0, :, :, i, p, m].ravel()
        e[:] = 0
    lam, vec = np.linalg.eig(M)
    k = np.argmax(lam.real)
    assert lam[k].real > 0.05
    f = np.zeros(o.shape, complex)
    f[0, :, :, i, p, m] = vec[:, k].reshape(16, 4)
    fl = o.fluxes(f, o.field_solve(f))
    assert fl[0, 1] > 0
    assert abs(fl[0, 0]) < 1e-12 * fl[0, 1]
