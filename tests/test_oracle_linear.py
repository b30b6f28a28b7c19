"""Pins for the oracle's linear terms: stencil exactness and order, the seam gather, the
velocity stencil, characteristic (energy) invariance of I+IV, reality symmetry, and advection
against its analytic solution."""
import numpy as np
import pytest

from oracle import gkref as G
from oracle.gkref import GkRef
from tests.util import small_cfg, rand_c, rel_l2


def _chain(nkx, m, ikx, start=None):
    """kx indices of the chain through `start` (default: the one containing the centre) for ky index m."""
    p = (nkx - 1) // 2 if start is None else start
    if m == 0:
        return [p]
    while p - m * ikx >= 0:
        p -= m * ikx
    out = []
    while p < nkx:
        out.append(p)
        p += m * ikx
    return out


def _lay_on_chain(o, cfg, m, fun, a=0):
    """f(j,l,i,p,m) = fun(theta_ext) on every chain of ky index m (theta_ext grows by 2 pi per link)."""
    g = cfg["grid"]
    f = np.zeros(o.shape, complex)
    th = o.table("theta")
    done = set()
    for p0 in range(g["nkx"]):
        ch = _chain(g["nkx"], m, g["ikxspace"], p0)
        if ch[0] in done:
            continue
        done.add(ch[0])
        # centre the extended angle on the middle link
        mid = len(ch) // 2
        for n, p in enumerate(ch):
            f[a, :, :, :, p, m] = fun(th + 2 * np.pi * (n - mid))[None, None, :]
    return f


def test_parallel_derivative_4th_order_across_the_seam():
    # term I only: rhs = -vR v_j F d/ds f.  A Gaussian in the extended angle, centred on a seam,
    # is differentiated through the kx connection; error must fall as ds^4.
    errs = []
    for ns in (16, 32, 64):
        cfg = small_cfg(nkx=9, nky=3, ns=ns, nvpar=4, nmu=1, ikxspace=1)
        o = GkRef(cfg, term_mask=G.T_I)
        sig = 0.9
        fun = lambda t: np.exp(-((t - np.pi) ** 2) / (2 * sig ** 2))          # centred ON the seam
        dfun = lambda t: -(t - np.pi) / sig ** 2 * fun(t)
        m = 1
        f = _lay_on_chain(o, cfg, m, fun)
        rhs, _ = o.rhs(f)
        v, F = o.table("vpar"), o.table("F")
        ch = _chain(9, m, 1)
        mid = len(ch) // 2
        th = o.table("theta")
        err = 0.0
        for n in (mid, mid + 1):  # the two links that meet at the seam theta_ext = pi
            exact = -v[:, None] * F[None, :] * 2 * np.pi * dfun(th + 2 * np.pi * (n - mid))[None, :]
            err = max(err, abs(rhs[0, :, 0, :, ch[n], m] - exact).max())
        errs.append(err)
    assert errs[0] / errs[1] > 12 and errs[1] / errs[2] > 13, errs


def test_boundary_classes_polynomial_exactness():
    # class 0: centred 4th order exact for quartics (dissipation: 4th difference kills cubics).
    # class != 0 (closure 0): 2nd-order upwind, exact for quadratics on the side that does not
    # look through the open end.  ky index m=3 with nkx=5: every chain is a single link.
    cfg = small_cfg(nkx=5, nky=4, ns=12, nvpar=4, nmu=1, ikxspace=1)
    o = GkRef(cfg, term_mask=G.T_I)
    s = o.table("s")
    v, F = o.table("vpar"), o.table("F")
    f = np.zeros(o.shape, complex)
    poly = lambda x: 1 + x - 2 * x ** 2
    dpoly = lambda x: 1 - 4 * x
    f[0, :, :, :, :, 3] = poly(s)[None, None, :, None]
    rhs, _ = o.rhs(f)
    exact = -v[:, None] * F[None, :] * dpoly(s)[None, :]
    got = rhs[0, :, 0, :, 2, 3].real
    # interior always exact; left end (i=0,1) exact for v<0 rows, right end for v>0 rows
    np.testing.assert_allclose(got[:, 2:-2], exact[:, 2:-2], atol=1e-12)
    np.testing.assert_allclose(got[v < 0][:, :2], exact[v < 0][:, :2], atol=1e-12)
    np.testing.assert_allclose(got[v > 0][:, -2:], exact[v > 0][:, -2:], atol=1e-12)
    # inflow side sees zero ghosts: at i=0, v>0 the upwind formula reduces to 3 f_0/(2 ds)
    ds = 1 / 12
    np.testing.assert_allclose(got[v > 0][:, 0], -v[v > 0] * F[0] * 1.5 * poly(s[0]) / ds, rtol=1e-12)
    # quartic exactness in the interior, periodic zonal chain untouched by classes
    q4 = lambda x: x ** 4 - x ** 3
    f[:] = 0
    f[0, :, :, :, :, 3] = q4(s)[None, None, :, None]
    rhs, _ = o.rhs(f)
    exact = -v[:, None] * F[None, :] * (4 * s ** 3 - 3 * s ** 2)[None, :]
    np.testing.assert_allclose(rhs[0, :, 0, 2:-2, 2, 3].real, exact[:, 2:-2], atol=1e-12)


def test_zero_ghost_closure_uses_centred_stencil_everywhere():
    cfg = small_cfg(nkx=5, nky=4, ns=12, nvpar=4, nmu=1, s_closure=1)
    o = GkRef(cfg, term_mask=G.T_I)
    np.testing.assert_allclose(o.table("dcoef")[0], o.table("dcoef")[2])
    np.testing.assert_allclose(o.table("dcoef")[2, 0] * 12, [1, -8, 0, 8, -1])


def test_velocity_stencil_and_mirror_coefficient():
    # term IV only: +vR mu B G d/dv f, centred 4th order, zero padding
    cfg = small_cfg(nkx=3, nky=2, ns=8, nvpar=16, nmu=2)
    o = GkRef(cfg, term_mask=G.T_IV)
    v, mu, BG = o.table("vpar"), o.table("mu"), o.table("BG")
    f = np.zeros(o.shape, complex)
    f[0] = (v ** 4 - 2 * v)[:, None, None, None, None] * (1 + 0.5j)
    rhs, _ = o.rhs(f)
    exact = (mu[None, :, None] * BG[None, None, :]) * (4 * v ** 3 - 2)[:, None, None] * (1 + 0.5j)
    np.testing.assert_allclose(rhs[0, 2:-2, :, :, 1, 1], exact[2:-2], rtol=1e-11, atol=1e-12)
    # zero padding at the edge: j=0 row uses only j=0,1,2
    dv = v[1] - v[0]
    g = (v ** 4 - 2 * v)
    edge = (8 * g[1] - g[2]) / (12 * dv)
    np.testing.assert_allclose(rhs[0, 0, 1, 3, 1, 1], mu[1] * BG[3] * edge * (1 + 0.5j), rtol=1e-12)


def test_energy_is_a_characteristic_invariant_of_I_plus_IV():
    # (-v F d_s + mu B G d_v) g(v^2 + 2 mu B(s)) = 0 because B G = F d_s B:
    # the two discrete terms must cancel to O(ds^4 + dv^4) although each is O(1).
    res = []
    for n in (16, 32):
        cfg = small_cfg(nkx=3, nky=1, ns=n, nvpar=2 * n, nmu=2, mu_grid=1)
        o = GkRef(cfg, term_mask=G.T_I | G.T_IV)
        oI = GkRef(cfg, term_mask=G.T_I)
        f = np.zeros(o.shape, complex)
        FM = o.table("FM")  # a function of the energy only
        f[0] = FM[:, :, :, None, None]
        both, _ = o.rhs(f)
        only, _ = oI.rhs(f)
        j = slice(2, -2)
        res.append(abs(both[0, j]).max() / abs(only[0, j]).max())
    assert res[0] < 2e-2 and res[1] < res[0] / 10, res


def test_linear_operator_preserves_ky0_reality():
    cfg = small_cfg(nkx=9, nky=3, ns=8, nvpar=8, nmu=2, nonlinear=0)
    o = GkRef(cfg)
    f = rand_c(np.random.default_rng(3), o.shape, True)
    rhs, phi = o.rhs(f)
    np.testing.assert_allclose(rhs[..., :, 0], np.conj(rhs[..., ::-1, 0]), atol=1e-12 * abs(rhs).max())
    np.testing.assert_allclose(phi[:, :, 0], np.conj(phi[:, ::-1, 0]), atol=1e-12 * abs(phi).max())
    assert phi[:, 4, 0].tolist() == [0] * 8                       # phi(kx=0,ky=0) = 0


def test_term_mask_is_additive():
    cfg = small_cfg(nkx=9, nky=3, ns=8, nvpar=8, nmu=2)
    f = rand_c(np.random.default_rng(4), GkRef(cfg).shape, True)
    full, _ = GkRef(cfg).rhs(f)
    acc = 0
    for bit in range(10):
        r, _ = GkRef(cfg, term_mask=1 << bit).rhs(f)
        acc = acc + r
    assert rel_l2(acc, full) < 1e-13


def test_advection_matches_analytic_translation():
    # term I alone on the periodic zonal chain: f(s,t) = f0(s - vR v F t).  RK4 + 4th-order stencil.
    cfg = small_cfg(nkx=3, nky=1, ns=64, nvpar=4, nmu=1, geom_q=None)
    cfg["geom"]["q"] = 0.05      # fast streaming so the shift is visible: F = 1/(2 pi q)
    o = GkRef(cfg, term_mask=G.T_I)
    s, v, F = o.table("s"), o.table("vpar"), o.table("F")[0]
    f0 = lambda x: np.exp(np.cos(2 * np.pi * x))
    f = np.zeros(o.shape, complex)
    f[0, :, 0, :, 2, 0] = f0(s)[None, :]
    T, n = 0.02, 40
    out = o.rk4_step(f, T / n, n)
    exact = f0(s[None, :] - v[:, None] * F * T)
    np.testing.assert_allclose(out[0, :, 0, :, 2, 0].real, exact, atol=3e-4)
    # and the sign: positive v moves the profile towards positive s
    assert np.argmax(out[0, 3, 0, :, 2, 0].real) > np.argmax(f[0, 3, 0, :, 2, 0].real)
