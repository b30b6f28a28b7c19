"""Pins for the oracle's circular (Lapillonne) geometry, eq. 1-4, reading R24.  Expected values come
from (i) the formulas the paper prints, (ii) NUMERICAL differentiation, written here, of the coordinate maps
(R, Z, phi) -> (psi, zeta, s) -- the oracle uses closed-form derivatives --, (iii) the eps -> 0 limit, which must be
the s-alpha model the other pins fix, and (iv) continuity along the extended field line."""
import numpy as np
import pytest

from oracle.gkref import GkRef
from tests.util import small_cfg, rand_c, rel_l2

Q, SHAT, EPS = 1.4, 0.78, 0.19


def circ_cfg(eps=EPS, **kw):
    base = dict(nkx=11, nky=4, ns=16, nvpar=4, nmu=2, ikxspace=2, ky0=0.13, mu_grid=1)
    base.update(kw)
    cfg = small_cfg(**base)
    cfg["geom"].update(q=Q, shat=SHAT, eps=eps)
    cfg["opts"]["geometry"] = 1
    return cfg


# ---- the coordinate maps, as functions of (eps, theta), and everything derived from them by finite differences ----
def q_of(eps, eps0):
    return Q * (eps / eps0) ** SHAT                      # (eps/q) dq/deps = shat at eps0


def s_of(eps, th):
    return (th + eps * np.sin(th)) / (2 * np.pi)


def zeta_of(eps, th, eps0, turns=0):
    a = np.arctan(np.sqrt((1 - eps) / (1 + eps)) * np.tan(th / 2)) + np.pi * turns   # branch-tracked
    return q_of(eps, eps0) / np.pi * a                    # the -phi/2pi part is added analytically below


def b_of(eps, th, eps0):
    q = q_of(eps, eps0)
    delta = np.sqrt(1 + eps ** 2 / (q ** 2 * (1 - eps ** 2)))
    return delta / (1 + eps * np.cos(th))                 # eq. 1


def derived(eps0, th, turns=0, h=1e-6):
    d_e = lambda f: (f(eps0 + h, th) - f(eps0 - h, th)) / (2 * h)
    d_t = lambda f: (f(eps0, th + h) - f(eps0, th - h)) / (2 * h)
    R = 1 + eps0 * np.cos(th)
    # gradients in the orthonormal frame (e_r, e_theta, e_phi): (d/deps, (1/eps) d/dtheta, (1/R) d/dphi)
    g_psi = np.array([1.0, 0.0, 0.0])
    fs = lambda e, t: s_of(e, t)
    fz = lambda e, t: zeta_of(e, t, eps0, turns)
    fb = lambda e, t: b_of(e, t, eps0)
    g_s = np.array([d_e(fs), d_t(fs) / eps0, 0.0])
    g_z = np.array([d_e(fz), d_t(fz) / eps0, -1 / (2 * np.pi * R)])
    B = fb(eps0, th)
    # derivatives of B at fixed (psi, s): invert the Jacobian of (eps, theta) -> (psi, s)
    J = np.array([[1.0, 0.0], [d_e(fs), d_t(fs)]])        # rows: d(psi), d(s) / d(eps, theta)
    dB = np.linalg.solve(J.T, np.array([d_e(fb), d_t(fb)]))   # (dB/dpsi|s, dB/ds|psi)
    gpp, gpz, gzz = g_psi @ g_psi, g_psi @ g_z, g_z @ g_z
    gps, gzs = g_psi @ g_s, g_z @ g_s
    pref = np.pi * (eps0 / (Q * np.sqrt(1 - eps0 ** 2))) / B ** 2          # pi dpf/dpsi / B^2
    Epz, Eps, Ezs = pref * (gpp * gzz - gpz ** 2), pref * (gpp * gzs - gps * gpz), pref * (gpz * gzs - gps * gzz)
    Dpsi = -2 * (Eps * dB[1]) / B                                          # eq. 4 (E^{psi psi} = 0)
    Dzeta = -2 * (-Epz * dB[0] + Ezs * dB[1]) / B
    return dict(B=B, dBds=dB[1], gpz=gpz, gzz=gzz, Dpsi=Dpsi, Dzeta=Dzeta, Epz=Epz, R=R)


def test_theta_grid_and_field_strength_follow_eq_1():
    o = GkRef(circ_cfg())
    s, th, B = o.table("s"), o.table("theta"), o.table("B")
    np.testing.assert_allclose(th + EPS * np.sin(th), 2 * np.pi * s, atol=1e-13)
    delta = np.sqrt(1 + EPS ** 2 / (Q ** 2 * (1 - EPS ** 2)))
    np.testing.assert_allclose(B, delta / (1 + EPS * np.cos(th)), rtol=1e-14)          # eq. 1
    b_ups = 1 / (2 * np.pi * Q * np.sqrt(1 - EPS ** 2))
    np.testing.assert_allclose(o.table("F"), b_ups / B, rtol=1e-14)
    # gfun = F d_s B / B: d_s B by differentiating B(s) numerically through the theta(s) inversion
    def b_at_s(sv):
        t = 2 * np.pi * sv
        for _ in range(60):
            t = t - (t + EPS * np.sin(t) - 2 * np.pi * sv) / (1 + EPS * np.cos(t))
        return delta / (1 + EPS * np.cos(t))
    h = 1e-6
    np.testing.assert_allclose(o.table("BG"), o.table("F") * (b_at_s(s + h) - b_at_s(s - h)) / (2 * h), rtol=1e-7, atol=1e-9)
    np.testing.assert_allclose(o.table("R"), (1 + EPS * np.cos(th)) / delta, rtol=1e-14)   # R B_t/B, bt_frac = 1/delta


def test_metric_and_drifts_against_numerical_differentiation_of_the_coordinate_maps():
    cfg = circ_cfg()
    o = GkRef(cfg)
    th = o.table("theta")
    kth = np.sqrt(derived(EPS, 0.0)["gzz"])
    np.testing.assert_allclose(o.table("kthnorm")[0], kth, rtol=1e-8)
    d = [derived(EPS, t) for t in th]
    np.testing.assert_allclose(o.table("gpz"), [x["gpz"] / kth for x in d], rtol=1e-7, atol=1e-9)
    np.testing.assert_allclose(o.table("gzz"), [x["gzz"] / kth ** 2 for x in d], rtol=1e-7)
    np.testing.assert_allclose(o.table("sth"), [-x["Dpsi"] for x in d], rtol=1e-6, atol=1e-8)
    np.testing.assert_allclose(o.table("cz"), [-x["Dzeta"] / kth for x in d], rtol=1e-6, atol=1e-8)
    np.testing.assert_allclose(o.table("ef"), [2 * x["Epz"] / kth for x in d], rtol=1e-7)
    # k_perp^2 (eq. 2) and kappa assembled from them
    kx = (np.arange(11) - 5) * o.table("dkx")[0]
    ky = np.arange(4) * 0.13
    kp2 = kx[None, :, None] ** 2 + 2 * kx[None, :, None] * ky[None, None, :] * o.table("gpz")[:, None, None] \
        + ky[None, None, :] ** 2 * o.table("gzz")[:, None, None]
    np.testing.assert_allclose(o.table("kperp2"), kp2, rtol=1e-13)
    kap = -(kx[None, :, None] * o.table("sth")[:, None, None] + ky[None, None, :] * o.table("cz")[:, None, None])
    np.testing.assert_allclose(o.table("kappa"), kap, rtol=1e-13, atol=1e-15)
    # the field line lies in the zeta = const surface: b . grad zeta = 0 with b = (B_t e_phi + B_p e_theta)/B,
    # B_t = 1/R, B_p = eps/(q sqrt(1-eps^2) R) -- ties the arctan form of zeta to eq. 1
    h = 1e-6
    for t in th[::3]:
        R = 1 + EPS * np.cos(t)
        z_th = (zeta_of(EPS, t + h, EPS) - zeta_of(EPS, t - h, EPS)) / (2 * h)
        assert abs((1 / R) * (-1 / (2 * np.pi * R)) + EPS / (Q * np.sqrt(1 - EPS ** 2) * R) * z_th / EPS) < 1e-8


def test_small_eps_limit_is_the_s_alpha_model():
    for eps in (1e-3, 1e-4):
        c1 = circ_cfg(eps)
        c0 = circ_cfg(eps)
        c0["opts"]["geometry"] = 0
        a, b = GkRef(c0), GkRef(c1)
        for name in ("B", "F", "BG", "sth", "cz", "gpz", "gzz", "ef", "dkx", "kthnorm", "R", "kperp2", "kappa"):
            x, y = a.table(name), b.table(name)
            assert np.abs(x - y).max() <= 3 * eps * max(np.abs(x).max(), 1e-30), (name, eps)


def test_kperp_and_kappa_are_continuous_along_the_extended_field_line():
    # Leaving at s = +1/2, (p, m) continues at s = -1/2 in (p + m ikxspace, m).  With the branch-tracked
    # arctan, g_psizeta grows by q' = shat q / eps per turn, so the link n of a chain at the principal-branch angle
    # theta must equal link 0 evaluated at the extended angle theta + 2 pi n.
    cfg = circ_cfg()
    o = GkRef(cfg)
    th = o.table("theta")
    kth, dkx = o.table("kthnorm")[0], o.table("dkx")[0]
    np.testing.assert_allclose(dkx, (SHAT * Q / EPS) / kth * 0.13 / 2, rtol=1e-12)      # R24
    kp2, kap = o.table("kperp2"), o.table("kappa")
    for m in (1, 2):
        ky = m * 0.13
        for p0 in range(2 * m):                       # chains start at p0 < m ikxspace
            kx0 = (p0 - 5) * dkx
            n = 0
            p = p0
            while p < 11:
                for i in (0, 5, 15):
                    d = derived(EPS, th[i], turns=n)
                    want = kx0 ** 2 + 2 * kx0 * ky * d["gpz"] / kth + ky ** 2 * d["gzz"] / kth ** 2
                    np.testing.assert_allclose(kp2[i, p, m], want, rtol=2e-6)
                    np.testing.assert_allclose(kap[i, p, m], kx0 * d["Dpsi"] + ky * d["Dzeta"] / kth, rtol=2e-5, atol=1e-7)
                p += 2 * m
                n += 1


def test_exb_factor_enters_drive_bracket_and_fluxes():
    # terms V and III and the fluxes carry E^{psi zeta} k_zeta = ef ky / 2: compare with the s-alpha operator given
    # the same phi-independent inputs, plane by plane
    from oracle import gkref as G
    cfg1 = circ_cfg(nkx=9, nky=4, ns=8, nvpar=4, nmu=2, ikxspace=1)
    cfg0 = circ_cfg(nkx=9, nky=4, ns=8, nvpar=4, nmu=2, ikxspace=1)
    cfg0["opts"]["geometry"] = 0
    o1 = GkRef(cfg1, term_mask=G.T_III, bracket_method=1)
    ef = o1.table("ef")
    # B = 2 pi dpf/dpsi grad psi x grad zeta, so E^{psi zeta} = pi dpf |grad psi x grad zeta|^2 / B^2 = 1/(4 pi dpf):
    # constant along the field line, closed form
    np.testing.assert_allclose(ef, Q * np.sqrt(1 - EPS ** 2) / (2 * np.pi * EPS * o1.table("kthnorm")[0]), rtol=1e-12)
    rng = np.random.default_rng(11)
    chi, fs = rand_c(rng, (9, 4), True), rand_c(rng, (9, 4), True)
    # the bracket of two slabs does not know the plane; rhs_slab applies ef[i]
    f = np.zeros(o1.shape, complex)
    f[0, 1, 0, 3] = fs
    phi = np.zeros(o1.phi_shape, complex)
    phi[3] = chi / o1.table("J0")[0, 0, 3]
    got = o1.rhs_slab(f, phi, 0, 1, 0, 3)
    np.testing.assert_allclose(got, ef[3] * o1.bracket_slab(chi, fs, 1), rtol=1e-12, atol=1e-14)
    # term V: diagonal closed form -i (ef ky / 2) chi F_M [R/Ln + (E - 3/2) R/LT]
    oV = GkRef(cfg1, term_mask=G.T_V)
    r = oV.rhs_slab(f, phi, 0, 1, 0, 3)
    v, mu, B, FM = oV.table("vpar"), oV.table("mu"), oV.table("B"), oV.table("FM")
    E = v[1] ** 2 + 2 * mu[0] * B[3]
    ky = np.arange(4) * 0.13
    want = -1j * (ef[3] * ky[None, :] / 2) * chi * FM[1, 0, 3] * (2.0 + (E - 1.5) * 7.0)
    np.testing.assert_allclose(r, want, rtol=1e-12, atol=1e-16)
