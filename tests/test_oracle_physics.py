"""Physics pins for the oracle's linear operator as a whole: eigenvalues of the operator built
from unit vectors through gkref_rhs must be roots of independently written textbook dispersion
relations (local kinetic toroidal ITG; slab parallel streaming), the time-stepped solution must
grow at the eigen-solve's rate, and the Rosenbluth-Hinton residual must match eq. 5 of the paper."""
import numpy as np
import pytest

from oracle import gkref as G
from oracle.gkref import GkRef
from tests.util import small_cfg, rel_l2


def _operator_matrix(o, sel, leak_tol=1e-12):
    """Dense matrix of f -> rhs(f) restricted to the index set `sel` (a boolean mask over f)."""
    idx = np.flatnonzero(sel.ravel())
    n = len(idx)
    M = np.empty((n, n), complex)
    e = np.zeros(o.shape, complex)
    for c, q in enumerate(idx):
        e.ravel()[q] = 1.0
        r, _ = o.rhs(e)
        # nothing may leak outside the selected subspace
        out = r.ravel().copy()
        M[:, c] = out[idx]
        out[idx] = 0
        assert abs(out).max() < leak_tol
        e.ravel()[q] = 0.0
    return M


def test_local_toroidal_itg_dispersion_relation():
    # q -> infinity removes parallel streaming (F = 1/(2 pi q)) and eps = 0 the mirror force, so each
    # (s_i, kx, ky>0) decouples and the linear operator on f(v_par, mu) is diagonal + rank one.  Its
    # eigenvalues lambda = -i omega are the roots of the textbook local kinetic dispersion relation
    #   D(omega) = 1 + Te/Ti... = (Z^2 n/T) + ne/Te - (Z^2 n/T) int J0^2 F_M (omega-omega_*T)/(omega-omega_d) d^3v
    # with omega_d = (T/Z)(v_par^2 + mu B) kappa, omega_*T = -(T/Z)(ky/2)[R/Ln + (E-3/2) R/LT]
    # (the integral as the discrete quadrature; Gamma0 analytic minus its quadrature is carried).
    cfg = small_cfg(nkx=3, nky=2, ns=4, nvpar=16, nmu=4, mu_grid=0, ky0=0.35, q=1e9, eps=0.0,
                    nonlinear=0)
    mask = G.T_ALL & ~G.T_HYP & ~G.T_III
    o = GkRef(cfg, term_mask=mask)
    v, mu, wmu, wv = o.table("vpar"), o.table("mu"), o.table("wmu"), o.table("wv")[0]
    B, J0, G0, FM, kap = o.table("B"), o.table("J0"), o.table("Gamma0"), o.table("FM"), o.table("kappa")
    ky = o.table("ky")
    sp = cfg["species"][0]
    unstable = []
    for (i, p, m) in [(2, 1, 1), (1, 2, 1), (0, 0, 1)]:
        sel = np.zeros(o.shape, bool)
        sel[0, :, :, i, p, m] = True
        lam = np.linalg.eigvals(_operator_matrix(o, sel, leak_tol=1e-7))   # residual streaming ~ 1/q
        E = v[:, None] ** 2 + 2 * mu[None, :] * B[i]
        ED = v[:, None] ** 2 + mu[None, :] * B[i]
        w_d = ED * kap[i, p, m]                                  # T = Z = 1
        w_s = -(ky[m] / 2) * (sp["rln"] + (E - 1.5) * sp["rlt"])
        W = 2 * np.pi * B[i] * wv * wmu[None, :] * J0[0, :, i, p, m][None, :] ** 2 * FM[:, :, i]
        g0 = G0[0, i, p, m]

        def D(om):
            return 1 + 1 - (g0 - W.sum()) - (W * (om - w_s) / (om - w_d)).sum()

        k = np.argmax(lam.real)
        om = 1j * lam[k]
        scale = abs((W * (w_d - w_s) / (om - w_d) ** 2).sum()) * abs(om)   # |omega dD/domega|
        assert abs(D(om)) < 1e-9 * max(scale, 1.0), (i, p, m, lam[k])
        unstable.append(lam[k].real)
    # bad-curvature side (theta ~ 0.79: kappa<0 ... i=2) is ITG unstable at R/LT = 7; the inboard
    # side (i=0, theta=-2.36, good curvature) is not.
    assert unstable[0] > 0.05 and unstable[2] < 1e-9, unstable


def test_slab_streaming_dispersion_relation():
    # terms I + VII + polarisation-only field solve on the periodic zonal chain with eps = 0:
    # plane waves exp(2 pi i n s) with effective wavenumber of the centred 4th-order stencil
    # k_n = [8 sin(2 pi n/ns) - sin(4 pi n/ns)]/(6 ds); textbook electrostatic slab dispersion
    #   D_n(omega) = (1 - Gamma0) - int J0^2 F_M k_n c/(omega - k_n c) d^3v,  c = vR v_par F
    # Collisionless + no dissipation: all omega real (Case-van Kampen modes).
    cfg = small_cfg(nkx=3, nky=1, ns=8, nvpar=12, nmu=2, mu_grid=0, eps=0.0, q=0.7, adiabatic=0,
                    nonlinear=0)
    o = GkRef(cfg, term_mask=G.T_I | G.T_VII)
    sel = np.zeros(o.shape, bool)
    sel[0, :, :, :, 2, 0] = True
    lam = np.linalg.eigvals(_operator_matrix(o, sel))
    assert abs(lam.real).max() < 1e-12 * abs(lam).max()
    v, wmu, wv = o.table("vpar"), o.table("wmu"), o.table("wv")[0]
    J0, G0, FM, F = o.table("J0"), o.table("Gamma0"), o.table("FM"), o.table("F")[0]
    ns, ds = 8, 1 / 8
    n = np.arange(ns)
    kn = (8 * np.sin(2 * np.pi * n / ns) - np.sin(4 * np.pi * n / ns)) / (6 * ds)
    c = v * F
    W = 2 * np.pi * wv * wmu[None, :] * J0[0, :, 0, 2, 0][None, :] ** 2 * FM[:, :, 0]
    g0 = G0[0, 0, 2, 0]
    bad = 0
    for om in (1j * lam):
        ok = False
        for k in kn:
            poles = k * c
            if abs(om - poles).min() < 1e-9:
                ok = True
                break
            Dn = (1 - g0) - (W * (k * c)[:, None] / (om - poles)[:, None]).sum()
            slope = abs((W * (k * c)[:, None] / (om - poles)[:, None] ** 2).sum())
            if abs(Dn) < 1e-8 * max(1.0, slope * abs(om)):
                ok = True
                break
        bad += not ok
    assert bad == 0


def test_time_stepped_growth_matches_eigen_solve():
    # Whole linear operator (all terms, seam connectivity, boundary classes, adiabatic field solve)
    # on one ky>0 family of chains of a config-1-sized grid: matrix from unit vectors ->
    # numpy.linalg.eigvals; the RK4-stepped solution must grow as |R(lambda dt)| per step,
    # R(z) = 1 + z + z^2/2 + z^3/6 + z^4/24.
    cfg = small_cfg(nkx=5, nky=2, ns=8, nvpar=8, nmu=2, ky0=0.3, ikxspace=1, nonlinear=0)
    o = GkRef(cfg)
    sel = np.zeros(o.shape, bool)
    sel[..., 1] = True                                    # all kx of ky index 1 (chains connect them)
    M = _operator_matrix(o, sel)
    lam = np.linalg.eigvals(M)
    dt = 0.01
    z = lam * dt
    amp = abs(1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24)
    k = np.argmax(amp)
    assert lam[k].real > 0.05                             # R/LT = 7: ITG unstable (sign check, R0)
    rng = np.random.default_rng(21)
    f = np.zeros(o.shape, complex)
    f[..., 1] = rng.standard_normal(o.shape[:-1]) + 1j * rng.standard_normal(o.shape[:-1])
    f = o.rk4_step(f, dt, 3000)
    n0 = np.linalg.norm(f)
    f = o.rk4_step(f, dt, 200)
    rate = (np.linalg.norm(f) / n0) ** (1 / 200)
    np.testing.assert_allclose(rate, amp[k], rtol=2e-5)
    # ballooning: the unstable mode peaks at the outboard midplane theta = 0 (centre of the s grid)
    prof = (abs(f[0, :, :, :, 2, 1]) ** 2).sum(axis=(0, 1))
    assert np.argmax(prof) in (3, 4)


def test_kinetic_electron_omega_h_mode_sets_the_smallest_stable_kperp():
    # Why BASELINE config 4 runs at ky0 = 0.2 (R5): with kinetic electrons the zonal
    # (ky=0, kx=dkx) chain carries the electrostatic omega_H mode, |lambda| ~ k_par v_te/(k_perp rho).
    # Explicit RK4 at dt = 0.002 amplifies it when k_perp = dkx is too small (PAPER.md:356 lists this
    # "field CFL" among the timestep limits).
    amp = {}
    for ky0 in (0.035, 0.2):
        cfg = small_cfg(nkx=3, nky=1, ns=32, nvpar=8, nmu=1, nspecies=2, adiabatic=0, mu_grid=1, ky0=ky0,
                        ikxspace=5, nonlinear=0)
        o = GkRef(cfg)
        sel = np.zeros(o.shape, bool)
        sel[:, :, :, :, 2, 0] = True
        z = np.linalg.eigvals(_operator_matrix(o, sel)) * 0.002
        amp[ky0] = abs(1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24).max()
    assert amp[0.035] > 10 and amp[0.2] < 1.0, amp


@pytest.mark.slow
def test_rosenbluth_hinton_residual():
    # PAPER.md:134, 460-468 (eq. 5): q=1.3, eps=0.05, shat=0.1592, s-alpha, k_psi rho = 0.025,
    # disp_par=0.01, zonal initial condition: phi(inf)/phi(0) = 1/(1+q^2 Theta/eps^2) = 0.07105.
    # Reduced resolution and run time (the paper uses 128x128x16 to t=100 and quotes 0.1 %): the
    # GAM (omega ~ 2.07 v_th/R, weakly damped at q=1.3) is removed by averaging over whole periods.
    # The v_par grid is the paper's (Nv = 128): DESIGN.md section 4 shows that the v_par resolution is the one knob
    # the residual depends on (recurrence time 2 pi q R / dv = 131 at Nv = 128; t = 60 stays below half of it), while
    # Ns = 32 and Nmu = 8 cost well under a per cent.  Measured: 0.07202 (+1.4 %); the round-1 grid 16 x 48 x 8
    # (recurrence at t = 49, inside the averaging window) gave -5.9 % and needed a 12 % tolerance.
    q, shat, eps = 1.3, 0.1592, 0.05
    cfg = small_cfg(nkx=3, nky=1, ns=32, nvpar=128, nmu=8, mu_grid=1, ky0=0.025 / (2 * np.pi * shat),
                    ikxspace=1, nonlinear=0, disp_par=0.01, disp_vp=0.0, disp_x=0.0, disp_y=0.0)
    cfg["geom"].update(q=q, shat=shat, eps=eps)
    cfg["species"][0].update(rlt=0.0, rln=0.0)
    o = GkRef(cfg)
    np.testing.assert_allclose(o.table("kx")[2], 0.025, rtol=1e-12)
    f = np.zeros(o.shape, complex)
    f[0, :, :, :, 0, 0] = f[0, :, :, :, 2, 0] = 1e-4 * o.table("FM")
    phi0 = o.field_solve(f)[:, 2, 0].mean()
    dt, blk = 0.025, 10
    tr = []
    for _ in range(int(60 / (dt * blk))):
        f = o.rk4_step(f, dt, blk)
        tr.append((o.field_solve(f)[:, 2, 0].mean() / phi0).real)
    tr = np.array(tr)
    t = (np.arange(len(tr)) + 1) * dt * blk
    theta = 1.6 * eps ** 1.5 + 0.5 * eps ** 2 + 0.36 * eps ** 2.5
    theory = 1 / (1 + q * q * theta / eps ** 2)
    assert abs(theory - 0.07105) < 1e-4
    # GAM frequency from a damped-cosine least-squares fit of the late signal (fluid theory with the
    # finite-q correction: omega^2 = (7/4 + Te/Ti)(1 + 46/(49 q^2)) v_th^2/R^2)
    from scipy.optimize import least_squares
    late = t > 10
    model = lambda p, x: p[0] + np.exp(-p[1] * x) * (p[2] * np.cos(p[3] * x) + p[4] * np.sin(p[3] * x))
    fit = least_squares(lambda p: model(p, t[late]) - tr[late], [0.07, 0.05, 0.5, 2.0, 0.0])
    omega = abs(fit.x[3])
    np.testing.assert_allclose(omega, np.sqrt(7 / 4 + 1) * np.sqrt(1 + 46 / (49 * q * q)), rtol=0.03)
    period = 2 * np.pi / omega
    nper = 6
    win = (t > 60 - nper * period)
    resid = tr[win].mean()
    assert abs(resid - theory) < 0.05 * theory, (resid, theory)
