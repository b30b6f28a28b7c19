"""GPU parity of the diagnostics folded into the stage launches: the CFL estimate
(R21-R23) and the flux triple reduced inside the first stage of a step,
on the generic kernel and on the production kernels of the BASELINE (kx, ky) planes."""
import numpy as np
import pytest

import gkinputs
from oracle.gkref import GkRef
from tests.util import small_cfg, rand_c, rel_l2

pytestmark = pytest.mark.gpu

MID = dict(nkx=21, nky=6, ns=8, nvpar=9, nmu=3, ikxspace=2, mu_grid=1, ky0=0.15)
PLANES = {
    "mid": (MID, 0), "mid_kinetic": (dict(nspecies=2, adiabatic=0, **MID), 0),
    "cfg2_plane": (dict(nkx=85, nky=16, ky0=0.07, ikxspace=5, ns=8, nvpar=8, nmu=2, mu_grid=1), 2),
    "cfg3_plane": (dict(nkx=85, nky=32, ky0=0.035, ikxspace=5, ns=8, nvpar=8, nmu=2, mu_grid=1), 2),
    "cfg3_plane_kinetic": (dict(nkx=85, nky=32, ky0=0.2, ikxspace=5, ns=8, nvpar=8, nmu=2, mu_grid=1, nspecies=2,
                                adiabatic=0), 2),
    "cfg5_plane": (dict(nkx=127, nky=64, ky0=0.0175, ikxspace=5, ns=8, nvpar=8, nmu=2, mu_grid=1), 5),
    "cfg3_plane_linear": (dict(nkx=85, nky=32, ky0=0.035, ikxspace=5, ns=8, nvpar=8, nmu=2, mu_grid=1, nonlinear=0), 3),
    "cfg5_plane_linear": (dict(nkx=127, nky=64, ky0=0.0175, ikxspace=5, ns=8, nvpar=8, nmu=2, mu_grid=1, nonlinear=0), 3),
    # tiny plane without term III: the point kernel, whose fluxes come from the separate gk_flux_kernel pass
    "tiny_linear": (dict(nkx=9, nky=4, ns=8, nvpar=8, nmu=2, nonlinear=0), 6),
}


def _ctx(case, **kw):
    from paper_2604_06085_b200 import GkContext
    grid, kind = PLANES[case]
    cfg = small_cfg(**grid)
    g = GkContext(cfg, **kw)
    assert g.plan()["kind"] == kind, g.plan()
    return cfg, g


@pytest.mark.parametrize("case", ["mid", "mid_kinetic", "cfg2_plane", "cfg3_plane", "cfg5_plane", "cfg3_plane_linear",
                                  "tiny_linear"])
def test_estimate_dt_parity(case):
    cfg, g = _ctx(case, full_workspace=False)
    p = g.plan()
    nl = bool(cfg["opts"]["nonlinear"])
    o = GkRef(cfg, pad=(p["mx"], p["my"]) if nl else (0, 0))
    # before any stage launch only the create-time bounds exist
    e0 = g.gk_estimate_dt()
    assert np.isinf(e0[1]) and e0[0] == min(e0[2], e0[3])
    f = rand_c(np.random.default_rng(81), o.shape, False).astype(np.complex64)     # asymmetric ky = 0 column (R15)
    rhs, phi = g.gk_rhs(g.to_state(f))
    est = g.gk_estimate_dt()
    ref = o.estimate_dt(phi.cpu().numpy().astype(np.complex128))
    if nl:
        np.testing.assert_allclose(est[1], ref[1], rtol=1e-5)
    else:
        assert np.isinf(est[1]) and np.isinf(ref[1])
    np.testing.assert_allclose(est[2], ref[2], rtol=1e-9)
    if np.isinf(ref[3]):
        assert np.isinf(est[3])
    else:
        np.testing.assert_allclose(est[3], ref[3], rtol=1e-9)
    np.testing.assert_allclose(est[0], ref[0], rtol=1e-5)
    # a weaker field gives a proportionally larger nonlinear bound, and the maximum is re-armed by every field solve
    if nl:
        g.gk_rhs(g.to_state(0.25 * f))
        np.testing.assert_allclose(g.gk_estimate_dt()[1], 4 * est[1], rtol=1e-5)


@pytest.mark.parametrize("case", ["mid", "cfg3_plane", "cfg5_plane"])
def test_a_bare_field_solve_keeps_the_nonlinear_bound(case):
    # The diagnostics loop "step, gk_field_solve (for spectra / fluxes), gk_estimate_dt" must still see the bound of
    # the step's last stage launch: only a field solve that a stage launch follows re-arms the maximum.
    cfg, g = _ctx(case)
    f = (0.05 * rand_c(np.random.default_rng(84), g.shape, True)).astype(np.complex64)
    fd = g.to_state(f)
    g.gk_rk4_steps(fd, 1e-3, 1)
    before = g.gk_estimate_dt()
    assert np.isfinite(before[1])
    phi = g.gk_field_solve(fd)
    g.gk_spectra(phi)
    g.gk_fluxes(fd, phi)
    assert np.array_equal(g.gk_estimate_dt(), before)
    # gk_reset_cfl: back to the linear-only estimate, e.g. before the context is reused for another state
    g.gk_reset_cfl()
    after = g.gk_estimate_dt()
    assert np.isinf(after[1]) and after[0] == min(before[2], before[3])
    g.gk_rhs(fd)
    assert np.isfinite(g.gk_estimate_dt()[1])


def test_cfl_adaptive_steps_follow_the_lagged_estimate():
    # dt_0 = min(dt_max, safety x linear-only bound); dt_k = min(dt_max, safety x min(linear, nonlinear bound of the
    # LAST stage of step k-1)).  The oracle replays the same rule with its own RK4 stages and its own estimate.
    # (The linear bound of PAPER.md:356 covers streaming and trapping only; at this amplitude the first step needs
    # the dt_max cap, as a production run started from noise would.)
    cfg, g = _ctx("mid")
    p = g.plan()
    o = GkRef(cfg, pad=(p["mx"], p["my"]))
    f = rand_c(np.random.default_rng(82), o.shape, True).astype(np.complex64)
    safety, nsteps, dt_max = 0.4, 4, 1e-3
    fd = g.to_state(f)
    dts, t = g.gk_rk4_steps_cfl(fd, nsteps, safety, dt_max=dt_max)
    y = f.astype(np.complex128)
    est = o.estimate_dt(np.zeros(o.phi_shape, complex))
    want = []
    nl_binding = 0
    for k in range(nsteps):
        dt = min(dt_max, safety * (min(est[2], est[3]) if k == 0 else est[0]))
        nl_binding += int(k > 0 and est[1] < min(est[2], est[3]) and safety * est[1] < dt_max)
        want.append(dt)
        k1, _ = o.rhs(y)
        k2, _ = o.rhs(y + 0.5 * dt * k1)
        k3, _ = o.rhs(y + 0.5 * dt * k2)
        k4, phi4 = o.rhs(y + dt * k3)
        y = y + dt / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        est = o.estimate_dt(phi4)
    assert want[0] == dt_max and nl_binding == nsteps - 1     # then the nonlinear bound sets every later step
    np.testing.assert_allclose(dts, want, rtol=2e-5)
    np.testing.assert_allclose(t, sum(want), rtol=2e-5)
    assert rel_l2(g.from_state(fd), y) < 1e-4
    # a fresh context without a cap: the first step is the linear-only estimate
    _, g2 = _ctx("mid")
    dts2, _ = g2.gk_rk4_steps_cfl(g2.to_state(1e-6 * f), 1, safety)
    e = g2.gk_estimate_dt()
    np.testing.assert_allclose(dts2, [safety * min(e[2], e[3])], rtol=1e-12)


@pytest.mark.parametrize("case", ["mid", "mid_kinetic", "cfg2_plane", "cfg3_plane", "cfg3_plane_kinetic", "cfg5_plane",
                                  "cfg3_plane_linear", "cfg5_plane_linear", "tiny_linear"])
def test_fluxes_from_the_stage_epilogue(case):
    import torch
    from paper_2604_06085_b200 import GkError
    cfg, g = _ctx(case)
    o = GkRef(cfg)
    amp = 0.003 if "kinetic" in case else 0.03
    f = (amp * rand_c(np.random.default_rng(83), o.shape, True)).astype(np.complex64)
    dt = 0.0005 if "kinetic" in case else 0.01
    with pytest.raises(GkError):
        g.gk_fluxes_last()                               # nothing recorded yet
    g.gk_set_diagnostics(True)
    fd = g.to_state(f)
    g.gk_rk4_steps(fd, dt, 1)
    got = g.gk_fluxes_last()
    ref = o.fluxes(f, o.field_solve(f))
    scale = np.abs(ref).max(axis=1, keepdims=True)
    np.testing.assert_allclose(got[:, 1:], ref[:, 1:], rtol=2e-4, atol=2e-5 * scale.max())
    if cfg["opts"]["adiabatic_electrons"]:
        assert abs(got[0, 0]) < 1e-4 * abs(got[0, 1])
    else:
        np.testing.assert_allclose(got[:, 0], ref[:, 0], rtol=5e-4, atol=2e-5 * scale.max())
    # the standalone pass agrees (same fp32 inputs, different summation order)
    f0d = g.to_state(f)
    alone = g.gk_fluxes(f0d, g.gk_field_solve(f0d))
    np.testing.assert_allclose(got, alone, rtol=2e-5, atol=1e-6 * np.abs(alone).max())
    # second step: fluxes of the state after the first step; bit-identical on repeat (no atomics)
    g.gk_set_diagnostics(True)
    f1 = fd.clone()
    g.gk_rk4_steps(fd, dt, 1)
    got1 = g.gk_fluxes_last()
    alone1 = g.gk_fluxes(f1, g.gk_field_solve(f1))
    np.testing.assert_allclose(got1, alone1, rtol=2e-5, atol=1e-6 * np.abs(alone1).max())
    fd2 = f1.clone()
    g.gk_rk4_steps(fd2, dt, 1)
    assert np.array_equal(g.gk_fluxes_last(), got1)
    assert torch.equal(fd, fd2)
    # diagnostics do not change the trajectory
    g.gk_set_diagnostics(False)
    fd3 = f1.clone()
    g.gk_rk4_steps(fd3, dt, 1)
    assert torch.equal(fd, fd3)
