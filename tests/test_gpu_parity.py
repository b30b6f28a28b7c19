"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Tolerances (BASELINE.json north_star): <= 1e-5 relative L2 per gk_rhs,
<= 1e-4 after 10 gk_rk4_step (fp32 arithmetic, complex64 storage), <= 1e-2 for half storage."""
import numpy as np
import pytest

import gkinputs
from oracle import gkref as G
from oracle.gkref import GkRef
from tests.util import max_abs_rel, small_cfg, rand_c, rel_l2

pytestmark = pytest.mark.gpu

TOL_RHS = 1e-5
TOL_RK10 = 1e-4
TOL_HALF = 1e-2


def _ctx(cfg, **kw):
    from paper_2604_06085_b200 import GkContext
    return GkContext(cfg, **kw)


MID = dict(nkx=21, nky=6, ns=8, nvpar=9, nmu=3, ikxspace=2, mu_grid=1, ky0=0.15)   # ragged sizes
MID2 = dict(nkx=37, nky=13, ns=6, nvpar=7, nmu=2, ikxspace=3, mu_grid=1, ky0=0.05)  # 64x48 padded grid


def test_create_time_tables_match_the_oracles():
    cfg = small_cfg(nspecies=2, adiabatic=0, **MID)
    g, o = _ctx(cfg), GkRef(cfg)
    for name in ("vpar", "mu", "wmu", "kx", "ky", "B", "F", "BG", "J0", "Gamma0", "FM"):
        np.testing.assert_allclose(g.gk_export_table(name), o.table(name).ravel(), rtol=1e-10, atol=1e-13,
                                   err_msg=name)
    cfg1 = gkinputs.config(1)   # Gauss-Laguerre grid
    g, o = _ctx(cfg1), GkRef(cfg1)
    for name in ("mu", "wmu", "J0"):
        np.testing.assert_allclose(g.gk_export_table(name), o.table(name).ravel(), rtol=1e-10, atol=1e-13)
    np.testing.assert_allclose(g.gk_export_table("den"), (o.table("Apol") + 1.0).ravel(), rtol=1e-12)


@pytest.mark.parametrize("case", ["cfg1", "mid_adiabatic", "mid_kinetic", "nky1"])
def test_field_solve_parity(case):
    cfg = {"cfg1": gkinputs.config(1), "mid_adiabatic": small_cfg(**MID),
           "mid_kinetic": small_cfg(nspecies=2, adiabatic=0, **MID),
           "nky1": small_cfg(nkx=5, nky=1, ns=4, nvpar=4, nmu=1)}[case]
    g, o = _ctx(cfg), GkRef(cfg)
    f = rand_c(np.random.default_rng(31), o.shape, True).astype(np.complex64)
    phi = g.gk_field_solve(g.to_state(f)).cpu().numpy()
    ref = o.field_solve(f)
    assert rel_l2(phi, ref) < TOL_RHS
    K = (cfg["grid"]["nkx"] - 1) // 2
    assert np.all(phi[:, K, 0] == 0)


@pytest.mark.parametrize("bit", range(10))
def test_rhs_parity_one_term_at_a_time(bit):
    # every term separately, relative to ITS OWN norm (the bracket is tiny next to the linear terms
    # at amplitude 1e-3 and would hide inside a whole-RHS norm)
    cfg = small_cfg(**MID)
    mask = 1 << bit
    g, o = _ctx(cfg, term_mask=mask), GkRef(cfg, term_mask=mask, bracket_method=1)
    f = rand_c(np.random.default_rng(32), o.shape, False).astype(np.complex64)   # asymmetric ky=0
    rhs, phi = g.gk_rhs(g.to_state(f))
    ref, _ = o.rhs(f)
    assert np.linalg.norm(ref) > 0
    assert rel_l2(rhs.cpu().numpy(), ref) < TOL_RHS, bit
    assert max_abs_rel(rhs.cpu().numpy(), ref) < 1e-4, bit


@pytest.mark.parametrize("case", ["cfg1", "mid", "mid2", "mid_kinetic", "closure1", "tiny"])
def test_rhs_parity_full(case):
    cfg = {"cfg1": gkinputs.config(1), "mid": small_cfg(**MID), "mid2": small_cfg(**MID2),
           "mid_kinetic": small_cfg(nspecies=2, adiabatic=0, **MID),
           "closure1": small_cfg(s_closure=1, **MID),
           "tiny": small_cfg(nkx=3, nky=2, ns=4, nvpar=4, nmu=1)}[case]
    g, o = _ctx(cfg), GkRef(cfg)
    f = gkinputs.initial_f(cfg, np.complex64) if case == "cfg1" else \
        rand_c(np.random.default_rng(33), o.shape, True).astype(np.complex64)
    rhs, phi = g.gk_rhs(g.to_state(f))
    ref, phiref = o.rhs(f)
    assert rel_l2(phi.cpu().numpy(), phiref) < TOL_RHS
    assert rel_l2(rhs.cpu().numpy(), ref) < TOL_RHS
    assert max_abs_rel(rhs.cpu().numpy(), ref) < 1e-4


@pytest.mark.parametrize("case,kind", [("chain", 6), ("mid", 6), ("mid2", 0), ("mid_kinetic", 6)])
def test_linear_runs_on_the_point_and_generic_kernels(case, kind):
    # term III off: planes of fewer than 256 modes take gk_stage_point_kernel (one thread per grid point; the
    # moment of the new state through gk_moment_kernel), larger odd shapes the generic kernel without the bracket
    cfg = {"chain": small_cfg(nkx=3, nky=1, ns=16, nvpar=12, nmu=3, mu_grid=1, nonlinear=0),
           "mid": small_cfg(nonlinear=0, **MID), "mid2": small_cfg(nonlinear=0, **MID2),
           "mid_kinetic": small_cfg(nspecies=2, adiabatic=0, nonlinear=0, **MID)}[case]
    g, o = _ctx(cfg), GkRef(cfg)
    assert g.plan()["kind"] == kind
    f = rand_c(np.random.default_rng(39), o.shape, False).astype(np.complex64)
    rhs, phi = g.gk_rhs(g.to_state(f))
    ref, phiref = o.rhs(f)
    assert rel_l2(phi.cpu().numpy(), phiref) < TOL_RHS
    assert rel_l2(rhs.cpu().numpy(), ref) < TOL_RHS
    assert max_abs_rel(rhs.cpu().numpy(), ref) < 1e-4
    dt = 0.0005 if case == "mid_kinetic" else 0.01
    fd = g.to_state(f)
    g.gk_rk4_steps(fd, dt, 10)
    assert rel_l2(g.from_state(fd), o.rk4_step(f, dt, 10)) < TOL_RK10


def test_bracket_independent_of_padded_size_and_matches_direct_convolution():
    cfg = small_cfg(**MID)     # K=10 -> 31, nky=6 -> 16: minimal supported 32 x 16
    o = GkRef(cfg, term_mask=G.T_III, bracket_method=1)
    f = rand_c(np.random.default_rng(34), o.shape, True).astype(np.complex64)
    ref, _ = o.rhs(f)
    for pad in [(32, 16), (48, 24), (64, 32), (32, 48)]:
        g = _ctx(cfg, term_mask=G.T_III, pad=pad)
        assert g.plan()["mx"] == pad[0] and g.plan()["my"] == pad[1]
        rhs, _ = g.gk_rhs(g.to_state(f))
        assert rel_l2(rhs.cpu().numpy(), ref) < TOL_RHS, pad


def test_bracket_antisymmetry_on_device():
    # sum_k P_m Re[conj(f_k) III_k] = 0 per slab (free-energy conservation of the nonlinearity)
    cfg = small_cfg(**MID)
    g = _ctx(cfg, term_mask=G.T_III)
    f = rand_c(np.random.default_rng(35), GkRef(cfg).shape, True).astype(np.complex64)
    rhs = g.gk_rhs(g.to_state(f))[0].cpu().numpy().astype(np.complex128)
    P = np.where(np.arange(6) == 0, 1.0, 2.0)
    num = (P * (np.conj(f) * rhs).real).sum(axis=(-1, -2))
    den = (P * abs(f) * abs(rhs)).sum(axis=(-1, -2))
    assert (abs(num) / den).max() < 2e-6


@pytest.mark.parametrize("case", ["cfg1", "mid"])
def test_rk4_ten_steps_parity(case):
    cfg = gkinputs.config(1) if case == "cfg1" else small_cfg(**MID)
    g, o = _ctx(cfg), GkRef(cfg)
    f = gkinputs.initial_f(cfg, np.complex64)
    dt = cfg["dt"]
    fd = g.to_state(f)
    for _ in range(10):
        g.gk_rk4_step(fd, dt)
    ref = o.rk4_step(f, dt, 10)
    assert rel_l2(g.from_state(fd), ref) < TOL_RK10
    # the multi-step entry point (moments carried between steps) gives the same trajectory
    fd2 = g.to_state(f)
    g.gk_rk4_steps(fd2, dt, 10)
    assert rel_l2(g.from_state(fd2), g.from_state(fd)) < 1e-6


def test_rk4_large_amplitude_nonlinear_step():
    # amplitude O(1): the bracket is as large as the linear terms
    cfg = small_cfg(**MID)
    g, o = _ctx(cfg), GkRef(cfg)
    f = rand_c(np.random.default_rng(36), o.shape, True).astype(np.complex64)
    fd = g.to_state(f)
    g.gk_rk4_steps(fd, 0.005, 2)
    ref = o.rk4_step(f, 0.005, 2)
    assert rel_l2(g.from_state(fd), ref) < TOL_RK10


@pytest.mark.parametrize("storage", [1, 2])
def test_half_storage_variant(storage):
    # BASELINE config 5 variant (R19): f, stage states and accumulator in complex fp16/bf16,
    # arithmetic fp32.  fp16 is compared after 10 steps, bf16 (8-bit mantissa) after 3.
    cfg = small_cfg(storage=storage, **MID)
    g = _ctx(cfg)
    o = GkRef(small_cfg(**MID))
    f = 30.0 * gkinputs.initial_f(cfg, np.complex64)       # 0.03: inside fp16's normal range
    fd = g.to_state(f)
    fq = g.from_state(fd)                                   # the rounded initial state
    rhs, _ = g.gk_rhs(fd)
    ref, _ = o.rhs(fq)
    assert rel_l2(g.from_state(rhs), ref) < TOL_HALF
    n = 10 if storage == 1 else 3
    g.gk_rk4_steps(fd, cfg["dt"], n)
    assert rel_l2(g.from_state(fd), o.rk4_step(fq, cfg["dt"], n)) < TOL_HALF


def test_rk4_step_host_buffers_equal_the_device_call():
    # gk_rk4_step_host = H2D + gk_rk4_step + D2H on the context stream: bit-identical to the device call
    import torch
    cfg = small_cfg(**MID)
    g = _ctx(cfg)
    f = rand_c(np.random.default_rng(43), gkinputs.f_shape(cfg), True).astype(np.complex64) * 1e-3
    fd = g.to_state(f)
    hin = fd.cpu().pin_memory()
    hout = torch.empty_like(hin).pin_memory()
    scratch = g.empty_state()
    g.gk_rk4_step_host(hin, hout, scratch, cfg["dt"])
    g.gk_rk4_step(fd, cfg["dt"])
    torch.cuda.synchronize()
    assert torch.equal(hout, fd.cpu())


def test_rk4_batch_host_pipeline_equals_single_steps():
    # gk_rk4_batch_host: three independent problems through two device buffers and three streams; each
    # result must be bit-identical to gk_rk4_step on the same input (also with nbatch = 0 and 1)
    import torch
    cfg = small_cfg(**MID)
    g = _ctx(cfg)
    shape = gkinputs.f_shape(cfg)
    ins, want = [], []
    for k in range(3):
        f = rand_c(np.random.default_rng(50 + k), shape, True).astype(np.complex64) * 1e-3
        fd = g.to_state(f)
        ins.append(fd.cpu().pin_memory())
        g.gk_rk4_step(fd, cfg["dt"])
        want.append(fd.cpu())
    outs = [torch.empty_like(t).pin_memory() for t in ins]
    d0, d1 = g.empty_state(), g.empty_state()
    g.gk_rk4_batch_host([], [], d0, d1, cfg["dt"])
    g.gk_rk4_batch_host(ins, outs, d0, d1, cfg["dt"])
    for o, w in zip(outs, want):
        assert torch.equal(o, w)
    g.gk_rk4_batch_host(ins[:1], outs[2:], d0, d1, cfg["dt"])
    assert torch.equal(outs[2], want[0])


def test_spectra_parity():
    # PAPER.md:113, 390; R20.  Both sides sum the same fp32 phi in double: agreement to rounding order.
    cfg = small_cfg(**MID)
    g, o = _ctx(cfg), GkRef(cfg)
    f = rand_c(np.random.default_rng(41), o.shape, True).astype(np.complex64)
    phi = g.gk_field_solve(g.to_state(f))
    kxs, kys = g.gk_spectra(phi)
    rx, ry = o.spectra(phi.cpu().numpy())
    np.testing.assert_allclose(kxs, rx, rtol=1e-12)
    np.testing.assert_allclose(kys, ry, rtol=1e-12)
    assert abs(kxs.sum() - kys.sum()) < 1e-12 * kxs.sum()


def test_fluxes_parity_and_particle_flux_invariant():
    cfg = small_cfg(**MID)
    g, o = _ctx(cfg), GkRef(cfg)
    f = rand_c(np.random.default_rng(37), o.shape, True).astype(np.complex64)
    fd = g.to_state(f)
    phi = g.gk_field_solve(fd)
    fl = g.gk_fluxes(fd, phi)
    ref = o.fluxes(f, o.field_solve(f))
    np.testing.assert_allclose(fl[:, 1:], ref[:, 1:], rtol=2e-4)
    assert abs(fl[0, 0]) < 1e-4 * abs(fl[0, 1])
    cfgk = small_cfg(nspecies=2, adiabatic=0, **MID)
    g, o = _ctx(cfgk), GkRef(cfgk)
    f = rand_c(np.random.default_rng(38), o.shape, True).astype(np.complex64)
    fd = g.to_state(f)
    np.testing.assert_allclose(g.gk_fluxes(fd, g.gk_field_solve(fd)), o.fluxes(f, o.field_solve(f)), rtol=5e-4)


def test_error_behaviour():
    from paper_2604_06085_b200 import GkError
    from paper_2604_06085_b200 import binding as b
    import ctypes as C
    with pytest.raises(GkError) as ei:
        _ctx(small_cfg(nkx=8))
    assert ei.value.code == b.GK_EINVAL
    with pytest.raises(GkError) as ei:
        _ctx(small_cfg(**MID), pad=(16, 16))                # violates the 3/2 rule
    assert ei.value.code == b.GK_EUNSUPPORTED
    g = _ctx(gkinputs.config(1), full_workspace=False)
    fd = g.to_state(gkinputs.initial_f(gkinputs.config(1)))
    with pytest.raises(GkError) as ei:                      # rk4 needs the full workspace
        g.gk_rk4_step(fd, 0.01)
    assert ei.value.code == b.GK_EINVAL
    assert g.lib.gk_rhs(g._h, C.c_void_p(fd.data_ptr()), None, None) == b.GK_EINVAL
    g.gk_rhs(fd)                                            # still usable after an EINVAL
    assert g.gk_launch_count() >= 4
    # gk_rk4_batch_host validates every argument before it enqueues anything: a null pointer in the LAST
    # problem leaves the outputs of the earlier ones untouched
    import torch
    g2 = _ctx(small_cfg(**MID))
    hin = g2.to_state(gkinputs.initial_f(small_cfg(**MID))).cpu().pin_memory()
    hout = torch.full_like(hin, 7.0).pin_memory()
    d0, d1 = g2.empty_state(), g2.empty_state()
    ins = (C.c_void_p * 2)(hin.data_ptr(), hin.data_ptr())
    outs = (C.c_void_p * 2)(hout.data_ptr(), None)
    rc = g2.lib.gk_rk4_batch_host(g2._h, ins, outs, 2, C.c_void_p(d0.data_ptr()), C.c_void_p(d1.data_ptr()), 0.01)
    torch.cuda.synchronize()
    assert rc == b.GK_EINVAL and bool((hout == 7.0).all())


# ---- circular (Lapillonne) geometry, PAPER.md:286-310 (R24): gk_opts.geometry = 1 ---------------------------------
def _circ(cfg):
    cfg["opts"]["geometry"] = 1
    cfg["geom"].update(q=1.4, shat=0.78, eps=0.19)
    return cfg


def test_circular_geometry_tables_match_the_oracles():
    # the product builds its geometry from gradient vectors and logarithmic derivatives, the oracle from closed forms
    cfg = _circ(small_cfg(**MID))
    g, o = _ctx(cfg), GkRef(cfg)
    for name in ("B", "F", "BG", "sth", "cz", "gpz", "gzz", "ef", "R", "kthnorm", "dkx", "kx", "J0", "Gamma0", "FM"):
        np.testing.assert_allclose(g.gk_export_table(name), o.table(name).ravel(), rtol=1e-10, atol=1e-13, err_msg=name)


@pytest.mark.parametrize("case", ["mid", "mid_kinetic", "mid_linear", "cfg3_plane", "cfg5_plane"])
def test_circular_geometry_rhs_steps_fluxes_and_cfl(case):
    import torch
    kw = {"mid": MID, "mid_kinetic": dict(nspecies=2, adiabatic=0, **MID), "mid_linear": dict(nonlinear=0, **MID),
          "cfg3_plane": dict(nkx=85, nky=32, ky0=0.035, ikxspace=5, ns=8, nvpar=8, nmu=2, mu_grid=1),
          "cfg5_plane": dict(nkx=127, nky=64, ky0=0.0175, ikxspace=5, ns=8, nvpar=8, nmu=2, mu_grid=1)}[case]
    cfg = _circ(small_cfg(**kw))
    g = _ctx(cfg)
    p = g.plan()
    nl = bool(cfg["opts"]["nonlinear"])
    o = GkRef(cfg, pad=(p["mx"], p["my"]) if nl else (0, 0))
    f = rand_c(np.random.default_rng(91), o.shape, False).astype(np.complex64)
    rhs, phi = g.gk_rhs(g.to_state(f))
    ref, phiref = o.rhs(f)
    assert rel_l2(phi.cpu().numpy(), phiref) < TOL_RHS
    assert rel_l2(rhs.cpu().numpy(), ref) < TOL_RHS
    assert max_abs_rel(rhs.cpu().numpy(), ref) < 1e-4
    est, eref = g.gk_estimate_dt(), o.estimate_dt(phi.cpu().numpy().astype(np.complex128))
    for k in range(4):
        if np.isinf(eref[k]):
            assert np.isinf(est[k])
        else:
            np.testing.assert_allclose(est[k], eref[k], rtol=1e-5)
    # a few RK4 steps with the flux triple folded into the first stage
    amp, dt = (0.003, 0.0005) if "kinetic" in case else (0.03, 0.01)
    f = (amp * rand_c(np.random.default_rng(92), o.shape, True)).astype(np.complex64)
    g.gk_set_diagnostics(True)
    fd = g.to_state(f)
    g.gk_rk4_steps(fd, dt, 1)
    fl = g.gk_fluxes_last()
    np.testing.assert_allclose(fl[:, 1:], o.fluxes(f, o.field_solve(f))[:, 1:], rtol=3e-4, atol=1e-9)
    g.gk_rk4_steps(fd, dt, 2)
    torch.cuda.synchronize()
    f0 = f.astype(np.complex128)
    got, want = g.from_state(fd).astype(np.complex128), o.rk4_step(f0, dt, 3)
    assert rel_l2(got, want) < TOL_RK10
    assert rel_l2(got - f0, want - f0) < 3e-5
