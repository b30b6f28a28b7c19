"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times: the
oracle computes sampled (species, vpar, mu, s) slabs one by one; phi is compared in full."""
import numpy as np
import pytest

import gkinputs
from oracle.gkref import GkRef
from tests.util import max_abs_rel, rel_l2

pytestmark = pytest.mark.gpu


def _sample_slabs(shape, n, seed):
    rng = np.random.default_rng(seed)
    nsp, nv, nmu, ns = shape[:4]
    picks = {(0, 0, 0, 0), (nsp - 1, nv - 1, nmu - 1, ns - 1), (0, 1, 0, ns - 2), (nsp - 1, nv - 2, nmu - 1, 1)}
    while len(picks) < n:
        picks.add((int(rng.integers(nsp)), int(rng.integers(nv)), int(rng.integers(nmu)), int(rng.integers(ns))))
    return sorted(picks)


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_rhs_sampled_slabs_full_size(n):
    import torch
    from paper_2604_06085_b200 import GkContext
    cfg = gkinputs.config(n)
    if n == 5:
        cfg["opts"]["storage"] = 0          # the complex64 leg of config 5
    f = gkinputs.initial_f(cfg, np.complex64)
    # scale so the bracket is not negligible next to the linear terms in the whole-RHS norm
    f *= 100.0
    g = GkContext(cfg, full_workspace=False)
    fd = g.to_state(f)
    rhs, phi = g.gk_rhs(fd)
    torch.cuda.synchronize()
    o = GkRef(cfg)
    f128 = f.astype(np.complex128)
    phiref = o.field_solve(f128)
    assert rel_l2(phi.cpu().numpy(), phiref) < 1e-5
    assert max_abs_rel(phi.cpu().numpy(), phiref) < 1e-4
    worst, worst_pt = 0.0, 0.0
    for (a, j, l, i) in _sample_slabs(o.shape, 12, 100 + n):
        ref = o.rhs_slab(f128, phiref, a, j, l, i)
        got = rhs[a, j, l, i].cpu().numpy()
        worst = max(worst, rel_l2(got, ref))
        worst_pt = max(worst_pt, max_abs_rel(got, ref))     # no single point of a slab off by 1e-4 of its largest value
    assert worst < 1e-5, worst
    assert worst_pt < 1e-4, worst_pt


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_configured_run_stays_bounded(n):
    # before timing, run the configured step count and assert ||f|| stays finite and
    # grows < 10x (config 5: complex64 leg).  Configs 3-5 are run for 10 steps here.
    import torch
    from paper_2604_06085_b200 import GkContext
    cfg = gkinputs.config(n)
    cfg["opts"]["storage"] = 0
    g = GkContext(cfg)
    fd = g.to_state(gkinputs.initial_f(cfg, np.complex64))
    n0 = float(torch.linalg.vector_norm(torch.view_as_real(fd)))
    g.gk_rk4_steps(fd, cfg["dt"], cfg["steps"] if n == 2 else 10)
    n1 = float(torch.linalg.vector_norm(torch.view_as_real(fd)))
    assert np.isfinite(n1) and n1 < 10 * n0, (n0, n1)


def test_config2_two_steps_full_grid():
    from paper_2604_06085_b200 import GkContext
    cfg = gkinputs.config(2)
    f = gkinputs.initial_f(cfg, np.complex64)
    g, o = GkContext(cfg), GkRef(cfg)
    fd = g.to_state(f)
    g.gk_rk4_steps(fd, cfg["dt"], 2)
    ref = o.rk4_step(f, cfg["dt"], 2)
    assert rel_l2(g.from_state(fd), ref) < 1e-4
    assert np.isfinite(g.from_state(fd)).all()


def test_config5_half_storage_against_complex64_run():
    # BASELINE config 5: f stored complex fp16 vs the same run with complex64 storage (R19).
    # 3 steps at full size; sampled slabs against the oracle would need the oracle to step the
    # 266M-point grid, so the reference here is the complex64 GPU run (itself oracle-checked above).
    import torch
    from paper_2604_06085_b200 import GkContext
    cfg32 = gkinputs.config(5)
    cfg32["opts"]["storage"] = 0
    cfg16 = gkinputs.config(5)
    cfg16["opts"]["storage"] = 1
    f = 30.0 * gkinputs.initial_f(cfg32, np.complex64)
    g16 = GkContext(cfg16)
    fd16 = g16.to_state(f)
    f_rounded = g16.from_state(fd16)
    g16.gk_rk4_steps(fd16, cfg16["dt"], 3)
    out16 = g16.from_state(fd16)
    del g16, fd16
    torch.cuda.empty_cache()
    g32 = GkContext(cfg32)
    fd32 = g32.to_state(f_rounded)
    g32.gk_rk4_steps(fd32, cfg32["dt"], 3)
    out32 = g32.from_state(fd32)
    assert np.isfinite(out16).all()
    assert rel_l2(out16, out32) < 1e-2


@pytest.mark.parametrize("n,linear", [(2, False), (3, False), (3, True), (5, False)])
def test_repeated_runs_are_bit_identical(n, linear):
    # The stage kernels use no atomics: every output has one writer and a fixed summation order, and the
    # roles of the warp-specialised kernels hand data over through named barriers, an mbarrier and L2
    # rings.  A missing or misplaced hand-off shows up as run-to-run differences; three runs of three
    # RK4 steps (12 stage launches, each streaming every slab through the rings) must agree bit for bit.
    import torch
    from paper_2604_06085_b200 import GkContext
    cfg = gkinputs.config(n)
    cfg["opts"]["storage"] = 0
    if linear:
        cfg["opts"]["nonlinear"] = 0
    g = GkContext(cfg)
    f0 = g.to_state(gkinputs.initial_f(cfg, np.complex64) * 100.0)
    outs = []
    for _ in range(3):
        fd = f0.clone()
        g.gk_rk4_steps(fd, cfg["dt"], 3)
        torch.cuda.synchronize()
        outs.append(fd)
    assert torch.equal(torch.view_as_real(outs[0]), torch.view_as_real(outs[1]))
    assert torch.equal(torch.view_as_real(outs[0]), torch.view_as_real(outs[2]))


# The stage kernels are specialised on (padded grid, nkx, nky) only: a grid with the production (kx,ky)
# plane and few points along s, vpar, mu runs exactly the production kernels (all RK modes, the register
# / gk_moment_kernel moments that feed the next stage's field solve, the seam planes: 4 of 8 here) at a
# size the oracle steps in seconds.
SPECIALISED = {
    "cfg2_plane": (dict(nkx=85, nky=16, ky0=0.07, ikxspace=5), 2),
    "cfg3_plane": (dict(nkx=85, nky=32, ky0=0.035, ikxspace=5), 2),
    "cfg5_plane": (dict(nkx=127, nky=64, ky0=0.0175, ikxspace=5), 5),
}


@pytest.mark.parametrize("case", ["cfg2_plane", "cfg3_plane", "cfg5_plane", "cfg3_plane_kinetic", "cfg3_plane_linear",
                                  "cfg5_plane_f16"])
def test_rk4_steps_parity_on_the_production_kernels(case):
    import torch
    from paper_2604_06085_b200 import GkContext
    from tests.util import small_cfg, rand_c
    base = case.replace("_kinetic", "").replace("_linear", "").replace("_f16", "")
    grid, kind = SPECIALISED[base]
    kw = dict(ns=8, nvpar=8, nmu=2, mu_grid=1, **grid)
    if case.endswith("_kinetic"):
        kw.update(nspecies=2, adiabatic=0, ky0=0.2)     # DESIGN.md R5: stable k_perp,min with kinetic electrons
    cfg = small_cfg(**kw)
    dt, nsteps = (0.0005, 2) if case.endswith("_kinetic") else (0.01, 3)
    if case.endswith("_linear"):
        cfg["opts"]["nonlinear"] = 0
        kind = 3
    if case.endswith("_f16"):
        cfg["opts"]["storage"] = 1
    g = GkContext(cfg)
    assert g.plan()["kind"] == kind, g.plan()
    o = GkRef(cfg)
    # white noise of amplitude 0.03 in every mode: the bracket is a few per cent of the increment and the three
    # steps stay bounded (amplitude 0.1 blows up within three steps, in the oracle as on the device)
    amp = 0.003 if case.endswith("_kinetic") else 0.03
    f = (rand_c(np.random.default_rng(61), o.shape, True) * amp).astype(np.complex64)
    fd = g.to_state(f)
    f0 = g.from_state(fd).astype(np.complex128)         # what the device holds (rounded for half storage)
    g.gk_rk4_steps(fd, dt, nsteps)
    torch.cuda.synchronize()
    got = g.from_state(fd).astype(np.complex128)
    ref = o.rk4_step(f0, dt, nsteps)
    assert np.isfinite(ref).all() and np.abs(ref).max() < 10 * np.abs(f0).max()
    if case.endswith("_f16"):
        assert rel_l2(got, ref) < 1e-2
    else:
        assert rel_l2(got, ref) < 1e-4                   # north_star: 1e-4 after RK4 steps
        # the increment itself (not masked by f0): fp32 rounding of f1 - f0 is ~1e-6 of it
        assert rel_l2(got - f0, ref - f0) < 2e-5, rel_l2(got - f0, ref - f0)
        assert max_abs_rel(got - f0, ref - f0) < 1e-4


# ---- round 2: gaps the round-1 verdict listed for the production kernels ------------------------------------------
def _plane_cfg(base, ns=8, nvpar=8, nmu=2, **kw):
    from tests.util import small_cfg
    grid, kind = SPECIALISED[base]
    args = dict(grid)
    args.update(kw)                      # e.g. ky0 = 0.2 with kinetic electrons (R5)
    return small_cfg(ns=ns, nvpar=nvpar, nmu=nmu, mu_grid=1, **args), kind


@pytest.mark.parametrize("case", ["cfg2_plane", "cfg3_plane", "cfg5_plane", "cfg3_plane_linear", "cfg5_plane_linear"])
def test_rhs_on_the_production_kernels_with_an_asymmetric_ky0_column(case):
    # R15 on the specialised kernels: the ky = 0 column of the input is NOT Hermitian in kx, so the `Re P(0)` branch
    # of the in-place / cluster kernels (Hermitian average inside the bracket) sees an imaginary part it must drop;
    # the linear cases run gk_stage_lin_kernel in mode 0 (gk_rhs), which round 1 never compared with the oracle.
    from paper_2604_06085_b200 import GkContext
    from tests.util import rand_c
    linear = case.endswith("_linear")
    cfg, kind = _plane_cfg(case.replace("_linear", ""))
    if linear:
        cfg["opts"]["nonlinear"] = 0
        kind = 3
    g, o = GkContext(cfg, full_workspace=False), GkRef(cfg)
    assert g.plan()["kind"] == kind, g.plan()
    f = rand_c(np.random.default_rng(71), o.shape, False).astype(np.complex64)      # amplitude O(1): bracket ~ linear terms
    rhs, phi = g.gk_rhs(g.to_state(f))
    ref, phiref = o.rhs(f)
    assert rel_l2(phi.cpu().numpy(), phiref) < 1e-5
    assert rel_l2(rhs.cpu().numpy(), ref) < 1e-5
    assert max_abs_rel(rhs.cpu().numpy(), ref) < 1e-4
    # the bracket alone, relative to its own norm
    if not linear:
        from oracle import gkref as G
        gb, ob = GkContext(cfg, term_mask=G.T_III, full_workspace=False), GkRef(cfg, term_mask=G.T_III)
        rb, _ = gb.gk_rhs(gb.to_state(f))
        refb, _ = ob.rhs(f)
        assert rel_l2(rb.cpu().numpy(), refb) < 1e-5


@pytest.mark.parametrize("case", ["cfg2_plane", "cfg3_plane", "cfg5_plane", "cfg3_plane_linear"])
def test_rk4_parity_with_many_work_items_per_cta(case):
    # Deep enough that every CTA (cluster) of the persistent kernels runs several work items: the chi ring wraps,
    # the bracket ring is reused across items and every RK mode passes through the hand-offs repeatedly.
    import torch
    from paper_2604_06085_b200 import GkContext
    from tests.util import rand_c
    linear = case.endswith("_linear")
    depth = {"cfg2_plane": dict(ns=32, nvpar=8, nmu=16), "cfg3_plane": dict(ns=32, nvpar=16, nmu=8),
             "cfg5_plane": dict(ns=16, nvpar=16, nmu=8), "cfg3_plane_linear": dict(ns=32, nvpar=8, nmu=16)}[
        case if case.endswith("_linear") else case.replace("_linear", "")]
    cfg, kind = _plane_cfg(case.replace("_linear", ""), **depth)
    if linear:
        cfg["opts"]["nonlinear"] = 0
        kind = 3
    g, o = GkContext(cfg), GkRef(cfg)
    p = g.plan()
    assert p["kind"] == kind, p
    nsu = depth["ns"]
    items = nsu * depth["nmu"] * p["nchunk"] * p["nsh"]
    assert items >= 3 * (p["stage_grid"] // p["cluster"]), (items, p)
    f = (rand_c(np.random.default_rng(72), o.shape, True) * 0.03).astype(np.complex64)
    fd = g.to_state(f)
    f0 = f.astype(np.complex128)
    nsteps = 2
    g.gk_rk4_steps(fd, 0.01, nsteps)
    torch.cuda.synchronize()
    got = g.from_state(fd).astype(np.complex128)
    ref = o.rk4_step(f0, 0.01, nsteps)
    assert rel_l2(got, ref) < 1e-4
    assert rel_l2(got - f0, ref - f0) < 2e-5, rel_l2(got - f0, ref - f0)
    assert max_abs_rel(got - f0, ref - f0) < 1e-4


def test_config2_ten_steps_full_grid():
    # north_star: 1e-4 after 10 RK4 steps, on a BASELINE config at full size (the oracle needs about two minutes)
    from paper_2604_06085_b200 import GkContext
    cfg = gkinputs.config(2)
    f = gkinputs.initial_f(cfg, np.complex64)
    g, o = GkContext(cfg), GkRef(cfg)
    fd = g.to_state(f)
    g.gk_rk4_steps(fd, cfg["dt"], 10)
    ref = o.rk4_step(f, cfg["dt"], 10)
    assert rel_l2(g.from_state(fd), ref) < 1e-4


@pytest.mark.parametrize("rlt", [5.0, 9.0])
def test_config3_gradient_scan_on_the_production_kernel(rlt):
    # BASELINE config 3 sweeps R/LT over {5, 7, 9}: 7 is the default of every other test
    import torch
    from paper_2604_06085_b200 import GkContext
    from tests.util import rand_c
    cfg, kind = _plane_cfg("cfg3_plane")
    cfg["species"][0]["rlt"] = rlt
    g, o = GkContext(cfg), GkRef(cfg)
    assert g.plan()["kind"] == kind
    f = (rand_c(np.random.default_rng(73), o.shape, True) * 0.03).astype(np.complex64)
    fd = g.to_state(f)
    g.gk_rk4_steps(fd, 0.01, 3)
    torch.cuda.synchronize()
    f0 = f.astype(np.complex128)
    got, ref = g.from_state(fd).astype(np.complex128), o.rk4_step(f0, 0.01, 3)
    assert rel_l2(got - f0, ref - f0) < 2e-5
    # the drive term really differs between the gradients (the test is not blind to rlt)
    cfg7, _ = _plane_cfg("cfg3_plane")
    assert rel_l2(GkRef(cfg7).rk4_step(f0, 0.01, 1) - f0, o.rk4_step(f0, 0.01, 1) - f0) > 3e-3


@pytest.mark.parametrize("case", ["cfg3_plane_bf16", "cfg5_plane_bf16", "cfg3_plane_linear_f16", "cfg2_plane_linear_f16",
                                  "cfg5_plane_linear_bf16"])
def test_half_storage_on_the_production_kernels(case):
    import torch
    from paper_2604_06085_b200 import GkContext
    from tests.util import rand_c
    base = case.split("_plane")[0] + "_plane"
    cfg, kind = _plane_cfg(base)
    cfg["opts"]["storage"] = 2 if case.endswith("bf16") else 1
    if "_linear" in case:
        cfg["opts"]["nonlinear"] = 0
        kind = 3
    g = GkContext(cfg)
    assert g.plan()["kind"] == kind
    o = GkRef(cfg)
    f = (rand_c(np.random.default_rng(74), o.shape, True) * 0.03).astype(np.complex64)
    fd = g.to_state(f)
    f0 = g.from_state(fd).astype(np.complex128)          # what the device holds after rounding to the storage type
    g.gk_rk4_steps(fd, 0.01, 2)
    torch.cuda.synchronize()
    assert rel_l2(g.from_state(fd).astype(np.complex128), o.rk4_step(f0, 0.01, 2)) < 1e-2


def test_fp16_storage_at_the_configured_amplitude():
    # BASELINE config 5 as stated: seed-Gaussian amplitude 1e-3 (no rescaling), f stored complex fp16.  The Gaussian
    # tails lie below fp16's smallest normal number (6.1e-5) and are kept as subnormals; the relative L2 error is set
    # by the 11-bit significand of the bulk.  Production plane of config 5, reduced depth, against the oracle started
    # from the same complex64 input (the initial rounding counts as error).
    import torch
    from paper_2604_06085_b200 import GkContext
    cfg, kind = _plane_cfg("cfg5_plane", ns=8, nvpar=8, nmu=2)
    cfg["opts"]["storage"] = 1
    cfg["amp"], cfg["seed"] = 1e-3, 1239
    g, o = GkContext(cfg), GkRef(cfg)
    assert g.plan()["kind"] == kind
    f = gkinputs.initial_f(cfg, np.complex64)
    assert (np.abs(f.real) < 6.1e-5).mean() > 0.05          # the subnormal range is really exercised
    fd = g.to_state(f)
    rhs, _ = g.gk_rhs(fd)
    ref, _ = o.rhs(f)
    assert rel_l2(g.from_state(rhs), ref) < 1e-2
    g.gk_rk4_steps(fd, cfg["dt"], 5)
    torch.cuda.synchronize()
    assert rel_l2(g.from_state(fd), o.rk4_step(f, cfg["dt"], 5)) < 1e-2


@pytest.mark.parametrize("storage", [1, 2])
def test_half_storage_multi_step_call_equals_single_steps(storage):
    # the moment of the new state is accumulated from the value as stored, so gk_rk4_steps(n) and n x gk_rk4_step
    # (which recomputes the moment from the stored state) walk the same trajectory bit for bit
    import torch
    from paper_2604_06085_b200 import GkContext
    from tests.util import rand_c
    for base in ("cfg3_plane", "cfg5_plane"):
        cfg, _ = _plane_cfg(base)
        cfg["opts"]["storage"] = storage
        g = GkContext(cfg)
        f = (rand_c(np.random.default_rng(75), gkinputs.f_shape(cfg), True) * 0.03).astype(np.complex64)
        a, b = g.to_state(f), g.to_state(f)
        g.gk_rk4_steps(a, 0.01, 3)
        for _ in range(3):
            g.gk_rk4_step(b, 0.01)
        torch.cuda.synchronize()
        assert rel_l2(g.from_state(a), g.from_state(b)) < 2e-3      # a few ulps of the storage type at most
        if storage == 1:
            assert torch.equal(a, b)


def test_two_contexts_of_different_generic_shapes_interleaved():
    # the dynamic shared-memory attribute belongs to the kernel symbol, not to a context: a small-plan context created
    # after a large-plan one must not break the first
    from paper_2604_06085_b200 import GkContext
    from tests.util import small_cfg, rand_c
    big = small_cfg(nkx=37, nky=13, ns=6, nvpar=7, nmu=2, ikxspace=3, mu_grid=1, ky0=0.05)     # 64 x 48 padded
    small = small_cfg(nkx=9, nky=4, ns=8, nvpar=8, nmu=2)                                        # 16 x 12 padded
    ga = GkContext(big)
    fa = rand_c(np.random.default_rng(76), gkinputs.f_shape(big), True).astype(np.complex64)
    ra0 = ga.gk_rhs(ga.to_state(fa))[0].cpu().numpy()
    gb = GkContext(small)
    fb = rand_c(np.random.default_rng(77), gkinputs.f_shape(small), True).astype(np.complex64)
    rb = gb.gk_rhs(gb.to_state(fb))[0].cpu().numpy()
    ra1 = ga.gk_rhs(ga.to_state(fa))[0].cpu().numpy()
    assert np.array_equal(ra0, ra1)
    assert rel_l2(ra1, GkRef(big).rhs(fa)[0]) < 1e-5 and rel_l2(rb, GkRef(small).rhs(fb)[0]) < 1e-5


@pytest.mark.parametrize("case", ["cfg3_plane", "cfg5_plane", "cfg3_plane_kinetic"])
def test_ten_rk4_steps_on_the_production_planes(case):
    # north_star: <= 1e-4 after 10 RK4 steps, on the kernels BASELINE configs 3, 4 and 5 run (their (kx, ky) planes at
    # reduced depth along s, vpar, mu; config 2 takes the ten steps at full size above)
    import torch
    from paper_2604_06085_b200 import GkContext
    from tests.util import rand_c
    kin = case.endswith("_kinetic")
    kw = dict(nspecies=2, adiabatic=0, ky0=0.2) if kin else {}
    cfg, kind = _plane_cfg(case.replace("_kinetic", ""), **kw)
    g, o = GkContext(cfg), GkRef(cfg)
    assert g.plan()["kind"] == kind
    amp, dt = (0.002, 0.0005) if kin else (0.01, 0.01)
    if kin:     # the step the CFL estimate allows (field bound of the omega_H mode, R23), with a safety factor
        est = o.estimate_dt(np.zeros(o.phi_shape, complex))
        dt = 0.4 * min(est[2], est[3])
    f = (rand_c(np.random.default_rng(78), o.shape, True) * amp).astype(np.complex64)
    fd = g.to_state(f)
    g.gk_rk4_steps(fd, dt, 10)
    torch.cuda.synchronize()
    f0 = f.astype(np.complex128)
    got, ref = g.from_state(fd).astype(np.complex128), o.rk4_step(f0, dt, 10)
    assert np.isfinite(ref).all() and np.abs(ref).max() < 10 * np.abs(f0).max()
    assert rel_l2(got, ref) < 1e-4
    assert rel_l2(got - f0, ref - f0) < 1e-4, rel_l2(got - f0, ref - f0)
