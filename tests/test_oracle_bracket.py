"""Pins for the oracle's term III (ExB bracket): the plain truncated convolution, a library
(numpy.fft) pseudospectral evaluation, a single-pair closed form, exact antisymmetry and the
independence of the padded size."""
import numpy as np
import pytest

from oracle.gkref import GkRef
from tests.util import small_cfg, rand_c, rel_l2


def _numpy_pseudospectral(chi, fs, dkx, ky0, mx, my):
    """1/2 (d_y chi d_x f - d_x chi d_y f) with numpy's irfft2/rfft2 on an (mx,my) padded grid.
    irfft2 discards the imaginary part that a non-Hermitian ky=0 column would produce, which is
    the paper's baseline behaviour."""
    nkx, nky = chi.shape
    K = (nkx - 1) // 2
    p = np.arange(-K, K + 1)
    kx = (p * dkx)[:, None]
    ky = (np.arange(nky) * ky0)[None, :]

    def to_real(g):
        a = np.zeros((mx, my // 2 + 1), complex)
        a[p % mx, :nky] = g
        return np.fft.irfft2(a, s=(mx, my)) * (mx * my)   # sum g e^{+i k x}

    dxc, dyc = to_real(1j * kx * chi), to_real(1j * ky * chi)
    dxf, dyf = to_real(1j * kx * fs), to_real(1j * ky * fs)
    prod = 0.5 * (dyc * dxf - dxc * dyf)
    P = np.fft.rfft2(prod) / (mx * my)
    return P[p % mx, :nky]


@pytest.mark.parametrize("herm", [True, False])
def test_direct_convolution_vs_own_fft_vs_numpy(herm):
    cfg = small_cfg()
    o = GkRef(cfg)
    rng = np.random.default_rng(5)
    chi = rand_c(rng, (9, 4), herm)
    fs = rand_c(rng, (9, 4), herm)
    direct = o.bracket_slab(chi, fs, method=1)
    fft = o.bracket_slab(chi, fs, method=0)
    dkx = np.diff(o.table("kx"))[0]
    lib = _numpy_pseudospectral(chi, fs, dkx, 0.1, 16, 12)
    assert rel_l2(fft, direct) < 1e-13
    assert rel_l2(lib, direct) < 1e-13
    # output ky=0 column is Hermitian in kx (real field)
    np.testing.assert_allclose(direct[:, 0], np.conj(direct[::-1, 0]), atol=1e-14 * abs(direct).max())


def test_padded_size_independence():
    o = GkRef(small_cfg())
    rng = np.random.default_rng(6)
    chi, fs = rand_c(rng, (9, 4)), rand_c(rng, (9, 4))
    ref = o.bracket_slab(chi, fs, method=1)
    for mx, my in [(13, 10), (14, 10), (16, 12), (16, 16), (20, 15), (27, 21)]:
        assert rel_l2(o.bracket_slab(chi, fs, 0, mx, my), ref) < 1e-13, (mx, my)
    # one point below the 3/2-rule minimum aliases (the rule is sharp)
    assert rel_l2(o.bracket_slab(chi, fs, 0, 12, 10), ref) > 1e-6


def test_single_pair_closed_form():
    # chi has the single mode k'=(p1,m1), f the single mode k''=(p2,m2) (plus their implied
    # conjugates).  Then III has exactly two modes in the half plane:
    #   k'+k'' : 1/2 (k'_x k''_y - k'_y k''_x) chi f
    #   k''-k' : 1/2 (-k'_x k''_y + k'_y k''_x) conj(chi) f     (needs m2 - m1 >= 0)
    cfg = small_cfg(nkx=11, nky=5)
    o = GkRef(cfg)
    kx, ky = o.table("kx"), o.table("ky")
    K = 5
    p1, m1, p2, m2 = 2, 1, -1, 2
    c, fv = 0.7 - 0.2j, -0.3 + 1.1j
    chi = np.zeros((11, 5), complex)
    fs = np.zeros((11, 5), complex)
    chi[p1 + K, m1] = c
    fs[p2 + K, m2] = fv
    out = o.bracket_slab(chi, fs, method=1)
    cross = kx[p1 + K] * ky[m2] - ky[m1] * kx[p2 + K]
    exp = np.zeros_like(out)
    exp[p1 + p2 + K, m1 + m2] = 0.5 * cross * c * fv
    exp[p2 - p1 + K, m2 - m1] = -0.5 * cross * np.conj(c) * fv
    np.testing.assert_allclose(out, exp, atol=1e-16)
    np.testing.assert_allclose(o.bracket_slab(chi, fs, method=0), exp, atol=1e-15)
    # the bracket of a field with itself vanishes
    g = rand_c(np.random.default_rng(1), (11, 5))
    assert abs(o.bracket_slab(g, g, method=1)).max() < 1e-13 * abs(g).max() ** 2


@pytest.mark.parametrize("method", [0, 1])
def test_antisymmetry_free_energy(method):
    # sum_k P_m Re[conj(f_k) III_k] = 0 and sum_k P_m Re[conj(chi_k) III_k] = 0 exactly
    # (the truncated Galerkin bracket conserves both quadratic invariants), P_m = 1, 2, 2, ...
    o = GkRef(small_cfg())
    rng = np.random.default_rng(7)
    chi, fs = rand_c(rng, (9, 4)), rand_c(rng, (9, 4))
    out = o.bracket_slab(chi, fs, method=method)
    P = np.array([1.0, 2, 2, 2])[None, :]
    scale = (P * abs(out) * abs(fs)).sum()
    assert abs((P * (np.conj(fs) * out).real).sum()) < 1e-13 * scale
    assert abs((P * (np.conj(chi) * out).real).sum()) < 1e-13 * scale


def test_ky0_column_uses_hermitian_average():
    # each mirror pair (kx,-kx) at ky=0 is replaced by its Hermitian average before
    # the transform.  Feeding the average explicitly must give the identical result.
    o = GkRef(small_cfg())
    rng = np.random.default_rng(8)
    chi, fs = rand_c(rng, (9, 4), False), rand_c(rng, (9, 4), False)

    def sym(g):
        g = g.copy()
        g[:, 0] = 0.5 * (g[:, 0] + np.conj(g[::-1, 0]))
        return g

    a = o.bracket_slab(chi, fs, method=1)
    b = o.bracket_slab(sym(chi), sym(fs), method=1)
    np.testing.assert_allclose(a, b, atol=1e-15 * abs(a).max())
