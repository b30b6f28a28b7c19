"""The seeded input generator (reading R16): deterministic, counter-based, ky=0 Hermitian."""
import numpy as np

import gkinputs


def test_initial_f_is_deterministic_and_chunk_independent():
    cfg = gkinputs.config(1)
    a = gkinputs.initial_f(cfg, np.complex128)
    b = gkinputs.initial_f(cfg, np.complex128, chunk=1000)
    assert a.shape == (1, 8, 2, 8, 9, 4)
    np.testing.assert_array_equal(a, b)
    c = gkinputs.initial_f(gkinputs.config(1, seed=99), np.complex128)
    assert abs(a - c).max() > 0


def test_initial_f_statistics_and_symmetry():
    cfg = gkinputs.config(1, nvpar=32, ns=16)
    f = gkinputs.initial_f(cfg, np.complex128)
    K = 4
    np.testing.assert_array_equal(f[..., :K, 0], np.conj(f[..., K + 1:, 0][..., ::-1]))
    assert np.all(f[..., K, 0].imag == 0)
    body = f[..., 1:]
    # re, im ~ N(0, amp^2/2): |f|^2 has mean amp^2
    np.testing.assert_allclose((abs(body) ** 2).mean(), 1e-6, rtol=0.03)
    assert abs(body.real.mean()) < 3e-5 and abs(body.imag.mean()) < 3e-5
    np.testing.assert_allclose(body.real.std(), 1e-3 / np.sqrt(2), rtol=0.03)


def test_five_baseline_configs_have_the_stated_sizes():
    n = {k: int(np.prod(gkinputs.f_shape(c))) for k, c in gkinputs.CONFIGS.items()}
    assert n == {1: 4608, 2: 5570560, 3: 66846720, 4: 133693440, 5: 266338304}
