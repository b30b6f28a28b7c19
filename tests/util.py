"""Helpers shared by the tests (no method arithmetic)."""
import copy

import numpy as np

import gkinputs


def small_cfg(nkx=9, nky=4, ns=8, nvpar=8, nmu=2, nspecies=1, adiabatic=1, mu_grid=0, ky0=0.1,
              ikxspace=1, **kw):
    """A config-1-like dictionary with arbitrary sizes (same geometry, gradients, dissipation)."""
    c = gkinputs.config(1)
    c["grid"].update(nkx=nkx, nky=nky, ns=ns, nvpar=nvpar, nmu=nmu, mu_grid=mu_grid, ky0=ky0,
                     ikxspace=ikxspace)
    if nspecies == 2:
        c["species"] = [copy.deepcopy(gkinputs.CONFIGS[4]["species"][0]),
                        copy.deepcopy(gkinputs.CONFIGS[4]["species"][1])]
    c["opts"]["adiabatic_electrons"] = adiabatic
    for k, v in kw.items():
        if k in c["grid"]:
            c["grid"][k] = v
        elif k in c["opts"]:
            c["opts"][k] = v
        elif k in c["geom"]:
            c["geom"][k] = v
        else:
            c[k] = v
    return c


def rel_l2(a, b):
    a = np.asarray(a)
    b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def max_abs_rel(a, b):
    """max |a - b| / max |b|: a handful of wrong points (a seam row, an open-end class) cannot hide in it the way
    they can in the relative L2 norm of 1e8 points."""
    a = np.asarray(a)
    b = np.asarray(b)
    worst = 0.0
    flat_a, flat_b = a.reshape(-1), b.reshape(-1)
    step = 1 << 24                                   # chunked: no full-size temporaries at 6.7e7 points
    for q in range(0, flat_a.size, step):
        worst = max(worst, float(np.abs(flat_a[q:q + step] - flat_b[q:q + step]).max()))
    return worst / max(float(np.abs(flat_b).max()), 1e-300)


def rand_c(rng, shape, hermitian_ky0=True):
    z = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    if hermitian_ky0:
        nkx = shape[-2]
        K = (nkx - 1) // 2
        z[..., :K, 0] = np.conj(z[..., K + 1:, 0][..., ::-1])
        z[..., K, 0] = z[..., K, 0].real
    return z
