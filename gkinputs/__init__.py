"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic: only (i) the five BASELINE.json workload
descriptions as plain parameter dictionaries and (ii) the counter-based random initial
condition of SURVEY.md §8(c) reading R16 (SplitMix64 of (seed, linear index) -> Box-Muller,
re/im ~ N(0, amp^2/2), then the ky=0 column made Hermitian in kx).  It imports neither
`oracle/` nor the CUDA package.

The paper's own workloads (GKW reference trajectories, the 46-equilibria validation set,
PAPER.md:107) are not available; these seeded grids stand in for them ("Inputs").
"""
from __future__ import annotations

import numpy as np

__all__ = ["CONFIGS", "config", "initial_f", "f_shape", "splitmix64_normal"]

_ION = dict(Z=1.0, mass=1.0, temp=1.0, dens=1.0, rlt=7.0, rln=2.0)
# BASELINE.json config 4: electrons, mass ratio 1/1836, Te = Ti
_ELECTRON = dict(Z=-1.0, mass=1.0 / 1836.0, temp=1.0, dens=1.0, rlt=7.0, rln=2.0)
_GEOM = dict(q=1.5, shat=0.8, eps=0.18)
# dissipation defaults of SURVEY R9
_DISS = dict(disp_par=1.0, disp_vp=0.2, disp_x=0.1, disp_y=0.1)


def _cfg(name, nkx, nky, ns, nvpar, nmu, ky0, ikxspace, mu_grid, species, adiabatic, dt, steps, seed,
         storage=0):
    return dict(
        name=name,
        grid=dict(nkx=nkx, nky=nky, ns=ns, nvpar=nvpar, nmu=nmu, ky0=ky0, ikxspace=ikxspace,
                  vpar_max=4.0, mu_grid=mu_grid, vperp_max=3.0),
        species=[dict(s) for s in species],
        geom=dict(_GEOM),
        opts=dict(adiabatic_electrons=adiabatic, te=1.0, ne=1.0, nonlinear=1, s_closure=0,
                  storage=storage, **_DISS),
        dt=dt, steps=steps, seed=seed, amp=1e-3,
    )


# mu_grid: 0 = Gauss-Laguerre (config 1, stated by BASELINE.json), 1 = uniform in v_perp (the
# paper's grid) -- SURVEY R3.  ky0/ikxspace for configs 3-5: SURVEY R5.
CONFIGS = {
    1: _cfg("cfg1_tiny_adiabatic", 9, 4, 8, 8, 2, 0.1, 1, 0, [_ION], 1, 0.01, 10, 1235),
    2: _cfg("cfg2_itg_adiabatic_5.6M", 85, 16, 16, 32, 8, 0.07, 5, 1, [_ION], 1, 0.02, 100, 1236),
    3: _cfg("cfg3_itg_adiabatic_67M", 85, 32, 32, 48, 16, 0.035, 5, 1, [_ION], 1, 0.02, 50, 1237),
    # config 4: ky0 = 0.2 (not SURVEY R5's 0.035): with kinetic electrons the electrostatic
    # omega_H mode of the smallest k_perp has |lambda| dt = 11 at ky0 = 0.035, dt = 0.002 -> explicit
    # RK4 blows up (oracle eigen-solve, tests/test_oracle_physics.py); k_perp,min = 0.2 is stable.
    # Only ky0 was changed (dt and grid counts are BASELINE's); R5.
    4: _cfg("cfg4_kinetic_electrons_134M", 85, 32, 32, 48, 16, 0.2, 5, 1, [_ION, _ELECTRON], 0,
            0.002, 50, 1238),
    5: _cfg("cfg5_large_266M", 127, 64, 32, 64, 16, 0.0175, 5, 1, [_ION], 1, 0.02, 20, 1239),
}


def config(n: int, **overrides) -> dict:
    """Deep copy of BASELINE config `n` (1..5); `overrides` may replace grid/opts entries by key."""
    import copy
    c = copy.deepcopy(CONFIGS[n])
    for k, v in overrides.items():
        if k in c["grid"]:
            c["grid"][k] = v
        elif k in c["opts"]:
            c["opts"][k] = v
        elif k in c["geom"]:
            c["geom"][k] = v
        else:
            c[k] = v
    return c


def f_shape(cfg: dict):
    g = cfg["grid"]
    return (len(cfg["species"]), g["nvpar"], g["nmu"], g["ns"], g["nkx"], g["nky"])


_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """One SplitMix64 output per 64-bit counter (vectorised, wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def splitmix64_normal(seed: int, start: int, count: int):
    """Standard-normal pairs (re, im) for linear indices start..start+count-1 (Box-Muller)."""
    idx = np.arange(start, start + count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        base = (np.uint64(seed) * np.uint64(0xD1342543DE82EF95)) & _M64
        c = (idx * np.uint64(2) + base) & _M64
        u1 = _splitmix64(c)
        u2 = _splitmix64((c + np.uint64(1)) & _M64)
    # 53-bit mantissas; u1 in (0,1], u2 in [0,1)
    a = ((u1 >> np.uint64(11)).astype(np.float64) + 1.0) * (1.0 / 9007199254740992.0)
    b = (u2 >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
    r = np.sqrt(-2.0 * np.log(a))
    return r * np.cos(2.0 * np.pi * b), r * np.sin(2.0 * np.pi * b)


def initial_f(cfg: dict, dtype=np.complex64, chunk: int = 1 << 24) -> np.ndarray:
    """Seed-Gaussian initial distribution (reading R16): shape (nsp,nvpar,nmu,ns,nkx,nky)."""
    shape = f_shape(cfg)
    n = int(np.prod(shape))
    out = np.empty(n, dtype=dtype)
    sig = cfg["amp"] / np.sqrt(2.0)
    for s in range(0, n, chunk):
        c = min(chunk, n - s)
        re, im = splitmix64_normal(cfg["seed"], s, c)
        out[s:s + c] = (sig * re + 1j * sig * im).astype(dtype)
    out = out.reshape(shape)
    # ky = 0 column Hermitian in kx: f(-p,0) = conj f(p,0), Im f(0,0) = 0  (kx index = p + K)
    nkx = shape[4]
    K = (nkx - 1) // 2
    pos = out[..., K + 1:, 0]
    out[..., :K, 0] = np.conj(pos[..., ::-1])
    out[..., K, 0] = out[..., K, 0].real
    return out
