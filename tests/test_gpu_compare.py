"""the library formulations of term III kept as MEASURED COMPARISONS (bench.py `compare` block,
`--compare cufft`) are correct implementations of the same operation: the r2c pipeline and the paper's packed-C2C
layout in complex64 and complex128, through torch.fft = cuFFT, against the oracle's bracket on the
(kx, ky) planes of configs 3 and 5 with asymmetric ky = 0 columns.  PAPER.md:438-440: the c2r inverse "discards the
imaginary output by construction" (no explicit average needed), the packed C2C path needs the Hermitian average of
the ky = 0 mirror pairs -- without it the error is O(1e-4) or worse, with it O(1e-6) in FP32 and O(1e-14) in FP64."""
import numpy as np
import pytest

from oracle.gkref import GkRef
from tests.util import rel_l2, small_cfg

PLANES = {
    "cfg3_plane": dict(nkx=85, nky=32, ky0=0.035, ikxspace=5, pad=(128, 96)),
    "cfg5_plane": dict(nkx=127, nky=64, ky0=0.0175, ikxspace=5, pad=(192, 192)),
    "small_ragged": dict(nkx=21, nky=6, ky0=0.15, ikxspace=2, pad=(32, 16)),
}


def _legs_against_the_oracle(case, device):
    import torch
    import bench
    g = dict(PLANES[case])
    mx, my = g.pop("pad")
    cfg = small_cfg(ns=8, nvpar=8, nmu=2, mu_grid=1, **g)
    o = GkRef(cfg, pad=(mx, my))
    kx = o.table("kx")
    K = (g["nkx"] - 1) // 2
    lb = bench.LibraryBracket(g["nkx"], g["nky"], mx, my, float(kx[K + 1] - kx[K]), g["ky0"], device)
    rng = np.random.default_rng(5)
    shape = (3, g["nkx"], g["nky"])
    fs = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)        # ky = 0 column NOT Hermitian in kx
    cs = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    ref = np.stack([o.bracket_slab(cs[q], fs[q], 0, mx, my) for q in range(3)])
    ft, ct = torch.from_numpy(fs).to(device), torch.from_numpy(cs).to(device)
    err = {
        "r2c_c64": rel_l2(lb.r2c(ft.to(torch.complex64), chib=ct.to(torch.complex64)).cpu().numpy(), ref),
        "r2c_c128": rel_l2(lb.r2c(ft, chib=ct).cpu().numpy(), ref),
        "packed_c64": rel_l2(lb.packed(ft, ct, torch.complex64).cpu().numpy(), ref),
        "packed_c128": rel_l2(lb.packed(ft, ct, torch.complex128).cpu().numpy(), ref),
        "packed_c128_no_average": rel_l2(lb.packed(ft, ct, torch.complex128, hermitian_average=False).cpu().numpy(), ref),
    }
    assert err["r2c_c64"] < 1e-5 and err["packed_c64"] < 1e-5, err
    assert err["r2c_c128"] < 1e-12 and err["packed_c128"] < 1e-12, err
    assert err["packed_c128_no_average"] > 1e-4, err            # the leakage PAPER.md:440 describes
    return err


def test_library_bracket_math_on_the_host():
    # the same torch.fft pipeline on the CPU (pocketfft instead of cuFFT): pins the comparison code's arithmetic
    # where no GPU is present
    _legs_against_the_oracle("small_ragged", "cpu")


@pytest.mark.gpu
@pytest.mark.parametrize("case", ["cfg3_plane", "cfg5_plane"])
def test_cufft_legs_match_the_oracle(case):
    import torch
    print(case, _legs_against_the_oracle(case, torch.device("cuda", 0)))


@pytest.mark.gpu
def test_bench_compare_block_is_bounded_and_complete():
    import bench
    from paper_2604_06085_b200 import GkContext
    cfg = small_cfg(ns=8, nvpar=8, nmu=2, mu_grid=1, nkx=85, nky=32, ky0=0.035, ikxspace=5)
    g = GkContext(cfg, full_workspace=False)
    blk = bench.library_compare_block(g, cfg, batches=2)
    for k in ("cufft_r2c_bracket_ms_per_stage", "cufft_packed_c2c_fp32_bracket_ms_per_stage",
              "cufft_packed_c2c_fp64_bracket_ms_per_stage"):
        assert blk[k] > 0
    assert blk["padded_fft"] == [128, 96] and "UNFUSED" in blk["what"]
