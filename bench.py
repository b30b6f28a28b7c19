#!/usr/bin/env python
"""bench.py -- throughput of the gyrokinetic RK stage (field solve -> linear terms -> ExB bracket
-> RK4 stage update) on synthetic seeded grids shaped like the paper's workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl gk|reference]

A "step" is one classical RK4 step = 4 passes of the whole hot path over the 5-D grid.
metric = 5-D grid-point RK-stage updates per second = points * 4 * steps / time.
N > 1 (torchrun): the paper has no grid parallelism -> independent replicas, one per
GPU, no data-path collective ("scaling": "weak").  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import gkinputs  # noqa: E402

METRIC = "5D grid-point RK-stage updates/s"
UNIT = "stage-updates/s"
# algorithmic HBM bytes per grid point per stage launch: classical RK4 with the
# accumulator initialised in stage 1: stages move 24, 40, 40, 24 B/pt (complex64) -> 32 on average
ALG_BYTES_PER_POINT_STAGE = {0: 32.0, 1: 16.0, 2: 16.0}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def _running_src_hash():
    """The csrc/ hash compiled into the loaded library (gk_version "... src:<hash>")."""
    from paper_2604_06085_b200 import load_library
    v = load_library().gk_version().decode()
    return v.rsplit("src:", 1)[1].strip() if "src:" in v else None


def _ncu_record(workload):
    """Per-launch counters of the stage kernel from the committed ncu capture (profiles/stage_traffic.json):
    ({"dram_gb": ..., "l1_wavefronts": ...} or None if this workload was not captured, stale).  A record belongs to
    the csrc/ tree it was captured from (`src_hash`); if the running library was built from another tree the
    counters are NOT quoted: (None, True)."""
    p = os.path.join(ROOT, "profiles", "stage_traffic.json")
    if not os.path.exists(p):
        return None, False
    with open(p) as fh:
        rec = json.load(fh).get(workload)
    if rec is None:
        return None, False
    if rec.get("src_hash") is None or rec.get("src_hash") != _running_src_hash():
        return None, True
    return rec, False


SM_COUNT, FP32_LANES, SM_MAX_MHZ = 148, 128, 1965.0      # B200 (B200_PROFILING.md)


def fp32_flops_per_point(grid, plan, nonlinear):
    """fp32 flop model of one stage per grid point: 5 n log2 n per complex
    length-n transform; a real 2-D transform = x transforms on the nky non-zero columns + half-cost (c2r / r2c) y
    transforms on the mx rows; three real 2-D transforms per slab (d_x f, d_y f inverse, bracket forward) plus the two
    of grad(chi) amortised over vpar, 3 flops per real-space point for the product, about 100 for the linear terms
    and the RK update."""
    lin = 100.0
    if not nonlinear:
        return lin
    mx, my, nkx, nky, nv = plan["mx"], plan["my"], grid["nkx"], grid["nky"], grid["nvpar"]
    t2d = nky * 5.0 * mx * np.log2(mx) + mx * 0.5 * 5.0 * my * np.log2(my)
    return ((3.0 + 2.0 / nv) * t2d + 3.0 * mx * my) / (nkx * nky) + lin


def stage_rooflines(cfg, plan, npts, storage, stage_avg_ms, sm_mhz, nonlinear):
    """The three ceilings of one stage-kernel launch: HBM (algorithmic bytes / measured copy bandwidth), fp32 FMA
    pipes (flop model / 148 SMs x 128 lanes x 2 x clock) and the L1 / shared-memory data pipe (wavefronts counted by
    ncu for this kernel / one 128-byte wavefront per SM per clock)."""
    peak, peak_src = _peaks()
    bpp = ALG_BYTES_PER_POINT_STAGE[storage]
    t = stage_avg_ms * 1e-3
    achieved = bpp * npts / t / 1e9
    key = cfg["name"] + ("" if nonlinear else "+linear") + ("" if storage == 0 else "+half")
    rec, stale = _ncu_record(key)
    rec = rec or {}
    clock = (sm_mhz or SM_MAX_MHZ) * 1e6
    fpp = fp32_flops_per_point(cfg["grid"], plan, nonlinear)
    fp32_peak = SM_COUNT * FP32_LANES * 2 * SM_MAX_MHZ * 1e6 / 1e12
    fp32 = fpp * npts / t / 1e12
    out = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
           "traffic": rec.get("dram_gb"), "traffic_stale": stale, "traffic_kernel": rec.get("kernel"),
           "traffic_unit": "GB of DRAM read+write per stage-kernel launch (ncu --set full, profiles/)",
           "peak_source": peak_src, "avg_launch_ms": stage_avg_ms, "alg_bytes_per_point": bpp,
           "fp32": {"bound": "alu", "achieved": fp32, "peak": fp32_peak, "unit": "TFLOP/s", "frac": fp32 / fp32_peak,
                    "flops_per_point": fpp, "peak_source": "148 SM x 128 lanes x 2 x 1.965 GHz (B200_PROFILING.md)"}}
    wf = rec.get("l1_wavefronts")
    if wf:
        cyc = t * clock
        out["l1_shared_pipe"] = {"bound": "l1", "achieved": wf / cyc / SM_COUNT, "peak": 1.0,
                                 "unit": "128-byte wavefronts per SM per clock", "frac": wf / cyc / SM_COUNT,
                                 "wavefronts_per_launch": wf,
                                 "source": "l1tex__data_pipe_lsu_wavefronts of the committed ncu capture / the live launch time"}
    return out


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region: start() returns once the
    first sample has arrived, mark() brackets the timed region on the host clock, stop() reports the
    samples that fall inside the marks (all samples of the run if the region was shorter than one
    sampling period, said so in `window`)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index, self.marks = [], None, index, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "25"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
            t0 = time.perf_counter()
            while not self.rows and time.perf_counter() - t0 < 5.0:
                time.sleep(0.01)
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))

    def mark(self):
        self.marks.append(time.perf_counter())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.proc.terminate()
        rows, window = [r for _, r in self.rows], "whole run"
        if len(self.marks) >= 2:
            inside = [r for t, r in self.rows if self.marks[0] <= t <= self.marks[-1] + 0.03]
            if inside:
                rows, window = inside, "timed region"
        sm = [float(r[0]) for r in rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            for k, n in enumerate(names):
                if len(r) > 3 + k and r[3 + k].lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "window": window}


class OracleSampler:
    """The oracle as it stands on the host cores, bounded samples of one workload: the context, the seeded input and
    one full field solve are made once; every sample() runs as many whole (species, vpar, mu, s) slabs of gk_rhs as
    fit in its budget, spread over `cores` threads (the oracle's own rhs loop is the same slab loop under OpenMP),
    and extrapolates to one stage."""

    def __init__(self, cfg):
        from oracle import gkref
        self.cores = os.cpu_count() or 1
        gkref.set_threads(self.cores)
        self.o = gkref.GkRef(cfg)
        self.f = gkinputs.initial_f(cfg, np.complex128)
        t0 = time.perf_counter()
        self.phi = self.o.field_solve(self.f)
        self.t_field = time.perf_counter() - t0
        nsp, nv, nmu, ns, nkx, nky = self.o.shape
        self.nslabs = nsp * nv * nmu * ns
        rng = np.random.default_rng(7)
        self.picks = [(int(rng.integers(nsp)), int(rng.integers(nv)), int(rng.integers(nmu)), int(rng.integers(ns)))
                      for _ in range(min(self.nslabs, 1 << 16))]
        self.pos = 0

    def sample(self, budget_s=15.0):
        from concurrent.futures import ThreadPoolExecutor
        o, f, phi, cores = self.o, self.f, self.phi, self.cores
        done, t1 = 0, time.perf_counter()
        batch = cores * 4
        with ThreadPoolExecutor(cores) as ex:
            while done < self.nslabs and time.perf_counter() - t1 < budget_s:
                qs = [self.picks[(self.pos + k) % len(self.picks)] for k in range(batch)]
                list(ex.map(lambda q: o.rhs_slab(f, phi, *q), qs))
                done += batch
                self.pos += batch
        t_slabs = time.perf_counter() - t1
        done = min(done, self.nslabs)
        est_stage = self.t_field + t_slabs * self.nslabs / done
        n = int(np.prod(o.shape))
        return {"value": n / est_stage, "unit": UNIT, "cores": cores, "kind": "oracle",
                "sample": f"full field solve ({self.t_field:.2f}s) + {done} of {self.nslabs} slabs of gk_rhs "
                          f"({t_slabs:.1f}s) on {cores} threads, extrapolated to one stage"}


def _oracle_sample(cfg, budget_s=15.0):
    return OracleSampler(cfg).sample(budget_s)


def replica_config(config_no: int, rank: int, storage=None, linear=False) -> dict:
    """Workload of one rank: the paper has no grid parallelism, so N GPUs run N
    independent replicas of the same configuration that differ only in their seed."""
    cfg = gkinputs.config(config_no)
    if storage is not None:
        cfg["opts"]["storage"] = storage
    if linear:
        cfg["opts"]["nonlinear"] = 0
    cfg["seed"] += rank
    return cfg


def max_over_ranks(value: float, world: int, device=None) -> float:
    """Timing rule of the bench contract: the slowest rank defines the step time."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(npts: int, steps: int, world: int, ms_max: float) -> float:
    """Whole-job stage-updates/s: every rank advanced npts points through 4 stages per step."""
    return world * npts * 4 * steps / (ms_max * 1e-3)


def run_reference(args, cfg, rank):
    if rank != 0:
        return
    per_step = max(2.0, min(20.0, 100.0 / max(args.steps + args.warmup, 1)))
    vals = []
    smp = OracleSampler(cfg)
    for s in range(args.warmup + args.steps):
        r = smp.sample(budget_s=per_step)
        if s >= args.warmup:
            vals.append(r)
    v = float(np.mean([r["value"] for r in vals]))
    n = int(np.prod(gkinputs.f_shape(cfg)))
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * 4 * n / v,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": cfg["name"], "grid": cfg["grid"], "nspecies": len(cfg["species"]), "points": n,
                       "nonlinear": bool(cfg["opts"]["nonlinear"]), "dt": cfg["dt"],
                       "note": "CPU oracle (double precision), a bounded sample of the same workload per step"},
            "cpu_baseline": {**vals[-1], "value": v},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


class LibraryBracket:
    """Term III of one (kx, ky) slab batch the LIBRARY way (torch.fft = cuFFT on a CUDA device), kept as a measured
    comparison (north_star) and checked against the oracle by tests/test_gpu_compare.py.

    This is an UNFUSED pipeline: padded spectra and real-space fields are materialised in HBM between torch ops.  It is
    not the paper's design either: PAPER.md:420-426 fuses (1) scatter + i kx / i ky + J0 + scaling into the inverse
    transform's load callback, (2) the bracket product into the forward transform's load callback and (3) the
    truncation into its store callback; this pipeline has none of the three -- only the paper's data LAYOUT (the
    two-for-one packing of D.3 with the Hermitian average of PAPER.md:440) is reproduced, in the `packed` leg.

      r2c     both gradients of a field as separate half spectra, batched c2r inverse (which "discards the imaginary
              output by construction"), pointwise product, r2c forward, truncation;
      packed  Z = d_x g + i d_y g as ONE full complex spectrum (Hermitian extension; ky = 0 mirror pairs (kx, -kx)
              replaced by their Hermitian average unless hermitian_average=False), one C2C inverse per field, bracket,
              one r2c forward; complex64 (the paper's MP bracket) or complex128 (its DP bracket).
    Inputs: half spectra [..., nkx, nky] (kx index -K..K, ky index 0..nky-1); output: the bracket
    (1/2)(d_y chi d_x f - d_x chi d_y f), truncated to the retained modes, as the oracle's bracket_slab returns it."""

    def __init__(self, nkx, nky, mx, my, dkx, ky0, device):
        self.nkx, self.nky, self.mx, self.my, self.dkx, self.ky0, self.dev = nkx, nky, mx, my, dkx, ky0, device
        self.K = (nkx - 1) // 2

    def _k(self, rdt):
        import torch
        kx = ((torch.arange(self.nkx, device=self.dev) - self.K).to(rdt) * self.dkx).view(self.nkx, 1)
        ky = (torch.arange(self.nky, device=self.dev).to(rdt) * self.ky0).view(1, self.nky)
        return kx, ky

    def _pad_half(self, src):
        """[..., nkx, nky] -> zero-padded half spectrum [..., mx, my//2+1] in FFT order along kx."""
        import torch
        K, mx, nky = self.K, self.mx, self.nky
        pad = torch.zeros(src.shape[:-2] + (mx, self.my // 2 + 1), dtype=src.dtype, device=self.dev)
        pad[..., :K + 1, :nky] = src[..., K:, :]
        pad[..., mx - K:, :nky] = src[..., :K, :]
        return pad

    def _truncate(self, out):
        import torch
        K, mx, nky = self.K, self.mx, self.nky
        return torch.cat((out[..., mx - K:, :nky], out[..., :K + 1, :nky]), dim=-2)

    def grad_real(self, gs):
        """Real-space (d_x g, d_y g) on the padded grid through c2r transforms."""
        import torch
        kx, ky = self._k(torch.float64 if gs.dtype == torch.complex128 else torch.float32)
        return (torch.fft.irfft2(self._pad_half(1j * kx * gs), s=(self.mx, self.my), norm="forward"),
                torch.fft.irfft2(self._pad_half(1j * ky * gs), s=(self.mx, self.my), norm="forward"))

    def r2c(self, fb, chib=None, gchi=None):
        """gchi: real-space grad(chi) to reuse over vpar (as the paper and the fused kernel do), else built from chib."""
        import torch
        if gchi is None:
            gchi = self.grad_real(chib)
        fx, fy = self.grad_real(fb)
        br = 0.5 * (gchi[1] * fx - gchi[0] * fy)
        return self._truncate(torch.fft.rfft2(br, norm="forward"))

    def packed_spectrum(self, gs, cdt, hermitian_average=True):
        """Half spectrum -> full padded 2-D spectrum [..., mx, my] of d_x g + i d_y g."""
        import torch
        K, mx, my, nkx, nky = self.K, self.mx, self.my, self.nkx, self.nky
        M = nky - 1
        gs = gs.to(cdt)
        kxv, kyv = self._k(torch.float64 if cdt == torch.complex128 else torch.float32)
        g0 = gs.clone()
        if hermitian_average:     # both members of a ky = 0 mirror pair become their Hermitian average
            g0[..., 0] = 0.5 * (gs[..., 0] + torch.conj(torch.flip(gs[..., 0], dims=(-1,))))
        zp = (1j * kxv - kyv) * g0                                   # ky >= 0: (i kx) g + i (i ky) g
        zm = torch.conj(torch.flip(g0, dims=(-2,)))                  # value at (kx, -ky) = conj g(-kx, ky)
        zmm = (1j * kxv + kyv) * zm                                  # (i kx) g(kx,-ky) + i (i (-ky)) g(kx,-ky)
        full = torch.zeros(gs.shape[:-2] + (mx, my), dtype=cdt, device=self.dev)
        for lo, hi, dst in ((K, nkx, slice(0, K + 1)), (0, K, slice(mx - K, mx))):
            full[..., dst, :nky] = zp[..., lo:hi, :]
            if M > 0:
                full[..., dst, my - M:] = torch.flip(zmm[..., lo:hi, 1:], dims=(-1,))
        return full

    def packed(self, fb, chib, cdt, hermitian_average=True, zc=None):
        """zc: the C2C inverse of chi's packed spectrum to reuse over vpar, else built from chib."""
        import torch
        if zc is None:
            zc = torch.fft.ifft2(self.packed_spectrum(chib, cdt, hermitian_average), norm="forward")
        zf = torch.fft.ifft2(self.packed_spectrum(fb, cdt, hermitian_average), norm="forward")   # Re = d_x f, Im = d_y f
        br = 0.5 * (zc.imag * zf.real - zc.real * zf.imag)
        return self._truncate(torch.fft.rfft2(br, norm="backward") / (self.mx * self.my))


def _time_cuda(fn, reps):
    import torch
    for _ in range(3):          # cuFFT plan creation and the caching allocator's first blocks stay outside
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def library_compare_block(g, cfg, batches=10):
    """Bounded measurement for the bench line: `batches` batches of 4 (mu, s) pairs x nv slabs of the workload's plane
    through the three library legs, extrapolated to the slabs of one stage (said so in the block).  grad(chi) / the
    packed chi field are built once per batch and reused over vpar, as the fused kernel does."""
    import torch
    dev = g.device
    nsp, nv, nmu, ns, nkx, nky = g.shape
    plan = g.plan()
    kxt = g.gk_export_table("kx")
    K = (nkx - 1) // 2
    lb = LibraryBracket(nkx, nky, plan["mx"], plan["my"], float(kxt[K + 1] - kxt[K]), cfg["grid"]["ky0"], dev)
    nli = 4
    nbatch = (nsp * nmu * ns + nli - 1) // nli
    gen = torch.Generator(device=dev).manual_seed(1)
    f = torch.view_as_complex(torch.randn(nli, nv, nkx, nky, 2, device=dev, generator=gen)) * 1e-3
    chi = torch.view_as_complex(torch.randn(nli, 1, nkx, nky, 2, device=dev, generator=gen)) * 1e-2
    scale = nbatch
    out = {"what": "term III only (no linear terms, RK update or field solve) through torch.fft (cuFFT) as an UNFUSED "
                   "library pipeline with padded arrays in HBM; not the paper's LTO-callback design (PAPER.md:420-426: "
                   "none of its three callback fusions), only its packed-C2C layout with the Hermitian average "
                   "(PAPER.md:428-442); parity of every leg against the oracle: tests/test_gpu_compare.py",
           "padded_fft": [plan["mx"], plan["my"]], "slabs_per_stage": nsp * nv * nmu * ns,
           "sample": f"{batches} timed batches of {nli * nv} slabs, extrapolated x{nbatch} to one stage"}
    out["cufft_r2c_bracket_ms_per_stage"] = scale * _time_cuda(lambda: lb.r2c(f, chib=chi), batches)
    out["cufft_packed_c2c_fp32_bracket_ms_per_stage"] = scale * _time_cuda(lambda: lb.packed(f, chi, torch.complex64), batches)
    out["cufft_packed_c2c_fp64_bracket_ms_per_stage"] = scale * _time_cuda(lambda: lb.packed(f, chi, torch.complex128), batches)
    del f, chi
    torch.cuda.empty_cache()
    return out


def run_cufft_compare(args, cfg):
    """`--compare cufft`: the library legs timed over ALL slabs of a stage (no extrapolation) beside the fused stage."""
    import torch
    from paper_2604_06085_b200 import GkContext
    dev = torch.device("cuda", 0)
    g = GkContext(cfg, device=dev)
    nsp, nv, nmu, ns, nkx, nky = g.shape
    nbatch = (nsp * nmu * ns + 3) // 4
    blk = library_compare_block(g, cfg, batches=max(1, args.steps) * nbatch)
    blk["sample"] = f"every slab of {max(1, args.steps)} stage(s), no extrapolation"
    fd = g.to_state(gkinputs.initial_f(cfg, np.complex64))
    g.gk_rk4_steps(fd, cfg["dt"], 3)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    g.gk_rk4_steps(fd, cfg["dt"], max(1, args.steps))
    e1.record()
    torch.cuda.synchronize()
    blk["fused_whole_stage_ms"] = e0.elapsed_time(e1) / (4 * max(1, args.steps))
    print(json.dumps({"compare": "cufft_bracket", "workload": cfg["name"], **blk}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config number 1..5 (default: the largest, config 5 with complex64 storage)")
    ap.add_argument("--impl", default="gk", choices=["gk", "reference"])
    ap.add_argument("--storage", type=int, default=None, help="override storage (0 c64, 1 fp16, 2 bf16)")
    ap.add_argument("--linear", action="store_true", help="switch term III off (HBM-bound variant)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--no-secondary", action="store_true", help="skip the config-3 stage timing that follows a config-5 run")
    ap.add_argument("--no-compare", action="store_true", help="skip the bounded cuFFT comparison block of the bench line")
    ap.add_argument("--compare", default=None, choices=["cufft"], help="measured comparison: term III through cuFFT, unfused")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "gk" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, replica_config(args.config, 0, args.storage, args.linear), rank)
        return
    cfg = replica_config(args.config, rank, args.storage, args.linear)
    if args.compare == "cufft":
        if rank == 0:
            run_cufft_compare(args, cfg)
        return

    import torch
    import torch.distributed as dist
    from paper_2604_06085_b200 import GkContext

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    g = GkContext(cfg, device=dev)
    f_host = gkinputs.initial_f(cfg, np.complex64)
    fd = g.to_state(f_host)
    del f_host
    npts = int(np.prod(g.shape))
    dt = cfg["dt"]
    storage = g.storage
    nl = bool(cfg["opts"]["nonlinear"])

    def timed_steps(ctx, state, steps):
        """EXACTLY `steps` RK4 steps in one timed region (CUDA events on the context stream = torch's current
        stream); an event after every step gives the per-step times (median of >= 5 repetitions)."""
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        ctx.gk_set_profiling(True)
        ctx.gk_stage_kernel_time(reset=True)
        l0 = ctx.gk_launch_count()
        ev[0].record()
        for k in range(steps):
            ctx.gk_rk4_steps(state, dt, 1)
            ev[k + 1].record()
        barrier()
        total = ev[0].elapsed_time(ev[-1])
        per = [ev[k].elapsed_time(ev[k + 1]) for k in range(steps)]
        n_launch = ctx.gk_launch_count() - l0
        stage_ms, stage_n = ctx.gk_stage_kernel_time(reset=True)
        ctx.gk_set_profiling(False)
        return total, per, n_launch, stage_ms, stage_n

    # ---- device-resident throughput ----
    g.gk_rk4_steps(fd, dt, args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    sampler.mark()
    ms, per_step, launches, stage_ms, stage_n = timed_steps(g, fd, args.steps)
    sampler.mark()
    clocks = sampler.stop()
    finite = bool(torch.isfinite(torch.view_as_real(fd) if storage == 0 else fd.float()).all().item())
    ms_max = max_over_ranks(ms, world, dev)
    value = aggregate_value(npts, args.steps, world, ms_max)

    # ---- end to end: host buffers, H2D of f and D2H of f_{n+1} inside the timed region ----
    e2e_steps = max(1, min(args.steps, 5))
    if args.no_e2e:
        e2e_steps = 0
    hbuf = torch.empty(fd.shape if e2e_steps else (1,), dtype=fd.dtype).pin_memory()
    if e2e_steps:
        hbuf.copy_(fd.cpu())
    # a time advance: one C-ABI call per step on HOST buffers, each step uploads its input and downloads its result
    # (H2D + 4 stages + D2H back to back on one stream; step k+1 depends on step k, nothing overlaps)
    for _ in range(2 if e2e_steps else 0):
        g.gk_rk4_step_host(hbuf, hbuf, fd, dt)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(e2e_steps):
        g.gk_rk4_step_host(hbuf, hbuf, fd, dt)
    e1.record()
    barrier()
    serial_ms = max_over_ranks(e0.elapsed_time(e1), world, dev) if e2e_steps else None
    # a batch of INDEPENDENT problems (an ensemble, not a time advance) as one C-ABI call: the upload of problem k+1
    # and the download of problem k-1 overlap the compute of problem k over two device buffers
    if e2e_steps:
        hout = torch.empty_like(hbuf).pin_memory()
        fd2 = g.empty_state()
        g.gk_rk4_batch_host([hbuf] * 2, [hout] * 2, fd, fd2, dt)
    barrier()
    e0.record()
    if e2e_steps:
        g.gk_rk4_batch_host([hbuf] * e2e_steps, [hout] * e2e_steps, fd, fd2, dt)
    e1.record()
    barrier()
    batch_ms = max_over_ranks(e0.elapsed_time(e1), world, dev)
    fbytes = fd.numel() * fd.element_size()
    plan = g.plan()
    kernel_names = {0: "gk_stage_kernel", 2: "gk_stage_ws2_kernel", 3: "gk_stage_lin_kernel", 5: "gk_stage_ws4_kernel", 6: "gk_stage_point_kernel"}

    # ---- the library formulation of term III beside the fused stage, after the timed regions ----
    compare = None
    if rank == 0 and world == 1 and nl and not args.no_compare:
        compare = library_compare_block(g, cfg)

    # ---- secondary workload (rank 0, N = 1): the stage kernel of BASELINE config 3 (the round-1 headline) ----
    secondary = None
    if rank == 0 and world == 1 and args.config == 5 and not args.no_secondary:
        del g, fd, hbuf
        if e2e_steps:
            del hout, fd2
        torch.cuda.empty_cache()
        cfg3 = replica_config(3, rank, None, args.linear)
        g3 = GkContext(cfg3, device=dev)
        f3 = g3.to_state(gkinputs.initial_f(cfg3, np.complex64))
        g3.gk_rk4_steps(f3, cfg3["dt"], args.warmup)
        barrier()
        ms3, per3, _, st3, sn3 = timed_steps(g3, f3, max(5, min(args.steps, 10)))
        n3 = int(np.prod(g3.shape))
        p3 = g3.plan()
        secondary = {"workload": cfg3["name"], "points": n3, "value": n3 * 4 * len(per3) / (ms3 * 1e-3), "unit": UNIT,
                     "ms_per_step_median": float(np.median(per3)), "kernel": kernel_names[p3["kind"]],
                     "roofline": stage_rooflines(cfg3, p3, n3, g3.storage, st3 / max(sn3, 1), clocks.get("sm_mhz"),
                                                 bool(cfg3["opts"]["nonlinear"]))}
        del g3, f3
        torch.cuda.empty_cache()

    if rank == 0:
        stage_avg_ms = stage_ms / max(stage_n, 1)
        roof = stage_rooflines(cfg, plan, npts, storage, stage_avg_ms, clocks.get("sm_mhz"), nl)
        roof.update({"kernel": kernel_names[plan["kind"]], "launches_timed": int(stage_n),
                     "stage_share_of_step": stage_ms / ms if ms > 0 else None})
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": {0: "f32", 1: "f32 (fp16 storage)", 2: "f32 (bf16 storage)"}[storage],
            "data": "synthetic",
            "config": {"workload": cfg["name"], "grid": cfg["grid"], "nspecies": len(cfg["species"]), "points": npts,
                       "nonlinear": nl, "dt": dt, "padded_fft": [plan["mx"], plan["my"]],
                       "launch": {"grid": plan["stage_grid"], "threads": plan["threads"], "cluster": plan["cluster"],
                                  "smem": plan["stage_smem"], "vpar_chunks": plan["nchunk"]},
                       "l2": "inputs larger than L2 (state + 3 work arrays)" if npts * 8 * 4 > 126e6 * 2
                       else "working set comparable to L2; not flushed",
                       "parallelism": "replicas only (paper has no grid parallelism)", "finite": finite,
                       # readings no number of the authors can pin (oracle/gkref.h header)
                       "unpinned_readings": ["R7", "R9", "R18"]},
            "step_ms": {"median": float(np.median(per_step)), "min": float(np.min(per_step)),
                        "max": float(np.max(per_step)), "repetitions": len(per_step)},
            "clocks": clocks,
            "e2e": {"value": aggregate_value(npts, e2e_steps, world, serial_ms) if e2e_steps else None, "unit": UNIT,
                    "h2d_bytes_per_step": fbytes, "d2h_bytes_per_step": fbytes, "steps": e2e_steps,
                    "call": "gk_rk4_step_host (pinned host buffers; a time advance: every step uploads f_n, runs 4 stages, "
                            "downloads f_n+1, nothing overlaps)",
                    "batch_value": aggregate_value(npts, e2e_steps, world, batch_ms) if e2e_steps else None,
                    "batch_call": "gk_rk4_batch_host (independent problems, copies pipelined with compute)"},
            "gpu_launches": int(launches),
            "roofline": roof,
        }
        if secondary:
            line["secondary"] = secondary
        if compare:
            compare["fused_whole_stage_ms"] = roof["avg_launch_ms"]
            line["compare"] = compare
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = _oracle_sample(cfg, budget_s=12.0)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
