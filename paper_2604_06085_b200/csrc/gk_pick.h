// gk_pick.h -- interface between the host side of libgk (gk_lib.cu) and the translation units that
// instantiate the stage kernels (gk_stage_inst.cu, compiled once per storage type so that the
// instantiations build in parallel).
#pragma once
#include <stddef.h>

enum {
  GK_KIND_GENERIC = 0,  // gk_stage_kernel: any shape, run-time sizes
  GK_KIND_WS2 = 2,      // gk_stage_ws2_kernel: in-place warp-specialised kernel (BASELINE grids 2-4)
  GK_KIND_LIN = 3,      // gk_stage_lin_kernel: term III off, streaming role only
  GK_KIND_WS4 = 5,      // gk_stage_ws4_kernel: 4-CTA cluster (BASELINE grid 5)
  GK_KIND_POINT = 6     // gk_chis_kernel + gk_stage_point_kernel: term III off on tiny (kx,ky) planes, one thread per point
};

// smem > 0: the kernel's own fixed shared-memory plan, 0: planned by gk_create (generic kernel)
// cluster: CTAs per thread-block cluster (1: none); a cluster works on one item at a time
// nsh: shares a (kx,ky) slab is split into, each a work item of its own (streaming kernel)
// chis_per_cta / nl_per_cta: float2 elements of per-CTA L2 scratch (chi, D_s chi; bracket ring)
struct StagePick {
  const void *fn;
  int threads;
  int kind;
  size_t smem;
  int cluster;
  int nsh;
  size_t chis_per_cta, nl_per_cta;
  const void *fn2 = nullptr;   // GK_KIND_POINT: gk_chis_kernel, launched before fn
};

// storage 0: complex64, 1: complex fp16, 2: complex bf16
StagePick gk_pick_stage_c64(int mx, int my, int nky, int nkx, bool nl);
StagePick gk_pick_stage_f16(int mx, int my, int nky, int nkx, bool nl);
StagePick gk_pick_stage_bf16(int mx, int my, int nky, int nkx, bool nl);

inline StagePick gk_pick_stage(int storage, int mx, int my, int nky, int nkx, bool nl) {
#ifdef GK_ONLY_C64
  if (storage != 0) return {nullptr, 0, 0, 0, 1, 1, 0, 0};
#else
  if (storage == 1) return gk_pick_stage_f16(mx, my, nky, nkx, nl);
  if (storage == 2) return gk_pick_stage_bf16(mx, my, nky, nkx, nl);
#endif
  return gk_pick_stage_c64(mx, my, nky, nkx, nl);
}
