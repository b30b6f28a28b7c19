// gk_pick.h -- interface between the host side of libgk (gk_lib.cu) and the translation units that
// instantiate gk_stage_kernel (gk_stage_inst.cu, compiled once per storage type so that the
// instantiations build in parallel).
#pragma once

// ws: FFT-role threads of the warp-specialised kernels (0: unified kernel); smem > 0: the kernel's own
// fixed shared-memory plan (gk_stage_ws2_kernel), 0: planned by gk_create
// kind: 0 gk_stage_kernel, 1 gk_stage_ws_kernel, 2 gk_stage_ws2_kernel, 3 gk_stage_lin_kernel
// 4 gk_stage_ws3_kernel.  gchi: elements of per-CTA grad(chi) scratch the kernel needs regardless of the
// shared-memory plan; host_moment: the kernel does not write the moment planes (gk_moment_kernel follows it)
struct StagePick { const void *fn; int threads; int occ; int ws; size_t smem; int kind; size_t gchi; int host_moment; };

// storage 0: complex64, 1: complex fp16, 2: complex bf16
StagePick gk_pick_stage_c64(int mx, int my, int nky, int nkx, bool nl, int force_occ, int force_thr, int ws_ntf);
StagePick gk_pick_stage_f16(int mx, int my, int nky, int nkx, bool nl, int force_occ, int force_thr, int ws_ntf);
StagePick gk_pick_stage_bf16(int mx, int my, int nky, int nkx, bool nl, int force_occ, int force_thr, int ws_ntf);

inline StagePick gk_pick_stage(int storage, int mx, int my, int nky, int nkx, bool nl, int force_occ, int force_thr, int ws_ntf) {
#ifdef GK_ONLY_C64
  if (storage != 0) return {nullptr, 0, 0, 0, 0, 0, 0, 0};
#else
  if (storage == 1) return gk_pick_stage_f16(mx, my, nky, nkx, nl, force_occ, force_thr, ws_ntf);
  if (storage == 2) return gk_pick_stage_bf16(mx, my, nky, nkx, nl, force_occ, force_thr, ws_ntf);
#endif
  return gk_pick_stage_c64(mx, my, nky, nkx, nl, force_occ, force_thr, ws_ntf);
}
