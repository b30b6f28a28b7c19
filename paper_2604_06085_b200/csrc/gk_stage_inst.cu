// gk_stage_inst.cu -- instantiations of gk_stage_kernel for one storage type (GK_ST_ID = 0 complex64,
// 1 complex fp16, 2 complex bf16).  Product path.
#include "gk_common.cuh"
#include "gk_stage.cuh"
#include "gk_stage_ws.cuh"
#include "gk_stage_ws2.cuh"
#include "gk_stage_ws3.cuh"
#include "gk_pick.h"

#ifndef GK_ST_ID
#define GK_ST_ID 0
#endif
#if GK_ST_ID == 0
#define GK_ST float2
#define GK_PICK_NAME gk_pick_stage_c64
#elif GK_ST_ID == 1
#define GK_ST __half2
#define GK_PICK_NAME gk_pick_stage_f16
#else
#define GK_ST __nv_bfloat162
#define GK_PICK_NAME gk_pick_stage_bf16
#endif

namespace {

// Stage-kernel instantiations: the four BASELINE shapes get compile-time sizes (index arithmetic and
// FFT radices fold to constants); everything else runs the generic kernel.  occ = 2 variants keep
// grad(chi) in global scratch so that two 256-thread CTAs share an SM.
template <class ST> StagePick pick_stage(int mx, int my, int nky, int nkx, bool nl, int want_occ, int want_thr) {
#define GK_SPEC(MX, MY, NKY, NKX, NT, OCC)                                                       \
  if (nl && mx == MX && my == MY && nky == NKY && nkx == NKX && want_occ == OCC && want_thr == NT) \
    return {(const void *)gk::gk_stage_kernel<ST, MX, MY, NKY, NKX, true, NT, OCC>, NT, OCC, 0, 0, 0}
  GK_SPEC(16, 12, 4, 9, 512, 1);
  GK_SPEC(128, 48, 16, 85, 1024, 1);
  GK_SPEC(128, 48, 16, 85, 512, 2);
  GK_SPEC(128, 96, 32, 85, 1024, 1);
  GK_SPEC(128, 96, 32, 85, 512, 2);
  GK_SPEC(128, 96, 32, 85, 512, 1);
  GK_SPEC(192, 192, 64, 127, 1024, 1);
  GK_SPEC(192, 192, 64, 127, 512, 1);
#undef GK_SPEC
  // term III switched off: a streaming stencil kernel
#define GK_SPEC_LIN(NKY, NKX)                                                                    \
  if (!nl && nky == NKY && nkx == NKX && want_occ == 1 && want_thr == 1024)                      \
    return {(const void *)gk::gk_stage_kernel<ST, 0, 0, NKY, NKX, false, 1024, 1>, 1024, 1, 0, 0, 0}
  GK_SPEC_LIN(16, 85);
  GK_SPEC_LIN(32, 85);
  GK_SPEC_LIN(64, 127);
#undef GK_SPEC_LIN
  return {nullptr, 0, 0, 0, 0, 0, 0, 0};
}
// preference order of (threads, occ) variants; the first one that exists and fits is used
// warp-specialised variants (FFT-role threads, epilogue-role threads)
template <class ST> StagePick pick_stage_ws(int mx, int my, int nky, int nkx, int ntf) {
#define GK_WS(MX, MY, NKY, NKX, NTF, NTE)                                         \
  if (mx == MX && my == MY && nky == NKY && nkx == NKX && ntf == NTF)             \
    return {(const void *)gk::gk_stage_ws_kernel<ST, MX, MY, NKY, NKX, NTF, NTE>, NTF + NTE, 1, NTF, 0, 1}
  GK_WS(128, 48, 16, 85, 512, 512);
  GK_WS(128, 96, 32, 85, 512, 512);
  GK_WS(128, 96, 32, 85, 768, 256);
  GK_WS(192, 192, 64, 127, 512, 512);
#undef GK_WS
  return {nullptr, 0, 0, 0, 0, 0, 0, 0};
}
// in-place variants (gk_stage_ws2_kernel): the padded field and grad(chi) both live in shared memory.
// `code` = FFT-role threads, +1, +2, ... for the alternative role splits (GK_WS_NTF, tuning).
template <class ST> StagePick pick_stage_ws2(int mx, int my, int nky, int nkx, int code) {
#define GK_WS2(CODE, MX, MY, NKY, NKX, NTF, NTE, RF, RE, NB)                      \
  if (mx == MX && my == MY && nky == NKY && nkx == NKX && code == CODE)           \
    return {(const void *)gk::gk_stage_ws2_kernel<ST, MX, MY, NKY, NKX, NTF, NTE, RF, RE, NB>, NTF + NTE, 1, NTF, \
            gk::ws2_smem_bytes<ST, MX, MY, NKY, NKX>(), 2}
  // measured on B200, cfg3 (ms per stage): 512+384 threads 1.42, 512+256 (2 points in flight) 1.42-1.43,
  // 768+256 1.46-1.48 (48/112 and 40/136 registers), 512+512 without setmaxnreg 1.84; the forward-x pass 2 moved
  // into the epilogue role 1.44-1.53
  GK_WS2(512, 128, 96, 32, 85, 512, 384, 56, 88, 1);
  GK_WS2(513, 128, 96, 32, 85, 512, 256, 56, 128, 2);
  GK_WS2(512, 128, 48, 16, 85, 512, 384, 56, 88, 1);
  GK_WS2(513, 128, 48, 16, 85, 512, 256, 56, 128, 2);
#undef GK_WS2
  return {nullptr, 0, 0, 0, 0, 0, 0, 0};
}
// term III off: lean streaming kernel (gk_stage_lin_kernel); `code` selects (threads, points in flight, CTAs per SM)
template <class ST> StagePick pick_stage_lin(int nky, int nkx, int code) {
#define GK_LIN(CODE, NKY, NKX, NT, NB, OCC)                                       \
  if (nky == NKY && nkx == NKX && code == CODE)                                   \
    return {(const void *)gk::gk_stage_lin_kernel<ST, NKY, NKX, NT, NB, OCC>, NT, OCC, 1, 0, 3}
  GK_LIN(0, 32, 85, 512, 2, 1);
  GK_LIN(1, 32, 85, 768, 1, 1);
  GK_LIN(0, 16, 85, 512, 2, 1);
  GK_LIN(0, 64, 127, 512, 2, 1);
#undef GK_LIN
  return {nullptr, 0, 0, 0, 0, 0, 0, 0};
}
// row-streaming variant (gk_stage_ws3_kernel): padded grids whose real-space field does not fit shared memory
template <class ST> StagePick pick_stage_ws3(int mx, int my, int nky, int nkx, int code) {
#define GK_WS3(CODE, MX, MY, NKY, NKX, RC, NTF, NTE)                              \
  if (mx == MX && my == MY && nky == NKY && nkx == NKX && code == CODE)           \
    return {(const void *)gk::gk_stage_ws3_kernel<ST, MX, MY, NKY, NKX, RC, NTF, NTE>, NTF + NTE, 1, NTF, \
            gk::ws3_smem_bytes<ST, MX, MY, NKY, NKX, RC>(), 4, (size_t)MX * MY, 1}
  GK_WS3(512, 192, 192, 64, 127, 24, 512, 512);
#undef GK_WS3
  return {nullptr, 0, 0, 0, 0, 0, 0, 0};
}
template <class ST> StagePick pick_stage_auto(int mx, int my, int nky, int nkx, bool nl, int force_occ, int force_thr, int ws_ntf) {
  const bool ws_old = ws_ntf < 0;  // negative: the chunked warp-specialised kernel (gk_stage_ws_kernel)
  if (ws_old) ws_ntf = -ws_ntf;
  if (nl && ws_ntf > 0) {
    StagePick p = ws_old ? StagePick{nullptr, 0, 0, 0, 0, 0, 0, 0} : pick_stage_ws2<ST>(mx, my, nky, nkx, ws_ntf);
    if (p.fn) return p;
    if (!ws_old) p = pick_stage_ws3<ST>(mx, my, nky, nkx, ws_ntf);
    if (p.fn) return p;
    p = pick_stage_ws<ST>(mx, my, nky, nkx, ws_ntf);
    if (p.fn) return p;
  }
  if (!nl && !force_occ && !force_thr) {
    StagePick p = pick_stage_lin<ST>(nky, nkx, ws_ntf >= 0 && ws_ntf < 16 ? ws_ntf : 0);
    if (p.fn) return p;
  }
  static const int pref[][2] = {{1024, 1}, {512, 2}, {512, 1}};
  for (auto &pr : pref) {
    if (force_thr && pr[0] != force_thr) continue;
    if (force_occ && pr[1] != force_occ) continue;
    StagePick p = pick_stage<ST>(mx, my, nky, nkx, nl, pr[1], pr[0]);
    if (p.fn) return p;
  }
  if (!nl) return {(const void *)gk::gk_stage_kernel<ST, 0, 0, 0, 0, false, 512, 1>, 512, 1, 0, 0, 0};
  return {(const void *)gk::gk_stage_kernel<ST, 0, 0, 0, 0, true, 512, 1>, 512, 1, 0, 0, 0};
}


}  // namespace

StagePick GK_PICK_NAME(int mx, int my, int nky, int nkx, bool nl, int force_occ, int force_thr, int ws_ntf) {
  return pick_stage_auto<GK_ST>(mx, my, nky, nkx, nl, force_occ, force_thr, ws_ntf);
}
