// gk_stage_inst.cu -- instantiations of the stage kernels for one storage type (GK_ST_ID = 0 complex64,
// 1 complex fp16, 2 complex bf16).  Product path.
#include "gk_common.cuh"
#include "gk_stage.cuh"
#include "gk_roles.cuh"
#include "gk_epilogue.cuh"
#include "gk_stage_ws2.cuh"
#include "gk_stage_ws4.cuh"
#include "gk_stage_point.cuh"
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

// The (kx, ky) planes of the BASELINE grids get kernels with compile-time sizes (index arithmetic, FFT radices
// and zero-padding tests fold to constants); every other shape runs the generic kernel.
template <class ST> StagePick pick_stage(int mx, int my, int nky, int nkx, bool nl) {
  const size_t slab = (size_t)nkx * nky;
  // in-place kernel: the padded field and grad(chi) both live in shared memory.  Measured on B200, cfg3 (ms per
  // stage): 512 FFT + 384 epilogue threads 1.42, 512 + 256 (2 points in flight) 1.42-1.43, 768 + 256 1.46-1.48,
  // 512 + 512 without the register split 1.84
#define GK_WS2(MX, MY, NKY, NKX, NTF, NTE, RF, RE, NB)                            \
  if (nl && mx == MX && my == MY && nky == NKY && nkx == NKX)                     \
    return {(const void *)gk::gk_stage_ws2_kernel<ST, MX, MY, NKY, NKX, NTF, NTE, RF, RE, NB>, NTF + NTE, GK_KIND_WS2, \
            gk::ws2_smem_bytes<ST, MX, MY, NKY, NKX>(), 1, 1, GK_WS_CHI_RING * 3 * slab, GK_WS_NL_RING * slab}
  GK_WS2(128, 96, 32, 85, 512, 384, 56, 88, 1);
  GK_WS2(128, 48, 16, 85, 512, 384, 56, 88, 1);
#undef GK_WS2
  // 4-CTA cluster: padded grids whose real-space field does not fit the shared memory of one SM
#define GK_WS4(MX, MY, NKY, NKX, NTF, NTE, RF, RE, NB)                            \
  if (nl && mx == MX && my == MY && nky == NKY && nkx == NKX)                     \
    return {(const void *)gk::gk_stage_ws4_kernel<ST, MX, MY, NKY, NKX, 4, NTF, NTE, RF, RE, NB>, NTF + NTE, GK_KIND_WS4, \
            gk::ws4_smem_bytes<ST, MX, MY, NKY, NKX, 4, NTE>(), 4, 1, gk::ws4_chis_elems<NKY, NKX, 4>(), GK_WS_NL_RING * slab}
  // register split measured on B200 (ms per stage): 56/152 11.56, 64/144 11.45, 72/128 11.16, 80/120 11.59, 88/104 12.33
  GK_WS4(192, 192, 64, 127, 384, 256, 72, 128, 1);
#undef GK_WS4
  // term III off: streaming kernel (threads, shares per slab, vector items in flight)
#define GK_LIN(NKY, NKX, NT, NSH, NB)                                             \
  if (!nl && nky == NKY && nkx == NKX)                                            \
    return {(const void *)gk::gk_stage_lin_kernel<ST, NKY, NKX, NT, NSH, NB>, NT, GK_KIND_LIN, \
            gk::lin_smem_bytes<ST, NKY, NKX, NT, NSH>(), 1, NSH, 0, 0}
  GK_LIN(32, 85, 352, 1, 2);
  GK_LIN(16, 85, 352, 1, 1);
  GK_LIN(64, 127, 512, 4, 2);   // both vector items of a thread in flight: 2.27 -> 2.06 ms per stage on cfg5
#undef GK_LIN
  // term III off on planes too small to occupy a CTA: one thread per grid point
  if (!nl && slab < 256)
    return {(const void *)gk::gk_stage_point_kernel<ST>, 256, GK_KIND_POINT, 0, 1, 1, 0, 0, (const void *)gk::gk_chis_kernel<ST>};
  if (!nl) return {(const void *)gk::gk_stage_kernel<ST, 0, 0, 0, 0, false, 512, 1>, 512, GK_KIND_GENERIC, 0, 1, 1, 3 * slab, 0};
  return {(const void *)gk::gk_stage_kernel<ST, 0, 0, 0, 0, true, 512, 1>, 512, GK_KIND_GENERIC, 0, 1, 1, 3 * slab, 0};
}

}  // namespace

StagePick GK_PICK_NAME(int mx, int my, int nky, int nkx, bool nl) { return pick_stage<GK_ST>(mx, my, nky, nkx, nl); }
