// gk_common.cuh -- what every CUDA translation unit of libgk shares: the device parameter block, the
// FFT building blocks, the term-mask bits and the storage-type accessors.  Product path.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "gk_dev.h"
#include "gk_fft.cuh"

#define GK_T_I 1
#define GK_T_II 2
#define GK_T_IV 4
#define GK_T_V 8
#define GK_T_VII 16
#define GK_T_VIII 32
#define GK_T_DISS_S 64
#define GK_T_DISS_V 128
#define GK_T_HYP 256
#define GK_T_III 512

namespace gk {

using gkfft::cadd;
using gkfft::cmul;
using gkfft::csub;

// ---- storage types: complex64 / complex fp16 / complex bf16, arithmetic always fp32 (R19) ----
// ld/st: plain; ldg: read-only path (data not written by this launch); ldcs/stcs: streaming
// (evict-first) for arrays that are touched once per stage (f_n, the RK accumulator, the new
// state), so that L2 keeps the stencil halos of the state being differentiated.
template <class ST> struct Cv;
template <> struct Cv<float2> {
  static __device__ __forceinline__ float2 ld(const void *p, long long i) { return ((const float2 *)p)[i]; }
  static __device__ __forceinline__ float2 ldg(const void *p, long long i) { return __ldg((const float2 *)p + i); }
  static __device__ __forceinline__ float2 ldcs(const void *p, long long i) { return __ldcs((const float2 *)p + i); }
  static __device__ __forceinline__ void st(void *p, long long i, float2 v) { ((float2 *)p)[i] = v; }
  static __device__ __forceinline__ void stcs(void *p, long long i, float2 v) { __stcs((float2 *)p + i, v); }
};
template <> struct Cv<__half2> {
  static __device__ __forceinline__ float2 ld(const void *p, long long i) { return __half22float2(((const __half2 *)p)[i]); }
  static __device__ __forceinline__ float2 ldg(const void *p, long long i) { return __half22float2(__ldg((const __half2 *)p + i)); }
  static __device__ __forceinline__ float2 ldcs(const void *p, long long i) { return __half22float2(__ldcs((const __half2 *)p + i)); }
  static __device__ __forceinline__ void st(void *p, long long i, float2 v) { ((__half2 *)p)[i] = __float22half2_rn(v); }
  static __device__ __forceinline__ void stcs(void *p, long long i, float2 v) { __stcs((__half2 *)p + i, __float22half2_rn(v)); }
};
template <> struct Cv<__nv_bfloat162> {
  static __device__ __forceinline__ float2 ld(const void *p, long long i) { return __bfloat1622float2(((const __nv_bfloat162 *)p)[i]); }
  static __device__ __forceinline__ float2 ldg(const void *p, long long i) { return __bfloat1622float2(__ldg((const __nv_bfloat162 *)p + i)); }
  static __device__ __forceinline__ float2 ldcs(const void *p, long long i) { return __bfloat1622float2(__ldcs((const __nv_bfloat162 *)p + i)); }
  static __device__ __forceinline__ void st(void *p, long long i, float2 v) { ((__nv_bfloat162 *)p)[i] = __float22bfloat162_rn(v); }
  static __device__ __forceinline__ void stcs(void *p, long long i, float2 v) { __stcs((__nv_bfloat162 *)p + i, __float22bfloat162_rn(v)); }
};

// the value a stored number has when it is read back (identity for complex64): the moment of the new state is
// accumulated from what the next stage will actually read
template <class ST> __device__ __forceinline__ float2 as_stored(float2 v) { return v; }
template <> __device__ __forceinline__ float2 as_stored<__half2>(float2 v) { return __half22float2(__float22half2_rn(v)); }
template <> __device__ __forceinline__ float2 as_stored<__nv_bfloat162>(float2 v) {
  return __bfloat1622float2(__float22bfloat162_rn(v));
}

// ---- diagnostics folded into a stage launch ---------------------------------------------------------------------
// CFL (PAPER.md:356 (i); R21): every thread that produces real-space grad(chi) = (d_x chi, d_y chi) keeps the largest
// |d_y chi| kx_max + |d_x chi| ky_max it has seen; one atomicMax per warp at the end of its role.
struct GmaxAcc {
  float v = 0.f;
  // ef: ExB factor of the plane the gradient belongs to
  __device__ __forceinline__ void add(const GkDev &P, float2 g, float ef) { v = fmaxf(v, ef * (fabsf(g.y) * P.kxmax + fabsf(g.x) * P.kymax)); }
  // all 32 lanes of the warp call
  __device__ __forceinline__ void flush(unsigned int *dst) const {
    if (!dst) return;
    const unsigned int b = __reduce_max_sync(0xffffffffu, __float_as_uint(v));
    if ((threadIdx.x & 31) == 0 && b) atomicMax(dst, b);
  }
};

// Fluxes (R18) of the state a stage-1 launch reads (y = f_n, chi = J0 phi(f_n) are in registers
// there).  A thread sums 2 m Im[conj(chi) f] over its points of a slab (P_m ky_m / ky0, zero at m = 0), the slab-uniform
// factors are applied once per slab, the three moments are reduced over the warp once per work item into per-warp
// DOUBLE slots in shared memory and written out when the species changes: one writer per slot, fixed order, no atomics.
struct FluxAcc {
  float s0 = 0.f, s1 = 0.f, s2 = 0.f;
  // psum = sum over the thread's points of 2 m Im[conj(chi) f]
  __device__ __forceinline__ void slab(const GkDev &P, int l, int i, int j, float psum) {
    const float vj = P.v[j], Bi = P.B[i];
    const float t = -0.5f * P.ef[i] * P.ky0 * Bi * P.wmu[l] * psum;
    s0 += t;
    s1 = fmaf(t, vj * vj + 2.f * P.mu[l] * Bi, s1);
    s2 = fmaf(t, vj * P.Rmaj[i], s2);
  }
  // end of a work item; all 32 lanes call.  slot: 3 doubles of this warp in shared memory
  __device__ __forceinline__ void item_end(double *slot) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      s0 += __shfl_xor_sync(0xffffffffu, s0, o);
      s1 += __shfl_xor_sync(0xffffffffu, s1, o);
      s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    if ((threadIdx.x & 31) == 0) { slot[0] += (double)s0; slot[1] += (double)s1; slot[2] += (double)s2; }
    s0 = s1 = s2 = 0.f;
  }
};
// lane 0 of a warp: write the warp's slot for species a (if any) and clear it
__device__ __forceinline__ void flux_flush(const GkDev &P, double *fluxp, int cta, int nwarps, int warp, int a, double *slot) {
  if (a < 0) return;
  double *dst = fluxp + (((size_t)cta * nwarps + warp) * P.nsp + a) * 3;
  dst[0] = slot[0]; dst[1] = slot[1]; dst[2] = slot[2];
  slot[0] = slot[1] = slot[2] = 0.0;
}

}  // namespace gk
