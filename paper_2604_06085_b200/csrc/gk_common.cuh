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

}  // namespace gk
