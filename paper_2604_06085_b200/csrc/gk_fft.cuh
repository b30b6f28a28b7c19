// gk_fft.cuh -- hand-written batched shared-memory FFT building blocks for the bracket kernel.
//
// Sizes N = 2^a * 3^b (b <= 1), 2 <= N <= 256, as two register-resident radix passes
// N = R1 * R2 with R1, R2 in {1,2,3,4,6,8,12,16}.  Each work item is one radix-R butterfly held
// entirely in registers (compile-time twiddles); passes exchange data through shared memory.
//
// Index convention (Cooley-Tukey, n = n1 + R1*n2, k = R2*k1 + k2):
//   nat2perm<N,S>: input in natural order, output element k = R2*k1 + k2 is left at position
//                  q = k1 + R1*k2 (in place, no transposition pass).
//   perm2nat<N,S>: the mirror image: input in that permuted order, output in natural order.
// The bracket only multiplies real-space fields pointwise, so the permuted order in real space is
// harmless and the forward transform undoes it for free (any self-consistent FFT
// convention gives the truncated convolution).  S = +1: exp(+2 pi i nk/N), S = -1: exp(-...).
#pragma once
#include <cuda_runtime.h>
#include <type_traits>

namespace gkfft {

template <int I> using IC = std::integral_constant<int, I>;

template <int B, int E, class F>
__device__ __forceinline__ void sfor(F &&f) {
  if constexpr (B < E) {
    f(IC<B>{});
    sfor<B + 1, E>(f);
  }
}

constexpr double kPi = 3.14159265358979323846264338327950288;
__host__ __device__ constexpr double cx_cos(double x) {  // |x| <= pi
  double s = 1, t = 1;
  for (int i = 1; i <= 30; ++i) { t *= -x * x / ((2.0 * i - 1) * (2.0 * i)); s += t; }
  return s;
}
__host__ __device__ constexpr double cx_sin(double x) {
  double s = x, t = x;
  for (int i = 1; i <= 30; ++i) { t *= -x * x / ((2.0 * i) * (2.0 * i + 1)); s += t; }
  return s;
}

// Complex arithmetic on the packed fp32x2 pipe of sm_100a (FADD2 / FMUL2 / FFMA2 take a complex
// number per instruction; the half-swap and per-half negation that multiplication by +-i needs are
// operand modifiers, and a real factor is a broadcast operand, so they cost nothing).
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
// a + s*b, s real
__device__ __forceinline__ float2 caxpy(float s, float2 b, float2 a) { return __ffma2_rn(b, make_float2(s, s), a); }
__device__ __forceinline__ float2 cscale(float s, float2 a) { return __fmul2_rn(a, make_float2(s, s)); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {   // a*b = a b.x + (i a) b.y
  return __ffma2_rn(make_float2(-a.y, a.x), make_float2(b.y, b.y), __fmul2_rn(a, make_float2(b.x, b.x)));
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) {  // a*conj(b)
  return __ffma2_rn(make_float2(a.y, -a.x), make_float2(b.y, b.y), __fmul2_rn(a, make_float2(b.x, b.x)));
}
// multiply by S*i
template <int S> __device__ __forceinline__ float2 muli(float2 a) {
  return S > 0 ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}

// a * exp(S * 2 pi i K / N), K and N compile-time
template <int N, int K, int S> __device__ __forceinline__ float2 mulw(float2 a) {
  constexpr int k = ((K % N) + N) % N;
  if constexpr (k == 0) return a;
  else if constexpr (4 * k == N) return muli<S>(a);
  else if constexpr (2 * k == N) return make_float2(-a.x, -a.y);
  else if constexpr (4 * k == 3 * N) return muli<-S>(a);
  else {
    constexpr double ang = 2.0 * kPi * (k > N / 2 ? k - N : k) / N;
    constexpr float c = (float)cx_cos(ang);
    constexpr float s = (float)(S * cx_sin(ang));
    return __ffma2_rn(make_float2(-a.y, a.x), make_float2(s, s), __fmul2_rn(a, make_float2(c, c)));
  }
}

// In-register DFT of R points, natural order in and out.
template <int R, int S> __device__ __forceinline__ void dft(float2 (&v)[R]) {
  if constexpr (R == 1) {
  } else if constexpr (R == 2) {
    float2 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
  } else if constexpr (R == 3) {
    const float2 t1 = cadd(v[1], v[2]);
    const float2 t2 = caxpy(-0.5f, t1, v[0]);
    const float2 d = muli<S>(csub(v[1], v[2]));
    v[0] = cadd(v[0], t1);
    v[1] = caxpy(0.86602540378443864676f, d, t2);
    v[2] = caxpy(-0.86602540378443864676f, d, t2);
  } else if constexpr (R == 4) {
    float2 s02 = cadd(v[0], v[2]), d02 = csub(v[0], v[2]);
    float2 s13 = cadd(v[1], v[3]), d13 = muli<S>(csub(v[1], v[3]));
    v[0] = cadd(s02, s13);
    v[2] = csub(s02, s13);
    v[1] = cadd(d02, d13);
    v[3] = csub(d02, d13);
  } else {
    constexpr int A = (R % 4 == 0) ? 4 : ((R % 2 == 0) ? 2 : 3);
    constexpr int B = R / A;
    float2 t[A][B];
    sfor<0, A>([&](auto n1c) {
      constexpr int n1 = decltype(n1c)::value;
      float2 u[B];
      sfor<0, B>([&](auto n2c) {
        constexpr int n2 = decltype(n2c)::value;
        u[n2] = v[n1 + A * n2];
      });
      dft<B, S>(u);
      sfor<0, B>([&](auto k2c) {
        constexpr int k2 = decltype(k2c)::value;
        t[n1][k2] = mulw<R, n1 * k2, S>(u[k2]);
      });
    });
    sfor<0, B>([&](auto k2c) {
      constexpr int k2 = decltype(k2c)::value;
      float2 u[A];
      sfor<0, A>([&](auto n1c) {
        constexpr int n1 = decltype(n1c)::value;
        u[n1] = t[n1][k2];
      });
      dft<A, S>(u);
      sfor<0, A>([&](auto k1c) {
        constexpr int k1 = decltype(k1c)::value;
        v[B * k1 + k2] = u[k1];
      });
    });
  }
}

// two-pass factorisation N = R1 * R2
template <int N> struct Fac;
#define GK_FAC(N_, A_, B_) \
  template <> struct Fac<N_> { static constexpr int R1 = A_, R2 = B_; }
GK_FAC(2, 2, 1); GK_FAC(3, 3, 1); GK_FAC(4, 4, 1); GK_FAC(6, 6, 1); GK_FAC(8, 8, 1);
GK_FAC(12, 12, 1); GK_FAC(16, 16, 1); GK_FAC(24, 4, 6); GK_FAC(32, 4, 8); GK_FAC(48, 6, 8);
GK_FAC(64, 8, 8); GK_FAC(96, 8, 12); GK_FAC(128, 8, 16); GK_FAC(192, 12, 16); GK_FAC(256, 16, 16);
#undef GK_FAC

// Batched transforms: element e of batch b lives at base[b*bstride + e*estride];
// tw[t] = exp(+2 pi i t/N), t < N.  All threads of the CTA must call; they end WITHOUT a barrier.
//
// Fused variants.  The natural-order side of a transform is produced / consumed by a functor that
// receives the index split as (run-time base, compile-time offset, compile-time span):
//     n = nbase + OFF,  0 <= nbase < SPAN
// so a caller with compile-time sizes can decide with `if constexpr` which elements are zero
// padding (never loaded) or not needed (never stored -> the dead arithmetic is eliminated).
//
// nat2perm_load:  natural-order input of batch b from LOAD(b, nbase, IC<OFF>, IC<SPAN>) (global
//   memory, or another shared array combined on the fly): the first radix pass doubles as the
//   load / zero-pad / pre-multiply pass.  Output digit-permuted in `base`.
struct CtaSync { __device__ __forceinline__ void operator()() const { __syncthreads(); } };
// barrier among the NTHR threads (a multiple of 32) that name the same id
template <int ID, int NTHR> struct NamedSync {
  __device__ __forceinline__ void operator()() const {
    asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(NTHR) : "memory");
  }
};

template <int N, int S, class LOAD, class SYNC = CtaSync>
__device__ __forceinline__ void nat2perm_load(float2 *base, int nb, int bstride, int estride,
                                              const float2 *tw, int tid, int nthr, LOAD load,
                                              SYNC sync = SYNC{}) {
  constexpr int R1 = Fac<N>::R1, R2 = Fac<N>::R2;
  if constexpr (R2 > 1) {
    for (int w = tid; w < nb * R1; w += nthr) {
      const int b = w % nb, n1 = w / nb;
      float2 *p = base + b * bstride + n1 * estride;
      float2 u[R2];
      sfor<0, R2>([&](auto n2c) {
        constexpr int n2 = decltype(n2c)::value;
        u[n2] = load(b, n1, IC<R1 * n2>{}, IC<R1>{});
      });
      dft<R2, S>(u);
#pragma unroll
      for (int k2 = 1; k2 < R2; ++k2) {
        const float2 t = tw[n1 * k2];
        u[k2] = S > 0 ? cmul(u[k2], t) : cmulc(u[k2], t);
      }
#pragma unroll
      for (int k2 = 0; k2 < R2; ++k2) p[k2 * R1 * estride] = u[k2];
    }
    sync();
    for (int w = tid; w < nb * R2; w += nthr) {
      const int b = w % nb, k2 = w / nb;
      float2 *p = base + b * bstride + k2 * R1 * estride;
      float2 u[R1];
#pragma unroll
      for (int n1 = 0; n1 < R1; ++n1) u[n1] = p[n1 * estride];
      dft<R1, S>(u);
#pragma unroll
      for (int k1 = 0; k1 < R1; ++k1) p[k1 * estride] = u[k1];
    }
  } else {
    for (int b = tid; b < nb; b += nthr) {
      float2 *p = base + b * bstride;
      float2 u[R1];
      sfor<0, R1>([&](auto n1c) {
        constexpr int n1 = decltype(n1c)::value;
        u[n1] = load(b, 0, IC<n1>{}, IC<1>{});
      });
      dft<R1, S>(u);
#pragma unroll
      for (int k1 = 0; k1 < R1; ++k1) p[k1 * estride] = u[k1];
    }
  }
}

// perm2nat_fused: digit-permuted input of batch b, position q, from LOADP(b, q) (may combine
//   several shared arrays: the pointwise bracket is evaluated here); natural-order output handed
//   to STORE(b, nbase, IC<OFF>, IC<SPAN>, value).  `base` is the exchange buffer between the
//   two radix passes; LOADP may read it at the positions its own work item overwrites.
template <int N, int S, class LOADP, class STORE, class SYNC = CtaSync>
__device__ __forceinline__ void perm2nat_fused(float2 *base, int nb, int bstride, int estride,
                                               const float2 *tw, int tid, int nthr, LOADP loadp,
                                               STORE store, SYNC sync = SYNC{}) {
  constexpr int R1 = Fac<N>::R1, R2 = Fac<N>::R2;
  if constexpr (R2 > 1) {
    for (int w = tid; w < nb * R2; w += nthr) {
      const int b = w % nb, k2 = w / nb;
      float2 *p = base + b * bstride + k2 * R1 * estride;
      float2 u[R1];
#pragma unroll
      for (int k1 = 0; k1 < R1; ++k1) u[k1] = loadp(b, k2 * R1 + k1);
      dft<R1, S>(u);
#pragma unroll
      for (int n1 = 1; n1 < R1; ++n1) {
        const float2 t = tw[n1 * k2];
        u[n1] = S > 0 ? cmul(u[n1], t) : cmulc(u[n1], t);
      }
#pragma unroll
      for (int n1 = 0; n1 < R1; ++n1) p[n1 * estride] = u[n1];
    }
    sync();
    for (int w = tid; w < nb * R1; w += nthr) {
      const int b = w % nb, n1 = w / nb;
      const float2 *p = base + b * bstride + n1 * estride;
      float2 u[R2];
#pragma unroll
      for (int k2 = 0; k2 < R2; ++k2) u[k2] = p[k2 * R1 * estride];
      dft<R2, S>(u);
      sfor<0, R2>([&](auto n2c) {
        constexpr int n2 = decltype(n2c)::value;
        store(b, n1, IC<R1 * n2>{}, IC<R1>{}, u[n2]);
      });
    }
  } else {
    for (int b = tid; b < nb; b += nthr) {
      float2 u[R1];
#pragma unroll
      for (int k1 = 0; k1 < R1; ++k1) u[k1] = loadp(b, k1);
      dft<R1, S>(u);
      sfor<0, R1>([&](auto n1c) {
        constexpr int n1 = decltype(n1c)::value;
        store(b, 0, IC<n1>{}, IC<1>{}, u[n1]);
      });
    }
  }
}

#define GK_FFT_SWITCH(n, CALL)                                                            \
  switch (n) {                                                                            \
    case 2: CALL(2); break;     case 3: CALL(3); break;     case 4: CALL(4); break;       \
    case 6: CALL(6); break;     case 8: CALL(8); break;     case 12: CALL(12); break;     \
    case 16: CALL(16); break;   case 24: CALL(24); break;   case 32: CALL(32); break;     \
    case 48: CALL(48); break;   case 64: CALL(64); break;   case 96: CALL(96); break;     \
    case 128: CALL(128); break; case 192: CALL(192); break; case 256: CALL(256); break;   \
    default: break;                                                                       \
  }

// Size dispatch: NC > 0 is a compile-time length (specialised kernels), NC == 0 switches on n.
template <int NC, class LOAD, class SYNC = CtaSync>
__device__ __forceinline__ void inv_nat2perm_load(int n, float2 *base, int nb, int bstride, int estride,
                                                  const float2 *tw, int tid, int nthr, LOAD load,
                                                  SYNC sync = SYNC{}) {
  if constexpr (NC > 0) {
    nat2perm_load<NC, +1>(base, nb, bstride, estride, tw, tid, nthr, load, sync);
  } else {
#define GK_CALL(N_) nat2perm_load<N_, +1>(base, nb, bstride, estride, tw, tid, nthr, load, sync)
    GK_FFT_SWITCH(n, GK_CALL)
#undef GK_CALL
  }
}
template <int NC, class LOADP, class STORE, class SYNC = CtaSync>
__device__ __forceinline__ void fwd_perm2nat_fused(int n, float2 *base, int nb, int bstride, int estride,
                                                   const float2 *tw, int tid, int nthr, LOADP loadp,
                                                   STORE store, SYNC sync = SYNC{}) {
  if constexpr (NC > 0) {
    perm2nat_fused<NC, -1>(base, nb, bstride, estride, tw, tid, nthr, loadp, store, sync);
  } else {
#define GK_CALL(N_) perm2nat_fused<N_, -1>(base, nb, bstride, estride, tw, tid, nthr, loadp, store, sync)
    GK_FFT_SWITCH(n, GK_CALL)
#undef GK_CALL
  }
}

// host helper: is n a supported transform length?
inline bool supported_len(int n) {
  switch (n) {
    case 2: case 3: case 4: case 6: case 8: case 12: case 16: case 24: case 32: case 48:
    case 64: case 96: case 128: case 192: case 256: return true;
    default: return false;
  }
}

}  // namespace gkfft
