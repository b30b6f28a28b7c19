// gk_kernels.cuh -- the CUDA kernels of libgk (sm_100a).  Product path; shares nothing with oracle/.
//
//   gk_moment_kernel   a1: J0-gyroaveraged velocity-space moment of f, per (species, mu, vpar-chunk)
//   gk_phi_kernel      a2: sum of the moment planes, Poisson division
//   gk_zonal_kernel    a2: flux-surface-average correction of the ky=0 column (adiabatic electrons)
//   gk_stage_kernel    a3-a6: gyro-average, linear terms, bracket (shared-memory 2-D FFT), RK stage
//                      update and the moment planes of the next stage, one pass over f
//   gk_flux_kernel     diagnostics
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
template <class ST> struct Cv;
template <> struct Cv<float2> {
  static __device__ __forceinline__ float2 ld(const void *p, long long i) { return ((const float2 *)p)[i]; }
  static __device__ __forceinline__ float2 ldg(const void *p, long long i) { return __ldg((const float2 *)p + i); }
  static __device__ __forceinline__ void st(void *p, long long i, float2 v) { ((float2 *)p)[i] = v; }
};
template <> struct Cv<__half2> {
  static __device__ __forceinline__ float2 ld(const void *p, long long i) { return __half22float2(((const __half2 *)p)[i]); }
  static __device__ __forceinline__ float2 ldg(const void *p, long long i) { return __half22float2(__ldg((const __half2 *)p + i)); }
  static __device__ __forceinline__ void st(void *p, long long i, float2 v) { ((__half2 *)p)[i] = __float22half2_rn(v); }
};
template <> struct Cv<__nv_bfloat162> {
  static __device__ __forceinline__ float2 ld(const void *p, long long i) { return __bfloat1622float2(((const __nv_bfloat162 *)p)[i]); }
  static __device__ __forceinline__ float2 ldg(const void *p, long long i) { return __bfloat1622float2(((const __nv_bfloat162 *)p)[i]); }
  static __device__ __forceinline__ void st(void *p, long long i, float2 v) { ((__nv_bfloat162 *)p)[i] = __float22bfloat162_rn(v); }
};

// =================================================================================================
// a1. Velocity-space moment.  One thread per (work item, slab element); a work
// item is (species a, mu l, vpar chunk c, s i).  Writes
//   mom[((a*nmu+l)*nchunk+c)][i][p][m] = Z_a n_a 2 pi B_i w_v w_mu,l J0_a(l,i,p,m) sum_{j in c} f
// Reads f exactly once, coalesced along (p,m).
// =================================================================================================
template <class ST>
__global__ void __launch_bounds__(256) gk_moment_kernel(const __grid_constant__ GkDev P,
                                                        const void *__restrict__ f,
                                                        float2 *__restrict__ mom) {
  const int nblk_slab = (int)((P.slab + 255) / 256);
  const int w = blockIdx.x / nblk_slab;
  const long long e = (long long)(blockIdx.x % nblk_slab) * 256 + threadIdx.x;
  if (e >= P.slab) return;
  const int i = w % P.ns;
  const int c = (w / P.ns) % P.nchunk;
  const int l = (w / (P.ns * P.nchunk)) % P.nmu;
  const int a = w / (P.ns * P.nchunk * P.nmu);
  const int j0 = c * P.jchunk, j1 = min(P.nv, j0 + P.jchunk);
  float2 acc = make_float2(0.f, 0.f);
  const long long jstride = (long long)P.nmu * P.ns * P.slab;
  long long idx = ((((long long)a * P.nv + j0) * P.nmu + l) * P.ns + i) * P.slab + e;
#pragma unroll 4
  for (int j = j0; j < j1; ++j, idx += jstride) acc = cadd(acc, Cv<ST>::ldg(f, idx));
  const float wgt = P.sp[a].momfac * P.wmu[l] * P.B[i] *
                    __ldg(&P.J0[(((long long)a * P.nmu + l) * P.ns + i) * P.slab + e]);
  mom[(((long long)a * P.nmu + l) * P.nchunk + c) * P.nphi + (long long)i * P.slab + e] =
      make_float2(acc.x * wgt, acc.y * wgt);
}

// a2. phi = (sum of planes) / denominator.  For adiabatic electrons the ky=0 column receives the
// plain division here and the flux-surface-average correction in gk_zonal_kernel (R10).
__global__ void __launch_bounds__(256) gk_phi_kernel(const __grid_constant__ GkDev P,
                                                     const float2 *__restrict__ mom,
                                                     float2 *__restrict__ phi) {
  const long long e = (long long)blockIdx.x * 256 + threadIdx.x;
  if (e >= P.nphi) return;
  float2 acc = make_float2(0.f, 0.f);
  for (int q = 0; q < P.nparts; ++q) acc = cadd(acc, __ldg(&mom[(long long)q * P.nphi + e]));
  const float d = P.dinv[e];
  phi[e] = make_float2(acc.x * d, acc.y * d);
}

// Zonal correction: phibar = <N/(A+a)>_s / <A/(A+a)>_s; phi_i = N_i/(A_i+a) + a phibar/(A_i+a).
// One warp per kx.
__global__ void __launch_bounds__(32) gk_zonal_kernel(const __grid_constant__ GkDev P,
                                                      float2 *__restrict__ phi) {
  const int ip = blockIdx.x;
  float2 s = make_float2(0.f, 0.f);
  for (int i = threadIdx.x; i < P.ns; i += 32) s = cadd(s, phi[((long long)i * P.nkx + ip) * P.nky]);
  for (int o = 16; o > 0; o >>= 1) {
    s.x += __shfl_xor_sync(0xffffffffu, s.x, o);
    s.y += __shfl_xor_sync(0xffffffffu, s.y, o);
  }
  const float sc = P.ae * P.zinv[ip] / (float)P.ns;
  for (int i = threadIdx.x; i < P.ns; i += 32) {
    const long long q = ((long long)i * P.nkx + ip) * P.nky;
    const float d = P.dinv[q];
    float2 v = phi[q];
    v.x += sc * s.x * d;
    v.y += sc * s.y * d;
    phi[q] = v;
  }
}

// =================================================================================================
// Linear terms at one point.  y is the stage state.
// =================================================================================================
struct PointCtx {  // quantities uniform over a slab (a, j, l, i)
  int a, j, l, i;
  float vj, mul, Bi, E, ED, fm, cpar, cmir, sthi, czi;
  int sg;  // 0: v>0, 1: v<0
  long long base;   // index of (a,j,l,i,0,0)
  long long jbase;  // J0 index of (a,l,i,0,0)
};

template <class ST>
__device__ __forceinline__ float2 linear_point(const GkDev &P, const void *__restrict__ y,
                                               const float2 *__restrict__ phi, const PointCtx &C,
                                               int ip, int m, float2 f0) {
  const GkSpeciesDev &S = P.sp[C.a];
  const long long e = (long long)ip * P.nky + m;
  const int mask = P.mask;
  const int shift = m * P.ikx;
  int cls = 2;
  if (m > 0) {
    if (C.i < 2 && ip - shift < 0) cls = C.i;                              // -2,-1 -> 0,1
    else if (C.i >= P.ns - 2 && ip + shift > P.nkx - 1) cls = C.i - (P.ns - 3) + 2;  // +1,+2 -> 3,4
  }
  const float2 chi0 = [&] {
    const float j0 = __ldg(&P.J0[C.jbase + e]);
    const float2 ph = __ldg(&phi[(long long)C.i * P.slab + e]);
    return make_float2(j0 * ph.x, j0 * ph.y);
  }();
  float2 dsf = make_float2(0.f, 0.f), d4f = dsf, dschi = dsf;
#pragma unroll
  for (int d = -2; d <= 2; ++d) {
    float2 fd, cd;
    if (d == 0) {
      fd = f0;
      cd = chi0;
    } else {
      int i2 = C.i + d, ip2 = ip;
      bool ok = true;
      if (i2 >= P.ns) { i2 -= P.ns; ip2 = ip + shift; ok = ip2 <= P.nkx - 1; }
      else if (i2 < 0) { i2 += P.ns; ip2 = ip - shift; ok = ip2 >= 0; }
      fd = make_float2(0.f, 0.f);
      cd = fd;
      if (ok) {
        const long long off = (long long)(i2 - C.i) * P.slab + (long long)(ip2 - ip) * P.nky;
        fd = Cv<ST>::ldg(y, C.base + e + off);
        const float j0 = __ldg(&P.J0[C.jbase + e + off]);
        const float2 ph = __ldg(&phi[(long long)C.i * P.slab + e + off]);
        cd = make_float2(j0 * ph.x, j0 * ph.y);
      }
    }
    const float cd1 = P.dcoef[cls][C.sg][d + 2], cd4 = P.discoef[cls][d + 2];
    dsf.x += cd1 * fd.x; dsf.y += cd1 * fd.y;
    d4f.x += cd4 * fd.x; d4f.y += cd4 * fd.y;
    dschi.x += cd1 * cd.x; dschi.y += cd1 * cd.y;
  }
  float2 r = make_float2(0.f, 0.f);
  {
    float cI = (mask & GK_T_I) ? -C.cpar * P.ds_inv : 0.f;
    float cD = (mask & GK_T_DISS_S) ? -P.nu_s * fabsf(C.cpar) * P.ds_inv : 0.f;
    float c7 = (mask & GK_T_VII) ? -S.ZoverT * C.cpar * C.fm * P.ds_inv : 0.f;
    r.x = cI * dsf.x + cD * d4f.x + c7 * dschi.x;
    r.y = cI * dsf.y + cD * d4f.y + c7 * dschi.y;
  }
  // vpar stencil, zero padding
  {
    const long long js = (long long)P.nmu * P.ns * P.slab;
    float2 z = make_float2(0.f, 0.f);
    float2 fm2 = (C.j >= 2) ? Cv<ST>::ldg(y, C.base + e - 2 * js) : z;
    float2 fm1 = (C.j >= 1) ? Cv<ST>::ldg(y, C.base + e - js) : z;
    float2 fp1 = (C.j + 1 < P.nv) ? Cv<ST>::ldg(y, C.base + e + js) : z;
    float2 fp2 = (C.j + 2 < P.nv) ? Cv<ST>::ldg(y, C.base + e + 2 * js) : z;
    const float k1 = 1.f / 12.f, k8 = 8.f / 12.f;
    float2 dvf = make_float2(k1 * (fm2.x - fp2.x) + k8 * (fp1.x - fm1.x),
                             k1 * (fm2.y - fp2.y) + k8 * (fp1.y - fm1.y));
    float2 d4v = make_float2(k1 * (fm2.x + fp2.x) - (4.f / 12.f) * (fm1.x + fp1.x) + 0.5f * f0.x,
                             k1 * (fm2.y + fp2.y) - (4.f / 12.f) * (fm1.y + fp1.y) + 0.5f * f0.y);
    float c4 = (mask & GK_T_IV) ? C.cmir * P.dv_inv : 0.f;
    float cD = (mask & GK_T_DISS_V) ? -P.nu_v * fabsf(C.cmir) * P.dv_inv : 0.f;
    r.x += c4 * dvf.x + cD * d4v.x;
    r.y += c4 * dvf.y + cD * d4v.y;
  }
  // diagonal terms: -i a f  ->  (a f.y, -a f.x)
  {
    const float kap = -(P.kx[ip] * C.sthi + P.ky[m] * C.czi);
    float a2 = (mask & GK_T_II) ? S.ToverZ * C.ED * kap : 0.f;
    float a5 = (mask & GK_T_V) ? 0.5f * P.ky[m] * C.fm * (S.rln + (C.E - 1.5f) * S.rlt) : 0.f;
    float a8 = (mask & GK_T_VIII) ? C.ED * kap * C.fm : 0.f;
    float ac = a5 + a8;
    r.x += a2 * f0.y + ac * chi0.y;
    r.y -= a2 * f0.x + ac * chi0.x;
    if (mask & GK_T_HYP) {
      const float h = P.hypx[ip] + P.hypy[m];
      r.x -= h * f0.x;
      r.y -= h * f0.y;
    }
  }
  return r;
}

__device__ __forceinline__ void make_ctx(const GkDev &P, int a, int j, int l, int i, PointCtx &C) {
  C.a = a; C.j = j; C.l = l; C.i = i;
  C.vj = P.v[j]; C.mul = P.mu[l]; C.Bi = P.B[i];
  C.E = C.vj * C.vj + 2.f * C.mul * C.Bi;
  C.ED = C.vj * C.vj + C.mul * C.Bi;
  C.fm = P.fmv[j] * P.fmm[l * P.ns + i];
  C.cpar = P.sp[a].vR * C.vj * P.F[i];
  C.cmir = P.sp[a].vR * C.mul * P.BG[i];
  C.sthi = P.sth[i]; C.czi = P.cz[i];
  C.sg = (C.vj > 0.f) ? 0 : 1;
  C.base = ((((long long)a * P.nv + j) * P.nmu + l) * P.ns + i) * P.slab;
  C.jbase = (((long long)a * P.nmu + l) * P.ns + i) * P.slab;
}

// =================================================================================================
// Bracket building blocks.  Shared-memory arrays:
//   A  [mx][ldx]   x-transformed half spectra; columns 0..nky-1: i kx g, nky..2nky-1: i ky g
//   W  [rc][ldy]   y-transform workspace for a chunk of rc rows (ldy odd: conflict-free rows)
//   G  [mx][ldy]   real-space (d_x chi, d_y chi) packed as (re, im); shared or per-CTA global
// Two real fields ride in one complex transform (re = d_x, im = d_y); the imaginary part the
// ky=0 column would leak is dropped, i.e. the column is Hermitian-averaged.
// =================================================================================================
struct Smem {
  float2 *twx, *twy, *A, *W, *G;
};

// spectral slab -> A (zero padded), multiplied by i kx / i ky.  LOADER(e) returns g at slab index e.
template <class LOADER>
__device__ __forceinline__ void load_gradients(const GkDev &P, const Smem &S, LOADER g, int tid, int nthr) {
  const int n_el = P.mx * P.nky;
  for (int q = tid; q < n_el; q += nthr) {
    const int n = q / P.nky, m = q - n * P.nky;
    int ip = -1;
    if (n <= P.K) ip = n + P.K;
    else if (n >= P.mx - P.K) ip = n - P.mx + P.K;
    float2 ax = make_float2(0.f, 0.f), ay = ax;
    if (ip >= 0) {
      const float2 v = g(ip * P.nky + m);
      const float kx = P.kx[ip], ky = P.ky[m];
      ax = make_float2(-kx * v.y, kx * v.x);
      ay = make_float2(-ky * v.y, ky * v.x);
    }
    S.A[n * P.ldx + m] = ax;
    S.A[n * P.ldx + P.nky + m] = ay;
  }
}

// rows [r0, r0+rc) of A -> packed Hermitian-extended rows in W
__device__ __forceinline__ void build_rows(const GkDev &P, const Smem &S, int r0, int tid, int nthr) {
  const int n_el = P.rc * P.my;
  for (int q = tid; q < n_el; q += nthr) {
    const int r = q / P.my, y = q - r * P.my;
    const float2 *row = S.A + (r0 + r) * P.ldx;
    float2 z = make_float2(0.f, 0.f);
    if (y == 0) {
      z = make_float2(row[0].x, row[P.nky].x);                 // real parts only (ky=0 column)
    } else if (y < P.nky) {
      const float2 ax = row[y], ay = row[P.nky + y];           // ax + i ay
      z = make_float2(ax.x - ay.y, ax.y + ay.x);
    } else if (y > P.my - P.nky) {
      const int m = P.my - y;                                   // conj(ax) + i conj(ay)
      const float2 ax = row[m], ay = row[P.nky + m];
      z = make_float2(ax.x + ay.y, ay.x - ax.y);
    }
    S.W[r * P.ldy + y] = z;
  }
}

// real-space gradients of one spectral slab for all rows, chunk by chunk; SINK(r0) consumes W.
template <class LOADER, class SINK>
__device__ __forceinline__ void gradients_to_real(const GkDev &P, const Smem &S, LOADER g, SINK sink,
                                                  int tid, int nthr) {
  load_gradients(P, S, g, tid, nthr);
  __syncthreads();
  gkfft::inv_nat2perm(P.mx, S.A, 2 * P.nky, 1, P.ldx, S.twx, tid, nthr);
  __syncthreads();
  for (int r0 = 0; r0 < P.mx; r0 += P.rc) {
    build_rows(P, S, r0, tid, nthr);
    __syncthreads();
    gkfft::inv_nat2perm(P.my, S.W, P.rc, P.ldy, 1, S.twy, tid, nthr);
    __syncthreads();
    sink(r0);
    __syncthreads();
  }
}

// =================================================================================================
// a3-a6. The fused stage kernel.  Persistent CTAs; a work item is (species a, mu l, s i, vpar chunk);
// consecutive items of a CTA share (a,l,i) so grad(chi) is transformed once per (a,l,i) and reused
// over vpar.  Per vpar slab: gradients of f -> real space -> Poisson bracket with grad(chi) ->
// forward transform -> truncate; then per point linear terms + RK stage update + moment of the
// new state, written once.
// =================================================================================================
#define GK_STAGE_THREADS 512
#define GK_EPT_MAX 16  // slab elements per thread for the moment accumulators (512*16 = 8192)

template <class ST, bool NL>
__global__ void __launch_bounds__(GK_STAGE_THREADS, 1)
gk_stage_kernel(const __grid_constant__ GkDev P, const __grid_constant__ GkStageArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, nthr = blockDim.x;
  Smem S;
  float2 *sp = (float2 *)smem_raw;
  float2 *stage = nullptr;  // per-element staging of the moment contribution
  if (NL) {
    S.twx = sp; sp += P.mx;
    S.twy = sp; sp += P.my;
    S.A = sp; sp += P.mx * P.ldx;
    S.W = sp; sp += P.rc * P.ldy;
    S.G = P.gchi_in_smem ? sp : A.gchi + (long long)blockIdx.x * P.mx * P.ldy;
    for (int t = tid; t < P.mx; t += nthr) S.twx[t] = P.twx[t];
    for (int t = tid; t < P.my; t += nthr) S.twy[t] = P.twy[t];
    stage = S.A + P.nky;  // the i*ky columns are free after the y-transforms
    __syncthreads();
  } else {
    stage = sp;
  }
  const int slab = (int)P.slab;
  const long long w0 = (long long)blockIdx.x * A.nwork / gridDim.x;
  const long long w1 = (long long)(blockIdx.x + 1) * A.nwork / gridDim.x;
  int cur = -1;
  const float scale = 0.25f * P.fftnorm;  // 1/2 (bracket) * 1/2 (two-for-one unpack) / (mx my)

  for (long long w = w0; w < w1; ++w) {
    const int c = (int)(w % P.nchunk);
    const int ali = (int)(w / P.nchunk);
    const int i = ali % P.ns, l = (ali / P.ns) % P.nmu, a = ali / (P.ns * P.nmu);
    if (NL && ali != cur) {
      cur = ali;
      const long long jb = (((long long)a * P.nmu + l) * P.ns + i) * P.slab;
      const float2 *ph = A.phi + (long long)i * P.slab;
      gradients_to_real(
          P, S,
          [&](int e) {
            const float j0 = __ldg(&P.J0[jb + e]);
            const float2 p = __ldg(&ph[e]);
            return make_float2(j0 * p.x, j0 * p.y);
          },
          [&](int r0) {
            for (int q = tid; q < P.rc * P.my; q += nthr) {
              const int r = q / P.my, y = q - r * P.my;
              S.G[(r0 + r) * P.ldy + y] = S.W[r * P.ldy + y];
            }
          },
          tid, nthr);
    }
    float2 macc[GK_EPT_MAX];
#pragma unroll
    for (int k = 0; k < GK_EPT_MAX; ++k) macc[k] = make_float2(0.f, 0.f);
    const int j1 = min(P.nv, (c + 1) * P.jchunk);
    for (int j = c * P.jchunk; j < j1; ++j) {
      PointCtx C;
      make_ctx(P, a, j, l, i, C);
      if (NL) {
        gradients_to_real(
            P, S, [&](int e) { return Cv<ST>::ldg(A.y, C.base + e); },
            [&](int r0) {
              // bracket d_y chi d_x f - d_x chi d_y f on row pairs, packed (row, row+1) -> (re, im)
              const int half = P.rc / 2;
              for (int q = tid; q < half * P.my; q += nthr) {
                const int rp = q / P.my, y = q - rp * P.my;
                const int r = 2 * rp;
                const float2 g0 = S.G[(r0 + r) * P.ldy + y], g1 = S.G[(r0 + r + 1) * P.ldy + y];
                const float2 f0 = S.W[r * P.ldy + y], f1 = S.W[(r + 1) * P.ldy + y];
                S.W[r * P.ldy + y] = make_float2(g0.y * f0.x - g0.x * f0.y, g1.y * f1.x - g1.x * f1.y);
              }
              __syncthreads();
              gkfft::fwd_perm2nat(P.my, S.W, half, 2 * P.ldy, 1, S.twy, tid, nthr);
              __syncthreads();
              // unpack the two real rows and keep only the retained ky: overwrite A's i*kx columns
              for (int q = tid; q < half * P.nky; q += nthr) {
                const int rp = q / P.nky, m = q - rp * P.nky;
                const float2 z = S.W[2 * rp * P.ldy + m];
                float2 zc = S.W[2 * rp * P.ldy + (m == 0 ? 0 : P.my - m)];
                zc.y = -zc.y;
                S.A[(r0 + 2 * rp) * P.ldx + m] = make_float2(z.x + zc.x, z.y + zc.y);
                S.A[(r0 + 2 * rp + 1) * P.ldx + m] = make_float2(z.y - zc.y, zc.x - z.x);
              }
            },
            tid, nthr);
        gkfft::fwd_perm2nat(P.mx, S.A, P.nky, 1, P.ldx, S.twx, tid, nthr);
        __syncthreads();
      }
      // ---- epilogue: linear terms + bracket + RK update, one coalesced pass over the slab ----
      const float momw = P.sp[a].momfac * P.wmu[l] * P.B[i];
      for (int e = tid; e < slab; e += nthr) {
        const int ip = e / P.nky, m = e - ip * P.nky;
        const float2 f0 = Cv<ST>::ldg(A.y, C.base + e);
        float2 k = linear_point<ST>(P, A.y, A.phi, C, ip, m, f0);
        if (NL) {
          const int n = (ip >= P.K) ? ip - P.K : P.mx + ip - P.K;
          const float2 nl = S.A[n * P.ldx + m];
          k.x += scale * nl.x;
          k.y += scale * nl.y;
        }
        float2 out;
        const long long g = C.base + e;
        if (A.mode == 0) {
          out = k;
        } else if (A.mode == 1) {
          Cv<ST>::st(A.acc, g, make_float2(f0.x + A.b * k.x, f0.y + A.b * k.y));
          out = make_float2(f0.x + A.c * k.x, f0.y + A.c * k.y);
        } else if (A.mode == 2) {
          const float2 fn = Cv<ST>::ldg(A.fn, g);
          const float2 ac = Cv<ST>::ld(A.acc, g);
          Cv<ST>::st(A.acc, g, make_float2(ac.x + A.b * k.x, ac.y + A.b * k.y));
          out = make_float2(fn.x + A.c * k.x, fn.y + A.c * k.y);
        } else {
          const float2 ac = Cv<ST>::ld(A.acc, g);
          out = make_float2(ac.x + A.b * k.x, ac.y + A.b * k.y);
        }
        Cv<ST>::st(A.out, g, out);
        if (A.mom) {
          const float wj = momw * __ldg(&P.J0[C.jbase + e]);
          stage[NL ? (ip * P.ldx + m) : e] = make_float2(wj * out.x, wj * out.y);
        }
      }
      if (A.mom) {  // same thread wrote these entries: no barrier needed
#pragma unroll
        for (int k = 0; k < GK_EPT_MAX; ++k) {
          const int e = tid + k * nthr;
          if (e < slab) {
            const int ip = e / P.nky, m = e - ip * P.nky;
            macc[k] = cadd(macc[k], stage[NL ? (ip * P.ldx + m) : e]);
          }
        }
      }
      __syncthreads();  // A / stage are rewritten by the next slab
    }
    if (A.mom) {
      float2 *dst = A.mom + (((long long)a * P.nmu + l) * P.nchunk + c) * P.nphi + (long long)i * P.slab;
#pragma unroll
      for (int k = 0; k < GK_EPT_MAX; ++k) {
        const int e = tid + k * nthr;
        if (e < slab) dst[e] = macc[k];
      }
    }
  }
}

// =================================================================================================
// Fluxes (R18).  out[3*a+q] accumulated with double atomics.
// =================================================================================================
template <class ST>
__global__ void __launch_bounds__(256) gk_flux_kernel(const __grid_constant__ GkDev P,
                                                      const void *__restrict__ f,
                                                      const float2 *__restrict__ phi, double *out) {
  const long long per_sp = P.ntot / P.nsp;
  double acc[3] = {0, 0, 0};
  const int a = blockIdx.y;
  for (long long q = (long long)blockIdx.x * 256 + threadIdx.x; q < per_sp; q += (long long)gridDim.x * 256) {
    const int e = (int)(q % P.slab);
    long long t = q / P.slab;
    const int i = (int)(t % P.ns); t /= P.ns;
    const int l = (int)(t % P.nmu);
    const int j = (int)(t / P.nmu);
    const int m = e % P.nky;
    const float2 fv = Cv<ST>::ldg(f, (long long)a * per_sp + q);
    const float j0 = P.J0[(((long long)a * P.nmu + l) * P.ns + i) * P.slab + e];
    const float2 ph = phi[(long long)i * P.slab + e];
    const float im = j0 * (ph.x * fv.y - ph.y * fv.x);  // Im[conj(chi) f]
    const float pw = (m == 0) ? 1.f : 2.f;
    const float wgt = -pw * 0.5f * P.ky[m] * P.B[i] * P.wmu[l] * im;
    const float vj = P.v[j];
    const float E = vj * vj + 2.f * P.mu[l] * P.B[i];
    acc[0] += wgt;
    acc[1] += wgt * E;
    acc[2] += wgt * vj * P.Rmaj[i];
  }
  __shared__ double red[3][8];
  for (int q = 0; q < 3; ++q) {
    double v = acc[q];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) red[q][threadIdx.x >> 5] = v;
  }
  __syncthreads();
  if (threadIdx.x < 3) {
    double v = 0;
    for (int w = 0; w < 8; ++w) v += red[threadIdx.x][w];
    atomicAdd(&out[3 * a + threadIdx.x], v);
  }
}

}  // namespace gk
