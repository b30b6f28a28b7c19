// gk_kernels.cuh -- the CUDA kernels of libgk (sm_100a).  Product path; shares nothing with oracle/.
//
//   gk_moment_kernel   a1: J0-gyroaveraged velocity-space moment of f, per (species, mu, vpar-chunk)
//   gk_phi_kernel      a2: sum of the moment planes, Poisson division
//   gk_zonal_kernel    a2: flux-surface-average correction of the ky=0 column (adiabatic electrons)
//   gk_stage_kernel    a3-a6: gyro-average, linear terms, bracket (shared-memory 2-D FFT), RK stage
//                      update and the moment planes of the next stage, one pass over f
//   gk_flux_kernel     diagnostics
#pragma once
#include "gk_common.cuh"

namespace gk {

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
// Also clears the CFL maximum that the stage launch following this field solve accumulates (GmaxAcc).
__global__ void __launch_bounds__(256) gk_phi_kernel(const __grid_constant__ GkDev P,
                                                     const float2 *__restrict__ mom,
                                                     float2 *__restrict__ phi, unsigned int *gmax) {
  const long long e = (long long)blockIdx.x * 256 + threadIdx.x;
  if (e == 0 && gmax) *gmax = 0u;
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
// Fluxes (R18) of a caller-supplied (f, phi): per-block partial sums
// part[(blockIdx.x * nsp + a) * 3 + q], summed in a fixed order by gk_flux_sum_kernel (no atomics).
// =================================================================================================
template <class ST>
__global__ void __launch_bounds__(256) gk_flux_kernel(const __grid_constant__ GkDev P,
                                                      const void *__restrict__ f,
                                                      const float2 *__restrict__ phi, double *part) {
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
    const float wgt = -pw * 0.5f * P.ef[i] * P.ky[m] * P.B[i] * P.wmu[l] * im;
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
    part[((size_t)blockIdx.x * P.nsp + a) * 3 + threadIdx.x] = v;
  }
}

// out[3 a + q] = sum over the `nslots` partial records part[slot][a][q] in slot order: one thread per output,
// deterministic.  The partials come from gk_flux_kernel (one slot per block) or from the flux diagnostics of a
// stage-1 launch (one slot per (CTA, warp): FluxAcc in gk_common.cuh).
__global__ void __launch_bounds__(32) gk_flux_sum_kernel(const __grid_constant__ GkDev P, const double *__restrict__ part,
                                                         int nslots, double *__restrict__ out) {
  const int t = threadIdx.x;
  if (t >= 3 * P.nsp) return;
  double acc = 0.0;
  for (int sl = 0; sl < nslots; ++sl) acc += part[(size_t)sl * 3 * P.nsp + t];
  out[t] = acc;
}

// Spectra of |phi|^2 (R20).  Block b < nkx sums row p = b over (s, ky) with the Parseval
// factor; block nkx + m sums column m over (s, kx).  One deterministic tree per output, double accumulation.
__global__ void __launch_bounds__(256) gk_spectra_kernel(const __grid_constant__ GkDev P,
                                                         const float2 *__restrict__ phi, double *out) {
  const int b = blockIdx.x;
  const bool row = b < P.nkx;
  const int fixed = row ? b : b - P.nkx;        // p (row) or m (column)
  const int nfree = row ? P.nky : P.nkx;
  double acc = 0.0;
  for (int q = threadIdx.x; q < P.ns * nfree; q += 256) {
    const int i = q / nfree, r = q - i * nfree;
    const int p = row ? fixed : r, m = row ? r : fixed;
    const float2 v = phi[(long long)i * P.slab + p * P.nky + m];
    const double a2 = (double)v.x * v.x + (double)v.y * v.y;
    acc += (m == 0 ? 1.0 : 2.0) * a2;
  }
  __shared__ double red[256];
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int h = 128; h > 0; h >>= 1) {
    if (threadIdx.x < h) red[threadIdx.x] += red[threadIdx.x + h];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[b] = red[0] / P.ns;
}

}  // namespace gk
