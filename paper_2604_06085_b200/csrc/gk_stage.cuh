// gk_stage.cuh -- the fused RK-stage kernel of libgk (steps a3-a6 of DESIGN.md):
// gyro-average, linear terms I,II,IV,V,VII,VIII + dissipation, dealiased ExB bracket through a
// hand-written shared-memory 2-D FFT, RK4 stage update and the velocity-space moment of the new
// state -- one pass over f per stage.  Product path; shares nothing with oracle/.
//
// Persistent CTAs; a work item is (species a, mu l, s i, vpar chunk); consecutive items of a CTA
// share (a,l,i), so chi = J0 phi, its parallel derivative and its real-space gradient are built
// once per (a,l,i) and reused over vpar.
//
// Shared memory (NL only):
//   A [mx][ldx]  x-transformed half spectra, columns 0..nky-1: X = Fx(i kx g), nky..2nky-1: Y0 = Fx(g)
//                (d/dy is the multiplication by i ky, applied when the rows are assembled)
//   W [rc][ldy]  y-transform workspace for a chunk of rc rows
//   G [mx][ldy]  real-space (d_x chi, d_y chi) packed as (re, im); per-CTA global scratch if it
//                does not fit
// ldx, ldy odd: row-parallel passes (lane = row) and column-parallel passes (lane = column) are
// both free of bank conflicts.  Two real fields ride in one complex transform; the imaginary
// part the ky=0 column would leak is dropped = Hermitian average of that column.
#pragma once

namespace gk {

#define GK_SLAB_MAX 8192  // largest nkx*nky a CTA handles (moment accumulators live in registers)

struct SlabCtx {  // quantities uniform over a slab (a, j, l, i)
  int a, j, l, i, sg;
  float E, ED, fm;
  float cI, cDs, c7;      // s-derivative terms, 1/ds folded in
  float c4, cDv;          // vpar-derivative terms, 1/dv folded in
  float a2, a5, a8;       // -i a f coefficients without the (kx,ky) dependent factor
  float sthi, czi;
  long long base, jbase;  // index of (a,j,l,i,0,0) in f, of (a,l,i,0,0) in J0
  long long om2, om1, op1, op2;  // vpar neighbour offsets (0 where outside the grid)
  float wm2, wm1, wp1, wp2;      // 1 inside, 0 outside (zero padding)
};

__device__ __forceinline__ void make_slab_ctx(const GkDev &P, int a, int j, int l, int i, SlabCtx &C) {
  const GkSpeciesDev &S = P.sp[a];
  const int mask = P.mask;
  C.a = a; C.j = j; C.l = l; C.i = i;
  const float vj = P.v[j], mul = P.mu[l], Bi = P.B[i];
  C.sg = (vj > 0.f) ? 0 : 1;
  C.E = vj * vj + 2.f * mul * Bi;
  C.ED = vj * vj + mul * Bi;
  C.fm = P.fmv[j] * P.fmm[l * P.ns + i];
  const float cpar = S.vR * vj * P.F[i];
  const float cmir = S.vR * mul * P.BG[i];
  C.cI = (mask & GK_T_I) ? -cpar * P.ds_inv : 0.f;
  C.cDs = (mask & GK_T_DISS_S) ? -P.nu_s * fabsf(cpar) * P.ds_inv : 0.f;
  C.c7 = (mask & GK_T_VII) ? -S.ZoverT * cpar * C.fm * P.ds_inv : 0.f;
  C.c4 = (mask & GK_T_IV) ? cmir * P.dv_inv : 0.f;
  C.cDv = (mask & GK_T_DISS_V) ? -P.nu_v * fabsf(cmir) * P.dv_inv : 0.f;
  C.a2 = (mask & GK_T_II) ? S.ToverZ * C.ED : 0.f;
  C.a5 = (mask & GK_T_V) ? 0.5f * C.fm * (S.rln + (C.E - 1.5f) * S.rlt) : 0.f;
  C.a8 = (mask & GK_T_VIII) ? C.ED * C.fm : 0.f;
  C.sthi = P.sth[i]; C.czi = P.cz[i];
  C.base = ((((long long)a * P.nv + j) * P.nmu + l) * P.ns + i) * P.slab;
  C.jbase = (((long long)a * P.nmu + l) * P.ns + i) * P.slab;
  const long long js = (long long)P.nmu * P.ns * P.slab;
  C.wm2 = (j >= 2) ? 1.f : 0.f; C.om2 = (j >= 2) ? -2 * js : 0;
  C.wm1 = (j >= 1) ? 1.f : 0.f; C.om1 = (j >= 1) ? -js : 0;
  C.wp1 = (j + 1 < P.nv) ? 1.f : 0.f; C.op1 = (j + 1 < P.nv) ? js : 0;
  C.wp2 = (j + 2 < P.nv) ? 1.f : 0.f; C.op2 = (j + 2 < P.nv) ? 2 * js : 0;
}

// stencil class of (i, ip, m): index into dcoef/discoef (2 = interior)    (R7)
__device__ __forceinline__ int stencil_class(const GkDev &P, int i, int ip, int m) {
  if (m > 0) {
    const int shift = m * P.ikx;
    if (i < 2 && ip - shift < 0) return i;
    if (i >= P.ns - 2 && ip + shift > P.nkx - 1) return i - (P.ns - 3) + 2;
  }
  return 2;
}
// offset (in elements of a [i][kx][ky] block) from (i,ip,m) to its parallel neighbour (i+d), through
// the kx connection at the seam (R6); false beyond an open chain end.
__device__ __forceinline__ bool seam_offset(const GkDev &P, int i, int d, int ip, int m, long long &off) {
  int i2 = i + d, ip2 = ip;
  bool ok = true;
  if (i2 >= P.ns) { i2 -= P.ns; ip2 = ip + m * P.ikx; ok = ip2 <= P.nkx - 1; }
  else if (i2 < 0) { i2 += P.ns; ip2 = ip - m * P.ikx; ok = ip2 >= 0; }
  off = ok ? (long long)(i2 - i) * P.slab + (long long)(ip2 - ip) * P.nky : 0;
  return ok;
}

// ---- one slab element: linear terms + bracket + RK update.  INTERIOR: 2 <= i < ns-2, where the
// parallel stencil never crosses the seam (28 of 32 planes in the BASELINE grids). ----
template <class ST, bool INTERIOR>
__device__ __forceinline__ float2 rhs_point(const GkDev &P, const GkStageArgs &A, const SlabCtx &C,
                                            const float2 *chis, int e, int ip, int m,
                                            int slab, float2 f0, float2 nl) {
  const long long g = C.base + e;
  // ---- all loads first (unconditional, clamped offsets) so they are in flight together ----
  float2 fs[5];
  float cd[5], c4s[5];
  if (INTERIOR) {
    fs[0] = Cv<ST>::ldg(A.y, g - 2 * (long long)slab);
    fs[1] = Cv<ST>::ldg(A.y, g - slab);
    fs[3] = Cv<ST>::ldg(A.y, g + slab);
    fs[4] = Cv<ST>::ldg(A.y, g + 2 * (long long)slab);
#pragma unroll
    for (int d = 0; d < 5; ++d) { cd[d] = P.dcoef[2][C.sg][d]; c4s[d] = P.discoef[2][d]; }
  } else {
    const int cls = stencil_class(P, C.i, ip, m);
#pragma unroll
    for (int d = 0; d < 5; ++d) {
      if (d == 2) { cd[d] = P.dcoef[cls][C.sg][d]; c4s[d] = P.discoef[cls][d]; continue; }
      long long off;
      const bool ok = seam_offset(P, C.i, d - 2, ip, m, off);
      fs[d] = Cv<ST>::ldg(A.y, g + off);
      cd[d] = ok ? P.dcoef[cls][C.sg][d] : 0.f;
      c4s[d] = ok ? P.discoef[cls][d] : 0.f;
    }
  }
  fs[2] = f0;
  const float2 fm2 = Cv<ST>::ldg(A.y, g + C.om2), fm1 = Cv<ST>::ldg(A.y, g + C.om1);
  const float2 fp1 = Cv<ST>::ldg(A.y, g + C.op1), fp2 = Cv<ST>::ldg(A.y, g + C.op2);
  const float2 chi0 = chis[e];
  const float2 dschi = chis[(1 + C.sg) * slab + e];

  float2 dsf = make_float2(0.f, 0.f), d4f = dsf;
#pragma unroll
  for (int d = 0; d < 5; ++d) {
    dsf.x += cd[d] * fs[d].x; dsf.y += cd[d] * fs[d].y;
    d4f.x += c4s[d] * fs[d].x; d4f.y += c4s[d] * fs[d].y;
  }
  float2 r;
  r.x = C.cI * dsf.x + C.cDs * d4f.x + C.c7 * dschi.x;
  r.y = C.cI * dsf.y + C.cDs * d4f.y + C.c7 * dschi.y;
  {
    const float k1 = 1.f / 12.f, k8 = 8.f / 12.f, k4 = 4.f / 12.f;
    const float ax = C.wm2 * fm2.x, ay = C.wm2 * fm2.y, bx = C.wm1 * fm1.x, by = C.wm1 * fm1.y;
    const float cx = C.wp1 * fp1.x, cy = C.wp1 * fp1.y, dx = C.wp2 * fp2.x, dy = C.wp2 * fp2.y;
    const float dvx = k1 * (ax - dx) + k8 * (cx - bx), dvy = k1 * (ay - dy) + k8 * (cy - by);
    const float d4x = k1 * (ax + dx) - k4 * (bx + cx) + 0.5f * f0.x;
    const float d4y = k1 * (ay + dy) - k4 * (by + cy) + 0.5f * f0.y;
    r.x += C.c4 * dvx + C.cDv * d4x;
    r.y += C.c4 * dvy + C.cDv * d4y;
  }
  {
    const float pk = (float)(ip - P.K), kxv = pk * P.dkx, kyv = (float)m * P.ky0;
    const float kap = -(kxv * C.sthi + kyv * C.czi);
    const float a2 = C.a2 * kap, ac = C.a5 * kyv + C.a8 * kap;
    r.x += a2 * f0.y + ac * chi0.y;       // -i a z = (a z.y, -a z.x)
    r.y -= a2 * f0.x + ac * chi0.x;
    const float rx = pk * P.invK, ry = (float)m * P.invM;
    const float h = P.hyp_x * (rx * rx) * (rx * rx) + P.hyp_y * (ry * ry) * (ry * ry);
    r.x -= h * f0.x;
    r.y -= h * f0.y;
  }
  r.x += nl.x;
  r.y += nl.y;
  return r;
}

// =================================================================================================
// NT threads per CTA, OCC resident CTAs per SM (OCC = 2: grad(chi) is kept in the per-CTA global
// scratch so that two CTAs fit one SM and their memory-bound and FFT phases overlap).
template <class ST, int MX_, int MY_, int NKY_, int NKX_, bool NL, int NT, int OCC>
__global__ void __launch_bounds__(NT, OCC)
gk_stage_kernel(const __grid_constant__ GkDev P, const __grid_constant__ GkStageArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr bool SPEC = (MX_ > 0);
  const int tid = threadIdx.x;
  constexpr int nthr = NT;
  constexpr int EPT = SPEC ? (NKX_ * NKY_ + NT - 1) / NT : GK_SLAB_MAX / NT;
  const int mx = SPEC ? MX_ : P.mx, my = SPEC ? MY_ : P.my;
  const int nky = SPEC ? NKY_ : P.nky, nkx = SPEC ? NKX_ : P.nkx;
  const int K = (nkx - 1) / 2, slab = nkx * nky;
  const int ldx = 2 * nky + 1, ldy = my | 1, rc = P.rc, half = rc / 2;

  float2 *sp = (float2 *)smem_raw;
  float2 *twx = nullptr, *twy = nullptr, *SA = nullptr, *SW = nullptr, *SG = nullptr, *stage = nullptr;
  if (NL) {
    twx = sp; sp += mx;
    twy = sp; sp += my;
    SA = sp; sp += mx * ldx;
    SW = sp; sp += rc * ldy;
    SG = P.gchi_in_smem ? sp : A.gchi + (long long)blockIdx.x * mx * ldy;
    for (int t = tid; t < mx; t += nthr) twx[t] = P.twx[t];
    for (int t = tid; t < my; t += nthr) twy[t] = P.twy[t];
    stage = SA + nky;  // the Y0 columns are free once the rows have been assembled
  } else {
    stage = sp;
  }
  float2 *chis = A.chis + (long long)blockIdx.x * 3 * slab;  // chi0, D_s chi (v>0), D_s chi (v<0)
  __syncthreads();

  constexpr int KC = (NKX_ - 1) / 2;  // compile-time K of the specialised kernels
  // real-space gradients of the spectral slab `g` (callable: slab index -> value), chunk by chunk
  auto to_real = [&](auto g, auto sink) {
    gkfft::inv_nat2perm_load<MX_>(mx, SA, 2 * nky, 1, ldx, twx, tid, nthr,
                                  [&](int c, int nbase, auto offc, auto spanc) {
      constexpr int off = decltype(offc)::value, hi = off + decltype(spanc)::value - 1;
      const int n = nbase + off;
      int p;
      if constexpr (SPEC && hi <= KC) {
        p = n;                                   // always a retained kx >= 0
      } else if constexpr (SPEC && (off > KC && hi < MX_ - KC)) {
        return make_float2(0.f, 0.f);            // always zero padding: nothing is loaded
      } else if constexpr (SPEC && off >= MX_ - KC) {
        p = n - mx;                              // always a retained kx < 0
      } else {
        if (n <= K) p = n;
        else if (n >= mx - K) p = n - mx;
        else return make_float2(0.f, 0.f);
      }
      const bool isx = c < nky;
      const int m = isx ? c : c - nky;
      float2 v = g((p + K) * nky + m);
      if (isx) {
        const float kxv = (float)p * P.dkx;
        v = make_float2(-kxv * v.y, kxv * v.x);
      }
      return v;
    });
    __syncthreads();
    for (int r0 = 0; r0 < mx; r0 += rc) {
      gkfft::inv_nat2perm_load<MY_>(my, SW, rc, ldy, 1, twy, tid, nthr,
                                    [&](int r, int nbase, auto offc, auto spanc) {
        constexpr int off = decltype(offc)::value, span = decltype(spanc)::value, hi = off + span - 1;
        const int y = nbase + off;
        const float2 *row = SA + (r0 + r) * ldx;
        auto lower = [&](int m) {                // X + i (i ky Y0)
          const float kyv = (float)m * P.ky0;
          const float2 ax = row[m], g0 = row[nky + m];
          return make_float2(ax.x - kyv * g0.x, ax.y - kyv * g0.y);
        };
        auto upper = [&](int m) {                // conj(X) + i conj(i ky Y0)
          const float kyv = (float)m * P.ky0;
          const float2 ax = row[m], g0 = row[nky + m];
          return make_float2(ax.x + kyv * g0.x, -(ax.y + kyv * g0.y));
        };
        if constexpr (SPEC && off == 0 && span == 1) {
          return make_float2(row[0].x, 0.f);     // ky = 0: real part only (R15)
        } else if constexpr (SPEC && off > 0 && hi < NKY_) {
          return lower(y);
        } else if constexpr (SPEC && off >= NKY_ && hi <= MY_ - NKY_) {
          return make_float2(0.f, 0.f);
        } else if constexpr (SPEC && off > MY_ - NKY_) {
          return upper(my - y);
        } else {
          if (y == 0) return make_float2(row[0].x, 0.f);
          if (y < nky) return lower(y);
          if (y > my - nky) return upper(my - y);
          return make_float2(0.f, 0.f);
        }
      });
      __syncthreads();
      sink(r0);
      __syncthreads();
    }
  };

  const long long w0 = (long long)blockIdx.x * A.nwork / gridDim.x;
  const long long w1 = (long long)(blockIdx.x + 1) * A.nwork / gridDim.x;
  int cur = -1;
  const float scale = 0.25f * P.fftnorm;  // 1/2 (bracket) * 1/2 (two-for-one unpack) / (mx my)

  for (long long w = w0; w < w1; ++w) {
    const int c = (int)(w % P.nchunk);
    const int ali = (int)(w / P.nchunk);
    const int i = ali % P.ns, l = (ali / P.ns) % P.nmu, a = ali / (P.ns * P.nmu);
    if (ali != cur) {
      cur = ali;
      // ---- chi = J0 phi and its parallel derivative for both streaming directions (VII) ----
      const long long jb = (((long long)a * P.nmu + l) * P.ns + i) * P.slab;
      const float2 *ph = A.phi + (long long)i * P.slab;
      for (int e = tid; e < slab; e += nthr) {
        const int ip = e / nky, m = e - ip * nky;
        const int cls = stencil_class(P, i, ip, m);
        float2 c0 = make_float2(0.f, 0.f), dp = c0, dn = c0;
#pragma unroll
        for (int d = 0; d < 5; ++d) {
          long long off;
          if (!seam_offset(P, i, d - 2, ip, m, off)) continue;
          const float j0 = __ldg(&P.J0[jb + e + off]);
          const float2 p = __ldg(&ph[e + off]);
          const float2 ch = make_float2(j0 * p.x, j0 * p.y);
          if (d == 2) c0 = ch;
          dp.x += P.dcoef[cls][0][d] * ch.x; dp.y += P.dcoef[cls][0][d] * ch.y;
          dn.x += P.dcoef[cls][1][d] * ch.x; dn.y += P.dcoef[cls][1][d] * ch.y;
        }
        chis[e] = c0;
        chis[slab + e] = dp;
        chis[2 * slab + e] = dn;
      }
      __syncthreads();
      if (NL) {
        to_real([&](int e) { return chis[e]; },
                [&](int r0) {
                  for (int q = tid; q < rc * my; q += nthr) {
                    const int r = q / my, y = q - r * my;
                    SG[(r0 + r) * ldy + y] = SW[r * ldy + y];
                  }
                });
      }
    }
    float2 macc[EPT];
#pragma unroll
    for (int k = 0; k < EPT; ++k) macc[k] = make_float2(0.f, 0.f);
    const int j1 = min(P.nv, (c + 1) * P.jchunk);
    for (int j = c * P.jchunk; j < j1; ++j) {
      SlabCtx C;
      make_slab_ctx(P, a, j, l, i, C);
      if (NL) {
        to_real([&](int e) { return Cv<ST>::ldg(A.y, C.base + e); },
                [&](int r0) {
                  // bracket d_y chi d_x f - d_x chi d_y f, rows (p, p+rc/2) packed as (re, im), evaluated
                  // inside the first pass of the forward y-transform; only the retained ky are stored
                  auto keep = [&](int p, int nbase, auto offc, auto spanc, float2 v) {
                    constexpr int off = decltype(offc)::value, hi = off + decltype(spanc)::value - 1;
                    const int m = nbase + off;
                    if constexpr (SPEC && off >= NKY_ && hi <= MY_ - NKY_) {
                    } else if constexpr (SPEC && (hi < NKY_ || off > MY_ - NKY_)) {
                      SW[p * ldy + m] = v;
                    } else {
                      if (m < nky || m > my - nky) SW[p * ldy + m] = v;
                    }
                  };
                  if (P.gchi_in_smem) {
                    gkfft::fwd_perm2nat_fused<MY_>(my, SW, half, ldy, 1, twy, tid, nthr,
                        [&](int p, int q) {
                          const float2 g0 = SG[(r0 + p) * ldy + q], g1 = SG[(r0 + p + half) * ldy + q];
                          const float2 f0 = SW[p * ldy + q], f1 = SW[(p + half) * ldy + q];
                          return make_float2(g0.y * f0.x - g0.x * f0.y, g1.y * f1.x - g1.x * f1.y);
                        }, keep);
                  } else {  // grad(chi) in global scratch: coalesced product pass (lane = y) first
                    for (int q = tid; q < half * my; q += nthr) {
                      const int p = q / my, y = q - p * my;
                      const float2 g0 = SG[(r0 + p) * ldy + y], g1 = SG[(r0 + p + half) * ldy + y];
                      const float2 f0 = SW[p * ldy + y], f1 = SW[(p + half) * ldy + y];
                      SW[p * ldy + y] = make_float2(g0.y * f0.x - g0.x * f0.y, g1.y * f1.x - g1.x * f1.y);
                    }
                    __syncthreads();
                    gkfft::fwd_perm2nat_fused<MY_>(my, SW, half, ldy, 1, twy, tid, nthr,
                        [&](int p, int q) { return SW[p * ldy + q]; }, keep);
                  }
                  __syncthreads();
                  // unpack the two real rows, keep only the retained ky: overwrite A's X columns
                  for (int q = tid; q < half * nky; q += nthr) {
                    const int p = q / nky, m = q - p * nky;
                    const float2 z = SW[p * ldy + m];
                    float2 zc = SW[p * ldy + (m == 0 ? 0 : my - m)];
                    zc.y = -zc.y;
                    SA[(r0 + p) * ldx + m] = make_float2(z.x + zc.x, z.y + zc.y);
                    SA[(r0 + p + half) * ldx + m] = make_float2(z.y - zc.y, zc.x - z.x);
                  }
                });
        // forward x-transform of the nky columns; only |p| <= K is stored
        gkfft::fwd_perm2nat_fused<MX_>(mx, SA, nky, 1, ldx, twx, tid, nthr,
            [&](int c, int q) { return SA[q * ldx + c]; },
            [&](int c, int nbase, auto offc, auto spanc, float2 v) {
              constexpr int off = decltype(offc)::value, hi = off + decltype(spanc)::value - 1;
              const int n = nbase + off;
              if constexpr (SPEC && (off > KC && hi < MX_ - KC)) {
              } else if constexpr (SPEC && (hi <= KC || off >= MX_ - KC)) {
                SA[n * ldx + c] = v;
              } else {
                if (n <= K || n >= mx - K) SA[n * ldx + c] = v;
              }
            });
        __syncthreads();
      }
      // ---- epilogue: one coalesced pass over the slab ----
      const bool interior = (i >= 2 && i < P.ns - 2);
      const float momw = P.sp[a].momfac * P.wmu[l] * P.B[i];
      for (int e = tid; e < slab; e += nthr) {
        const int ip = e / nky, m = e - ip * nky;
        const long long g = C.base + e;
        const float2 f0 = Cv<ST>::ldg(A.y, g);
        float2 nlv = make_float2(0.f, 0.f);
        if (NL) {
          const int n = (ip >= K) ? ip - K : mx + ip - K;
          nlv = SA[n * ldx + m];
          nlv.x *= scale;
          nlv.y *= scale;
        }
        // operands of the RK update and of the moment are requested before the stencil arithmetic
        float2 fn = f0, ac = make_float2(0.f, 0.f);
        if (A.mode == 2) fn = Cv<ST>::ldg(A.fn, g);
        if (A.mode >= 2) ac = Cv<ST>::ld(A.acc, g);
        const float j0 = A.mom ? __ldg(&P.J0[C.jbase + e]) : 0.f;
        const float2 k = interior ? rhs_point<ST, true>(P, A, C, chis, e, ip, m, slab, f0, nlv)
                                  : rhs_point<ST, false>(P, A, C, chis, e, ip, m, slab, f0, nlv);
        float2 out;
        if (A.mode == 0) {
          out = k;
        } else if (A.mode == 1) {
          Cv<ST>::st(A.acc, g, make_float2(f0.x + A.b * k.x, f0.y + A.b * k.y));
          out = make_float2(f0.x + A.c * k.x, f0.y + A.c * k.y);
        } else if (A.mode == 2) {
          Cv<ST>::st(A.acc, g, make_float2(ac.x + A.b * k.x, ac.y + A.b * k.y));
          out = make_float2(fn.x + A.c * k.x, fn.y + A.c * k.y);
        } else {
          out = make_float2(ac.x + A.b * k.x, ac.y + A.b * k.y);
        }
        Cv<ST>::st(A.out, g, out);
        if (A.mom) {
          const float wj = momw * j0;
          stage[NL ? (ip * ldx + m) : e] = make_float2(wj * out.x, wj * out.y);
        }
      }
      if (A.mom) {  // the same thread wrote these entries: no barrier needed
#pragma unroll
        for (int k = 0; k < EPT; ++k) {
          const int e = tid + k * nthr;
          if (e < slab) {
            const int ip = e / nky, m = e - ip * nky;
            macc[k] = cadd(macc[k], stage[NL ? (ip * ldx + m) : e]);
          }
        }
      }
      __syncthreads();  // A / stage are rewritten by the next slab
    }
    if (A.mom) {
      float2 *dst = A.mom + (((long long)a * P.nmu + l) * P.nchunk + c) * P.nphi + (long long)i * P.slab;
#pragma unroll
      for (int k = 0; k < EPT; ++k) {
        const int e = tid + k * nthr;
        if (e < slab) dst[e] = macc[k];
      }
    }
  }
}

}  // namespace gk
