// gk_stage.cuh -- the fused RK-stage kernel of libgk (steps a3-a6 of DESIGN.md):
// gyro-average, linear terms I,II,IV,V,VII,VIII + dissipation, dealiased ExB bracket through a
// hand-written shared-memory 2-D FFT, RK4 stage update and the velocity-space moment of the new
// state -- one pass over f per stage.  Product path; shares nothing with oracle/.
//
// Persistent CTAs.  A work item is (species a, mu l, vpar chunk c, s i) with i fastest, dealt
// round-robin: the CTAs resident at one time cover whole s-chains of a few (a,l,c), so the
// parallel-stencil halos (i +- 1, i +- 2, through the kx connection at the seam) that one CTA reads
// are the slabs its neighbours stream at the same moment and come from L2, not from HBM.  Inside
// an item the CTA marches along vpar: chi = J0 phi, its parallel derivative and its real-space
// gradient are built once and reused, and the vpar halos are the CTA's own recent slabs.
//
// Shared memory (NL only):
//   A [mx][ldx]  x-transformed half spectra, columns 0..nky-1: P = Fx((i kx - ky) g),
//                nky..2nky-1: Q = Fx((i kx + ky) g); the Hermitian-extended row of d_x g + i d_y g
//                is  P(m) at y = m  and  conj Q(m) at y = my - m
//   W [rc][ldy]  y-transform workspace for a chunk of rc rows
//   G [mx][ldy]  real-space (d_x chi, d_y chi) packed as (re, im); per-CTA global scratch if it
//                does not fit
// ldx, ldy odd: row-parallel passes (lane = row) and column-parallel passes (lane = column) are
// both free of bank conflicts.  Two real fields ride in one complex transform; the imaginary
// part the ky=0 column would leak is dropped = Hermitian average of that column.
#pragma once

namespace gk {

struct ItemCtx {  // quantities uniform over a work item (a, l, i)
  int a, l, i;
  float cparF;   // v_R F_i            (times v_j: parallel streaming speed)
  float cmir;    // v_R mu_l B_i G_i   (mirror force)
  float muB;     // mu_l B_i
  float fmm;     // exp(-2 mu B)
  float ZoverT, ToverZ, rln, rlt;
  float ksx, kcz;  // kappa = -(pk ksx + m kcz):  ksx = dkx sin(theta), kcz = ky0 (cos + shat theta sin)
  float hx4, hy4;  // hyper-viscosity: hx4 (p/K)^4 + hy4 (m/(nky-1))^4
  long long base0; // index of (a, 0, l, i, 0, 0) in f
  long long jstride;
};

struct SlabCtx {  // quantities uniform over a slab (a, j, l, i)
  int sg;
  float ws[5];            // parallel stencil on f, interior class: I + dissipation (centre included)
  float wv[5];            // vpar stencil on f: IV + dissipation, zero padding folded in
  float cI, cDs, c7;      // s-derivative terms, 1/ds folded in
  float a2, a5, a8;       // -i a f coefficients without the (kx,ky) dependent factor
  long long base;         // index of (a,j,l,i,0,0) in f
  long long ov[4];        // vpar neighbour offsets j-2, j-1, j+1, j+2 (0 where outside the grid)
};

__device__ __forceinline__ void make_item_ctx(const GkDev &P, int a, int l, int i, ItemCtx &I) {
  const GkSpeciesDev &S = P.sp[a];
  const int mask = P.mask;
  I.a = a; I.l = l; I.i = i;
  const float mul = P.mu[l], Bi = P.B[i];
  I.cparF = S.vR * P.F[i];
  I.cmir = S.vR * mul * P.BG[i];
  I.muB = mul * Bi;
  I.fmm = P.fmm[l * P.ns + i];
  I.ZoverT = S.ZoverT; I.ToverZ = S.ToverZ; I.rln = S.rln; I.rlt = S.rlt;
  I.ksx = P.dkx * P.sth[i];
  I.kcz = P.ky0 * P.cz[i];
  I.hx4 = (mask & GK_T_HYP) ? P.hyp_x * (P.invK * P.invK) * (P.invK * P.invK) : 0.f;
  I.hy4 = (mask & GK_T_HYP) ? P.hyp_y * (P.invM * P.invM) * (P.invM * P.invM) : 0.f;
  I.jstride = (long long)P.nmu * P.ns * P.slab;
  I.base0 = (((long long)a * P.nv * P.nmu + l) * P.ns + i) * P.slab;
}

__device__ __forceinline__ void make_slab_ctx(const GkDev &P, const ItemCtx &I, int j, SlabCtx &C) {
  const int mask = P.mask;
  const float vj = P.v[j];
  C.sg = (vj > 0.f) ? 0 : 1;
  const float E = vj * vj + 2.f * I.muB, ED = vj * vj + I.muB;
  const float fm = P.fmv[j] * I.fmm;
  const float cpar = I.cparF * vj;
  C.cI = (mask & GK_T_I) ? -cpar * P.ds_inv : 0.f;
  C.cDs = (mask & GK_T_DISS_S) ? -P.nu_s * fabsf(cpar) * P.ds_inv : 0.f;
  C.c7 = (mask & GK_T_VII) ? -I.ZoverT * cpar * fm * P.ds_inv : 0.f;
  const float c4 = (mask & GK_T_IV) ? I.cmir * P.dv_inv : 0.f;
  const float cDv = (mask & GK_T_DISS_V) ? -P.nu_v * fabsf(I.cmir) * P.dv_inv : 0.f;
  C.a2 = (mask & GK_T_II) ? I.ToverZ * ED : 0.f;
  C.a5 = (mask & GK_T_V) ? 0.5f * P.ef[I.i] * fm * (I.rln + (E - 1.5f) * I.rlt) : 0.f;
  C.a8 = (mask & GK_T_VIII) ? ED * fm : 0.f;
#pragma unroll
  for (int d = 0; d < 5; ++d) C.ws[d] = C.cI * P.dcoef[2][C.sg][d] + C.cDs * P.discoef[2][d];
  // D_v = (1,-8,0,8,-1)/12, delta^4_v/12 = (1,-4,6,-4,1)/12; ghosts outside the grid are zero
  const float k1 = 1.f / 12.f, k8 = 8.f / 12.f, k4 = 4.f / 12.f;
  const bool m2 = j >= 2, m1 = j >= 1, p1 = j + 1 < P.nv, p2 = j + 2 < P.nv;
  C.wv[0] = m2 ? (c4 * k1 + cDv * k1) : 0.f;
  C.wv[1] = m1 ? (-c4 * k8 - cDv * k4) : 0.f;
  C.wv[2] = cDv * 0.5f;
  C.wv[3] = p1 ? (c4 * k8 - cDv * k4) : 0.f;
  C.wv[4] = p2 ? (-c4 * k1 + cDv * k1) : 0.f;
  C.base = I.base0 + (long long)j * I.jstride;
  C.ov[0] = m2 ? -2 * I.jstride : 0;
  C.ov[1] = m1 ? -I.jstride : 0;
  C.ov[2] = p1 ? I.jstride : 0;
  C.ov[3] = p2 ? 2 * I.jstride : 0;
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
__device__ __forceinline__ bool seam_offset(const GkDev &P, int i, int d, int ip, int m, int &off) {
  int i2 = i + d, ip2 = ip;
  bool ok = true;
  if (i2 >= P.ns) { i2 -= P.ns; ip2 = ip + m * P.ikx; ok = ip2 <= P.nkx - 1; }
  else if (i2 < 0) { i2 += P.ns; ip2 = ip - m * P.ikx; ok = ip2 >= 0; }
  off = ok ? (i2 - i) * (int)P.slab + (ip2 - ip) * P.nky : 0;
  return ok;
}

// Operand pointers of one slab's epilogue.
template <class ST> struct EpiPtrs {
  const ST *yb;                    // state slab (a,j,l,i)
  const ST *yv0, *yv1, *yv3, *yv4; // vpar neighbours j-2, j-1, j+1, j+2 (== yb where outside the grid)
  const ST *fnb;                   // f_n slab
  ST *accb, *outb;                 // accumulator and output slabs
  const float2 *chi0, *dsch;       // chi and D_s chi (for the sign of v_j) of this (a,l,i)
};
template <class ST>
__device__ __forceinline__ void make_epi_ptrs(const GkStageArgs &A, const SlabCtx &C, const float2 *chis,
                                              int slab, EpiPtrs<ST> &Q) {
  Q.yb = (const ST *)A.y + C.base;
  Q.yv0 = Q.yb + C.ov[0]; Q.yv1 = Q.yb + C.ov[1]; Q.yv3 = Q.yb + C.ov[2]; Q.yv4 = Q.yb + C.ov[3];
  Q.fnb = (const ST *)A.fn + C.base;
  Q.accb = (ST *)A.acc + C.base;
  Q.outb = (ST *)A.out + C.base;
  Q.chi0 = chis;
  Q.dsch = chis + (1 + C.sg) * slab;
}

// ---- one slab element: linear terms + bracket + RK update.  The operands (own value, 4 parallel
// and 4 vpar neighbours, f_n, accumulator, chi, D_s chi) are all requested before the arithmetic;
// the arithmetic is one packed-fp32 FMA per operand.  INTERIOR: 2 <= i < ns-2, where the parallel
// stencil never crosses the seam (28 of 32 planes in the BASELINE grids).  nlv: bracket value
// (unscaled) of this element. ----
template <class ST, int MODE, bool INTERIOR>
__device__ __forceinline__ float2 rhs_point(const GkDev &P, const GkStageArgs &A, const ItemCtx &I,
                                            const SlabCtx &C, const EpiPtrs<ST> &Q, int slab, int e,
                                            int ip, int m, float pk, float fmf, float2 nlv, float scale,
                                            float &fsum) {
  const float2 f0 = Cv<ST>::ldg(Q.yb, e);
  float2 fs[5];
  float wsd[5];
  if constexpr (INTERIOR) {
    fs[0] = Cv<ST>::ldg(Q.yb, e - 2 * slab);
    fs[1] = Cv<ST>::ldg(Q.yb, e - slab);
    fs[3] = Cv<ST>::ldg(Q.yb, e + slab);
    fs[4] = Cv<ST>::ldg(Q.yb, e + 2 * slab);
#pragma unroll
    for (int d = 0; d < 5; ++d) wsd[d] = C.ws[d];
  } else {
    const int cls = stencil_class(P, I.i, ip, m);
#pragma unroll
    for (int d = 0; d < 5; ++d) {
      const float wgt = C.cI * P.dcoef[cls][C.sg][d] + C.cDs * P.discoef[cls][d];
      if (d == 2) { wsd[d] = wgt; continue; }
      int off;
      const bool ok = seam_offset(P, I.i, d - 2, ip, m, off);
      fs[d] = Cv<ST>::ldg(Q.yb, e + off);
      wsd[d] = ok ? wgt : 0.f;
    }
  }
  const float2 fv0 = Cv<ST>::ldg(Q.yv0, e), fv1 = Cv<ST>::ldg(Q.yv1, e);
  const float2 fv3 = Cv<ST>::ldg(Q.yv3, e), fv4 = Cv<ST>::ldg(Q.yv4, e);
  float2 fn = f0, ac = make_float2(0.f, 0.f);
  if constexpr (MODE == 2) fn = Cv<ST>::ldcs(Q.fnb, e);
  if constexpr (MODE >= 2) ac = Cv<ST>::ldcs(Q.accb, e);
  const float2 chi0 = __ldcg(&Q.chi0[e]);   // written by this CTA earlier in the launch: L2, not the
  const float2 dschi = __ldcg(&Q.dsch[e]);  // read-only path
  // kappa and the hyper-viscosity rate of this (kx, ky)
  const float kap = -(pk * I.ksx + fmf * I.kcz);
  const float pk2 = pk * pk, fm2 = fmf * fmf;
  const float wc = wsd[2] + C.wv[2] - (I.hx4 * (pk2 * pk2) + I.hy4 * (fm2 * fm2));
  float2 r = gkfft::cscale(wc, f0);
  r = gkfft::caxpy(wsd[0], fs[0], r);
  r = gkfft::caxpy(wsd[1], fs[1], r);
  r = gkfft::caxpy(wsd[3], fs[3], r);
  r = gkfft::caxpy(wsd[4], fs[4], r);
  r = gkfft::caxpy(C.wv[0], fv0, r);
  r = gkfft::caxpy(C.wv[1], fv1, r);
  r = gkfft::caxpy(C.wv[3], fv3, r);
  r = gkfft::caxpy(C.wv[4], fv4, r);
  r = gkfft::caxpy(C.c7, dschi, r);
  // -i a z = a (z.y, -z.x)
  r = gkfft::caxpy(C.a2 * kap, make_float2(f0.y, -f0.x), r);
  r = gkfft::caxpy(C.a5 * (fmf * P.ky0) + C.a8 * kap, make_float2(chi0.y, -chi0.x), r);
  r = gkfft::caxpy(scale, nlv, r);
  float2 out;
  if constexpr (MODE == 0) {
    out = r;
  } else if constexpr (MODE == 1) {
    Cv<ST>::stcs(Q.accb, e, gkfft::caxpy(A.b, r, f0));
    out = gkfft::caxpy(A.c, r, f0);
    fsum = fmaf(2.f * fmf, chi0.x * f0.y - chi0.y * f0.x, fsum);   // flux diagnostics (FluxAcc)
  } else if constexpr (MODE == 2) {
    Cv<ST>::stcs(Q.accb, e, gkfft::caxpy(A.b, r, ac));
    out = gkfft::caxpy(A.c, r, fn);
  } else {
    out = gkfft::caxpy(A.b, r, ac);
  }
  Cv<ST>::stcs(Q.outb, e, out);
  return out;
}

// chi = J0 phi and its parallel derivative for both streaming directions (VII), into the per-CTA
// scratch `chis` (chi0, D_s chi for v>0, D_s chi for v<0)
__device__ __forceinline__ void build_chis(const GkDev &P, const GkStageArgs &A, int a, int l, int i,
                                           int slab, int nky, float2 *chis, int tid, int nthr) {
  const long long jb = (((long long)a * P.nmu + l) * P.ns + i) * P.slab;
  const float2 *ph = A.phi + (long long)i * P.slab;
  for (int e = tid; e < slab; e += nthr) {
    const int ip = e / nky, m = e - ip * nky;
    const int cls = stencil_class(P, i, ip, m);
    float2 c0 = make_float2(0.f, 0.f), dp = c0, dn = c0;
#pragma unroll
    for (int d = 0; d < 5; ++d) {
      int off;
      if (!seam_offset(P, i, d - 2, ip, m, off)) continue;
      const float j0 = __ldg(&P.J0[jb + e + off]);
      const float2 ph0 = __ldg(&ph[e + off]);
      const float2 ch = make_float2(j0 * ph0.x, j0 * ph0.y);
      if (d == 2) c0 = ch;
      dp.x += P.dcoef[cls][0][d] * ch.x; dp.y += P.dcoef[cls][0][d] * ch.y;
      dn.x += P.dcoef[cls][1][d] * ch.x; dn.y += P.dcoef[cls][1][d] * ch.y;
    }
    chis[e] = c0;
    chis[slab + e] = dp;
    chis[2 * slab + e] = dn;
  }
}

// =================================================================================================
// NT threads per CTA, OCC resident CTAs per SM (OCC = 2: grad(chi) is kept in the per-CTA global
// scratch so that two CTAs fit one SM and their memory-bound and FFT phases overlap).
template <class ST, int MX_, int MY_, int NKY_, int NKX_, bool NL, int NT, int OCC>
__global__ void __launch_bounds__(NT, OCC)
gk_stage_kernel(const __grid_constant__ GkDev P, const __grid_constant__ GkStageArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr bool SPEC = (NKX_ > 0);
  const int tid = threadIdx.x;
  constexpr int nthr = NT;
  constexpr int EPT = SPEC ? (NKX_ * NKY_ + NT - 1) / NT : GK_SLAB_MAX / NT;
  const int mx = SPEC ? MX_ : P.mx, my = SPEC ? MY_ : P.my;
  const int nky = SPEC ? NKY_ : P.nky, nkx = SPEC ? NKX_ : P.nkx;
  const int K = (nkx - 1) / 2, slab = nkx * nky;
  const int ldx = 2 * nky + 1, ldy = my | 1, rc = P.rc, half = rc / 2;
  // the (kx, ky) of a thread's k-th element is tid-derived when a CTA row of threads spans whole ky rows
  constexpr bool ROWMAP = SPEC && (NT % (NKY_ > 0 ? NKY_ : 1) == 0);

  float2 *sp = (float2 *)smem_raw;
  float2 *twx = nullptr, *twy = nullptr, *SA = nullptr, *SW = nullptr, *SG = nullptr, *stage = nullptr;
  if constexpr (NL) {
    twx = sp; sp += mx;
    twy = sp; sp += my;
    SA = sp; sp += mx * ldx;
    SW = sp; sp += rc * ldy;
    SG = P.gchi_in_smem ? sp : A.gchi + (long long)blockIdx.x * mx * ldy;
    for (int t = tid; t < mx; t += nthr) twx[t] = P.twx[t];
    for (int t = tid; t < my; t += nthr) twy[t] = P.twy[t];
    stage = SA + nky;  // the Q columns are free once the rows have been assembled
  } else {
    stage = sp;
  }
  // per-CTA scratch: chi0, D_s chi (v>0), D_s chi (v<0)
  float2 *chis = A.chis + (long long)blockIdx.x * 3 * slab;
  __syncthreads();

  constexpr int KC = (NKX_ - 1) / 2;  // compile-time K of the specialised kernels
  // real-space gradients of the spectral slab `g` (callable: slab index -> value), chunk by chunk
  auto to_real = [&](auto g, auto sink) {
    gkfft::inv_nat2perm_load<MX_>(mx, SA, 2 * nky, 1, ldx, twx, tid, nthr,
                                  [&](int c, int nbase, auto offc, auto spanc) {
      constexpr int off = decltype(offc)::value, hi = off + decltype(spanc)::value - 1;
      const int n = nbase + off;
      int p = 0;
      if constexpr (SPEC && MX_ > 0 && hi <= KC) {
        p = n;                                   // always a retained kx >= 0
      } else if constexpr (SPEC && MX_ > 0 && (off > KC && hi < MX_ - KC)) {
        return make_float2(0.f, 0.f);            // always zero padding: nothing is loaded
      } else if constexpr (SPEC && MX_ > 0 && off >= MX_ - KC) {
        p = n - mx;                              // always a retained kx < 0
      } else {
        if (n <= K) p = n;
        else if (n >= mx - K) p = n - mx;
        else return make_float2(0.f, 0.f);
      }
      const bool isp = c < nky;
      const int m = isp ? c : c - nky;
      const float2 v = g((p + K) * nky + m);
      const float kxv = (float)p * P.dkx;
      const float kyv = isp ? -(float)m * P.ky0 : (float)m * P.ky0;
      // (i kx -+ ky) v
      return gkfft::caxpy(kyv, v, gkfft::cscale(kxv, make_float2(-v.y, v.x)));
    });
    __syncthreads();
    for (int r0 = 0; r0 < mx; r0 += rc) {
      gkfft::inv_nat2perm_load<MY_>(my, SW, rc, ldy, 1, twy, tid, nthr,
                                    [&](int r, int nbase, auto offc, auto spanc) {
        constexpr int off = decltype(offc)::value, span = decltype(spanc)::value, hi = off + span - 1;
        const int y = nbase + off;
        const float2 *row = SA + (r0 + r) * ldx;
        auto upper = [&](int m) {                // conj Q
          const float2 q = row[nky + m];
          return make_float2(q.x, -q.y);
        };
        if constexpr (SPEC && MY_ > 0 && off == 0 && span == 1) {
          return make_float2(row[0].x, 0.f);     // ky = 0: real part only (R15)
        } else if constexpr (SPEC && MY_ > 0 && off > 0 && hi < NKY_) {
          return row[y];
        } else if constexpr (SPEC && MY_ > 0 && off >= NKY_ && hi <= MY_ - NKY_) {
          return make_float2(0.f, 0.f);
        } else if constexpr (SPEC && MY_ > 0 && off > MY_ - NKY_) {
          return upper(my - y);
        } else {
          if (y == 0) return make_float2(row[0].x, 0.f);
          if (y < nky) return row[y];
          if (y > my - nky) return upper(my - y);
          return make_float2(0.f, 0.f);
        }
      });
      __syncthreads();
      sink(r0);
      __syncthreads();
    }
  };

  const float scale = 0.25f * P.fftnorm;  // 1/2 (bracket) * 1/2 (two-for-one unpack) / (mx my)

  // diagnostics folded into the launch (gk_common.cuh): CFL maximum of grad(chi), fluxes of the stage-1 state
  GmaxAcc gm;
  __shared__ double fslots[(NT / 32) * 3];
  const bool want_flux = A.fluxp != nullptr && A.mode == 1;
  double *fslot = fslots + (tid >> 5) * 3;
  if ((tid & 31) == 0) fslot[0] = fslot[1] = fslot[2] = 0.0;
  FluxAcc fx;
  int a_prev = -1;

  for (int w = blockIdx.x; w < A.nwork; w += gridDim.x) {
    const int i = w % P.ns;
    const int c = (w / P.ns) % P.nchunk;
    const int al = w / (P.ns * P.nchunk);
    const int l = al % P.nmu, a = al / P.nmu;
    if (want_flux && a != a_prev) {
      if ((tid & 31) == 0) flux_flush(P, A.fluxp, blockIdx.x, NT / 32, tid >> 5, a_prev, fslot);
      a_prev = a;
    }
    ItemCtx I;
    make_item_ctx(P, a, l, i, I);
    {
      build_chis(P, A, a, l, i, slab, nky, chis, tid, nthr);
      __syncthreads();
      if constexpr (NL) {
        to_real([&](int e) { return chis[e]; },
                [&](int r0) {
                  for (int q = tid; q < rc * my; q += nthr) {
                    const int r = q / my, y = q - r * my;
                    const float2 gv = SW[r * ldy + y];
                    SG[(r0 + r) * ldy + y] = gv;
                    gm.add(P, gv, P.ef[i]);
                  }
                });
      }
    }
    float2 macc[EPT];
#pragma unroll
    for (int k = 0; k < EPT; ++k) macc[k] = make_float2(0.f, 0.f);
    const bool interior = (i >= 2 && i < P.ns - 2);
    const int j1 = min(P.nv, (c + 1) * P.jchunk);
    for (int j = c * P.jchunk; j < j1; ++j) {
      SlabCtx C;
      make_slab_ctx(P, I, j, C);
      const ST *yb = (const ST *)A.y + C.base;
      if constexpr (NL) {
        // L2 prefetch of what the epilogue will read from HBM for the first time (the slab j+2 of
        // the state, f_n and the accumulator of this slab): their latency hides behind the FFTs
        if (P.prefetch) {
          const int nline = (slab * (int)sizeof(ST) + 127) / 128;
          if (tid < nline) {
            const char *p0 = (const char *)(yb + C.ov[3]) + tid * 128;
            const char *p1 = (const char *)((const ST *)A.fn + C.base) + tid * 128;
            const char *p2 = (const char *)((const ST *)A.acc + C.base) + tid * 128;
            if (C.ov[3] != 0) asm volatile("prefetch.global.L2 [%0];" ::"l"(p0));
            if (A.mode == 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(p1));
            if (A.mode >= 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(p2));
          }
        }
        to_real([&](int e) { return Cv<ST>::ldg(yb, e); },
                [&](int r0) {
                  // bracket d_y chi d_x f - d_x chi d_y f, rows (p, p+rc/2) packed as (re, im), evaluated
                  // inside the first pass of the forward y-transform; only the retained ky are stored
                  auto keep = [&](int p, int nbase, auto offc, auto spanc, float2 v) {
                    constexpr int off = decltype(offc)::value, hi = off + decltype(spanc)::value - 1;
                    const int m = nbase + off;
                    if constexpr (SPEC && MY_ > 0 && off >= NKY_ && hi <= MY_ - NKY_) {
                    } else if constexpr (SPEC && MY_ > 0 && (hi < NKY_ || off > MY_ - NKY_)) {
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
                  // unpack the two real rows, keep only the retained ky: overwrite A's P columns
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
              if constexpr (SPEC && MX_ > 0 && (off > KC && hi < MX_ - KC)) {
              } else if constexpr (SPEC && MX_ > 0 && (hi <= KC || off >= MX_ - KC)) {
                SA[n * ldx + c] = v;
              } else {
                if (n <= K || n >= mx - K) SA[n * ldx + c] = v;
              }
            });
        __syncthreads();
      }

      // ---- epilogue: linear terms + bracket + RK update, one coalesced pass over the slab ----
      // The operands (own value, 4 parallel and 4 vpar neighbours, f_n, accumulator, chi, D_s chi)
      // are all requested before the arithmetic; the arithmetic is one packed-fp32 FMA per operand.
      EpiPtrs<ST> Q;
      make_epi_ptrs<ST>(A, C, chis, slab, Q);
      float fsum = 0.f;
      auto point = [&](auto modec, auto intc, int e, int ip, int m, float pk, float fmf) -> float2 {
        float2 nlv = make_float2(0.f, 0.f);
        if constexpr (NL) {
          const int n = (ip >= K) ? ip - K : mx + ip - K;
          nlv = SA[n * ldx + m];
        }
        return rhs_point<ST, decltype(modec)::value, decltype(intc)::value != 0>(
            P, A, I, C, Q, slab, e, ip, m, pk, fmf, nlv, scale * P.ef[i], fsum);
      };
      auto epilogue = [&](auto modec, auto intc) {
        if constexpr (ROWMAP) {
          constexpr int RS = NT / (NKY_ > 0 ? NKY_ : 1);  // kx rows per sweep of the CTA
          const int m = tid % nky, ip0 = tid / nky;
          const float fmf = (float)m, pk0 = (float)(ip0 - K);
#pragma unroll
          for (int k = 0; k < EPT; ++k) {
            const int e = tid + k * NT;
            if (k + 1 < EPT || e < slab) {
              const float2 out = point(modec, intc, e, ip0 + k * RS, m, pk0 + (float)(k * RS), fmf);
              macc[k] = cadd(macc[k], as_stored<ST>(out));   // what the next stage will read back
            }
          }
        } else {
          for (int e = tid; e < slab; e += nthr) {
            const int ip = e / nky, m = e - ip * nky;
            const float2 out = point(modec, intc, e, ip, m, (float)(ip - K), (float)m);
            if (A.mom) stage[NL ? (ip * ldx + m) : e] = as_stored<ST>(out);
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
        }
      };
      auto by_plane = [&](auto modec) {
        if (interior) epilogue(modec, gkfft::IC<1>{});
        else epilogue(modec, gkfft::IC<0>{});
      };
      switch (A.mode) {
        case 0: by_plane(gkfft::IC<0>{}); break;
        case 1: by_plane(gkfft::IC<1>{}); break;
        case 2: by_plane(gkfft::IC<2>{}); break;
        default: by_plane(gkfft::IC<3>{}); break;
      }
      if (want_flux) fx.slab(P, l, i, j, fsum);
      __syncthreads();  // A / stage are rewritten by the next slab
    }
    if (want_flux) fx.item_end(fslot);
    if (A.mom) {
      // moment plane of this item: Z n 2 pi w_v B_i w_mu J0 sum_j f   (a1 of the next stage)
      const float momw = P.sp[a].momfac * P.wmu[l] * P.B[i];
      const float *j0p = P.J0 + (((long long)a * P.nmu + l) * P.ns + i) * P.slab;
      float2 *dst = A.mom + (((long long)a * P.nmu + l) * P.nchunk + c) * P.nphi + (long long)i * P.slab;
#pragma unroll
      for (int k = 0; k < EPT; ++k) {
        const int e = tid + k * nthr;
        if (e < slab) dst[e] = gkfft::cscale(momw * __ldg(&j0p[e]), macc[k]);
      }
    }
  }
  if constexpr (NL) gm.flush(A.gmax);
  if (want_flux && (tid & 31) == 0) flux_flush(P, A.fluxp, blockIdx.x, NT / 32, tid >> 5, a_prev, fslot);
}

}  // namespace gk
