// gk_epilogue.cuh -- the streaming part of one RK stage (steps a4 + a6 of DESIGN.md and the velocity-space
// moment of the new state) on a SHARE of a (kx,ky) slab: kx rows [row0, row0+nrows) x all ky.  Used by the
// kernels whose threads have registers to spare for it (gk_stage_lin_kernel: term III off; gk_stage_ws4_kernel:
// the 4-CTA-cluster kernel of the largest grid).  Product path; shares nothing with oracle/.
//
// What differs from the epilogue role of gk_stage_ws2.cuh:
//  * 128-bit accesses: a thread owns PV adjacent ky (2 complex64 / 4 complex-half) of EPT kx rows, so every
//    operand of an interior plane moves as one LDG.128 / STG.128 ("strided addressing";
//    north_star "128-bit vectorised complex loads").  Only the four planes next to the s boundary, whose kx
//    connection shifts each ky by a different amount, fall back to one access per point.
//  * the vpar stencil (term IV + its dissipation) reads a REGISTER WINDOW: the thread marches
//    along vpar with y[j-2..j+1] of its points in registers and loads only y[j+2] per slab, so the state is
//    read once for the vpar direction instead of five times ("velocity-axis tiling ...
//    sequential streaming reads").  Values outside the vpar grid are zeros in the window (zero padding).
//  * where chi = J0 phi and D_s chi come from, where the bracket comes from and how a slab is handed over
//    between roles is left to a hook object H (see the two kernels).
#pragma once

namespace gk {

// ---- PV complex numbers of storage type ST per 128-bit access ----
template <class ST> struct Vec;
template <> struct Vec<float2> {
  static constexpr int PV = 2;
  static __device__ __forceinline__ void unpack(const float4 r, float2 (&v)[2]) {
    v[0] = make_float2(r.x, r.y); v[1] = make_float2(r.z, r.w);
  }
  static __device__ __forceinline__ void ldg(const float2 *p, float2 (&v)[2]) { unpack(__ldg((const float4 *)p), v); }
  static __device__ __forceinline__ void ldcs(const float2 *p, float2 (&v)[2]) { unpack(__ldcs((const float4 *)p), v); }
  static __device__ __forceinline__ void stcs(float2 *p, const float2 (&v)[2]) {
    __stcs((float4 *)p, make_float4(v[0].x, v[0].y, v[1].x, v[1].y));
  }
};
template <> struct Vec<__half2> {
  static constexpr int PV = 4;
  static __device__ __forceinline__ void unpack(const uint4 r, float2 (&v)[4]) {
    v[0] = __half22float2(*(const __half2 *)&r.x); v[1] = __half22float2(*(const __half2 *)&r.y);
    v[2] = __half22float2(*(const __half2 *)&r.z); v[3] = __half22float2(*(const __half2 *)&r.w);
  }
  static __device__ __forceinline__ void ldg(const __half2 *p, float2 (&v)[4]) { unpack(__ldg((const uint4 *)p), v); }
  static __device__ __forceinline__ void ldcs(const __half2 *p, float2 (&v)[4]) { unpack(__ldcs((const uint4 *)p), v); }
  static __device__ __forceinline__ void stcs(__half2 *p, const float2 (&v)[4]) {
    uint4 r;
    *(__half2 *)&r.x = __float22half2_rn(v[0]); *(__half2 *)&r.y = __float22half2_rn(v[1]);
    *(__half2 *)&r.z = __float22half2_rn(v[2]); *(__half2 *)&r.w = __float22half2_rn(v[3]);
    __stcs((uint4 *)p, r);
  }
};
template <> struct Vec<__nv_bfloat162> {
  static constexpr int PV = 4;
  static __device__ __forceinline__ void unpack(const uint4 r, float2 (&v)[4]) {
    v[0] = __bfloat1622float2(*(const __nv_bfloat162 *)&r.x); v[1] = __bfloat1622float2(*(const __nv_bfloat162 *)&r.y);
    v[2] = __bfloat1622float2(*(const __nv_bfloat162 *)&r.z); v[3] = __bfloat1622float2(*(const __nv_bfloat162 *)&r.w);
  }
  static __device__ __forceinline__ void ldg(const __nv_bfloat162 *p, float2 (&v)[4]) { unpack(__ldg((const uint4 *)p), v); }
  static __device__ __forceinline__ void ldcs(const __nv_bfloat162 *p, float2 (&v)[4]) { unpack(__ldcs((const uint4 *)p), v); }
  static __device__ __forceinline__ void stcs(__nv_bfloat162 *p, const float2 (&v)[4]) {
    uint4 r;
    *(__nv_bfloat162 *)&r.x = __float22bfloat162_rn(v[0]); *(__nv_bfloat162 *)&r.y = __float22bfloat162_rn(v[1]);
    *(__nv_bfloat162 *)&r.z = __float22bfloat162_rn(v[2]); *(__nv_bfloat162 *)&r.w = __float22bfloat162_rn(v[3]);
    __stcs((uint4 *)p, r);
  }
};
// layout of the slab-uniform coefficient block (floats)
#define GK_EB_WS 0     // [5] parallel stencil, interior class (centre: I + dissipation)
#define GK_EB_WO 5     // [5] parallel stencil at an open chain end of this plane (ghost weights 0)
#define GK_EB_WV 10    // [4] vpar stencil j-2, j-1, j+1, j+2 (zero padding folded in)
#define GK_EB_WVC 14   // vpar stencil centre
#define GK_EB_C7 15
#define GK_EB_A2 16
#define GK_EB_A5 17    // a5 * ky0
#define GK_EB_A8 18
#define GK_EB_N 20

// Slab-uniform coefficients of the linear terms of slab (a, j, l, i), by one thread.
__device__ __forceinline__ void epi_coefficients(const GkDev &P, int a, int l, int i, int j, float *eb) {
  const int mask = P.mask;
  const GkSpeciesDev &Sp = P.sp[a];
  const float vj = P.v[j];
  const int sg = (vj > 0.f) ? 0 : 1;
  const bool m2 = j >= 2, m1 = j >= 1, p1 = j + 1 < P.nv, p2 = j + 2 < P.nv;
  const float mul = P.mu[l], muB = mul * P.B[i];
  const float E = vj * vj + 2.f * muB, ED = vj * vj + muB;
  const float fm = P.fmv[j] * P.fmm[l * P.ns + i];
  const float cpar = Sp.vR * P.F[i] * vj;
  const float cmir = Sp.vR * mul * P.BG[i];
  const float cI = (mask & GK_T_I) ? -cpar * P.ds_inv : 0.f;
  const float cDs = (mask & GK_T_DISS_S) ? -P.nu_s * fabsf(cpar) * P.ds_inv : 0.f;
  const float c4 = (mask & GK_T_IV) ? cmir * P.dv_inv : 0.f;
  const float cDv = (mask & GK_T_DISS_V) ? -P.nu_v * fabsf(cmir) * P.dv_inv : 0.f;
  const int cls = i < 2 ? i : (i >= P.ns - 2 ? i - (P.ns - 3) + 2 : 2);
#pragma unroll
  for (int d = 0; d < 5; ++d) {
    eb[GK_EB_WS + d] = cI * P.dcoef[2][sg][d] + cDs * P.discoef[2][d];
    const int i2 = i + d - 2;
    const bool ghost = (i2 < 0) || (i2 >= P.ns);
    eb[GK_EB_WO + d] = ghost ? 0.f : cI * P.dcoef[cls][sg][d] + cDs * P.discoef[cls][d];
  }
  // D_v = (1,-8,0,8,-1)/12, delta^4_v/12 = (1,-4,6,-4,1)/12; ghosts outside the grid are zero
  const float k1 = 1.f / 12.f, k8 = 8.f / 12.f, k4 = 4.f / 12.f;
  eb[GK_EB_WV + 0] = m2 ? (c4 * k1 + cDv * k1) : 0.f;
  eb[GK_EB_WV + 1] = m1 ? (-c4 * k8 - cDv * k4) : 0.f;
  eb[GK_EB_WV + 2] = p1 ? (c4 * k8 - cDv * k4) : 0.f;
  eb[GK_EB_WV + 3] = p2 ? (-c4 * k1 + cDv * k1) : 0.f;
  eb[GK_EB_WVC] = cDv * 0.5f;
  eb[GK_EB_C7] = (mask & GK_T_VII) ? -Sp.ZoverT * cpar * fm * P.ds_inv : 0.f;
  eb[GK_EB_A2] = (mask & GK_T_II) ? Sp.ToverZ * ED : 0.f;
  eb[GK_EB_A5] = (mask & GK_T_V) ? 0.5f * P.ef[i] * fm * (Sp.rln + (E - 1.5f) * Sp.rlt) * P.ky0 : 0.f;
  eb[GK_EB_A8] = (mask & GK_T_VIII) ? ED * fm : 0.f;
}

// Thread-to-point map of a share: NTE threads, PV adjacent ky per thread, RS kx rows per sweep of the threads,
// EPT sweeps ("vector items") per thread.
template <class ST, int NKY_, int NTE, int ROWS> struct EpiMap {
  static constexpr int PV = Vec<ST>::PV;
  static constexpr int VPR = NKY_ / PV;               // vector items per kx row
  static_assert(NKY_ % PV == 0, "a 128-bit access stays inside a kx row");
  static_assert(NTE % VPR == 0, "a sweep of the threads covers whole kx rows");
  static constexpr int RS = NTE / VPR;                // kx rows per sweep
  static constexpr int EPT = (ROWS + RS - 1) / RS;    // vector items per thread
  static constexpr int KS = RS * NKY_;                // slab elements between a thread's items
};

// One work item of the streaming role: share (row0, nrows) of the slabs (a, j0..j1-1, l, i).
// H supplies
//   static constexpr bool NL          a bracket is added (term III)
//   float *coef(int u, int et)        the coefficient block this thread reads for slab u
//   bool   makes_coef(int et)         this thread computes it
//   void   begin(int u), end(int u)   hand-over of slab u (barriers); begin() also publishes the coefficient block
//   void   chi(int k, int el, int sg, float2 (&chi)[PV], float2 (&dsc)[PV])   el: index inside the share
//   void   nl(int u, int e, float2 (&v)[PV])                                   e: index inside the slab
//   float2 *macc(int k)               PV moment accumulators of the thread's item k (shared memory, thread-private)
//   static constexpr bool FLUX        the flux diagnostics are folded into this role (else the host runs gk_flux_kernel)
//   double *fluxslot()                3 doubles of the thread's warp in shared memory (flux diagnostics, FluxAcc)
// u counts the slabs this CTA has processed since the start of the launch (ring slots).
template <class ST, int NKY_, int NKX_, int NTE, int ROWS, int NB, class H>
__device__ __forceinline__ void epi_item(const GkDev &P, const GkStageArgs &A, H &h, const int et, const int a,
                                         const int l, const int i, const int c, const int row0, const int nrows,
                                         int &u) {
  using M = EpiMap<ST, NKY_, NTE, ROWS>;
  constexpr int nky = NKY_, nkx = NKX_, K = (nkx - 1) / 2, slab = nkx * nky;
  constexpr int PV = M::PV, RS = M::RS, EPT = M::EPT, KS = M::KS;
  constexpr bool NL = H::NL;
  const int m0 = (et % M::VPR) * PV, r0 = et / M::VPR;
  // a thread whose first row lies beyond a short share (r0 >= nrows: it has no valid item at all) addresses row 0 of
  // the share instead: every address it forms stays inside the slab, and nothing it computes is stored
  const int r0a = r0 < nrows ? r0 : 0;
  const int el0 = r0a * nky + m0;             // index of item 0 inside the share
  const int e0 = row0 * nky + el0;            // ... inside the slab
  const int ip0 = row0 + r0a;                 // kx row of item 0
  const float scale = 0.25f * P.ef[i] * P.fftnorm;      // ef/2 (bracket) * 1/2 (two-for-one unpack) / (mx my)
  const long long jstride = (long long)P.nmu * P.ns * P.slab;
  const int js = (int)jstride;
  const long long base0 = (((long long)a * P.nv * P.nmu + l) * P.ns + i) * P.slab + e0;
  const int mask = P.mask;
  const float ksx = P.dkx * P.sth[i], kcz = P.ky0 * P.cz[i];
  const float hx4 = (mask & GK_T_HYP) ? P.hyp_x * (P.invK * P.invK) * (P.invK * P.invK) : 0.f;
  const float hy4 = (mask & GK_T_HYP) ? P.hyp_y * (P.invM * P.invM) * (P.invM * P.invM) : 0.f;
  // parallel neighbours of this plane: uniform element offset + (wrap * kx shift of the ky) per point
  const bool lowp = i < 2, seam = (i < 2) || (i >= P.ns - 2);
  const int j0 = c * P.jchunk, j1 = min(P.nv, (c + 1) * P.jchunk);

  // ---- register window along vpar; the moment accumulators live in thread-private shared-memory slots ----
  float2 win[EPT][4][PV];
  const bool want_flux = H::FLUX && A.fluxp != nullptr && A.mode == 1;
  FluxAcc fx;
  const ST *y0 = (const ST *)A.y + base0;
#pragma unroll
  for (int k = 0; k < EPT; ++k) {
#pragma unroll
    for (int v = 0; v < PV; v += 2) *(float4 *)(h.macc(k) + v) = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      const int jj = j0 - 2 + t;
#pragma unroll
      for (int v = 0; v < PV; ++v) win[k][t][v] = make_float2(0.f, 0.f);
      // (rows beyond the share repeat item 0: every thread runs the same straight-line code, only stores are predicated)
      if (jj >= 0 && jj < P.nv) Vec<ST>::ldg(y0 + (long long)jj * jstride + (r0 + k * RS < nrows ? k * KS : 0), win[k][t]);
    }
  }

  for (int j = j0; j < j1; ++j, ++u) {
    const int sg = (P.v[j] > 0.f) ? 0 : 1;
    const bool p2 = j + 2 < P.nv;
    float *eb = h.coef(u, et);
    if (h.makes_coef(et)) epi_coefficients(P, a, l, i, j, eb);
    const ST *yp = y0 + (long long)j * jstride;
    const ST *fnp = (const ST *)A.fn + base0 + (long long)j * jstride;
    ST *accp = (ST *)A.acc + base0 + (long long)j * jstride;
    ST *outp = (ST *)A.out + base0 + (long long)j * jstride;
    // L2 prefetch of the single-use operands of the NEXT slab (y[j+3], f_n and the accumulator of slab j+1)
    if (P.prefetch && j + 1 < j1) {
#pragma unroll
      for (int k = 0; k < EPT; ++k) {
        if (r0 + k * RS < nrows && (m0 * (int)sizeof(ST)) % 128 == 0) {
          if (j + 3 < P.nv) asm volatile("prefetch.global.L2 [%0];" ::"l"(yp + 3 * js + k * KS));
          if (A.mode == 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(fnp + js + k * KS));
          if (A.mode >= 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(accp + js + k * KS));
        }
      }
    }
    h.begin(u);
    float fsum = 0.f;     // flux diagnostics: sum of 2 m Im[conj(chi) f] over the thread's points of this slab
    auto sweep = [&](auto modec, auto seamc) {
      constexpr int MODE = decltype(modec)::value;
      constexpr bool SEAM = decltype(seamc)::value != 0;
#pragma unroll
      for (int k0 = 0; k0 < EPT; k0 += NB) {
        float2 yn[NB][PV], fs[NB][4][PV], fn[NB][PV], ac[NB][PV], chi0[NB][PV], dschi[NB][PV];
        bool open[NB][PV];
        // all loads of the batch are requested before its arithmetic
#pragma unroll
        for (int q = 0; q < NB; ++q) {
          const int k = k0 + q;
#pragma unroll
          for (int v = 0; v < PV; ++v) {
            open[q][v] = false;
            yn[q][v] = make_float2(0.f, 0.f);
            ac[q][v] = make_float2(0.f, 0.f);
          }
          if (k < EPT) {
            const int eo = (r0 + k * RS < nrows) ? k * KS : 0;
            if (p2) Vec<ST>::ldg(yp + 2 * js + eo, yn[q]);
            if constexpr (!SEAM) {
              Vec<ST>::ldg(yp + eo - 2 * slab, fs[q][0]);
              Vec<ST>::ldg(yp + eo - slab, fs[q][1]);
              Vec<ST>::ldg(yp + eo + slab, fs[q][2]);
              Vec<ST>::ldg(yp + eo + 2 * slab, fs[q][3]);
            } else {
              const int ip = ip0 + k * RS;
#pragma unroll
              for (int v = 0; v < PV; ++v) {
                const int m = m0 + v, mk = m * P.ikx;
                open[q][v] = lowp ? (ip < mk) : (ip + mk > nkx - 1);
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                  const int d = s < 2 ? s - 2 : s - 1;
                  int i2 = i + d, wrap = 0;
                  if (i2 >= P.ns) { i2 -= P.ns; wrap = 1; }
                  else if (i2 < 0) { i2 += P.ns; wrap = -1; }
                  // the kx connection shifts ky index m by m * ikxspace rows across the s boundary; neighbours
                  // beyond an open end carry weight 0: any valid address will do
                  const bool beyond = open[q][v] && wrap != 0;
                  const int off = beyond ? 0 : (i2 - i) * slab + wrap * mk * nky;
                  fs[q][s][v] = Cv<ST>::ldg(yp, eo + v + off);
                }
              }
            }
            if constexpr (MODE == 2) Vec<ST>::ldcs(fnp + eo, fn[q]);
            if constexpr (MODE >= 2) Vec<ST>::ldcs(accp + eo, ac[q]);
            h.chi(k, el0 + eo, sg, chi0[q], dschi[q]);
          }
        }
        asm volatile("" ::: "memory");      // coefficient loads stay behind the operand loads
#pragma unroll
        for (int q = 0; q < NB; ++q) {
          const int k = k0 + q;
          if (k < EPT) {
            const bool valid = r0 + k * RS < nrows;
            const int eo = valid ? k * KS : 0;
            const float pk = (float)(ip0 + k * RS - K);
            const float pk2 = pk * pk;
            const float4 *eb4 = (const float4 *)eb;
            const float4 wa0 = eb4[0];                     // ws0..ws3
            const float4 wb0 = eb4[1];                     // ws4, wo0..wo2
            const float4 wc = eb4[2], wd = eb4[3], we = eb4[4];  // wo3 wo4 wv0 wv1 | wv2 wv3 wvc c7 | a2 a5 a8 -
            float2 rr[PV], f0[PV];
#pragma unroll
            for (int v = 0; v < PV; ++v) {
              float4 wa = wa0;
              float wb = wb0.x;
              if constexpr (SEAM) {
                if (open[q][v]) { wa = make_float4(wb0.y, wb0.z, wb0.w, wc.x); wb = wc.y; }
              }
              const float fmf = (float)(m0 + v), fm2 = fmf * fmf;
              const float kap = -(pk * ksx + fmf * kcz);
              f0[v] = win[k][2][v];
              float2 r = gkfft::cscale(wa.x, fs[q][0][v]);
              r = gkfft::caxpy(wa.y, fs[q][1][v], r);
              r = gkfft::caxpy(wa.w, fs[q][2][v], r);
              r = gkfft::caxpy(wb, fs[q][3][v], r);
              r = gkfft::caxpy(wa.z + wd.z - (hx4 * (pk2 * pk2) + hy4 * (fm2 * fm2)), f0[v], r);
              r = gkfft::caxpy(wc.z, win[k][0][v], r);
              r = gkfft::caxpy(wc.w, win[k][1][v], r);
              r = gkfft::caxpy(wd.x, win[k][3][v], r);
              r = gkfft::caxpy(wd.y, yn[q][v], r);
              r = gkfft::caxpy(wd.w, dschi[q][v], r);
              // -i a z = a (z.y, -z.x)
              r = gkfft::caxpy(we.x * kap, make_float2(f0[v].y, -f0[v].x), r);
              r = gkfft::caxpy(we.y * fmf + we.z * kap, make_float2(chi0[q][v].y, -chi0[q][v].x), r);
              rr[v] = r;
              if constexpr (MODE == 1 && H::FLUX) {
                if (valid) fsum = fmaf(2.f * fmf, chi0[q][v].x * f0[v].y - chi0[q][v].y * f0[v].x, fsum);
              }
              // the window moves on by one slab
              win[k][0][v] = win[k][1][v];
              win[k][1][v] = f0[v];
              win[k][2][v] = win[k][3][v];
              win[k][3][v] = yn[q][v];
            }
            if constexpr (NL) {
              // the bracket is fetched only now: its CL partial sums are many registers in flight, and the
              // linear operands above are dead by this point
              float2 nlv[PV];
              h.nl(u, e0 + eo, nlv);
#pragma unroll
              for (int v = 0; v < PV; ++v) rr[v] = gkfft::caxpy(scale, nlv[v], rr[v]);
            }
            float2 outv[PV], accv[PV];
#pragma unroll
            for (int v = 0; v < PV; ++v) {
              if constexpr (MODE == 0) {
                outv[v] = rr[v];
              } else if constexpr (MODE == 1) {
                accv[v] = gkfft::caxpy(A.b, rr[v], f0[v]);
                outv[v] = gkfft::caxpy(A.c, rr[v], f0[v]);
              } else if constexpr (MODE == 2) {
                accv[v] = gkfft::caxpy(A.b, rr[v], ac[q][v]);
                outv[v] = gkfft::caxpy(A.c, rr[v], fn[q][v]);
              } else {
                outv[v] = gkfft::caxpy(A.b, rr[v], ac[q][v]);
              }
            }
            if (valid) {
              if constexpr (MODE == 1 || MODE == 2) Vec<ST>::stcs(accp + eo, accv);
              Vec<ST>::stcs(outp + eo, outv);
            }
            if (A.mom) {   // moment of what the next stage will read back
              float4 *ma = (float4 *)h.macc(k);
#pragma unroll
              for (int v = 0; v < PV; v += 2) {
                const float2 o0 = as_stored<ST>(outv[v]), o1 = as_stored<ST>(outv[v + 1]);
                float4 t = ma[v / 2];
                t.x += o0.x; t.y += o0.y; t.z += o1.x; t.w += o1.y;
                ma[v / 2] = t;
              }
            }
          }
        }
        asm volatile("" ::: "memory");      // the next batch's loads stay below this one's arithmetic
      }
    };
    auto by_plane = [&](auto modec) {
      if (seam) sweep(modec, gkfft::IC<1>{});
      else sweep(modec, gkfft::IC<0>{});
    };
    switch (A.mode) {
      case 0: by_plane(gkfft::IC<0>{}); break;
      case 1: by_plane(gkfft::IC<1>{}); break;
      case 2: by_plane(gkfft::IC<2>{}); break;
      default: by_plane(gkfft::IC<3>{}); break;
    }
    if constexpr (H::FLUX) { if (want_flux) fx.slab(P, l, i, j, fsum); }
    h.end(u);
  }
  if constexpr (H::FLUX) { if (want_flux) fx.item_end(h.fluxslot()); }
  if (A.mom) {
    // moment plane of this item: Z n 2 pi w_v B_i w_mu J0 sum_j f   (a1 of the next stage)
    const float momw = P.sp[a].momfac * P.wmu[l] * P.B[i];
    const float *j0p = P.J0 + (((long long)a * P.nmu + l) * P.ns + i) * P.slab + e0;
    float2 *dst = A.mom + (((long long)a * P.nmu + l) * P.nchunk + c) * P.nphi + (long long)i * P.slab + e0;
#pragma unroll
    for (int k = 0; k < EPT; ++k) {
      if (r0 + k * RS < nrows) {
#pragma unroll
        for (int v = 0; v < PV; v += 2) {
          const float4 t = *(const float4 *)(h.macc(k) + v);
          const float w0 = momw * __ldg(&j0p[k * KS + v]), w1 = momw * __ldg(&j0p[k * KS + v + 1]);
          *(float4 *)(dst + k * KS + v) = make_float4(w0 * t.x, w0 * t.y, w1 * t.z, w1 * t.w);
        }
      }
    }
  }
}

// chi = J0 phi and its parallel derivative for both streaming directions (term VII) at the thread's own points
// of a share, handed to store(k, which, values): which = 0 chi, 1 D_s chi (v > 0), 2 D_s chi (v < 0)
template <class ST, int NKY_, int NTE, int ROWS, class STORE>
__device__ __forceinline__ void epi_build_chis(const GkDev &P, const GkStageArgs &A, int a, int l, int i, int row0,
                                               int nrows, int et, STORE store) {
  using M = EpiMap<ST, NKY_, NTE, ROWS>;
  constexpr int PV = M::PV, RS = M::RS, EPT = M::EPT, nky = NKY_;
  const int m0 = (et % M::VPR) * PV, r0 = et / M::VPR;
  const long long jb = (((long long)a * P.nmu + l) * P.ns + i) * P.slab;
  const float2 *ph = A.phi + (long long)i * P.slab;
#pragma unroll
  for (int k = 0; k < EPT; ++k) {
    if (r0 + k * RS >= nrows) continue;
    const int ip = row0 + r0 + k * RS;
    float2 c0[PV], dp[PV], dn[PV];
#pragma unroll
    for (int v = 0; v < PV; ++v) {
      const int m = m0 + v, e = ip * nky + m;
      const int cls = stencil_class(P, i, ip, m);
      c0[v] = make_float2(0.f, 0.f); dp[v] = c0[v]; dn[v] = c0[v];
#pragma unroll
      for (int d = 0; d < 5; ++d) {
        int off;
        if (!seam_offset(P, i, d - 2, ip, m, off)) continue;
        const float j0 = __ldg(&P.J0[jb + e + off]);
        const float2 ph0 = __ldg(&ph[e + off]);
        const float2 ch = make_float2(j0 * ph0.x, j0 * ph0.y);
        if (d == 2) c0[v] = ch;
        dp[v].x += P.dcoef[cls][0][d] * ch.x; dp[v].y += P.dcoef[cls][0][d] * ch.y;
        dn[v].x += P.dcoef[cls][1][d] * ch.x; dn[v].y += P.dcoef[cls][1][d] * ch.y;
      }
    }
    store(k, 0, c0);
    store(k, 1, dp);
    store(k, 2, dn);
  }
}

// =================================================================================================
// Term III switched off: every thread of the CTA runs the streaming role (stencils + RK update + moment).
// A work item is (species, mu, vpar chunk, share of the slab, s); warps march along vpar on their own: a thread
// reads chi / D_s chi only at its own points (shared memory, written by itself), so no CTA-wide barrier exists.
// NSH shares per slab keep the register window of a thread small on large (kx,ky) planes.
template <class ST, int NKY_, int NKX_, int NT, int NSH, int NB>
struct LinHooks {
  static constexpr bool NL = false;
  static constexpr bool FLUX = false;   // 168 registers per thread are all taken: fluxes through gk_flux_kernel
  using M = EpiMap<ST, NKY_, NT, (NKX_ + NSH - 1) / NSH>;
  float2 *chis;   // [4][EPT][NT][PV] shared memory: chi, D_s chi (v > 0), D_s chi (v < 0), moment accumulators
  float *eblk;    // [NT/32][GK_EB_N]
  int et;
  __device__ __forceinline__ double *fluxslot() const { return nullptr; }
  __device__ __forceinline__ float *coef(int, int t) const { return eblk + (t >> 5) * GK_EB_N; }
  __device__ __forceinline__ bool makes_coef(int t) const {
    __syncwarp();                  // the warp has finished reading the previous slab's block
    return (t & 31) == 0;
  }
  __device__ __forceinline__ void begin(int) const { __syncwarp(); }
  __device__ __forceinline__ void end(int) const {}
  __device__ __forceinline__ float2 *slot(int which, int k) const {
    return chis + ((size_t)(which * M::EPT + k) * NT + et) * M::PV;
  }
  __device__ __forceinline__ void chi(int k, int, int sg, float2 (&c)[M::PV], float2 (&d)[M::PV]) const {
    const float4 *pc = (const float4 *)slot(0, k), *pd = (const float4 *)slot(1 + sg, k);
#pragma unroll
    for (int v = 0; v < M::PV; v += 2) {
      const float4 x = pc[v / 2], y = pd[v / 2];
      c[v] = make_float2(x.x, x.y); c[v + 1] = make_float2(x.z, x.w);
      d[v] = make_float2(y.x, y.y); d[v + 1] = make_float2(y.z, y.w);
    }
  }
  __device__ __forceinline__ void nl(int, int, float2 (&)[M::PV]) const {}
  __device__ __forceinline__ float2 *macc(int k) const { return slot(3, k); }
};

template <class ST, int NKY_, int NKX_, int NT, int NSH>
constexpr size_t lin_smem_bytes() {
  using M = EpiMap<ST, NKY_, NT, (NKX_ + NSH - 1) / NSH>;
  return (size_t)4 * M::EPT * NT * M::PV * 8;
}

template <class ST, int NKY_, int NKX_, int NT, int NSH, int NB>
__global__ void __launch_bounds__(NT, 1)
gk_stage_lin_kernel(const __grid_constant__ GkDev P, const __grid_constant__ GkStageArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(16) float eblk[(NT / 32) * GK_EB_N];
  constexpr int ROWS = (NKX_ + NSH - 1) / NSH;
  using HK = LinHooks<ST, NKY_, NKX_, NT, NSH, NB>;
  HK h{(float2 *)smem_raw, eblk, (int)threadIdx.x};
  const int et = threadIdx.x;
  int u = 0;
  for (int w = blockIdx.x; w < A.nwork; w += gridDim.x) {
    const int i = w % P.ns;
    const int sh = (w / P.ns) % NSH;
    const int c = (w / (P.ns * NSH)) % P.nchunk;
    const int al = w / (P.ns * NSH * P.nchunk);
    const int l = al % P.nmu, a = al / P.nmu;
    const int row0 = sh * ROWS, nrows = min(ROWS, NKX_ - row0);
    epi_build_chis<ST, NKY_, NT, ROWS>(P, A, a, l, i, row0, nrows, et, [&](int k, int which, const float2 (&v)[HK::M::PV]) {
      float4 *p = (float4 *)h.slot(which, k);
#pragma unroll
      for (int q = 0; q < HK::M::PV; q += 2) p[q / 2] = make_float4(v[q].x, v[q].y, v[q + 1].x, v[q + 1].y);
    });
    epi_item<ST, NKY_, NKX_, NT, ROWS, NB>(P, A, h, et, a, l, i, c, row0, nrows, u);
  }
}

}  // namespace gk
