// gk_stage_ws2.cuh -- second warp-specialised form of the fused RK-stage kernel (steps a3-a6 of
// DESIGN.md) for the shapes whose padded field fits shared memory twice.  Product path; shares
// nothing with oracle/.
//
// FFT role: the whole bracket (term III) of a slab runs IN PLACE in one array S[mx][my] (row stride
// LD odd: lane = row and lane = column passes are both conflict-free):
//   columns 0..nky-1        P(m)  = Fx[(i kx - ky) g](x, m)
//   columns my-nky+1..my-1  Q(m') = Fx[(i kx + ky) g](x, m') stored at column my - m', i.e. where
//                           the Hermitian extension of the row needs conj Q(m')
// so the y transforms need no row assembly and no workspace, all passes span the whole slab
// (7 named barriers per slab, no row chunks) and every item map has compile-time divisors:
//   X1  inverse x pass 1   slab (staged by one bulk async copy) -> S, zero padding never loaded
//   X2  inverse x pass 2   in place
//   Y1  inverse y pass 1   in place, only the 2 nky - 1 non-zero inputs of a row are read
//   YF  inverse y pass 2 + pointwise bracket with grad(chi) (SG[mx][my], built once per
//       (species, mu, s)) + two real rows packed into one complex row + forward y pass 1,
//       all in registers
//   F2  forward y pass 2   only the retained ky are stored
//   XF1 forward x pass 1   the two-for-one unpack (Z(m), conj Z(my-m)) is done in its loads;
//                          output to the dead columns nky..2nky-1
//   XF2 forward x pass 2   retained kx -> the bracket ring in L2 for the epilogue role
// Twiddles come from compile-time tables in constant memory (warp-uniform indices).
// Epilogue role: ws_epilogue_role2 below.
#pragma once

namespace gk {

// Twiddle tables of the two-pass transforms N = R1 R2 in constant memory (compile-time initialised; warp-uniform
// indices, so the loads go through the constant cache and not through the shared-memory/L1 data pipe that bounds
// the kernel):  a[n1 R2 + k2] = b[k2 R1 + n1] = exp(+2 pi i n1 k2 / N)
template <int N> struct TwTab { float2 a[N]; float2 b[N]; };
template <int N> constexpr TwTab<N> make_tw() {
  TwTab<N> t{};
  constexpr int R1 = gkfft::Fac<N>::R1, R2 = gkfft::Fac<N>::R2;
  for (int n1 = 0; n1 < R1; ++n1)
    for (int k2 = 0; k2 < R2; ++k2) {
      const int k = (n1 * k2) % N;
      const double ang = 2.0 * gkfft::kPi * (k > N / 2 ? k - N : k) / N;
      const float c = (float)gkfft::cx_cos(ang), sn = (float)gkfft::cx_sin(ang);
      t.a[n1 * R2 + k2].x = c; t.a[n1 * R2 + k2].y = sn;
      t.b[k2 * R1 + n1].x = c; t.b[k2 * R1 + n1].y = sn;
    }
  return t;
}
static __constant__ TwTab<128> c_tw128 = make_tw<128>();
static __constant__ TwTab<96> c_tw96 = make_tw<96>();
static __constant__ TwTab<48> c_tw48 = make_tw<48>();
static __constant__ TwTab<192> c_tw192 = make_tw<192>();
template <int N> __device__ __forceinline__ const TwTab<N> &tw_tab() {
  if constexpr (N == 128) return c_tw128;
  else if constexpr (N == 192) return c_tw192;
  else if constexpr (N == 96) return c_tw96;
  else { static_assert(N == 48, "no twiddle table for this length"); return c_tw48; }
}

// u[k] *= T[k] (S > 0) or conj T[k] (S < 0), k = 1..R-1
template <int R, int S>
__device__ __forceinline__ void twiddle_row(float2 (&u)[R], const float2 *T) {
#pragma unroll
  for (int k = 1; k < R; ++k) {
    const float2 t = T[k];
    u[k] = S > 0 ? gkfft::cmul(u[k], t) : gkfft::cmulc(u[k], t);
  }
}

// shared-memory bytes of the kernel below
template <class ST, int MX_, int MY_, int NKY_, int NKX_>
constexpr size_t ws2_smem_bytes() {
  return (size_t)(2 * MX_ * (MY_ | 1)) * 8 + (size_t)NKX_ * NKY_ * sizeof(ST) + 16 + 2 * GK_EB_N * 4;
}

// ---- lean epilogue role ------------------------------------------------------------------------
// The slab-uniform coefficients of the linear terms are computed once per slab by one thread and
// kept in a small shared block (2-slot ring); every point then needs 14 operands and one packed FMA
// per operand.  Parallel-stencil planes next to the s boundary run the same branch-free code with
// the kx connection folded into one per-thread offset (R6) and one predicate per point
// (open chain end: PAPER.md:350, 362; R7).  The velocity-space moment of the new state is accumulated
// in registers over the vpar march (one float2 per point of the thread).
template <class ST, int NKY_, int NKX_, int NTF, int NTE, int NB>
__device__ __forceinline__ void ws_epilogue_role2(const GkDev &P, const GkStageArgs &A, float2 *chis_cta,
                                                  const float2 *nl_cta, float *eblk, double *fslots, int tid) {
  constexpr int NT = NTF + NTE;
  constexpr int nky = NKY_, nkx = NKX_;
  constexpr int K = (nkx - 1) / 2, slab = nkx * nky;
  constexpr int BAR_FULL = GK_WS_BAR_FULL, BAR_FREE = GK_WS_BAR_FREE;
  static_assert(NTE % NKY_ == 0, "an epilogue sweep covers whole ky rows");
  const int et = tid - NTF;
  constexpr int EPT = (slab + NTE - 1) / NTE;
  constexpr int RS = NTE / nky;  // kx rows per sweep of the role's threads
  const int m = et % nky, ip0 = et / nky;
  const float fmf = (float)m, pk0 = (float)(ip0 - K);
  const int mk = m * P.ikx;      // kx shift of this ky across the s boundary
  const float scale = 0.25f * P.fftnorm;  // 1/2 (bracket) * 1/2 (two-for-one unpack) / (mx my)
  const long long jstride = (long long)P.nmu * P.ns * P.slab;
  const float fm2 = fmf * fmf;
  // flux diagnostics of the state a stage-1 launch reads (FluxAcc, gk_common.cuh)
  const bool want_flux = A.fluxp != nullptr && A.mode == 1;
  double *fslot = fslots + (et >> 5) * 3;
  if ((et & 31) == 0) fslot[0] = fslot[1] = fslot[2] = 0.0;
  FluxAcc fx;
  int u = 0, it = 0, a_prev = -1;
  for (int w = blockIdx.x; w < A.nwork; w += gridDim.x, ++it) {
    const int i = w % P.ns;
    const int c = (w / P.ns) % P.nchunk;
    const int al = w / (P.ns * P.nchunk);
    const int l = al % P.nmu, a = al / P.nmu;
    if (want_flux && a != a_prev) {
      if ((et & 31) == 0) flux_flush(P, A.fluxp, blockIdx.x, NTE / 32, et >> 5, a_prev, fslot);
      a_prev = a;
    }
    const long long base0 = (((long long)a * P.nv * P.nmu + l) * P.ns + i) * P.slab;
    const float2 *chip = chis_cta + (it % GK_WS_CHI_RING) * 3 * slab + et;
    // per item: kappa = -(pk ksx + m kcz), hyper-viscosity hx4 (p/K)^4 + hy4 (m/(nky-1))^4
    const int mask = P.mask;
    const float ksx = P.dkx * P.sth[i], kcz = P.ky0 * P.cz[i];
    const float hx4 = (mask & GK_T_HYP) ? P.hyp_x * (P.invK * P.invK) * (P.invK * P.invK) : 0.f;
    const float hyp_m = (mask & GK_T_HYP) ? P.hyp_y * (P.invM * P.invM) * (P.invM * P.invM) * (fm2 * fm2) : 0.f;
    const float kap_m = fmf * kcz;
    const float scale_i = scale * P.ef[i];   // ExB factor of this plane
    // parallel neighbours of this plane: uniform element offset + (wrap * kx shift) per thread
    const bool lowp = i < 2, seam = (i < 2) || (i >= P.ns - 2);
    int soff[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int d = q < 2 ? q - 2 : q - 1;
      int i2 = i + d, wrap = 0;
      if (i2 >= P.ns) { i2 -= P.ns; wrap = 1; }
      else if (i2 < 0) { i2 += P.ns; wrap = -1; }
      soff[q] = (i2 - i) * slab + wrap * mk * nky;
    }
    float2 macc[EPT];
#pragma unroll
    for (int k = 0; k < EPT; ++k) macc[k] = make_float2(0.f, 0.f);
    const int j0 = c * P.jchunk, j1 = min(P.nv, (c + 1) * P.jchunk);
    for (int j = j0; j < j1; ++j, ++u) {
      // coefficient block: one per slab parity, published by BAR_FULL
      float *eb = eblk + (u & 1) * GK_EB_N;
      const bool m2 = j >= 2, m1 = j >= 1, p1 = j + 1 < P.nv, p2 = j + 2 < P.nv;
      const int sg = (P.v[j] > 0.f) ? 0 : 1;
      if (et == 0) epi_coefficients(P, a, l, i, j, eb);
      const long long sb = base0 + (long long)j * jstride;
      const ST *yp = (const ST *)A.y + sb + et;
      const ST *fnp = (const ST *)A.fn + sb + et;
      ST *accp = (ST *)A.acc + sb + et;
      ST *outp = (ST *)A.out + sb + et;
      const int js = (int)jstride;  // vpar neighbours as element offsets (outside the grid: weight 0, own address)
      const int ov0 = m2 ? -2 * js : 0, ov1 = m1 ? -js : 0, ov3 = p1 ? js : 0, ov4 = p2 ? 2 * js : 0;
      // L2 prefetch of what the NEXT slab reads from HBM for the first time (slab j+3 of the
      // state, f_n and the accumulator of slab j+1)
      if (P.prefetch && j + 1 < j1) {
        constexpr int nline = (slab * (int)sizeof(ST) + 127) / 128;
        for (int t = et; t < nline; t += NTE) {
          const long long nb = sb + jstride;
          if (j + 3 < P.nv) asm volatile("prefetch.global.L2 [%0];" ::"l"((const char *)((const ST *)A.y + sb + 3 * jstride) + t * 128));
          if (A.mode == 2) asm volatile("prefetch.global.L2 [%0];" ::"l"((const char *)((const ST *)A.fn + nb) + t * 128));
          if (A.mode >= 2) asm volatile("prefetch.global.L2 [%0];" ::"l"((const char *)((const ST *)A.acc + nb) + t * 128));
        }
      }
      const float2 *nlr = nl_cta + (u & 1) * slab + et;
      const float2 *dsp = chip + (1 + sg) * slab;
      bar_sync_n(BAR_FULL + (u & 1), NT);   // also publishes eb to the role's other threads
      float fsum = 0.f;
      auto sweep = [&](auto modec, auto seamc) {
        constexpr int MODE = decltype(modec)::value;
        constexpr bool SEAM = decltype(seamc)::value != 0;
        // NB points per thread are in flight at once (14 operands each): the loads of a batch are all
        // requested before its arithmetic, and batches do not overlap (register budget)
#pragma unroll
        for (int k0 = 0; k0 < EPT; k0 += NB) {
          float2 f0[NB], fs0[NB], fs1[NB], fs3[NB], fs4[NB], fv0[NB], fv1[NB], fv3[NB], fv4[NB], fn[NB], ac[NB], chi0[NB], dschi[NB], nlv[NB];
          bool open[NB];
#pragma unroll
          for (int q = 0; q < NB; ++q) {
            const int k = k0 + q, eo = k * NTE;
            open[q] = false;
            if (k < EPT && (k + 1 < EPT || et + eo < slab)) {
              const int ip = ip0 + k * RS;
              int o0 = -2 * slab, o1 = -slab, o3 = slab, o4 = 2 * slab;
              if constexpr (SEAM) {
                open[q] = lowp ? (ip < mk) : (ip + mk > nkx - 1);
                o0 = soff[0]; o1 = soff[1]; o3 = soff[2]; o4 = soff[3];
                if (open[q]) {  // neighbours beyond the open end carry weight 0: any valid address will do
                  if (lowp) { if (i - 2 < 0) o0 = 0; if (i - 1 < 0) o1 = 0; }
                  else { if (i + 1 >= P.ns) o3 = 0; if (i + 2 >= P.ns) o4 = 0; }
                }
              }
              f0[q] = Cv<ST>::ldg(yp, eo);
              fs0[q] = Cv<ST>::ldg(yp, eo + o0); fs1[q] = Cv<ST>::ldg(yp, eo + o1);
              fs3[q] = Cv<ST>::ldg(yp, eo + o3); fs4[q] = Cv<ST>::ldg(yp, eo + o4);
              fv0[q] = Cv<ST>::ldg(yp, eo + ov0); fv1[q] = Cv<ST>::ldg(yp, eo + ov1);
              fv3[q] = Cv<ST>::ldg(yp, eo + ov3); fv4[q] = Cv<ST>::ldg(yp, eo + ov4);
              fn[q] = f0[q]; ac[q] = make_float2(0.f, 0.f);
              if constexpr (MODE == 2) fn[q] = Cv<ST>::ldcs(fnp, eo);
              if constexpr (MODE >= 2) ac[q] = Cv<ST>::ldcs(accp, eo);
              chi0[q] = __ldcg(chip + eo);    // written by this CTA earlier in the launch: L2, not the
              dschi[q] = __ldcg(dsp + eo);    // read-only path
              nlv[q] = __ldcg(nlr + eo);
            }
          }
          asm volatile("" ::: "memory");      // coefficient loads stay behind the operand loads
#pragma unroll
          for (int q = 0; q < NB; ++q) {
            const int k = k0 + q, eo = k * NTE;
            if (k < EPT && (k + 1 < EPT || et + eo < slab)) {
              const float pk = pk0 + (float)(k * RS);
              const float4 *eb4 = (const float4 *)eb;
              float4 wa = eb4[0];                      // ws0..ws3
              float4 wb = eb4[1];                      // ws4, wo0..wo2
              const float4 wc = eb4[2], wd = eb4[3], we = eb4[4];  // wo3 wo4 wv0 wv1 | wv2 wv3 wvc c7 | a2 a5 a8 -
              if constexpr (SEAM) {
                if (open[q]) { wa = make_float4(wb.y, wb.z, wb.w, wc.x); wb.x = wc.y; }
              }
              const float kap = -(pk * ksx + kap_m);
              const float pk2 = pk * pk;
              float2 r = gkfft::cscale(wa.x, fs0[q]);
              r = gkfft::caxpy(wa.y, fs1[q], r);
              r = gkfft::caxpy(wa.w, fs3[q], r);
              r = gkfft::caxpy(wb.x, fs4[q], r);
              r = gkfft::caxpy(wa.z + wd.z - (hx4 * (pk2 * pk2) + hyp_m), f0[q], r);
              r = gkfft::caxpy(wc.z, fv0[q], r);
              r = gkfft::caxpy(wc.w, fv1[q], r);
              r = gkfft::caxpy(wd.x, fv3[q], r);
              r = gkfft::caxpy(wd.y, fv4[q], r);
              r = gkfft::caxpy(wd.w, dschi[q], r);
              // -i a z = a (z.y, -z.x)
              r = gkfft::caxpy(we.x * kap, make_float2(f0[q].y, -f0[q].x), r);
              r = gkfft::caxpy(we.y * fmf + we.z * kap, make_float2(chi0[q].y, -chi0[q].x), r);
              r = gkfft::caxpy(scale_i, nlv[q], r);
              float2 out;
              if constexpr (MODE == 0) {
                out = r;
              } else if constexpr (MODE == 1) {
                Cv<ST>::stcs(accp, eo, gkfft::caxpy(A.b, r, f0[q]));
                out = gkfft::caxpy(A.c, r, f0[q]);
                fsum = fmaf(2.f * fmf, chi0[q].x * f0[q].y - chi0[q].y * f0[q].x, fsum);
              } else if constexpr (MODE == 2) {
                Cv<ST>::stcs(accp, eo, gkfft::caxpy(A.b, r, ac[q]));
                out = gkfft::caxpy(A.c, r, fn[q]);
              } else {
                out = gkfft::caxpy(A.b, r, ac[q]);
              }
              Cv<ST>::stcs(outp, eo, out);
              macc[k] = cadd(macc[k], as_stored<ST>(out));   // what the next stage will read back
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
      if (want_flux) fx.slab(P, l, i, j, fsum);
      bar_arrive_n(BAR_FREE + (u & 1), NT);
    }
    if (want_flux) fx.item_end(fslot);
    if (A.mom) {
      // moment plane of this item: Z n 2 pi w_v B_i w_mu J0 sum_j f   (a1 of the next stage)
      const float momw = P.sp[a].momfac * P.wmu[l] * P.B[i];
      const float *j0p = P.J0 + (((long long)a * P.nmu + l) * P.ns + i) * P.slab;
      float2 *dst = A.mom + (((long long)a * P.nmu + l) * P.nchunk + c) * P.nphi + (long long)i * P.slab;
#pragma unroll
      for (int k = 0; k < EPT; ++k) {
        const int e = et + k * NTE;
        if (e < slab) dst[e] = gkfft::cscale(momw * __ldg(&j0p[e]), macc[k]);
      }
    }
  }
  if (want_flux && (et & 31) == 0) flux_flush(P, A.fluxp, blockIdx.x, NTE / 32, et >> 5, a_prev, fslot);
}

// RF, RE: registers per thread of the FFT / epilogue role after setmaxnreg (0: the launch allocation is
// kept); NB: points an epilogue thread keeps in flight.
template <class ST, int MX_, int MY_, int NKY_, int NKX_, int NTF, int NTE, int RF, int RE, int NB>
__global__ void __launch_bounds__(NTF + NTE, 1)
gk_stage_ws2_kernel(const __grid_constant__ GkDev P, const __grid_constant__ GkStageArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using gkfft::IC;
  using gkfft::sfor;
  using gkfft::dft;
  constexpr int NT = NTF + NTE;
  constexpr int K = (NKX_ - 1) / 2, slab = NKX_ * NKY_;
  constexpr int LD = MY_ | 1;
  constexpr int RX1 = gkfft::Fac<MX_>::R1, RX2 = gkfft::Fac<MX_>::R2;  // mx = RX1 * RX2
  constexpr int RY1 = gkfft::Fac<MY_>::R1, RY2 = gkfft::Fac<MY_>::R2;  // my = RY1 * RY2
  constexpr int NC = 2 * NKY_;   // x-transformed columns: P(0..nky-1), Q(0..nky-1); Q(0) is never used
  constexpr int H = MX_ / 2;     // row pairs (p, p + H) of the forward transform
  static_assert(NTF % 128 == 0 && NTE % 128 == 0, "roles are whole warpgroups (setmaxnreg)");
  // setmaxnreg moves registers inside the pool the CTA was LAUNCHED with (threads x registers per thread at
  // launch, itself limited by 16 K registers per SM sub-partition): a split that needs more never completes
  constexpr int WPS = ((NTF + NTE) / 32 + 3) / 4, RL = (16384 / (WPS * 32)) / 8 * 8;
  static_assert(RF == 0 || (RF % 8 == 0 && RE % 8 == 0 && NTF * RF + NTE * RE <= (NTF + NTE) * (RL < 255 ? RL : 255)), "register split");
  static_assert(RX2 > 1 && RY2 > 1 && RX2 % 2 == 0 && RY2 % 2 == 0 && RX1 % 2 == 0 && RY1 % 2 == 0, "two-pass even radices");
  static_assert(H % RX1 == 0, "a forward-x item lies in one half of the row pairs");
  static_assert(2 * NKY_ <= MY_ - NKY_ + 1, "dead columns hold the forward-x exchange");
  static_assert((slab * sizeof(ST)) % 16 == 0, "bulk copy size");
  constexpr int BAR_FFT = GK_WS_BAR_FFT, BAR_FULL = GK_WS_BAR_FULL, BAR_FREE = GK_WS_BAR_FREE;
  const int tid = threadIdx.x;
  float2 *chis_cta = A.chis + (long long)blockIdx.x * (GK_WS_CHI_RING * 3 * slab);
  float2 *nl_cta = A.nlbuf + (long long)blockIdx.x * (GK_WS_NL_RING * slab);

  float2 *sp = (float2 *)smem_raw;
  float2 *S = sp; sp += MX_ * LD;
  float2 *SG = sp; sp += MX_ * LD;
  ST *stg = (ST *)sp;            // the slab being transformed, landed by the bulk copy
  uint64_t *mbar = (uint64_t *)((unsigned char *)stg + slab * sizeof(ST));
  float *eblk = (float *)(mbar + 2);  // 16-byte aligned: slab-uniform epilogue coefficients, 2 slots
  __shared__ double fslots[(NTE / 32) * 3];
  if (tid == 0) { mbar_init(mbar, 1); mbar_init_fence(); }
  __syncthreads();

  if (tid < NTF) {
    // =============================== FFT role =====================================
    if constexpr (RF > 0) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(RF));
    const gkfft::NamedSync<BAR_FFT, NTF> fsync;
    // With 512 FFT threads and mx = 128 the item maps below keep two groups of warps (even / odd warp index)
    // closed under Y1 -> YF -> F2 (rows p, p + H with p < 32 / p >= 32) and, when a warp spans 32 of the 2 nky
    // columns, under X1 -> X2 (P / Q columns): those hand-offs need only a barrier among the 256 threads of a
    // group, and the two groups drift apart and fill each other's latency gaps.
    constexpr bool GRP = (NTF == 512 && MX_ == 128), GRPX = GRP && (NC == 64);
    auto gsync = [&]() { asm volatile("bar.sync %0, %1;" ::"r"(6 + ((tid >> 5) & 1)), "n"(NTF / 2) : "memory"); };
    // ---- X1: inverse x pass 1 of the spectral slab g (callable: slab index -> value) ----
    auto x1 = [&](auto g) {
      for (int w = tid; w < NC * RX1; w += NTF) {
        const int c = w % NC, n1 = w / NC;
        if (c == NKY_) continue;
        const bool isp = c < NKY_;
        const int m = isp ? c : c - NKY_;
        const int col = isp ? m : MY_ - m;
        const float kyv = isp ? -(float)m * P.ky0 : (float)m * P.ky0;
        float2 u[RX2];
        sfor<0, RX2>([&](auto n2c) {
          constexpr int off = RX1 * decltype(n2c)::value, hi = off + RX1 - 1;
          const int n = n1 + off;
          int p = 0;
          bool zero = false;
          if constexpr (hi <= K) p = n;                          // always a retained kx >= 0
          else if constexpr (off > K && hi < MX_ - K) zero = true;  // always zero padding: nothing is loaded
          else if constexpr (off >= MX_ - K) p = n - MX_;        // always a retained kx < 0
          else {
            if (n <= K) p = n;
            else if (n >= MX_ - K) p = n - MX_;
            else zero = true;
          }
          if (zero) {
            u[decltype(n2c)::value] = make_float2(0.f, 0.f);
          } else {
            const float2 v = g((p + K) * NKY_ + m);
            u[decltype(n2c)::value] = gkfft::caxpy(kyv, v, gkfft::cscale((float)p * P.dkx, make_float2(-v.y, v.x)));  // (i kx -+ ky) v
          }
        });
        dft<RX2, +1>(u);
        twiddle_row<RX2, +1>(u, tw_tab<MX_>().a + n1 * RX2);
        float2 *q = S + n1 * LD + col;
#pragma unroll
        for (int k2 = 0; k2 < RX2; ++k2) q[k2 * RX1 * LD] = u[k2];
      }
    };
    // ---- X2: inverse x pass 2, in place ----
    auto x2 = [&]() {
      // two items per thread when the item count allows (same column, k2 and k2 + NTF/NC): both are loaded
      // before either is transformed, so one shared-memory round trip covers both (the passes are
      // latency-bound at 4 FFT warps per scheduler)
      constexpr int ITEMS = NC * RX2, B = (ITEMS % (2 * NTF) == 0 && NTF % NC == 0) ? 2 : 1;
      constexpr int BOFF = (NTF / NC) * RX1 * LD;
      for (int w = tid; w < ITEMS; w += B * NTF) {
        const int c = w % NC, k2 = w / NC;
        if (c == NKY_) continue;
        const int col = c < NKY_ ? c : MY_ - (c - NKY_);
        float2 *q = S + k2 * RX1 * LD + col;
        float2 u[B][RX1];
#pragma unroll
        for (int b = 0; b < B; ++b)
#pragma unroll
          for (int n1 = 0; n1 < RX1; ++n1) u[b][n1] = q[b * BOFF + n1 * LD];
#pragma unroll
        for (int b = 0; b < B; ++b) {
          dft<RX1, +1>(u[b]);
#pragma unroll
          for (int k1 = 0; k1 < RX1; ++k1) q[b * BOFF + k1 * LD] = u[b][k1];
        }
      }
    };
    // ---- Y1: inverse y pass 1, in place; the Hermitian-extended row is P(y) for 0 < y < nky,
    // conj of what sits at y > my - nky, Re P(0) at y = 0 (R15) and zero in between ----
    auto y1 = [&]() {
      auto load = [&](const float2 *row, int n1, float2 (&u)[RY2]) {
        sfor<0, RY2>([&](auto n2c) {
          constexpr int n2 = decltype(n2c)::value, off = RY1 * n2, hi = off + RY1 - 1;
          const int y = n1 + off;
          float2 v;
          if constexpr (off >= NKY_ && hi <= MY_ - NKY_) {
            v = make_float2(0.f, 0.f);
          } else if constexpr (off > 0 && hi < NKY_) {
            v = row[off];
          } else if constexpr (off > MY_ - NKY_) {
            v = row[off];
            v.y = -v.y;
          } else {
            v = make_float2(0.f, 0.f);
            if (y < NKY_ || y > MY_ - NKY_) v = row[off];
            if (y == 0) v.y = 0.f;
            if (y > MY_ - NKY_) v.y = -v.y;
          }
          u[n2] = v;
        });
      };
      // two items per thread when the item count allows (same row, n1 and n1 + NTF/mx): the second item's
      // loads are issued between the first item's butterfly and its twiddle/store tail
      constexpr int ITEMS = MX_ * RY1, B = (ITEMS % (2 * NTF) == 0 && NTF % MX_ == 0) ? 2 : 1;
      constexpr int DN = NTF / MX_;
      for (int w = tid; w < ITEMS; w += B * NTF) {
        const int r = w % MX_, n1 = w / MX_;
        float2 *row = S + r * LD + n1;
        float2 u[RY2];
        load(row, n1, u);
        dft<RY2, +1>(u);
        if constexpr (B == 2) {
          float2 v[RY2];
          load(row + DN, n1 + DN, v);
          twiddle_row<RY2, +1>(u, tw_tab<MY_>().a + n1 * RY2);
#pragma unroll
          for (int k2 = 0; k2 < RY2; ++k2) row[k2 * RY1] = u[k2];
          dft<RY2, +1>(v);
          twiddle_row<RY2, +1>(v, tw_tab<MY_>().a + (n1 + DN) * RY2);
#pragma unroll
          for (int k2 = 0; k2 < RY2; ++k2) row[DN + k2 * RY1] = v[k2];
        } else {
          twiddle_row<RY2, +1>(u, tw_tab<MY_>().a + n1 * RY2);
#pragma unroll
          for (int k2 = 0; k2 < RY2; ++k2) row[k2 * RY1] = u[k2];
        }
      }
    };
    // ---- Y2: inverse y pass 2, S -> dst (grad(chi) of the work item) ----
    GmaxAcc gm;
    float ef_item = 1.f;   // ExB factor of the work item's plane
    auto y2_to = [&](float2 *dst) {
      for (int w = tid; w < MX_ * RY2; w += NTF) {
        const int r = w % MX_, k2 = w / MX_;
        const float2 *q = S + r * LD + k2 * RY1;
        float2 u[RY1];
#pragma unroll
        for (int n1 = 0; n1 < RY1; ++n1) u[n1] = q[n1];
        dft<RY1, +1>(u);
        float2 *d = dst + r * LD + k2 * RY1;
#pragma unroll
        for (int k1 = 0; k1 < RY1; ++k1) { d[k1] = u[k1]; gm.add(P, u[k1], ef_item); }
      }
    };
    // ---- YF: inverse y pass 2 of rows p and p + H, bracket d_y chi d_x f - d_x chi d_y f (real space
    // holds d_x + i d_y of f in S and (d_x chi, d_y chi) in SG), the two real rows packed as
    // (re, im), forward y pass 1; result in row p ----
    auto yf = [&]() {
      for (int w = tid; w < H * RY2; w += NTF) {
        const int p = w % H, k2 = w / H;
        float2 *q0 = S + p * LD + k2 * RY1;
        const float2 *q1 = q0 + H * LD;
        const float2 *g0 = SG + p * LD + k2 * RY1, *g1 = g0 + H * LD;
        float2 u[RY1];
        float br[RY1];
#pragma unroll
        for (int n1 = 0; n1 < RY1; ++n1) u[n1] = q0[n1];
        dft<RY1, +1>(u);
#pragma unroll
        for (int k1 = 0; k1 < RY1; ++k1) {
          const float2 g = g0[k1];
          br[k1] = g.y * u[k1].x - g.x * u[k1].y;
        }
#pragma unroll
        for (int n1 = 0; n1 < RY1; ++n1) u[n1] = q1[n1];
        dft<RY1, +1>(u);
#pragma unroll
        for (int k1 = 0; k1 < RY1; ++k1) {
          const float2 g = g1[k1];
          u[k1] = make_float2(br[k1], g.y * u[k1].x - g.x * u[k1].y);
        }
        dft<RY1, -1>(u);
        twiddle_row<RY1, -1>(u, tw_tab<MY_>().b + k2 * RY1);
#pragma unroll
        for (int n1 = 0; n1 < RY1; ++n1) q0[n1] = u[n1];
      }
    };
    // ---- F2: forward y pass 2 of the packed rows, in place; only the retained ky (and their
    // mirror images, needed by the unpack) are stored ----
    auto f2 = [&]() {
      for (int w = tid; w < H * RY1; w += NTF) {
        const int p = w % H, n1 = w / H;
        float2 *row = S + p * LD + n1;
        float2 u[RY2];
#pragma unroll
        for (int k2 = 0; k2 < RY2; ++k2) u[k2] = row[k2 * RY1];
        dft<RY2, -1>(u);
        sfor<0, RY2>([&](auto n2c) {
          constexpr int n2 = decltype(n2c)::value, off = RY1 * n2, hi = off + RY1 - 1;
          if constexpr (off >= NKY_ && hi <= MY_ - NKY_) {
          } else if constexpr (hi < NKY_ || off > MY_ - NKY_) {
            row[off] = u[n2];
          } else {
            const int y = n1 + off;
            if (y < NKY_ || y > MY_ - NKY_) row[off] = u[n2];
          }
        });
      }
    };
    // ---- XF1: forward x pass 1 of the nky retained columns.  Row r < H is the first real row of a
    // pair, A(m) = Z(m) + conj Z(my-m); row r >= H the second, B(m) = -i (Z(m) - conj Z(my-m)) (the
    // factor 1/2 is in the epilogue's scale).  Output to the dead columns nky..2nky-1. ----
    auto xf1 = [&]() {
      for (int w = tid; w < NKY_ * RX2; w += NTF) {
        const int m = w % NKY_, k2 = w / NKY_;
        const int mm = (m == 0) ? 0 : MY_ - m;
        const bool hi = (k2 * RX1 >= H);
        const float2 *q = S + (k2 * RX1 - (hi ? H : 0)) * LD;
        float2 u[RX1];
#pragma unroll
        for (int k1 = 0; k1 < RX1; ++k1) {
          const float2 z = q[k1 * LD + m];
          const float2 zc = q[k1 * LD + mm];   // conj applied below
          u[k1] = hi ? make_float2(z.y + zc.y, zc.x - z.x) : make_float2(z.x + zc.x, z.y - zc.y);
        }
        dft<RX1, -1>(u);
        twiddle_row<RX1, -1>(u, tw_tab<MX_>().b + k2 * RX1);
        float2 *d = S + k2 * RX1 * LD + NKY_ + m;
#pragma unroll
        for (int n1 = 0; n1 < RX1; ++n1) d[n1 * LD] = u[n1];
      }
    };
    // ---- XF2: forward x pass 2; the retained kx go to the bracket ring slot `nlw` in slab order ----
    auto xf2 = [&](float2 *nlw) {
      for (int w = tid; w < NKY_ * RX1; w += NTF) {
        const int m = w % NKY_, n1 = w / NKY_;
        const float2 *q = S + n1 * LD + NKY_ + m;
        float2 u[RX2];
#pragma unroll
        for (int k2 = 0; k2 < RX2; ++k2) u[k2] = q[k2 * RX1 * LD];
        dft<RX2, -1>(u);
        sfor<0, RX2>([&](auto n2c) {
          constexpr int n2 = decltype(n2c)::value, off = RX1 * n2, hi = off + RX1 - 1;
          const int n = n1 + off;
          if constexpr (off > K && hi < MX_ - K) {
          } else if constexpr (hi <= K) {
            __stcg(&nlw[(n + K) * NKY_ + m], u[n2]);
          } else if constexpr (off >= MX_ - K) {
            __stcg(&nlw[(n - MX_ + K) * NKY_ + m], u[n2]);
          } else {
            if (n <= K) __stcg(&nlw[(n + K) * NKY_ + m], u[n2]);
            else if (n >= MX_ - K) __stcg(&nlw[(n - MX_ + K) * NKY_ + m], u[n2]);
          }
        });
      }
    };

    const long long jstride = (long long)P.nmu * P.ns * P.slab;
    uint32_t parity = 0;
    int u = 0, it = 0;
    for (int w = blockIdx.x; w < A.nwork; w += gridDim.x, ++it) {
      const int i = w % P.ns;
      const int c = (w / P.ns) % P.nchunk;
      const int al = w / (P.ns * P.nchunk);
      const int l = al % P.nmu, a = al / P.nmu;
      const long long base0 = (((long long)a * P.nv * P.nmu + l) * P.ns + i) * P.slab;
      const int j0 = c * P.jchunk, j1 = min(P.nv, (c + 1) * P.jchunk);
      // the first slab of the item lands while grad(chi) is built (the staging buffer was last read
      // by the X1 of the previous slab, which every thread of the role has left)
      if (tid == 0) bulk_load(stg, (const ST *)A.y + (base0 + (long long)j0 * jstride), slab * sizeof(ST), mbar);
      float2 *chis = chis_cta + (it % GK_WS_CHI_RING) * 3 * slab;
      ef_item = P.ef[i];
      build_chis(P, A, a, l, i, slab, NKY_, chis, tid, NTF);
      fsync();
      x1([&](int e) { return __ldcg(&chis[e]); });
      fsync();
      x2();
      fsync();
      y1();
      fsync();
      y2_to(SG);
      fsync();
      for (int j = j0; j < j1; ++j, ++u) {
        mbar_wait(mbar, parity);
        parity ^= 1u;
        x1([&](int e) { return Cv<ST>::ld(stg, e); });
        if constexpr (GRPX) gsync(); else fsync();
        x2();
        fsync();
        // every thread has left X1: the staging buffer may take the next slab
        if (tid == 0 && j + 1 < j1)
          bulk_load(stg, (const ST *)A.y + (base0 + (long long)(j + 1) * jstride), slab * sizeof(ST), mbar);
        y1();
        if constexpr (GRP) gsync(); else fsync();
        yf();
        if constexpr (GRP) gsync(); else fsync();
        f2();
        fsync();
        xf1();
        fsync();
        // ring slot must have been consumed by the epilogue of slab u-2
        if (u >= GK_WS_NL_RING) bar_sync_n(BAR_FREE + (u & 1), NT);
        xf2(nl_cta + (u & 1) * slab);
        // XF2 reads only the dead columns, which X1/X2 of the next slab do not write: no barrier here
        bar_arrive_n(BAR_FULL + (u & 1), NT);
      }
    }
    // consume the epilogue's last arrivals so that no barrier is left half-way at exit
    for (int v = max(0, u - GK_WS_NL_RING); v < u; ++v) bar_sync_n(BAR_FREE + (v & 1), NT);
    gm.flush(A.gmax);
  } else {
    if constexpr (RE > 0) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(RE));
    ws_epilogue_role2<ST, NKY_, NKX_, NTF, NTE, NB>(P, A, chis_cta, nl_cta, eblk, fslots, tid);
  }
}

}  // namespace gk
