// gk_stage_ws3.cuh -- row-streaming form of the warp-specialised RK-stage kernel (steps a3-a6 of
// DESIGN.md) for padded grids of which not even one real-space field fits shared memory (BASELINE
// grid 5: 192 x 192, 296 KB per field).  Product path; shares nothing with oracle/.
//
// Same passes as gk_stage_ws2_kernel, but only the x-transformed half spectra stay resident:
//   XA [mx][2 nky - 1]   column c < nky: P(c) = Fx[(i kx - ky) g], column nky-1+m': Q(m'), m' >= 1
//   W  [RC][my]          the y transforms of RC rows at a time (rows are independent once the x
//                        transform is done); the unpacked bracket rows overwrite XA's P columns
//   grad(chi)            per-CTA scratch in L2, stored in the order the fused pass reads it:
//                        [chunk][k2][k1][row of the chunk] -> lanes read consecutive addresses
// per slab: X1, X2, then per chunk Y1 (XA -> W), YF (inverse y pass 2 + bracket + forward y pass 1,
// in registers), F2U (forward y pass 2 + two-for-one unpack into XA, partners exchanged by shuffles); XF1, XF2 -> bracket ring for the epilogue
// role (ws_epilogue_role2 without register moments: gk_moment_kernel runs on the new state).
#pragma once

namespace gk {

template <class ST, int MX_, int MY_, int NKY_, int NKX_, int RC_>
constexpr size_t ws3_smem_bytes() {
  return (size_t)(MX_ * (2 * NKY_ - 1) + RC_ * (MY_ | 1)) * 8 + 2 * GK_EB_N * 4;
}
// elements of the per-CTA grad(chi) scratch
template <int MX_, int MY_> constexpr size_t ws3_gchi_elems() { return (size_t)MX_ * MY_; }

template <class ST, int MX_, int MY_, int NKY_, int NKX_, int RC_, int NTF, int NTE>
__global__ void __launch_bounds__(NTF + NTE, 1)
gk_stage_ws3_kernel(const __grid_constant__ GkDev P, const __grid_constant__ GkStageArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using gkfft::sfor;
  using gkfft::dft;
  constexpr int NT = NTF + NTE;
  constexpr int K = (NKX_ - 1) / 2, slab = NKX_ * NKY_;
  constexpr int LDX = 2 * NKY_ - 1, LDW = MY_ | 1;
  constexpr int RX1 = gkfft::Fac<MX_>::R1, RX2 = gkfft::Fac<MX_>::R2;
  constexpr int RY1 = gkfft::Fac<MY_>::R1, RY2 = gkfft::Fac<MY_>::R2;
  constexpr int NC = 2 * NKY_ - 1;   // columns of XA
  constexpr int HC = RC_ / 2;        // row pairs (p, p + HC) of a chunk
  constexpr int NCH = MX_ / RC_;
  static_assert(MX_ % RC_ == 0 && RC_ % 2 == 0, "chunks of whole row pairs");
  static_assert(NTF % 32 == 0 && NTE % 32 == 0, "roles are whole warps");
  constexpr int BAR_FFT = GK_WS_BAR_FFT, BAR_FULL = GK_WS_BAR_FULL, BAR_FREE = GK_WS_BAR_FREE;
  const int tid = threadIdx.x;
  // chi / D_s chi and grad(chi) live in scratch indexed by (species, mu, s), not by CTA: the CTAs that work on the
  // vpar chunks of one (species, mu, s) at the same time write identical values and share the L2 lines
  float2 *nl_cta = A.nlbuf + (long long)blockIdx.x * (GK_WS_NL_RING * slab);
  float2 *SGg = A.gchi;

  float2 *XA = (float2 *)smem_raw;
  float2 *W = XA + MX_ * LDX;
  float *eblk = (float *)(W + RC_ * LDW);

  if (tid < NTF) {
    // =============================== FFT role =====================================
    const gkfft::NamedSync<BAR_FFT, NTF> fsync;
    // ---- X1: inverse x pass 1 of the spectral slab g (callable: slab index -> value) ----
    auto x1 = [&](auto g) {
      for (int w = tid; w < NC * RX1; w += NTF) {
        const int c = w % NC, n1 = w / NC;
        const bool isp = c < NKY_;
        const int m = isp ? c : c - NKY_ + 1;
        const float kyv = isp ? -(float)m * P.ky0 : (float)m * P.ky0;
        float2 u[RX2];
        sfor<0, RX2>([&](auto n2c) {
          constexpr int off = RX1 * decltype(n2c)::value, hi = off + RX1 - 1;
          const int n = n1 + off;
          int p = 0;
          bool zero = false;
          if constexpr (hi <= K) p = n;
          else if constexpr (off > K && hi < MX_ - K) zero = true;
          else if constexpr (off >= MX_ - K) p = n - MX_;
          else {
            if (n <= K) p = n;
            else if (n >= MX_ - K) p = n - MX_;
            else zero = true;
          }
          if (zero) {
            u[decltype(n2c)::value] = make_float2(0.f, 0.f);
          } else {
            const float2 v = g((p + K) * NKY_ + m);
            u[decltype(n2c)::value] = gkfft::caxpy(kyv, v, gkfft::cscale((float)p * P.dkx, make_float2(-v.y, v.x)));
          }
        });
        dft<RX2, +1>(u);
        twiddle_row<RX2, +1>(u, tw_tab<MX_>().a + n1 * RX2);
        float2 *q = XA + n1 * LDX + c;
#pragma unroll
        for (int k2 = 0; k2 < RX2; ++k2) q[k2 * RX1 * LDX] = u[k2];
      }
    };
    // ---- X2: inverse x pass 2, in place ----
    auto x2 = [&]() {
      for (int w = tid; w < NC * RX2; w += NTF) {
        const int c = w % NC, k2 = w / NC;
        float2 *q = XA + k2 * RX1 * LDX + c;
        float2 u[RX1];
#pragma unroll
        for (int n1 = 0; n1 < RX1; ++n1) u[n1] = q[n1 * LDX];
        dft<RX1, +1>(u);
#pragma unroll
        for (int k1 = 0; k1 < RX1; ++k1) q[k1 * LDX] = u[k1];
      }
    };
    // ---- Y1: inverse y pass 1 of rows r0 .. r0+RC-1, XA -> W.  Hermitian-extended row: Re P(0) at y = 0
    // (R15), P(y) for 0 < y < nky, conj Q(my - y) for y > my - nky, zero in between ----
    auto y1 = [&](int r0) {
      for (int w = tid; w < RC_ * RY1; w += NTF) {
        const int r = w % RC_, n1 = w / RC_;
        const float2 *row = XA + (r0 + r) * LDX;
        float2 u[RY2];
        sfor<0, RY2>([&](auto n2c) {
          constexpr int n2 = decltype(n2c)::value, off = RY1 * n2, hi = off + RY1 - 1;
          const int y = n1 + off;
          float2 v;
          if constexpr (off >= NKY_ && hi <= MY_ - NKY_) {
            v = make_float2(0.f, 0.f);
          } else if constexpr (off > 0 && hi < NKY_) {
            v = row[y];
          } else if constexpr (off > MY_ - NKY_) {
            v = row[NKY_ - 1 + MY_ - y];
            v.y = -v.y;
          } else {
            v = make_float2(0.f, 0.f);
            if (y < NKY_) v = row[y];
            if (y > MY_ - NKY_) { v = row[NKY_ - 1 + MY_ - y]; v.y = -v.y; }
            if (y == 0) v.y = 0.f;
          }
          u[n2] = v;
        });
        dft<RY2, +1>(u);
        twiddle_row<RY2, +1>(u, tw_tab<MY_>().a + n1 * RY2);
        float2 *q = W + r * LDW + n1;
#pragma unroll
        for (int k2 = 0; k2 < RY2; ++k2) q[k2 * RY1] = u[k2];
      }
    };
    // position of real-space element (chunk ch, row r of the chunk, y position k2 RY1 + k1) in the scratch
    auto sg_index = [](int ch, int r, int k2, int k1) { return ((ch * RY2 + k2) * RY1 + k1) * RC_ + r; };
    // ---- Y2: inverse y pass 2 of the chunk in W -> grad(chi) scratch ----
    auto y2_to_sg = [&](int ch) {
      for (int w = tid; w < RC_ * RY2; w += NTF) {
        const int r = w % RC_, k2 = w / RC_;
        const float2 *q = W + r * LDW + k2 * RY1;
        float2 u[RY1];
#pragma unroll
        for (int n1 = 0; n1 < RY1; ++n1) u[n1] = q[n1];
        dft<RY1, +1>(u);
#pragma unroll
        for (int k1 = 0; k1 < RY1; ++k1) __stcg(&SGg[sg_index(ch, r, k2, k1)], u[k1]);
      }
    };
    // ---- YF: inverse y pass 2 of rows p and p + HC of the chunk, bracket d_y chi d_x f - d_x chi d_y f
    // against grad(chi) (re = d_x chi, im = d_y chi) from the L2 scratch, the two real rows packed as
    // (re, im), forward y pass 1; result in row p of W ----
    auto yf = [&](int ch) {
      for (int w = tid; w < HC * RY2; w += NTF) {
        const int p = w % HC, k2 = w / HC;
        float2 *q0 = W + p * LDW + k2 * RY1;
        const float2 *q1 = q0 + HC * LDW;
        const float2 *g0 = SGg + sg_index(ch, p, k2, 0);
        float2 u[RY1], g[RY1];
        float br[RY1];
#pragma unroll
        for (int k1 = 0; k1 < RY1; ++k1) g[k1] = __ldcg(g0 + k1 * RC_);
#pragma unroll
        for (int n1 = 0; n1 < RY1; ++n1) u[n1] = q0[n1];
        dft<RY1, +1>(u);
#pragma unroll
        for (int k1 = 0; k1 < RY1; ++k1) br[k1] = g[k1].y * u[k1].x - g[k1].x * u[k1].y;
#pragma unroll
        for (int k1 = 0; k1 < RY1; ++k1) g[k1] = __ldcg(g0 + k1 * RC_ + HC);
#pragma unroll
        for (int n1 = 0; n1 < RY1; ++n1) u[n1] = q1[n1];
        dft<RY1, +1>(u);
#pragma unroll
        for (int k1 = 0; k1 < RY1; ++k1) u[k1] = make_float2(br[k1], g[k1].y * u[k1].x - g[k1].x * u[k1].y);
        dft<RY1, -1>(u);
        twiddle_row<RY1, -1>(u, tw_tab<MY_>().b + k2 * RY1);
#pragma unroll
        for (int n1 = 0; n1 < RY1; ++n1) q0[n1] = u[n1];
      }
    };
    // ---- F2U: forward y pass 2 of the packed rows fused with the two-for-one unpack.  A warp holds PW pairs x
    // RY1 residues n1; the thread (p, n1) ends with Z(n1 + RY1 n2) and needs Z(my - y) for its retained
    // y = n1 + RY1 n2 < nky, which is output RY2-1-n2 of the thread (p, RY1 - n1) (its own output RY2 - n2
    // when n1 = 0): one shuffle per retained value.  Row r0+p of XA gets A(m) = Z(m) + conj Z(my-m), row
    // r0+p+HC gets B(m) = -i (Z(m) - conj Z(my-m)) (factor 1/2 in the epilogue's scale). ----
    auto f2u = [&](int r0) {
      constexpr int PW = 32 / RY1, NLOW = (NKY_ + RY1 - 1) / RY1;
      static_assert(PW >= 1 && HC % PW == 0 && NLOW < RY2, "pairs per warp");
      const int lane = tid & 31, wq = lane / RY1, n1 = lane - wq * RY1;
      const bool active = lane < PW * RY1;
      const int n1p = (n1 == 0) ? 0 : RY1 - n1;
      const int src = active ? wq * RY1 + n1p : lane;
      for (int wp = tid >> 5; wp < HC / PW; wp += NTF / 32) {
        const int p = wp * PW + (active ? wq : 0);
        const float2 *row = W + p * LDW + n1;
        float2 u[RY2];
#pragma unroll
        for (int k2 = 0; k2 < RY2; ++k2) u[k2] = active ? row[k2 * RY1] : make_float2(0.f, 0.f);
        dft<RY2, -1>(u);
        float2 *da = XA + (r0 + p) * LDX + n1, *db = da + HC * LDX;
        sfor<0, NLOW>([&](auto n2c) {
          constexpr int n2 = decltype(n2c)::value;
          const float2 mine = (n1 == 0) ? u[n2 == 0 ? 0 : RY2 - n2] : u[RY2 - 1 - n2];   // what my partner needs
          float2 zc;
          zc.x = __shfl_sync(0xffffffffu, mine.x, src);
          zc.y = __shfl_sync(0xffffffffu, mine.y, src);
          const float2 z = u[n2];
          if (active && n1 + RY1 * n2 < NKY_) {
            da[RY1 * n2] = make_float2(z.x + zc.x, z.y - zc.y);
            db[RY1 * n2] = make_float2(z.y + zc.y, zc.x - z.x);
          }
        });
      }
    };
    // ---- XF1: forward x pass 1 of the nky retained columns, in place ----
    auto xf1 = [&]() {
      for (int w = tid; w < NKY_ * RX2; w += NTF) {
        const int m = w % NKY_, k2 = w / NKY_;
        float2 *q = XA + k2 * RX1 * LDX + m;
        float2 u[RX1];
#pragma unroll
        for (int k1 = 0; k1 < RX1; ++k1) u[k1] = q[k1 * LDX];
        dft<RX1, -1>(u);
        twiddle_row<RX1, -1>(u, tw_tab<MX_>().b + k2 * RX1);
#pragma unroll
        for (int n1 = 0; n1 < RX1; ++n1) q[n1 * LDX] = u[n1];
      }
    };
    // ---- XF2: forward x pass 2; the retained kx go to the bracket ring slot `nlw` in slab order ----
    auto xf2 = [&](float2 *nlw) {
      for (int w = tid; w < NKY_ * RX1; w += NTF) {
        const int m = w % NKY_, n1 = w / NKY_;
        const float2 *q = XA + n1 * LDX + m;
        float2 u[RX2];
#pragma unroll
        for (int k2 = 0; k2 < RX2; ++k2) u[k2] = q[k2 * RX1 * LDX];
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
    int u = 0, it = 0;
    for (int w = blockIdx.x; w < A.nwork; w += gridDim.x, ++it) {
      const int i = w % P.ns;
      const int c = (w / P.ns) % P.nchunk;
      const int al = w / (P.ns * P.nchunk);
      const int l = al % P.nmu, a = al / P.nmu;
      const long long base0 = (((long long)a * P.nv * P.nmu + l) * P.ns + i) * P.slab;
      const int j0 = c * P.jchunk, j1 = min(P.nv, (c + 1) * P.jchunk);
      const long long item_li = ((long long)a * P.nmu + l) * P.ns + i;
      float2 *chis = A.chis + item_li * (3 * slab);
      SGg = A.gchi + item_li * (MX_ * MY_);
      build_chis(P, A, a, l, i, slab, NKY_, chis, tid, NTF);
      fsync();   // also: every thread has left the XF2 of the previous slab (XA is free)
      x1([&](int e) { return __ldcg(&chis[e]); });
      fsync();
      x2();
      fsync();
      for (int ch = 0; ch < NCH; ++ch) {
        y1(ch * RC_);
        fsync();
        y2_to_sg(ch);
        fsync();
      }
      for (int j = j0; j < j1; ++j, ++u) {
        const ST *yb = (const ST *)A.y + (base0 + (long long)j * jstride);
        x1([&](int e) { return Cv<ST>::ldg(yb, e); });
        fsync();
        x2();
        fsync();
        for (int ch = 0; ch < NCH; ++ch) {
          y1(ch * RC_);
          fsync();
          yf(ch);
          fsync();
          f2u(ch * RC_);
          fsync();
        }
        xf1();
        fsync();
        // ring slot must have been consumed by the epilogue of slab u-2
        if (u >= GK_WS_NL_RING) bar_sync_n(BAR_FREE + (u & 1), NT);
        xf2(nl_cta + (u & 1) * slab);
        fsync();   // XA is rewritten by the next slab's X1
        bar_arrive_n(BAR_FULL + (u & 1), NT);
      }
    }
    // consume the epilogue's last arrivals so that no barrier is left half-way at exit
    for (int v = max(0, u - GK_WS_NL_RING); v < u; ++v) bar_sync_n(BAR_FREE + (v & 1), NT);
  } else {
    ws_epilogue_role2<ST, NKY_, NKX_, NTF, NTE, 1, false, true>(P, A, A.chis, nl_cta, eblk, tid);
  }
}

}  // namespace gk
