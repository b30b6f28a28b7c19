// gk_stage_ws4.cuh -- the fused RK-stage kernel (steps a3-a6 of DESIGN.md) for padded grids of which not even
// one real-space field fits the shared memory of an SM (BASELINE grid 5: 192 x 192, 296 KB per field), as a
// thread-block CLUSTER of CL = 4 CTAs.  Product path; shares nothing with oracle/.
//
// The x transform is split by decimation: CTA q of the cluster owns the real-space rows r = CL s + q,
//   inverse   G[CL s + q] = sum_{n1 < mx/CL} { w^{n1 q} sum_{t < CL} g[n1 + (mx/CL) t] i^{t q} } w_{mx/CL}^{n1 s}
//             = a length-(mx/CL) transform of a folded, pre-twiddled input: every CTA reads the whole spectral
//             slab (65 KB, one bulk copy each) and does a quarter of the arithmetic; no exchange.
//   forward   N[k] = sum_q w^{-q k} C_q[k mod (mx/CL)],  C_q = length-(mx/CL) transform of the CTA's rows:
//             every CTA writes its PARTIAL sum for all retained (kx, ky) to a 2-slot ring in L2 and the
//             epilogue roles add the CL partials in a fixed order (deterministic).
// So a CTA holds only its quarter of the rows: S[mx/4][my] (the slab in flight, transformed in place exactly
// as in gk_stage_ws2_kernel) and SG[mx/4][my] (real-space grad(chi), built once per (species, mu, s) and
// resident over the vpar march: "no intermediate HBM round-trips"), 2 x 74 KB + 65 KB staging.
// Real space is only multiplied pointwise, so which rows a CTA owns never matters.
//
// Roles per CTA (setmaxnreg split): NTF FFT threads; NTE streaming threads that run epi_item (gk_epilogue.cuh)
// on the CTA's quarter of the (kx, ky) slab: 128-bit accesses, vpar register window, moments in registers.
// Hand-over across the cluster by mbarriers in shared memory (remote arrive, release/acquire at cluster
// scope): FULL[b] counts the CL FFT roles that have written their partial of ring slot b, FREE[b] the CL
// streaming roles that have consumed it.
#pragma once

namespace gk {

// exp(+2 pi i t / 192)
struct W192Tab { float2 w[192]; };
constexpr W192Tab make_w192() {
  W192Tab t{};
  for (int k = 0; k < 192; ++k) {
    const double ang = 2.0 * gkfft::kPi * (k > 96 ? k - 192 : k) / 192;
    t.w[k].x = (float)gkfft::cx_cos(ang);
    t.w[k].y = (float)gkfft::cx_sin(ang);
  }
  return t;
}
static __constant__ W192Tab c_w192 = make_w192();

template <class ST, int MX_, int MY_, int NKY_, int NKX_, int CL, int NTE>
constexpr size_t ws4_smem_bytes() {
  return (size_t)(2 * (MX_ / CL) * (MY_ | 1)) * 8 + (size_t)NKX_ * NKY_ * sizeof(ST) + 8 * 8 + (NTE / 32) * GK_EB_N * 4 +
         (size_t)EpiMap<ST, NKY_, NTE, (NKX_ + CL - 1) / CL>::EPT * NTE * Vec<ST>::PV * 8;
}
// per-CTA scratch (float2 elements) for chi, D_s chi (v > 0), D_s chi (v < 0) on the CTA's share of the slab
template <int NKY_, int NKX_, int CL> constexpr size_t ws4_chis_elems() {
  return (size_t)3 * ((NKX_ + CL - 1) / CL) * NKY_;
}

template <class ST, int NKY_, int NKX_, int CL, int NTE>
struct Ws4Hooks {
  static constexpr bool NL = true;
  static constexpr bool FLUX = true;
  static constexpr int ROWS = (NKX_ + CL - 1) / CL, SHARE = ROWS * NKY_, slab = NKX_ * NKY_;
  using M = EpiMap<ST, NKY_, NTE, ROWS>;
  float2 *chis;          // this CTA's scratch [3][SHARE] (L2), written and read by the same thread
  const float2 *nlring;  // the cluster's ring [2][CL][slab]
  uint64_t *full, *free_;  // [2] each
  float *eblk;           // [NTE/32][GK_EB_N]
  float2 *maccs;         // [EPT][NTE][PV] shared memory: moment accumulators, thread-private slots
  double *fslots;        // [NTE/32][3]
  int et;
  __device__ __forceinline__ double *fluxslot() const { return fslots + (et >> 5) * 3; }
  __device__ __forceinline__ float *coef(int, int t) const { return eblk + (t >> 5) * GK_EB_N; }
  __device__ __forceinline__ bool makes_coef(int t) const {
    __syncwarp();
    return (t & 31) == 0;
  }
  __device__ __forceinline__ void begin(int u) const {
    __syncwarp();
    mbar_wait_cluster(full + (u & 1), (u >> 1) & 1);
  }
  __device__ __forceinline__ void end(int u) const {
    bar_sync_n(GK_WS_BAR_EPI, NTE);     // every thread of the role has consumed ring slot u & 1
    if (et == 0) {
#pragma unroll
      for (int r = 0; r < CL; ++r) mbar_arrive_remote(free_ + (u & 1), r);
    }
  }
  __device__ __forceinline__ void chi(int, int el, int sg, float2 (&c)[M::PV], float2 (&d)[M::PV]) const {
    const float4 *pc = (const float4 *)(chis + el), *pd = (const float4 *)(chis + (1 + sg) * SHARE + el);
#pragma unroll
    for (int v = 0; v < M::PV; v += 2) {
      const float4 x = __ldcg(pc + v / 2), y = __ldcg(pd + v / 2);
      c[v] = make_float2(x.x, x.y); c[v + 1] = make_float2(x.z, x.w);
      d[v] = make_float2(y.x, y.y); d[v + 1] = make_float2(y.z, y.w);
    }
  }
  __device__ __forceinline__ float2 *macc(int k) const { return maccs + ((size_t)k * NTE + et) * M::PV; }
  __device__ __forceinline__ void nl(int u, int e, float2 (&o)[M::PV]) const {
    const float2 *base = nlring + (size_t)(u & 1) * CL * slab + e;
#pragma unroll
    for (int v = 0; v < M::PV; v += 2) {
      float4 p[CL];
#pragma unroll
      for (int r = 0; r < CL; ++r) p[r] = __ldcg((const float4 *)(base + (size_t)r * slab + v));
      float4 s = p[0];
#pragma unroll
      for (int r = 1; r < CL; ++r) { s.x += p[r].x; s.y += p[r].y; s.z += p[r].z; s.w += p[r].w; }
      o[v] = make_float2(s.x, s.y); o[v + 1] = make_float2(s.z, s.w);
    }
  }
};

// multiply by i^e, e in 0..3 (uniform over the CTA)
__device__ __forceinline__ float2 mul_ipow(float2 a, int e) {
  const float2 b = (e & 1) ? make_float2(-a.y, a.x) : a;
  return (e & 2) ? make_float2(-b.x, -b.y) : b;
}

template <class ST, int MX_, int MY_, int NKY_, int NKX_, int CL, int NTF, int NTE, int RF, int RE, int NB>
__global__ void __launch_bounds__(NTF + NTE, 1)
gk_stage_ws4_kernel(const __grid_constant__ GkDev P, const __grid_constant__ GkStageArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using gkfft::sfor;
  using gkfft::dft;
  static_assert(CL == 4 && MX_ == 192, "the folding below is written for 4 CTAs and the 192-point table");
  constexpr int K = (NKX_ - 1) / 2, slab = NKX_ * NKY_;
  constexpr int MQ = MX_ / CL;   // real-space rows of a CTA
  constexpr int LD = MY_ | 1;
  constexpr int RX1 = gkfft::Fac<MQ>::R1, RX2 = gkfft::Fac<MQ>::R2;    // mx/CL = RX1 * RX2
  constexpr int RY1 = gkfft::Fac<MY_>::R1, RY2 = gkfft::Fac<MY_>::R2;  // my = RY1 * RY2
  constexpr int NC = 2 * NKY_;   // x-transformed columns: P(0..nky-1), Q(0..nky-1); Q(0) is never used
  constexpr int H = MQ / 2;      // row pairs (p, p + H) of the forward transform
  constexpr int ROWS = (NKX_ + CL - 1) / CL;   // kx rows of a CTA's share of the streaming work
  static_assert(NTF % 128 == 0 && NTE % 128 == 0, "roles are whole warpgroups (setmaxnreg)");
  // setmaxnreg moves registers inside the pool the CTA was LAUNCHED with (threads x registers per thread at
  // launch, itself limited by 16 K registers per SM sub-partition): a split that needs more never completes
  constexpr int WPS = ((NTF + NTE) / 32 + 3) / 4, RL = (16384 / (WPS * 32)) / 8 * 8;
  static_assert(RF % 8 == 0 && RE % 8 == 0 && NTF * RF + NTE * RE <= (NTF + NTE) * (RL < 255 ? RL : 255), "register split");
  static_assert(RX2 > 1 && RY2 > 1 && H % RX1 == 0, "two-pass transforms; a forward-x item lies in one half of the row pairs");
  static_assert(2 * NKY_ <= MY_ - NKY_ + 1, "dead columns hold the forward-x exchange");
  static_assert((slab * sizeof(ST)) % 16 == 0, "bulk copy size");
  static_assert(2 * K + 1 == NKX_ && 3 * K + 1 <= MX_ && K < 2 * MQ && K >= MQ, "folding ranges");
  const int tid = threadIdx.x;
  const int q = (int)cluster_ctarank();
  const int cid = (int)cluster_id_x(), ncl = (int)cluster_count_x();

  float2 *sp = (float2 *)smem_raw;
  float2 *S = sp; sp += MQ * LD;
  float2 *SG = sp; sp += MQ * LD;
  ST *stg = (ST *)sp;            // the slab being transformed, landed by the bulk copy
  uint64_t *mbar = (uint64_t *)((unsigned char *)stg + slab * sizeof(ST));  // [0] staging, [2..3] FULL, [4..5] FREE
  uint64_t *full = mbar + 2, *free_ = mbar + 4;
  float *eblk = (float *)(mbar + 8);
  __shared__ double fslots[(NTE / 32) * 3];
  if (tid == 0) {
    mbar_init(mbar, 1);
    mbar_init(full, CL); mbar_init(full + 1, CL);
    mbar_init(free_, CL); mbar_init(free_ + 1, CL);
    mbar_init_fence();
  }
  cluster_sync_all();   // nobody arrives at a barrier that is not initialised yet
  float2 *nlring = A.nlbuf + (size_t)cid * (GK_WS_NL_RING * CL * slab);

  if (tid < NTF) {
    // =============================== FFT role =====================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(RF));
    const gkfft::NamedSync<GK_WS_BAR_FFT, NTF> fsync;
    // ---- X1: folding + inverse x pass 1 of the spectral slab g (callable: slab index -> value) ----
    // h[n1] = w^{n1 q} sum_t i^{t q} (i kx -+ ky) g[n1 + MQ t]; the padding (K < n < mx - K) is never loaded
    // The items of a warp share n1a (NC is a multiple of 32): the body is instantiated once per n1a, so that which of
    // the CL fold terms exist, their kx and their slab rows are compile-time constants (no predicate arithmetic, no
    // dead loads); only the rotations by the CTA rank q stay run-time (uniform).
    auto x1 = [&](auto g) {
      for (int w = tid; w < NC * RX1; w += NTF) {
        const int c = w % NC, n1a = w / NC;
        if (c == NKY_) continue;
        const bool isp = c < NKY_;
        const int m = isp ? c : c - NKY_;
        const int col = isp ? m : MY_ - m;
        const float kyv = isp ? -(float)m * P.ky0 : (float)m * P.ky0;
        float2 u[RX2];
        float dkx = P.dkx;
        int qq = q;                     // opaque copies: the products p * dkx and the twiddles w^{n1 q} are formed where
        asm volatile("" : "+f"(dkx), "+r"(qq));   // they are used, not hoisted out of the item loop (and spilled)
        sfor<0, RX1>([&](auto n1ac) {
          constexpr int N1A = decltype(n1ac)::value;
          if (n1a != N1A) return;
          sfor<0, RX2>([&](auto n2c) {
            constexpr int n2 = decltype(n2c)::value, n1 = N1A + RX1 * n2;
            float2 acc = make_float2(0.f, 0.f);
            sfor<0, CL>([&](auto tc) {
              constexpr int t = decltype(tc)::value, n = n1 + MQ * t;
              // t = 0: n < MQ <= K always retained (kx >= 0); t = CL-1: n >= mx - MQ >= mx - K always retained (kx < 0)
              constexpr bool pos = (t == 0) || (t < CL - 1 && n <= K);
              constexpr bool neg = (t == CL - 1) || (t > 0 && n >= MX_ - K);
              if constexpr (pos || neg) {
                constexpr int p = pos ? n : n - MX_;
                const float2 v = g((p + K) * NKY_ + m);
                const float2 d = gkfft::caxpy(kyv, v, gkfft::cscale((float)p * dkx, make_float2(-v.y, v.x)));  // (i kx -+ ky) v
                acc = cadd(acc, mul_ipow(d, t * qq));
              }
            });
            u[n2] = gkfft::cmul(acc, c_w192.w[(n1 * qq) % MX_]);
          });
        });
        dft<RX2, +1>(u);
        twiddle_row<RX2, +1>(u, tw_tab<MQ>().a + n1a * RX2);
        float2 *o = S + n1a * LD + col;
#pragma unroll
        for (int k2 = 0; k2 < RX2; ++k2) o[k2 * RX1 * LD] = u[k2];
      }
    };
    // ---- X2: inverse x pass 2, in place ----
    auto x2 = [&]() {
      for (int w = tid; w < NC * RX2; w += NTF) {
        const int c = w % NC, k2 = w / NC;
        if (c == NKY_) continue;
        const int col = c < NKY_ ? c : MY_ - (c - NKY_);
        float2 *o = S + k2 * RX1 * LD + col;
        float2 u[RX1];
#pragma unroll
        for (int n1 = 0; n1 < RX1; ++n1) u[n1] = o[n1 * LD];
        dft<RX1, +1>(u);
#pragma unroll
        for (int k1 = 0; k1 < RX1; ++k1) o[k1 * LD] = u[k1];
      }
    };
    // ---- Y1: inverse y pass 1, in place; the Hermitian-extended row is P(y) for 0 < y < nky,
    // conj of what sits at y > my - nky, Re P(0) at y = 0 (R15) and zero in between ----
    auto y1 = [&]() {
      for (int w = tid; w < MQ * RY1; w += NTF) {
        const int r = w % MQ, n1 = w / MQ;
        float2 *row = S + r * LD + n1;
        float2 u[RY2];
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
        dft<RY2, +1>(u);
        twiddle_row<RY2, +1>(u, tw_tab<MY_>().a + n1 * RY2);
#pragma unroll
        for (int k2 = 0; k2 < RY2; ++k2) row[k2 * RY1] = u[k2];
      }
    };
    // ---- Y2: inverse y pass 2, S -> SG (grad(chi) of the work item) ----
    GmaxAcc gm;
    float ef_item = 1.f;   // ExB factor of the work item's plane
    auto y2_to_sg = [&]() {
      for (int w = tid; w < MQ * RY2; w += NTF) {
        const int r = w % MQ, k2 = w / MQ;
        const float2 *o = S + r * LD + k2 * RY1;
        float2 u[RY1];
#pragma unroll
        for (int n1 = 0; n1 < RY1; ++n1) u[n1] = o[n1];
        dft<RY1, +1>(u);
        float2 *d = SG + r * LD + k2 * RY1;
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
          const float2 gg = g0[k1];
          br[k1] = gg.y * u[k1].x - gg.x * u[k1].y;
        }
#pragma unroll
        for (int n1 = 0; n1 < RY1; ++n1) u[n1] = q1[n1];
        dft<RY1, +1>(u);
#pragma unroll
        for (int k1 = 0; k1 < RY1; ++k1) {
          const float2 gg = g1[k1];
          u[k1] = make_float2(br[k1], gg.y * u[k1].x - gg.x * u[k1].y);
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
        const float2 *o = S + (k2 * RX1 - (hi ? H : 0)) * LD;
        float2 u[RX1];
#pragma unroll
        for (int k1 = 0; k1 < RX1; ++k1) {
          const float2 z = o[k1 * LD + m];
          const float2 zc = o[k1 * LD + mm];   // conj applied below
          u[k1] = hi ? make_float2(z.y + zc.y, zc.x - z.x) : make_float2(z.x + zc.x, z.y - zc.y);
        }
        dft<RX1, -1>(u);
        twiddle_row<RX1, -1>(u, tw_tab<MQ>().b + k2 * RX1);
        float2 *d = S + k2 * RX1 * LD + NKY_ + m;
#pragma unroll
        for (int n1 = 0; n1 < RX1; ++n1) d[n1 * LD] = u[n1];
      }
    };
    // ---- XF2: forward x pass 2; C[kap], kap = n1 + RX1 n2, feeds every retained k = kap + MQ t with the factor
    // w^{-q k}: this CTA's partial of the bracket, to its part of ring slot `nlw`, in slab order ----
    auto xf2 = [&](float2 *nlw) {
      for (int w = tid; w < NKY_ * RX1; w += NTF) {
        const int m = w % NKY_, n1 = w / NKY_;
        const float2 *o = S + n1 * LD + NKY_ + m;
        float2 u[RX2];
#pragma unroll
        for (int k2 = 0; k2 < RX2; ++k2) u[k2] = o[k2 * RX1 * LD];
        dft<RX2, -1>(u);
        int qq = q;
        asm volatile("" : "+r"(qq));    // see X1
        // n1 is uniform over a warp (NKY_ is a multiple of 32): one instantiation per n1, retained kx compile-time
        sfor<0, RX1>([&](auto n1c) {
          constexpr int N1 = decltype(n1c)::value;
          if (n1 != N1) return;
          sfor<0, RX2>([&](auto n2c) {
            constexpr int n2 = decltype(n2c)::value, kap = N1 + RX1 * n2;
            sfor<0, CL>([&](auto tc) {
              constexpr int t = decltype(tc)::value, k = kap + MQ * t;
              constexpr bool pos = (t == 0) || (t < CL - 1 && k <= K);
              constexpr bool neg = (t == CL - 1) || (t > 0 && k >= MX_ - K);
              if constexpr (pos || neg) {
                constexpr int p = pos ? k : k - MX_;
                __stcg(&nlw[(p + K) * NKY_ + m], gkfft::cmulc(u[n2], c_w192.w[(k * qq) % MX_]));
              }
            });
          });
        });
      }
    };

    const long long jstride = (long long)P.nmu * P.ns * P.slab;
    uint32_t parity = 0;
    int u = 0;
    for (int w = cid; w < A.nwork; w += ncl) {
      const int i = w % P.ns;
      const int c = (w / P.ns) % P.nchunk;
      const int al = w / (P.ns * P.nchunk);
      const int l = al % P.nmu, a = al / P.nmu;
      const long long base0 = (((long long)a * P.nv * P.nmu + l) * P.ns + i) * P.slab;
      const int j0 = c * P.jchunk, j1 = min(P.nv, (c + 1) * P.jchunk);
      ef_item = P.ef[i];
      // the first slab of the item lands while grad(chi) is built (the staging buffer was last read
      // by the X1 of the previous slab, which every thread of the role has left)
      if (tid == 0) bulk_load(stg, (const ST *)A.y + (base0 + (long long)j0 * jstride), slab * sizeof(ST), mbar);
      {
        const float *j0p = P.J0 + (((long long)a * P.nmu + l) * P.ns + i) * P.slab;
        const float2 *php = A.phi + (long long)i * P.slab;
        x1([&](int e) { return gkfft::cscale(__ldg(j0p + e), __ldg(php + e)); });   // chi = J0 phi (a3)
      }
      fsync();
      x2();
      fsync();
      y1();
      fsync();
      y2_to_sg();
      fsync();
      for (int j = j0; j < j1; ++j, ++u) {
        mbar_wait(mbar, parity);
        parity ^= 1u;
        x1([&](int e) { return Cv<ST>::ld(stg, e); });
        fsync();
        // every thread has left X1: the staging buffer may take the next slab
        if (tid == 0 && j + 1 < j1)
          bulk_load(stg, (const ST *)A.y + (base0 + (long long)(j + 1) * jstride), slab * sizeof(ST), mbar);
        x2();
        fsync();
        y1();
        fsync();
        yf();
        fsync();
        f2();
        fsync();
        xf1();
        fsync();
        // ring slot must have been consumed by the streaming roles of all CTAs (slab u - 2)
        if (u >= GK_WS_NL_RING) mbar_wait_cluster(free_ + (u & 1), ((u >> 1) - 1) & 1);
        xf2(nlring + ((size_t)(u & 1) * CL + q) * slab);
        // XF2 reads only the dead columns, which X1/X2 of the next slab do not write; the barrier orders the
        // partial of every thread before the release below
        fsync();
        if (tid == 0) {
          asm volatile("fence.acq_rel.cluster;" ::: "memory");
#pragma unroll
          for (int r = 0; r < CL; ++r) mbar_arrive_remote(full + (u & 1), r);
        }
      }
    }
    gm.flush(A.gmax);
  } else {
    // =============================== streaming role ===============================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(RE));
    using HK = Ws4Hooks<ST, NKY_, NKX_, CL, NTE>;
    const int et = tid - NTF;
    HK h{A.chis + (size_t)blockIdx.x * (3 * HK::SHARE), nlring, full, free_, eblk,
         (float2 *)(eblk + (NTE / 32) * GK_EB_N), fslots, et};
    const int row0 = q * ROWS, nrows = min(ROWS, NKX_ - row0);
    const bool want_flux = A.fluxp != nullptr && A.mode == 1;
    if ((et & 31) == 0) { double *fs = h.fluxslot(); fs[0] = fs[1] = fs[2] = 0.0; }
    int u = 0, a_prev = -1;
    for (int w = cid; w < A.nwork; w += ncl) {
      const int i = w % P.ns;
      const int c = (w / P.ns) % P.nchunk;
      const int al = w / (P.ns * P.nchunk);
      const int l = al % P.nmu, a = al / P.nmu;
      if (want_flux && a != a_prev) {   // species are visited in increasing order: one write per (warp, species)
        if ((et & 31) == 0) flux_flush(P, A.fluxp, blockIdx.x, NTE / 32, et >> 5, a_prev, h.fluxslot());
        a_prev = a;
      }
      // chi and D_s chi at the thread's own points: written and read back by the same thread (L2 scratch)
      epi_build_chis<ST, NKY_, NTE, ROWS>(P, A, a, l, i, row0, nrows, et, [&](int k, int which, const float2 (&v)[HK::M::PV]) {
        const int el = (et / HK::M::VPR + k * HK::M::RS) * NKY_ + (et % HK::M::VPR) * HK::M::PV;
        float4 *o = (float4 *)(h.chis + which * HK::SHARE + el);
#pragma unroll
        for (int x = 0; x < HK::M::PV; x += 2) __stcg(o + x / 2, make_float4(v[x].x, v[x].y, v[x + 1].x, v[x + 1].y));
      });
      epi_item<ST, NKY_, NKX_, NTE, ROWS, NB>(P, A, h, et, a, l, i, c, row0, nrows, u);
    }
    if (want_flux && (et & 31) == 0) flux_flush(P, A.fluxp, blockIdx.x, NTE / 32, et >> 5, a_prev, h.fluxslot());
  }
  // no CTA leaves while its peers may still arrive at its barriers
  cluster_sync_all();
}

}  // namespace gk
