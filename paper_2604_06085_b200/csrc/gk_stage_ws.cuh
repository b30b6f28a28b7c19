// gk_stage_ws.cuh -- warp-specialised form of the fused RK-stage kernel for the nonlinear
// BASELINE shapes (steps a3-a6 of DESIGN.md).  Product path; shares nothing with oracle/.
//
// One persistent CTA per SM, two roles:
//   FFT warps (NTF threads)      bracket (term III) of slab u: shared-memory 2-D FFTs exactly as in
//                                gk_stage_kernel; the retained spectrum goes to a 2-deep ring in
//                                the CTA's global scratch (L2-resident, 21 KB per slab on cfg3)
//   epilogue warps (NTE threads) linear terms + RK update + moment of slab u-1: the HBM/L2-latency
//                                bound part (13 operands per point), which in the unspecialised
//                                kernel was a phase of its own during which the FFT pipes idle
// so the memory phase of one slab runs under the arithmetic of the next.  Hand-off by named
// barriers: FULL[b] (FFT arrives, epilogue waits), FREE[b] (epilogue arrives, FFT waits before it
// overwrites ring slot b two slabs later).  chi / D_s chi of an item live in a 3-deep ring so the
// FFT warps may start the next item while the epilogue warps finish the previous one.
#pragma once

namespace gk {

__device__ __forceinline__ void bar_sync_n(int id, int n) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory");
}
__device__ __forceinline__ void bar_arrive_n(int id, int n) {
  __threadfence_block();  // the other role reads what this thread wrote (global scratch rings)
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory");
}

#define GK_WS_CHI_RING 3
#define GK_WS_NL_RING 2
#define GK_WS_BAR_FFT 1
#define GK_WS_BAR_FULL 2
#define GK_WS_BAR_FREE 4

// Epilogue role of the warp-specialised kernels: linear terms + RK update + moment of slab u once the
// FFT role has published its bracket in ring slot u & 1 (BAR_FULL), then releases the slot (BAR_FREE).
template <class ST, int NKY_, int NKX_, int NTF, int NTE>
__device__ __forceinline__ void ws_epilogue_role(const GkDev &P, const GkStageArgs &A, const float2 *chis_cta,
                                                 const float2 *nl_cta, int tid) {
  constexpr int NT = NTF + NTE;
  constexpr int nky = NKY_, nkx = NKX_;
  constexpr int K = (nkx - 1) / 2, slab = nkx * nky;
  constexpr int BAR_FULL = GK_WS_BAR_FULL, BAR_FREE = GK_WS_BAR_FREE;
  static_assert(NTE % NKY_ == 0, "an epilogue sweep covers whole ky rows");
  // =============================== epilogue role ================================
  const int et = tid - NTF;
  constexpr int EPT = (slab + NTE - 1) / NTE;
  constexpr int RS = NTE / nky;  // kx rows per sweep of the role's threads
  const int m = et % nky, ip0 = et / nky;
  const float fmf = (float)m, pk0 = (float)(ip0 - K);
  const float scale = 0.25f * P.fftnorm;  // 1/2 (bracket) * 1/2 (two-for-one unpack) / (mx my)
  int u = 0, it = 0;
  for (int w = blockIdx.x; w < A.nwork; w += gridDim.x, ++it) {
    const int i = w % P.ns;
    const int c = (w / P.ns) % P.nchunk;
    const int al = w / (P.ns * P.nchunk);
    const int l = al % P.nmu, a = al / P.nmu;
    ItemCtx I;
    make_item_ctx(P, a, l, i, I);
    const float2 *chis = chis_cta + (it % GK_WS_CHI_RING) * 3 * slab;
    float2 macc[EPT];
#pragma unroll
    for (int k = 0; k < EPT; ++k) macc[k] = make_float2(0.f, 0.f);
    const bool interior = (i >= 2 && i < P.ns - 2);
    const int j1 = min(P.nv, (c + 1) * P.jchunk);
    for (int j = c * P.jchunk; j < j1; ++j, ++u) {
      SlabCtx C;
      make_slab_ctx(P, I, j, C);
      EpiPtrs<ST> Q;
      make_epi_ptrs<ST>(A, C, chis, slab, Q);
      // L2 prefetch of what the NEXT slab reads from HBM for the first time (slab j+3 of the
      // state, f_n and the accumulator of slab j+1)
      if (P.prefetch && j + 1 < j1) {
        constexpr int nline = (slab * (int)sizeof(ST) + 127) / 128;
        for (int t = et; t < nline; t += NTE) {
          const long long nb = C.base + I.jstride;
          if (j + 3 < P.nv) asm volatile("prefetch.global.L2 [%0];" ::"l"((const char *)(Q.yb + 3 * I.jstride) + t * 128));
          if (A.mode == 2) asm volatile("prefetch.global.L2 [%0];" ::"l"((const char *)((const ST *)A.fn + nb) + t * 128));
          if (A.mode >= 2) asm volatile("prefetch.global.L2 [%0];" ::"l"((const char *)((const ST *)A.acc + nb) + t * 128));
        }
      }
      const float2 *nlr = nl_cta + (u & 1) * slab;
      bar_sync_n(BAR_FULL + (u & 1), NT);
      auto sweep = [&](auto modec, auto intc) {
#pragma unroll
        for (int k = 0; k < EPT; ++k) {
          const int e = et + k * NTE;
          if (k + 1 < EPT || e < slab) {
            const float2 out = rhs_point<ST, decltype(modec)::value, decltype(intc)::value != 0>(
                P, A, I, C, Q, slab, e, ip0 + k * RS, m, pk0 + (float)(k * RS), fmf, __ldcg(&nlr[e]), scale);
            macc[k] = cadd(macc[k], out);
            // one point's 13 operands in flight per thread is all the registers allow: keep the
            // compiler from hoisting the next point's loads above this one's arithmetic
            asm volatile("" ::: "memory");
          }
        }
      };
      auto by_plane = [&](auto modec) {
        if (interior) sweep(modec, gkfft::IC<1>{});
        else sweep(modec, gkfft::IC<0>{});
      };
      switch (A.mode) {
        case 0: by_plane(gkfft::IC<0>{}); break;
        case 1: by_plane(gkfft::IC<1>{}); break;
        case 2: by_plane(gkfft::IC<2>{}); break;
        default: by_plane(gkfft::IC<3>{}); break;
      }
      bar_arrive_n(BAR_FREE + (u & 1), NT);
    }
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
}

template <class ST, int MX_, int MY_, int NKY_, int NKX_, int NTF, int NTE>
__global__ void __launch_bounds__(NTF + NTE, 1)
gk_stage_ws_kernel(const __grid_constant__ GkDev P, const __grid_constant__ GkStageArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NT = NTF + NTE;
  constexpr int mx = MX_, my = MY_, nky = NKY_, nkx = NKX_;
  constexpr int K = (nkx - 1) / 2, slab = nkx * nky;
  constexpr int ldx = 2 * nky + 1, ldy = my | 1;
  static_assert(NTF % 32 == 0 && NTE % 32 == 0, "roles are whole warps");
  static_assert(NTE % NKY_ == 0, "an epilogue sweep covers whole ky rows");
  constexpr int BAR_FFT = GK_WS_BAR_FFT, BAR_FULL = GK_WS_BAR_FULL, BAR_FREE = GK_WS_BAR_FREE;
  const int tid = threadIdx.x;
  float2 *chis_cta = A.chis + (long long)blockIdx.x * (GK_WS_CHI_RING * 3 * slab);
  float2 *nl_cta = A.nlbuf + (long long)blockIdx.x * (GK_WS_NL_RING * slab);

  if (tid < NTF) {
    // =============================== FFT role =====================================
    const int rc = P.rc, half = rc / 2;
    const gkfft::NamedSync<BAR_FFT, NTF> fsync;
    float2 *sp = (float2 *)smem_raw;
    float2 *twx = sp; sp += mx;
    float2 *twy = sp; sp += my;
    float2 *SA = sp; sp += mx * ldx;
    float2 *SW = sp; sp += rc * ldy;
    float2 *SG = P.gchi_in_smem ? sp : A.gchi + (long long)blockIdx.x * mx * ldy;
    for (int t = tid; t < mx; t += NTF) twx[t] = P.twx[t];
    for (int t = tid; t < my; t += NTF) twy[t] = P.twy[t];
    fsync();

    // real-space gradients of the spectral slab `g` (callable: slab index -> value), chunk by chunk
    auto to_real = [&](auto g, auto sink) {
      gkfft::nat2perm_load<MX_, +1>(SA, 2 * nky, 1, ldx, twx, tid, NTF,
                                    [&](int c, int nbase, auto offc, auto spanc) {
        constexpr int off = decltype(offc)::value, hi = off + decltype(spanc)::value - 1;
        const int n = nbase + off;
        int p = 0;
        if constexpr (hi <= K) {
          p = n;                                   // always a retained kx >= 0
        } else if constexpr (off > K && hi < MX_ - K) {
          return make_float2(0.f, 0.f);            // always zero padding: nothing is loaded
        } else if constexpr (off >= MX_ - K) {
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
        return gkfft::caxpy(kyv, v, gkfft::cscale(kxv, make_float2(-v.y, v.x)));  // (i kx -+ ky) v
      }, fsync);
      fsync();
      for (int r0 = 0; r0 < mx; r0 += rc) {
        gkfft::nat2perm_load<MY_, +1>(SW, rc, ldy, 1, twy, tid, NTF,
                                      [&](int r, int nbase, auto offc, auto spanc) {
          constexpr int off = decltype(offc)::value, span = decltype(spanc)::value, hi = off + span - 1;
          const int y = nbase + off;
          const float2 *row = SA + (r0 + r) * ldx;
          auto upper = [&](int m) {                // conj Q
            const float2 q = row[nky + m];
            return make_float2(q.x, -q.y);
          };
          if constexpr (off == 0 && span == 1) {
            return make_float2(row[0].x, 0.f);     // ky = 0: real part only (R15)
          } else if constexpr (off > 0 && hi < NKY_) {
            return row[y];
          } else if constexpr (off >= NKY_ && hi <= MY_ - NKY_) {
            return make_float2(0.f, 0.f);
          } else if constexpr (off > MY_ - NKY_) {
            return upper(my - y);
          } else {
            if (y == 0) return make_float2(row[0].x, 0.f);
            if (y < nky) return row[y];
            if (y > my - nky) return upper(my - y);
            return make_float2(0.f, 0.f);
          }
        }, fsync);
        fsync();
        sink(r0);
        fsync();
      }
    };

    int u = 0, it = 0;
    for (int w = blockIdx.x; w < A.nwork; w += gridDim.x, ++it) {
      const int i = w % P.ns;
      const int c = (w / P.ns) % P.nchunk;
      const int al = w / (P.ns * P.nchunk);
      const int l = al % P.nmu, a = al / P.nmu;
      float2 *chis = chis_cta + (it % GK_WS_CHI_RING) * 3 * slab;
      build_chis(P, A, a, l, i, slab, nky, chis, tid, NTF);
      fsync();
      to_real([&](int e) { return __ldcg(&chis[e]); },
              [&](int r0) {
                for (int q = tid; q < rc * my; q += NTF) {
                  const int r = q / my, y = q - r * my;
                  SG[(r0 + r) * ldy + y] = SW[r * ldy + y];
                }
              });
      const long long jstride = (long long)P.nmu * P.ns * P.slab;
      const long long base0 = (((long long)a * P.nv * P.nmu + l) * P.ns + i) * P.slab;
      const int j1 = min(P.nv, (c + 1) * P.jchunk);
      for (int j = c * P.jchunk; j < j1; ++j, ++u) {
        const ST *yb = (const ST *)A.y + (base0 + (long long)j * jstride);
        to_real([&](int e) { return Cv<ST>::ldg(yb, e); },
                [&](int r0) {
                  // bracket d_y chi d_x f - d_x chi d_y f, rows (p, p+rc/2) packed as (re, im), evaluated
                  // inside the first pass of the forward y-transform; only the retained ky are stored
                  auto keep = [&](int p, int nbase, auto offc, auto spanc, float2 v) {
                    constexpr int off = decltype(offc)::value, hi = off + decltype(spanc)::value - 1;
                    const int m = nbase + off;
                    if constexpr (off >= NKY_ && hi <= MY_ - NKY_) {
                    } else if constexpr (hi < NKY_ || off > MY_ - NKY_) {
                      SW[p * ldy + m] = v;
                    } else {
                      if (m < nky || m > my - nky) SW[p * ldy + m] = v;
                    }
                  };
                  if (P.gchi_in_smem) {
                    gkfft::perm2nat_fused<MY_, -1>(SW, half, ldy, 1, twy, tid, NTF,
                        [&](int p, int q) {
                          const float2 g0 = SG[(r0 + p) * ldy + q], g1 = SG[(r0 + p + half) * ldy + q];
                          const float2 f0 = SW[p * ldy + q], f1 = SW[(p + half) * ldy + q];
                          return make_float2(g0.y * f0.x - g0.x * f0.y, g1.y * f1.x - g1.x * f1.y);
                        }, keep, fsync);
                  } else {  // grad(chi) in global scratch: coalesced product pass (lane = y) first
                    for (int q = tid; q < half * my; q += NTF) {
                      const int p = q / my, y = q - p * my;
                      const float2 g0 = SG[(r0 + p) * ldy + y], g1 = SG[(r0 + p + half) * ldy + y];
                      const float2 f0 = SW[p * ldy + y], f1 = SW[(p + half) * ldy + y];
                      SW[p * ldy + y] = make_float2(g0.y * f0.x - g0.x * f0.y, g1.y * f1.x - g1.x * f1.y);
                    }
                    fsync();
                    gkfft::perm2nat_fused<MY_, -1>(SW, half, ldy, 1, twy, tid, NTF,
                        [&](int p, int q) { return SW[p * ldy + q]; }, keep, fsync);
                  }
                  fsync();
                  // unpack the two real rows, keep only the retained ky: overwrite A's P columns
                  for (int q = tid; q < half * nky; q += NTF) {
                    const int p = q / nky, m = q - p * nky;
                    const float2 z = SW[p * ldy + m];
                    float2 zc = SW[p * ldy + (m == 0 ? 0 : my - m)];
                    zc.y = -zc.y;
                    SA[(r0 + p) * ldx + m] = make_float2(z.x + zc.x, z.y + zc.y);
                    SA[(r0 + p + half) * ldx + m] = make_float2(z.y - zc.y, zc.x - z.x);
                  }
                });
        // ring slot must have been consumed by the epilogue of slab u-2
        if (u >= GK_WS_NL_RING) bar_sync_n(BAR_FREE + (u & 1), NT);
        float2 *nlw = nl_cta + (u & 1) * slab;
        // forward x-transform of the nky columns; only |p| <= K is stored, in slab order
        gkfft::perm2nat_fused<MX_, -1>(SA, nky, 1, ldx, twx, tid, NTF,
            [&](int cc, int q) { return SA[q * ldx + cc]; },
            [&](int cc, int nbase, auto offc, auto spanc, float2 v) {
              constexpr int off = decltype(offc)::value, hi = off + decltype(spanc)::value - 1;
              const int n = nbase + off;
              if constexpr (off > K && hi < MX_ - K) {
              } else if constexpr (hi <= K) {
                __stcg(&nlw[(n + K) * nky + cc], v);
              } else if constexpr (off >= MX_ - K) {
                __stcg(&nlw[(n - mx + K) * nky + cc], v);
              } else {
                if (n <= K) __stcg(&nlw[(n + K) * nky + cc], v);
                else if (n >= mx - K) __stcg(&nlw[(n - mx + K) * nky + cc], v);
              }
            }, fsync);
        fsync();  // SA is rewritten by the next slab
        bar_arrive_n(BAR_FULL + (u & 1), NT);
      }
    }
    // consume the epilogue's last arrivals so that no barrier is left half-way at exit
    for (int v = max(0, u - GK_WS_NL_RING); v < u; ++v) bar_sync_n(BAR_FREE + (v & 1), NT);
  } else {
    ws_epilogue_role<ST, NKY_, NKX_, NTF, NTE>(P, A, chis_cta, nl_cta, tid);
  }
}

}  // namespace gk
