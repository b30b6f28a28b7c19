// gk_stage_point.cuh -- the RK stage with term III off on SMALL (kx, ky) planes (nkx * nky < 256: the zonal-flow and
// single-mode linear benchmarks, run 3 x 1 or a few x 1 modes against 128 x 128 x 16 points
// along s, vpar, mu).  A slab cannot occupy a CTA there, so one THREAD takes one grid point: chi = J0 phi and D_s chi
// of every (species, mu, s) plane are built by a small kernel first (steps a3), then the point kernel evaluates the
// linear terms and the RK update (a4, a6) with the same per-point routine as the generic kernel (rhs_point); the
// velocity-space moment of the new state (a1 of the next stage) is left to gk_moment_kernel.
// Product path; shares nothing with oracle/.
#pragma once

namespace gk {

// chis[((a nmu + l) ns + i)][3][slab]: chi, D_s chi for v > 0, D_s chi for v < 0.  One CTA per (a, l, i).
// (A template only so that every storage type's translation unit gets its own copy.)
template <class ST>
__global__ void __launch_bounds__(128) gk_chis_kernel(const __grid_constant__ GkDev P, const __grid_constant__ GkStageArgs A) {
  const int w = blockIdx.x;
  const int i = w % P.ns, l = (w / P.ns) % P.nmu, a = w / (P.ns * P.nmu);
  build_chis(P, A, a, l, i, (int)P.slab, P.nky, A.chis + (size_t)w * 3 * P.slab, threadIdx.x, 128);
}

template <class ST>
__global__ void __launch_bounds__(256) gk_stage_point_kernel(const __grid_constant__ GkDev P, const __grid_constant__ GkStageArgs A) {
  const long long idx = (long long)blockIdx.x * 256 + threadIdx.x;
  if (idx >= P.ntot) return;
  const int slab = (int)P.slab;
  const int e = (int)(idx % slab);
  long long t = idx / slab;
  const int i = (int)(t % P.ns); t /= P.ns;
  const int l = (int)(t % P.nmu); t /= P.nmu;
  const int j = (int)(t % P.nv);
  const int a = (int)(t / P.nv);
  ItemCtx I;
  make_item_ctx(P, a, l, i, I);
  SlabCtx C;
  make_slab_ctx(P, I, j, C);
  EpiPtrs<ST> Q;
  make_epi_ptrs<ST>(A, C, A.chis + ((size_t)(a * P.nmu + l) * P.ns + i) * 3 * slab, slab, Q);
  const int ip = e / P.nky, m = e - ip * P.nky;
  const float pk = (float)(ip - P.K), fmf = (float)m;
  const float2 zero = make_float2(0.f, 0.f);
  float fsum = 0.f;
  switch (A.mode) {
    case 0: rhs_point<ST, 0, false>(P, A, I, C, Q, slab, e, ip, m, pk, fmf, zero, 0.f, fsum); break;
    case 1: rhs_point<ST, 1, false>(P, A, I, C, Q, slab, e, ip, m, pk, fmf, zero, 0.f, fsum); break;
    case 2: rhs_point<ST, 2, false>(P, A, I, C, Q, slab, e, ip, m, pk, fmf, zero, 0.f, fsum); break;
    default: rhs_point<ST, 3, false>(P, A, I, C, Q, slab, e, ip, m, pk, fmf, zero, 0.f, fsum); break;
  }
}

}  // namespace gk
