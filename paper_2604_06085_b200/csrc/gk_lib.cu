// gk_lib.cu -- C ABI of libgk (include/gk.h): context, table upload, launch logic.
// Product path.  No CPU fallback: every entry point needs a CUDA device.
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <new>
#include <stdexcept>
#include <string>
#include <vector>

#include "../../include/gk.h"
#include "../../include/gk_debug.h"
#include "gk_kernels.cuh"
#include "gk_pick.h"
#include "gk_tables.h"

namespace {

constexpr size_t kSmemMax = 232448;  // 227 KB opt-in shared memory per CTA on sm_100 (static + dynamic)
constexpr size_t kSmemDyn = kSmemMax - 1024;  // dynamic part the generic kernel may plan with (it has some static arrays)

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

template <class T> struct DevBuf {
  T *p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
};

}  // namespace

struct gk_ctx {
  gk_grid grid;
  gk_salpha geo;
  gk_opts opts;
  std::vector<gk_species> species;
  gkt::Tables T;
  GkDev P;
  cudaStream_t stream = nullptr;
  std::vector<void *> dev_allocs;
  std::string err;
  bool poisoned = false;
  int num_sms = 0;
  int stage_grid = 0;
  int stage_threads = 512, stage_kind = 0, stage_cluster = 1, stage_nsh = 1;
  size_t stage_smem = 0;
  size_t elem_bytes = 8;
  // workspace
  void *ws = nullptr;
  size_t ws_bytes = 0;
  size_t off_mom = 0, off_phi = 0, off_gchi = 0, off_chis = 0, off_nl = 0, off_ya = 0, off_yb = 0, off_acc = 0;
  const void *stage_fn = nullptr;  // the stage-kernel instantiation chosen at create time
  const void *stage_fn2 = nullptr; // GK_KIND_POINT: gk_chis_kernel
  int stage_nwork = 0;
  size_t need_rhs = 0, need_full = 0;
  bool mom_valid_for_f = false;  // inside gk_rk4_steps only
  long long launches = 0;
  // profiling of the stage kernel
  bool profiling = false;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev;
  // gk_rk4_batch_host: copy streams and per-buffer events, created on first use
  cudaStream_t s_up = nullptr, s_down = nullptr;
  cudaEvent_t e_in[2] = {nullptr, nullptr}, e_done[2] = {nullptr, nullptr}, e_out[2] = {nullptr, nullptr};
  size_t ev_used = 0;
  // diagnostics: one context-owned device block (allocated by gk_create, never by a hot call):
  // [gmax | flux_out 3*nsp | spectra nkx+nky | flux partials part_slots x nsp x 3]
  unsigned int *d_gmax = nullptr;
  double *d_flux_out = nullptr, *d_spec = nullptr, *d_part = nullptr;
  int part_slots = 0;
  bool diag = false;            // gk_set_diagnostics: fluxes of f_n folded into every stage-1 launch
  bool flux_valid = false;
  double dt_lin = 0, dt_field = 0;   // create-time CFL bounds (R22, R23)
};

namespace {

int fail(gk_ctx *c, int code, const std::string &msg) {
  if (c) {
    c->err = msg;
    if (code == GK_ECUDA) c->poisoned = true;
  }
  return code;
}

#define GK_CUDA(ctx, call)                                                                   \
  do {                                                                                       \
    cudaError_t e_ = (call);                                                                 \
    if (e_ != cudaSuccess)                                                                   \
      return fail(ctx, GK_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));        \
  } while (0)

template <class T>
int upload(gk_ctx *c, const std::vector<double> &src, const T **dst) {
  std::vector<T> tmp(src.size());
  for (size_t i = 0; i < src.size(); ++i) tmp[i] = (T)src[i];
  void *p = nullptr;
  cudaError_t e = cudaMalloc(&p, std::max<size_t>(tmp.size(), 1) * sizeof(T));
  if (e != cudaSuccess) return fail(c, e == cudaErrorMemoryAllocation ? GK_ENOMEM : GK_ECUDA,
                                    std::string("cudaMalloc(table): ") + cudaGetErrorString(e));
  c->dev_allocs.push_back(p);
  GK_CUDA(c, cudaMemcpy(p, tmp.data(), tmp.size() * sizeof(T), cudaMemcpyHostToDevice));
  *dst = (const T *)p;
  return GK_OK;
}

int smallest_pad(int nmin) {  // smallest supported 2^a 3^b (b<=1) length >= nmin
  static const int sizes[] = {2, 3, 4, 6, 8, 12, 16, 24, 32, 48, 64, 96, 128, 192, 256};
  for (int s : sizes)
    if (s >= nmin) return s;
  return -1;
}

template <class ST> void launch_moment(gk_ctx *c, const void *f, float2 *mom) {
  const GkDev &P = c->P;
  const int nblk_slab = (int)((P.slab + 255) / 256);
  const long long nwork = (long long)P.nsp * P.nmu * P.nchunk * P.ns;
  gk::gk_moment_kernel<ST><<<(unsigned)(nwork * nblk_slab), 256, 0, c->stream>>>(P, f, mom);
  ++c->launches;
}

void stage_config(const gk_ctx *c, cudaLaunchConfig_t &cfg, cudaLaunchAttribute &attr) {
  std::memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(c->stage_grid);
  cfg.blockDim = dim3(c->stage_threads);
  cfg.dynamicSmemBytes = c->stage_smem;
  cfg.stream = c->stream;
  if (c->stage_cluster > 1) {   // thread-block cluster: the CTAs of a cluster share one work item
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = c->stage_cluster;
    attr.val.clusterDim.y = 1;
    attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
  }
}

void launch_stage(gk_ctx *c, const GkStageArgs &A) {
  void *args[2] = {(void *)&c->P, (void *)&A};
  if (c->stage_kind == GK_KIND_POINT) {   // tiny (kx,ky) planes: chi planes first, then one thread per grid point
    cudaLaunchKernel(c->stage_fn2, dim3(c->P.nsp * c->P.nmu * c->P.ns), dim3(128), args, 0, c->stream);
    cudaLaunchKernel(c->stage_fn, dim3((unsigned)((c->P.ntot + 255) / 256)), dim3(256), args, 0, c->stream);
    c->launches += 2;
    return;
  }
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute attr;
  stage_config(c, cfg, attr);
  cudaLaunchKernelExC(&cfg, c->stage_fn, args);
  ++c->launches;
}

constexpr int kFluxBlocks = 4096;   // most blocks (per species) gk_flux_kernel is launched with

template <class ST> void launch_flux(gk_ctx *c, const void *f, const float2 *phi) {
  dim3 grid((unsigned)std::min<long long>(kFluxBlocks, (c->P.ntot / c->P.nsp + 255) / 256), c->P.nsp);
  gk::gk_flux_kernel<ST><<<grid, 256, 0, c->stream>>>(c->P, f, phi, c->d_part);
  gk::gk_flux_sum_kernel<<<1, 32, 0, c->stream>>>(c->P, c->d_part, (int)grid.x, c->d_flux_out);
  c->launches += 2;
}

#ifdef GK_ONLY_C64  // developer builds (GK_FAST_BUILD=1): complex64 storage only, 3x faster to compile
#define GK_BY_STORAGE(ctx, CALL) do { CALL(float2); } while (0)
#else
#define GK_BY_STORAGE(ctx, CALL)                         \
  do {                                                   \
    if ((ctx)->opts.storage == 0) { CALL(float2); }      \
    else if ((ctx)->opts.storage == 1) { CALL(__half2); } \
    else { CALL(__nv_bfloat162); }                       \
  } while (0)
#endif

int check_launch(gk_ctx *c, const char *what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(c, GK_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
  return GK_OK;
}

void stage_launch(gk_ctx *c, const GkStageArgs &A) {
  const bool prof = c->profiling;
  if (prof) {
    if (c->ev_used == c->ev.size()) {
      cudaEvent_t a, b;
      cudaEventCreate(&a);
      cudaEventCreate(&b);
      c->ev.push_back({a, b});
    }
    cudaEventRecord(c->ev[c->ev_used].first, c->stream);
  }
  launch_stage(c, A);
  if (c->stage_kind == GK_KIND_POINT && A.mom) {   // this kind leaves the moment of the new state to the moment kernel
#define GK_CALL(ST) launch_moment<ST>(c, A.out, A.mom)
    GK_BY_STORAGE(c, GK_CALL);
#undef GK_CALL
  }
  if (prof) {
    cudaEventRecord(c->ev[c->ev_used].second, c->stream);
    ++c->ev_used;
  }
}

// `gmax`: the CFL maximum to clear for the stage launch that follows this field solve (GmaxAcc), or nullptr if
// none follows (the public gk_field_solve: the bound of the most recent stage launch must survive it).
int solve_phi_from_planes(gk_ctx *c, float2 *mom, float2 *phi, unsigned int *gmax) {
  const GkDev &P = c->P;
  gk::gk_phi_kernel<<<(unsigned)((P.nphi + 255) / 256), 256, 0, c->stream>>>(P, mom, phi, gmax);
  ++c->launches;
  if (P.adiabatic) {
    gk::gk_zonal_kernel<<<P.nkx, 32, 0, c->stream>>>(P, phi);
    ++c->launches;
  }
  return check_launch(c, "field solve");
}

int usable(gk_ctx *c) {
  if (!c) return GK_EINVAL;
  if (c->poisoned) return GK_ECUDA;
  return GK_OK;
}

}  // namespace

extern "C" {

#ifndef GK_SRC_HASH
#define GK_SRC_HASH "unknown"
#endif
// "src:<hash>" = build.py's src_hash() of csrc/ at compile time (bench.py matches ncu captures against it)
const char *gk_version(void) { return "gk-b200 0.1 (sm_100a) src:" GK_SRC_HASH; }

const char *gk_last_error(const gk_ctx *c) { return c ? c->err.c_str() : "null context"; }

}  // extern "C"

namespace {

int create_impl(const gk_grid *g, const gk_species *sp, const gk_salpha *geo, const gk_opts *o,
                void *cuda_stream, gk_ctx **out) {
  if (!g || !sp || !geo || !o || !out) return GK_EINVAL;
  *out = nullptr;
  if (g->nkx < 1 || g->nkx % 2 == 0 || g->ns < 4 || g->nvpar < 4 || g->nky < 1 || g->nmu < 1 ||
      g->ikxspace < 1 || o->nspecies < 1 || o->nspecies > GK_MAX_SPECIES || o->storage < 0 ||
      o->storage > 2 || !(g->vpar_max > 0) || (g->mu_grid != 0 && g->mu_grid != 1) ||
      (o->geometry != 0 && o->geometry != 1) || !(geo->eps > 0) || !(geo->eps < 1) || !(geo->q > 0))
    return GK_EINVAL;
  for (int a = 0; a < o->nspecies; ++a)
    if (sp[a].Z == 0 || !(sp[a].mass > 0) || !(sp[a].temp > 0)) return GK_EINVAL;
#ifdef GK_ONLY_C64
  if (o->storage != 0) return GK_EUNSUPPORTED;
#endif
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return GK_ECUDA;  // no CPU fallback

  gk_ctx *c = new (std::nothrow) gk_ctx();
  if (!c) return GK_ENOMEM;
  *out = c;  // returned even on failure so that gk_last_error() can be read; caller destroys it
  c->grid = *g; c->geo = *geo; c->opts = *o;
  c->species.assign(sp, sp + o->nspecies);
  c->stream = (cudaStream_t)cuda_stream;
  c->elem_bytes = (o->storage == 0) ? 8 : 4;
  int dev = 0;
  GK_CUDA(c, cudaGetDevice(&dev));
  GK_CUDA(c, cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev));

  gkt::build_tables(*g, sp, *geo, *o, c->T);
  const gkt::Tables &T = c->T;
  GkDev &P = c->P;
  std::memset(&P, 0, sizeof(P));
  P.nsp = T.nsp; P.nv = T.nv; P.nmu = T.nmu; P.ns = T.ns; P.nkx = T.nkx; P.nky = T.nky; P.K = T.K;
  P.ikx = g->ikxspace;
  P.adiabatic = o->adiabatic_electrons ? 1 : 0;
  P.mask = (o->term_mask <= 0) ? GK_T_ALL : o->term_mask;
  if (!o->nonlinear) P.mask &= ~GK_T_III;
  P.hyp_x = (P.mask & GK_T_HYP) ? (float)o->disp_x : 0.f;
  P.hyp_y = (P.mask & GK_T_HYP) ? (float)o->disp_y : 0.f;
  P.storage = o->storage;
  P.ds_inv = (float)(1.0 / T.ds); P.dv_inv = (float)(1.0 / T.dv);
  P.nu_s = (float)o->disp_par; P.nu_v = (float)o->disp_vp;
  P.dkx = (float)T.dkx; P.ky0 = (float)g->ky0;
  P.kxmax = (float)(T.K * T.dkx); P.kymax = (float)((T.nky - 1) * g->ky0);
  P.invK = T.K > 0 ? (float)(1.0 / T.K) : 0.f;
  P.invM = T.nky > 1 ? (float)(1.0 / (T.nky - 1)) : 0.f;
  P.ae = o->adiabatic_electrons ? (float)(o->ne / o->te) : 0.f;
  P.slab = (long long)T.nkx * T.nky;
  P.nphi = (long long)T.ns * P.slab;
  P.ntot = (long long)T.nsp * T.nv * T.nmu * P.nphi;
  if (P.slab > (long long)GK_SLAB_MAX)
    return fail(c, GK_EUNSUPPORTED, "nkx*nky exceeds the per-CTA slab capacity (8192)");
  for (int a = 0; a < T.nsp; ++a) {
    GkSpeciesDev &S = P.sp[a];
    S.Z = (float)sp[a].Z; S.T = (float)sp[a].temp; S.mass = (float)sp[a].mass; S.dens = (float)sp[a].dens;
    S.vR = (float)T.vR[a]; S.rlt = (float)sp[a].rlt; S.rln = (float)sp[a].rln;
    S.ToverZ = (float)(sp[a].temp / sp[a].Z); S.ZoverT = (float)(sp[a].Z / sp[a].temp);
    S.momfac = (float)(sp[a].Z * sp[a].dens * 2.0 * gkt::kPi * T.wv);
  }
  for (int q = 0; q < 50; ++q) (&P.dcoef[0][0][0])[q] = (float)(&T.dcoef[0][0][0])[q];
  for (int q = 0; q < 25; ++q) (&P.discoef[0][0])[q] = (float)(&T.discoef[0][0])[q];

  // padded grid of the bracket (3/2 rule; R14); without term III no padded grid exists
  const bool nl = (P.mask & GK_T_III) != 0;
  const int need_x = 3 * T.K + 1, need_y = 3 * (T.nky - 1) + 1;
  if (nl) {
    P.mx = o->pad_mx > 0 ? o->pad_mx : smallest_pad(std::max(need_x, 2));
    P.my = o->pad_my > 0 ? o->pad_my : smallest_pad(std::max(need_y, 2));
    if (P.mx < need_x || P.my < need_y || !gkfft::supported_len(P.mx) || !gkfft::supported_len(P.my))
      return fail(c, GK_EUNSUPPORTED, "padded grid must be 2^a*3^b (b<=1), <=256 and satisfy the 3/2 rule");
    if (P.mx % 2) return fail(c, GK_EUNSUPPORTED, "padded x size must be even (row pairs)");
  } else {
    P.mx = P.my = 2;
  }
  P.fftnorm = (float)(1.0 / ((double)P.mx * P.my));
  P.prefetch = 1;
  P.ldx = 2 * T.nky + 1;
  P.ldy = P.my | 1;

  // Kernel by shape (gk_stage_inst.cu) and its launch plan.
  const StagePick pick = gk_pick_stage(o->storage, P.mx, P.my, P.nky, P.nkx, nl);
  if (!pick.fn) return fail(c, GK_EUNSUPPORTED, "this build has no stage kernel for the requested storage");
  c->stage_fn = pick.fn;
  c->stage_fn2 = pick.fn2;
  c->stage_threads = pick.threads;
  c->stage_kind = pick.kind;
  c->stage_cluster = pick.cluster;
  c->stage_nsh = pick.nsh;
  P.rc = nl ? P.mx : 2;
  P.gchi_in_smem = 1;
  if (pick.kind == GK_KIND_GENERIC && nl) {
    // shared-memory plan of the generic kernel: x-transformed spectra + a chunk of rc rows for the y transforms,
    // grad(chi) in shared memory if it fits next to at least 16 rows, else in per-CTA global scratch
    const size_t fixed = ((size_t)P.mx + P.my + (size_t)P.mx * P.ldx) * 8;
    const size_t gbytes = (size_t)P.mx * P.ldy * 8;
    int rc_best = 0, in_smem = 0;
    for (int pass = 0; pass < 2 && !rc_best; ++pass) {
      const size_t base = fixed + (pass == 0 ? gbytes : 0);
      for (int rc = P.mx; rc >= 2; rc /= 2) {
        if (P.mx % rc || rc % 2) continue;
        if (base + (size_t)rc * P.ldy * 8 <= kSmemDyn) {
          if (pass == 0 && rc < std::min(16, P.mx)) break;
          rc_best = rc;
          in_smem = (pass == 0);
          break;
        }
      }
    }
    if (!rc_best) return fail(c, GK_EUNSUPPORTED, "padded grid does not fit the shared-memory strategy");
    P.rc = rc_best;
    P.gchi_in_smem = in_smem;
    c->stage_smem = fixed + (in_smem ? gbytes : 0) + (size_t)P.rc * P.ldy * 8;
  } else if (pick.kind == GK_KIND_GENERIC) {
    c->stage_smem = (size_t)P.slab * 8;
  } else if (pick.kind == GK_KIND_POINT) {
    c->stage_smem = 0;
  } else {
    c->stage_smem = pick.smem;
  }
  if (pick.kind != GK_KIND_POINT) {
    // The attribute belongs to the kernel symbol, not to this context: the generic kernel (one symbol, plan by
    // shape) always gets the opt-in maximum so that contexts of different shapes can coexist.
    const size_t attr_smem = pick.kind == GK_KIND_GENERIC ? kSmemDyn : c->stage_smem;
    cudaError_t e = cudaFuncSetAttribute(c->stage_fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)attr_smem);
    if (e != cudaSuccess) return fail(c, GK_ECUDA, std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e));
  }
  // persistent launch: one CTA per SM, or as many clusters as the device keeps resident at once
  int resident = c->num_sms;   // units that take one work item at a time (CTAs or clusters)
  if (pick.cluster > 1) {
    c->stage_grid = c->num_sms / pick.cluster * pick.cluster;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr;
    stage_config(c, cfg, attr);
    int ncl = 0;
    cudaError_t e = cudaOccupancyMaxActiveClusters(&ncl, c->stage_fn, &cfg);
    if (e != cudaSuccess || ncl < 1)
      return fail(c, GK_ECUDA, std::string("cudaOccupancyMaxActiveClusters: ") + cudaGetErrorString(e));
    resident = std::min(ncl, c->num_sms / pick.cluster);
  }
  // work decomposition: items (a, l, vpar chunk, share, i) are dealt round-robin to the resident units.
  // Cost of a split = rounds x (slabs per item + the per-item set-up in slab units: chi / grad(chi) build,
  // and the 4 slabs that fill the vpar register window); chunks stay >= 4 long so that the set-up is amortised.
  long long nwork = 0;
  {
    const long long ali = (long long)T.nsp * T.nmu * T.ns * pick.nsh;
    const double setup = pick.kind == GK_KIND_LIN ? 1.5 : (pick.kind == GK_KIND_WS4 ? 1.7 : (nl ? 0.7 : 0.3));
    double best = 1e300;
    for (int nch = 1; nch <= std::max(1, T.nv / 4); ++nch) {
      const int jc = (T.nv + nch - 1) / nch;
      const int nce = (T.nv + jc - 1) / jc;
      const long long rounds = (ali * nce + resident - 1) / resident;
      const double cost = (double)rounds * (jc + setup);
      if (cost < best - 1e-9) { best = cost; P.jchunk = jc; P.nchunk = nce; }
    }
    P.nparts = T.nsp * T.nmu * P.nchunk;
    nwork = ali * P.nchunk;
  }
  c->stage_nwork = (int)nwork;
  c->stage_grid = (int)std::min<long long>(nwork, resident) * pick.cluster;

  // tables -> device
  int rcode;
#define UP(T_, field, vec) if ((rcode = upload<T_>(c, vec, &P.field)) != GK_OK) return rcode
  UP(float, v, T.v); UP(float, fmv, T.fmv); UP(float, mu, T.mu); UP(float, wmu, T.wmu);
  UP(float, fmm, T.fmm); UP(float, B, T.B); UP(float, F, T.F); UP(float, BG, T.BG);
  UP(float, sth, T.sth); UP(float, cz, T.cz); UP(float, Rmaj, T.Rmaj); UP(float, ef, T.ef); UP(float, kx, T.kx);
  UP(float, ky, T.ky); UP(float, hypx, T.hypx); UP(float, hypy, T.hypy); UP(float, J0, T.J0);
  UP(float, dinv, T.dinv); UP(float, zinv, T.zinv);
#undef UP
  for (int dir = 0; dir < 2; ++dir) {
    const int n = dir ? P.my : P.mx;
    std::vector<float2> tw(n);
    for (int t = 0; t < n; ++t)
      tw[t] = make_float2((float)std::cos(2.0 * gkt::kPi * t / n), (float)std::sin(2.0 * gkt::kPi * t / n));
    void *p = nullptr;
    GK_CUDA(c, cudaMalloc(&p, n * sizeof(float2)));
    c->dev_allocs.push_back(p);
    GK_CUDA(c, cudaMemcpy(p, tw.data(), n * sizeof(float2), cudaMemcpyHostToDevice));
    (dir ? P.twy : P.twx) = (const float2 *)p;
  }

  // create-time CFL bounds and the context-owned diagnostics block
  gkt::cfl_static(T, sp, *o, P.mask, &c->dt_lin, &c->dt_field);
  {
    c->part_slots = std::max(kFluxBlocks, c->stage_grid * ((c->stage_threads + 31) / 32));
    const size_t nspec = (size_t)P.nkx + P.nky;
    const size_t bytes = 256 + (16 + nspec + (size_t)c->part_slots * 3 * P.nsp) * sizeof(double);
    void *p = nullptr;
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) return fail(c, e == cudaErrorMemoryAllocation ? GK_ENOMEM : GK_ECUDA,
                                      std::string("cudaMalloc(diagnostics): ") + cudaGetErrorString(e));
    c->dev_allocs.push_back(p);
    GK_CUDA(c, cudaMemset(p, 0, bytes));
    c->d_gmax = (unsigned int *)p;
    c->d_flux_out = (double *)((char *)p + 256);
    c->d_spec = c->d_flux_out + 16;
    c->d_part = c->d_spec + nspec;
  }

  // workspace layout
  size_t off = 0;
  c->off_mom = off; off += align256((size_t)P.nparts * P.nphi * 8);
  c->off_phi = off; off += align256((size_t)P.nphi * 8);
  c->off_gchi = off;
  if (nl && !P.gchi_in_smem) off += align256((size_t)c->stage_grid * P.mx * P.ldy * 8);
  c->off_chis = off;
  off += align256(pick.kind == GK_KIND_POINT ? (size_t)P.nsp * P.nmu * P.ns * 3 * P.slab * 8
                                              : (size_t)c->stage_grid * pick.chis_per_cta * 8);
  c->off_nl = off; off += align256((size_t)c->stage_grid * pick.nl_per_cta * 8);
  c->need_rhs = off;
  c->off_ya = off; off += align256((size_t)P.ntot * c->elem_bytes);
  c->off_yb = off; off += align256((size_t)P.ntot * c->elem_bytes);
  c->off_acc = off; off += align256((size_t)P.ntot * c->elem_bytes);
  c->need_full = off;
  return GK_OK;
}

}  // namespace

// No exception crosses the ABI: an allocation failure of host-side containers maps to GK_ENOMEM, anything else to
// GK_EINVAL.  The context, if there is one, is poisoned (it may be half-built or half-updated) and carries the text
// where that text can still be stored.
namespace {
int caught(gk_ctx *c, int code, const char *what) noexcept {
  if (c) {
    c->poisoned = true;
    try { c->err = what; } catch (...) {}
  }
  return code;
}
template <class F> int guarded(gk_ctx *c, F &&body) noexcept {
  try {
    return body();
  } catch (const std::bad_alloc &) {
    return caught(c, GK_ENOMEM, "out of host memory");
  } catch (const std::exception &e) {
    return caught(c, GK_EINVAL, e.what());
  } catch (...) {
    return caught(c, GK_EINVAL, "internal error");
  }
}
}  // namespace

extern "C" {

int gk_create(const gk_grid *g, const gk_species *sp, const gk_salpha *geo, const gk_opts *o,
              void *cuda_stream, gk_ctx **out) {
  try {
    return create_impl(g, sp, geo, o, cuda_stream, out);
  } catch (const std::bad_alloc &) {   // *out, if set, is half-built: unusable from here on, caller destroys it
    return caught(out ? *out : nullptr, GK_ENOMEM, "gk_create: out of host memory");
  } catch (const std::exception &e) {
    return caught(out ? *out : nullptr, GK_EINVAL, e.what());
  } catch (...) {
    return caught(out ? *out : nullptr, GK_EINVAL, "gk_create: internal error");
  }
}

int gk_destroy(gk_ctx *c) {
  if (!c) return GK_EINVAL;
  for (void *p : c->dev_allocs) cudaFree(p);
  for (auto &e : c->ev) { cudaEventDestroy(e.first); cudaEventDestroy(e.second); }
  if (c->s_up) cudaStreamDestroy(c->s_up);
  if (c->s_down) cudaStreamDestroy(c->s_down);
  for (int b = 0; b < 2; ++b)
    for (cudaEvent_t e : {c->e_in[b], c->e_done[b], c->e_out[b]})
      if (e) cudaEventDestroy(e);
  delete c;
  return GK_OK;
}

size_t gk_workspace_bytes(const gk_ctx *c) { return c ? c->need_full : 0; }
size_t gk_workspace_bytes_rhs(const gk_ctx *c) { return c ? c->need_rhs : 0; }

int gk_set_workspace(gk_ctx *c, void *dev, size_t bytes) {
  if (int r = usable(c)) return r;
  if (!dev || ((uintptr_t)dev & 255) || bytes < c->need_rhs) return fail(c, GK_EINVAL, "workspace null, misaligned or too small");
  c->ws = dev;
  c->ws_bytes = bytes;
  return GK_OK;
}

}  // extern "C"

namespace {
int field_solve(gk_ctx *c, const void *f, void *phi, unsigned int *gmax) {
  if (int r = usable(c)) return r;
  if (!f || !phi || !c->ws) return fail(c, GK_EINVAL, "gk_field_solve: null pointer or no workspace");
  float2 *mom = (float2 *)((char *)c->ws + c->off_mom);
#define GK_CALL(ST) launch_moment<ST>(c, f, mom)
  GK_BY_STORAGE(c, GK_CALL);
#undef GK_CALL
  return solve_phi_from_planes(c, mom, (float2 *)phi, gmax);
}
}  // namespace

extern "C" {

// A field solve on its own is followed by no stage launch: it leaves the CFL maximum of the last one alone, so
// that step -> gk_field_solve (for gk_spectra / gk_fluxes) -> gk_estimate_dt still sees the nonlinear bound.
int gk_field_solve(gk_ctx *c, const void *f, void *phi) { return field_solve(c, f, phi, nullptr); }

int gk_rhs(gk_ctx *c, const void *f, void *phi, void *rhs) {
  return guarded(c, [&]() -> int {
  if (int r = usable(c)) return r;
  if (!f || !phi || !rhs || rhs == f || !c->ws) return fail(c, GK_EINVAL, "gk_rhs: bad pointers or no workspace");
  if (((uintptr_t)f | (uintptr_t)rhs) & 15) return fail(c, GK_EINVAL, "gk_rhs: f and rhs must be 16-byte aligned");
  if (int r = field_solve(c, f, phi, c->d_gmax)) return r;
  GkStageArgs A;
  std::memset(&A, 0, sizeof(A));
  A.y = f; A.out = rhs; A.phi = (const float2 *)phi; A.mode = 0;
  A.gchi = (float2 *)((char *)c->ws + c->off_gchi);
  A.chis = (float2 *)((char *)c->ws + c->off_chis);
  A.nlbuf = (float2 *)((char *)c->ws + c->off_nl);
  A.nwork = c->stage_nwork;
  A.gmax = c->d_gmax;
  stage_launch(c, A);
  return check_launch(c, "stage kernel");
  });
}

int gk_rk4_steps(gk_ctx *c, void *f, double dt, int nsteps) {
  return guarded(c, [&]() -> int {
  if (int r = usable(c)) return r;
  if (!f || !c->ws || nsteps < 0) return fail(c, GK_EINVAL, "gk_rk4_steps: bad arguments or no workspace");
  if ((uintptr_t)f & 15) return fail(c, GK_EINVAL, "gk_rk4_steps: f must be 16-byte aligned (bulk copies of whole slabs)");
  if (c->ws_bytes < c->need_full) return fail(c, GK_EINVAL, "workspace too small for gk_rk4_step");
  char *ws = (char *)c->ws;
  float2 *mom = (float2 *)(ws + c->off_mom);
  float2 *phi = (float2 *)(ws + c->off_phi);
  void *ya = ws + c->off_ya, *yb = ws + c->off_yb, *acc = ws + c->off_acc;
  GkStageArgs A;
  std::memset(&A, 0, sizeof(A));
  A.phi = phi; A.mom = mom; A.acc = acc;
  A.gchi = (float2 *)(ws + c->off_gchi);
  A.chis = (float2 *)(ws + c->off_chis);
  A.nlbuf = (float2 *)(ws + c->off_nl);
  A.nwork = c->stage_nwork;
  A.gmax = c->d_gmax;
  const float h = (float)dt;
  const size_t part_bytes = (size_t)c->part_slots * 3 * c->P.nsp * sizeof(double);
  for (int s = 0; s < nsteps; ++s) {
    if (s == 0) {  // later steps reuse the moment planes written by the previous stage 4
#define GK_CALL(ST) launch_moment<ST>(c, f, mom)
      GK_BY_STORAGE(c, GK_CALL);
#undef GK_CALL
    }
    // classical RK4: acc = f + dt/6 k1, then += dt/3 k2, += dt/3 k3, f = acc + dt/6 k4
    if (int r = solve_phi_from_planes(c, mom, phi, c->d_gmax)) return r;
    A.mode = 1; A.y = f; A.fn = f; A.out = ya; A.c = 0.5f * h; A.b = h / 6.f;
    const bool fused_diag = c->diag && c->stage_kind != GK_KIND_POINT && c->stage_kind != GK_KIND_LIN;
    if (c->diag && !fused_diag) {   // point kernel: no streaming role; streaming kernel: no registers to spare
#define GK_CALL(ST) launch_flux<ST>(c, f, phi)
      GK_BY_STORAGE(c, GK_CALL);
#undef GK_CALL
      c->flux_valid = true;
    }
    if (fused_diag) {   // fluxes of (f_n, phi(f_n)) from the registers of this launch's streaming role
      GK_CUDA(c, cudaMemsetAsync(c->d_part, 0, part_bytes, c->stream));
      A.fluxp = c->d_part;
    }
    stage_launch(c, A);
    if (fused_diag) {
      A.fluxp = nullptr;
      gk::gk_flux_sum_kernel<<<1, 32, 0, c->stream>>>(c->P, c->d_part, c->stage_grid * ((c->stage_threads + 31) / 32),
                                                      c->d_flux_out);
      ++c->launches;
      c->flux_valid = true;
    }
    if (int r = solve_phi_from_planes(c, mom, phi, c->d_gmax)) return r;
    A.mode = 2; A.y = ya; A.fn = f; A.out = yb; A.c = 0.5f * h; A.b = h / 3.f;
    stage_launch(c, A);
    if (int r = solve_phi_from_planes(c, mom, phi, c->d_gmax)) return r;
    A.mode = 2; A.y = yb; A.fn = f; A.out = ya; A.c = h; A.b = h / 3.f;
    stage_launch(c, A);
    if (int r = solve_phi_from_planes(c, mom, phi, c->d_gmax)) return r;
    A.mode = 3; A.y = ya; A.fn = f; A.out = f; A.c = 0.f; A.b = h / 6.f;
    stage_launch(c, A);
    if (int r = check_launch(c, "stage kernel")) return r;
  }
  return GK_OK;
  });
}

int gk_rk4_step(gk_ctx *c, void *f, double dt) { return gk_rk4_steps(c, f, dt, 1); }

int gk_rk4_step_host(gk_ctx *c, const void *f_host_in, void *f_host_out, void *f_dev, double dt) {
  if (int r = usable(c)) return r;
  if (!f_host_in || !f_host_out || !f_dev) return fail(c, GK_EINVAL, "gk_rk4_step_host: null pointer");
  if (!c->ws || c->ws_bytes < c->need_full || ((uintptr_t)f_dev & 15))   // checked before the upload is queued
    return fail(c, GK_EINVAL, "gk_rk4_step_host: workspace too small for gk_rk4_step or f_dev not 16-byte aligned");
  const size_t bytes = (size_t)c->P.ntot * c->elem_bytes;
  GK_CUDA(c, cudaMemcpyAsync(f_dev, f_host_in, bytes, cudaMemcpyHostToDevice, c->stream));
  if (int r = gk_rk4_steps(c, f_dev, dt, 1)) return r;
  GK_CUDA(c, cudaMemcpyAsync(f_host_out, f_dev, bytes, cudaMemcpyDeviceToHost, c->stream));
  return GK_OK;
}

int gk_rk4_batch_host(gk_ctx *c, const void *const *f_in, void *const *f_out, int nbatch, void *dev0, void *dev1,
                      double dt) {
  if (int r = usable(c)) return r;
  // everything is validated BEFORE anything is enqueued: no copy is in flight when an argument error is returned
  if (!f_in || !f_out || !dev0 || !dev1 || dev0 == dev1 || nbatch < 0)
    return fail(c, GK_EINVAL, "gk_rk4_batch_host: bad arguments");
  for (int k = 0; k < nbatch; ++k)
    if (!f_in[k] || !f_out[k]) return fail(c, GK_EINVAL, "gk_rk4_batch_host: null host pointer");
  if (!c->ws || c->ws_bytes < c->need_full) return fail(c, GK_EINVAL, "gk_rk4_batch_host: workspace too small for gk_rk4_step");
  if (((uintptr_t)dev0 | (uintptr_t)dev1) & 15) return fail(c, GK_EINVAL, "gk_rk4_batch_host: device buffers must be 16-byte aligned");
  if (!c->s_up) {
    GK_CUDA(c, cudaStreamCreateWithFlags(&c->s_up, cudaStreamNonBlocking));
    GK_CUDA(c, cudaStreamCreateWithFlags(&c->s_down, cudaStreamNonBlocking));
    for (int b = 0; b < 2; ++b) {
      GK_CUDA(c, cudaEventCreateWithFlags(&c->e_in[b], cudaEventDisableTiming));
      GK_CUDA(c, cudaEventCreateWithFlags(&c->e_done[b], cudaEventDisableTiming));
      GK_CUDA(c, cudaEventCreateWithFlags(&c->e_out[b], cudaEventDisableTiming));
    }
  }
  const size_t bytes = (size_t)c->P.ntot * c->elem_bytes;
  void *dev[2] = {dev0, dev1};
  // a failure past this point (a CUDA error) leaves no copy in flight either: the three streams are drained first
  auto drained = [&](int rc) {
    cudaStreamSynchronize(c->s_up);
    cudaStreamSynchronize(c->stream);
    cudaStreamSynchronize(c->s_down);
    return rc;
  };
#define GK_CUDA_D(call)                                                                                   \
  do {                                                                                                    \
    cudaError_t e_ = (call);                                                                              \
    if (e_ != cudaSuccess) return drained(fail(c, GK_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_))); \
  } while (0)
  // the copy streams start after whatever the caller queued on the context stream
  GK_CUDA_D(cudaEventRecord(c->e_done[0], c->stream));
  GK_CUDA_D(cudaStreamWaitEvent(c->s_up, c->e_done[0], 0));
  for (int k = 0; k < nbatch; ++k) {
    const int b = k & 1;
    if (k >= 2) GK_CUDA_D(cudaStreamWaitEvent(c->s_up, c->e_out[b], 0));   // buffer b has been downloaded
    GK_CUDA_D(cudaMemcpyAsync(dev[b], f_in[k], bytes, cudaMemcpyHostToDevice, c->s_up));
    GK_CUDA_D(cudaEventRecord(c->e_in[b], c->s_up));
    GK_CUDA_D(cudaStreamWaitEvent(c->stream, c->e_in[b], 0));
    if (int r = gk_rk4_steps(c, dev[b], dt, 1)) return drained(r);
    GK_CUDA_D(cudaEventRecord(c->e_done[b], c->stream));
    GK_CUDA_D(cudaStreamWaitEvent(c->s_down, c->e_done[b], 0));
    GK_CUDA_D(cudaMemcpyAsync(f_out[k], dev[b], bytes, cudaMemcpyDeviceToHost, c->s_down));
    GK_CUDA_D(cudaEventRecord(c->e_out[b], c->s_down));
  }
#undef GK_CUDA_D
  GK_CUDA(c, cudaStreamSynchronize(c->s_up));
  GK_CUDA(c, cudaStreamSynchronize(c->stream));
  GK_CUDA(c, cudaStreamSynchronize(c->s_down));
  return GK_OK;
}

namespace {
// species factors of the flux triple: -(1/ns) 2 pi w_v  x {1, T_a, m_a vR_a}
void flux_factors(const gk_ctx *c, double *out_host) {
  for (int a = 0; a < c->P.nsp; ++a) {
    const double base = 2.0 * gkt::kPi * c->T.wv / c->T.ns;
    out_host[3 * a + 0] *= base;
    out_host[3 * a + 1] *= base * c->species[a].temp;
    out_host[3 * a + 2] *= base * c->species[a].mass * c->T.vR[a];
  }
}
}  // namespace

int gk_fluxes(gk_ctx *c, const void *f, const void *phi, double *out_host) {
  if (int r = usable(c)) return r;
  if (!f || !phi || !out_host) return fail(c, GK_EINVAL, "gk_fluxes: null pointer");
#define GK_CALL(ST) launch_flux<ST>(c, f, (const float2 *)phi)
  GK_BY_STORAGE(c, GK_CALL);
#undef GK_CALL
  c->flux_valid = false;    // the output slot now holds this call's result, not a step's
  cudaError_t e = cudaMemcpyAsync(out_host, c->d_flux_out, 3 * c->P.nsp * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return fail(c, GK_ECUDA, std::string("gk_fluxes: ") + cudaGetErrorString(e));
  flux_factors(c, out_host);
  return GK_OK;
}

int gk_set_diagnostics(gk_ctx *c, int on) {
  if (int r = usable(c)) return r;
  c->diag = on != 0;
  if (!c->diag) c->flux_valid = false;
  return GK_OK;
}

int gk_fluxes_last(gk_ctx *c, double *out_host) {
  if (int r = usable(c)) return r;
  if (!out_host) return fail(c, GK_EINVAL, "gk_fluxes_last: null pointer");
  if (!c->flux_valid) return fail(c, GK_EINVAL, "gk_fluxes_last: no step has run with diagnostics enabled");
  cudaError_t e = cudaMemcpyAsync(out_host, c->d_flux_out, 3 * c->P.nsp * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return fail(c, GK_ECUDA, std::string("gk_fluxes_last: ") + cudaGetErrorString(e));
  flux_factors(c, out_host);
  return GK_OK;
}

int gk_estimate_dt(gk_ctx *c, double *out_host) {
  if (int r = usable(c)) return r;
  if (!out_host) return fail(c, GK_EINVAL, "gk_estimate_dt: null pointer");
  unsigned int bits = 0;
  cudaError_t e = cudaMemcpyAsync(&bits, c->d_gmax, sizeof(bits), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return fail(c, GK_ECUDA, std::string("gk_estimate_dt: ") + cudaGetErrorString(e));
  float g = 0.f;
  std::memcpy(&g, &bits, sizeof(g));
  // R21: lambda_NL = (1/2) max(|d_y chi| kx_max + |d_x chi| ky_max); RK4 is stable on the imaginary axis to 2 sqrt 2
  const bool nl = (c->P.mask & GK_T_III) != 0;
  out_host[1] = (nl && g > 0.f) ? 2.0 * std::sqrt(2.0) / (0.5 * (double)g) : HUGE_VAL;
  out_host[2] = c->dt_lin;
  out_host[3] = c->dt_field;
  out_host[0] = std::min(out_host[1], std::min(out_host[2], out_host[3]));
  return GK_OK;
}

int gk_reset_cfl(gk_ctx *c) {
  if (int r = usable(c)) return r;
  GK_CUDA(c, cudaMemsetAsync(c->d_gmax, 0, sizeof(unsigned int), c->stream));
  return GK_OK;
}

int gk_rk4_steps_cfl(gk_ctx *c, void *f, int nsteps, double safety, double dt_max, double *dt_used_host,
                     double *t_advanced_host) {
  if (int r = usable(c)) return r;
  if (!f || nsteps < 0 || !(safety > 0.0)) return fail(c, GK_EINVAL, "gk_rk4_steps_cfl: bad arguments");
  double t = 0.0;
  for (int s = 0; s < nsteps; ++s) {
    // one-step lag: the nonlinear bound comes from the grad(chi) of the most recent stage launch;
    // before the first one only the linear bounds exist ("conservative linear-only estimate")
    double est[4];
    if (int r = gk_estimate_dt(c, est)) return r;
    double dt = safety * est[0];
    if (dt_max > 0.0) dt = std::min(dt, dt_max);
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail(c, GK_EINVAL, "gk_rk4_steps_cfl: no finite step (give dt_max)");
    if (int r = gk_rk4_steps(c, f, dt, 1)) return r;
    if (dt_used_host) dt_used_host[s] = dt;
    t += dt;
  }
  if (t_advanced_host) *t_advanced_host = t;
  return GK_OK;
}

int gk_spectra(gk_ctx *c, const void *phi, double *kx_spec, double *ky_spec) {
  if (int r = usable(c)) return r;
  if (!phi || !kx_spec || !ky_spec) return fail(c, GK_EINVAL, "gk_spectra: null pointer");
  const int n = c->P.nkx + c->P.nky;
  gk::gk_spectra_kernel<<<n, 256, 0, c->stream>>>(c->P, (const float2 *)phi, c->d_spec);
  ++c->launches;
  std::vector<double> h;
  try { h.resize(n); } catch (const std::bad_alloc &) { return fail(c, GK_ENOMEM, "gk_spectra: out of host memory"); }
  cudaError_t e = cudaMemcpyAsync(h.data(), c->d_spec, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return fail(c, GK_ECUDA, std::string("gk_spectra: ") + cudaGetErrorString(e));
  std::memcpy(kx_spec, h.data(), c->P.nkx * sizeof(double));
  std::memcpy(ky_spec, h.data() + c->P.nkx, c->P.nky * sizeof(double));
  return GK_OK;
}

size_t gk_export_table(const gk_ctx *c, const char *which, double *out, size_t maxn) {
  if (!c || !which) return 0;
  try {
  const gkt::Tables &T = c->T;
  const std::string w(which);
  std::vector<double> tmp;
  const std::vector<double> *src = nullptr;
  if (w == "vpar") src = &T.v; else if (w == "mu") src = &T.mu; else if (w == "wmu") src = &T.wmu;
  else if (w == "kx") src = &T.kx; else if (w == "ky") src = &T.ky; else if (w == "B") src = &T.B;
  else if (w == "F") src = &T.F; else if (w == "BG") src = &T.BG; else if (w == "J0") src = &T.J0;
  else if (w == "ef") src = &T.ef; else if (w == "gpz") src = &T.gpz; else if (w == "gzz") src = &T.gzz;
  else if (w == "sth") src = &T.sth; else if (w == "cz") src = &T.cz; else if (w == "R") src = &T.Rmaj;
  else if (w == "kthnorm") { tmp = {T.kthnorm}; src = &tmp; } else if (w == "dkx") { tmp = {T.dkx}; src = &tmp; }
  else if (w == "Gamma0") src = &T.G0; else if (w == "den") src = &T.den; else if (w == "zonal") src = &T.zinv;
  else if (w == "FM") {
    tmp.resize((size_t)T.nv * T.nmu * T.ns);
    for (int j = 0; j < T.nv; ++j)
      for (int l = 0; l < T.nmu; ++l)
        for (int i = 0; i < T.ns; ++i)
          tmp[((size_t)j * T.nmu + l) * T.ns + i] = T.fmv[j] * T.fmm[(size_t)l * T.ns + i];
    src = &tmp;
  } else if (w == "pad") {
    tmp = {(double)c->P.mx, (double)c->P.my, (double)c->P.rc, (double)c->P.gchi_in_smem,
           (double)c->P.jchunk, (double)c->P.nchunk, (double)c->stage_grid, (double)c->stage_smem,
           (double)c->stage_threads, (double)c->stage_cluster, (double)c->stage_nsh, (double)c->stage_kind};
    src = &tmp;
  } else return 0;
  if (out) std::memcpy(out, src->data(), std::min(maxn, src->size()) * sizeof(double));
  return src->size();
  } catch (...) {   // host allocation failure of a temporary: reported as "no such table"
    return 0;
  }
}

long long gk_launch_count(const gk_ctx *c) { return c ? c->launches : 0; }

int gk_set_profiling(gk_ctx *c, int on) {
  if (int r = usable(c)) return r;
  c->profiling = on != 0;
  return GK_OK;
}

int gk_stage_kernel_time(gk_ctx *c, double *ms_total, long long *n, int reset) {
  if (int r = usable(c)) return r;
  GK_CUDA(c, cudaStreamSynchronize(c->stream));
  double tot = 0;
  for (size_t q = 0; q < c->ev_used; ++q) {
    float ms = 0;
    GK_CUDA(c, cudaEventElapsedTime(&ms, c->ev[q].first, c->ev[q].second));
    tot += ms;
  }
  if (ms_total) *ms_total = tot;
  if (n) *n = (long long)c->ev_used;
  if (reset) c->ev_used = 0;
  return GK_OK;
}

}  // extern "C"
