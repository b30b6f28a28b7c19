/* gk.h -- C ABI of libgk, the B200 (sm_100a) hot path of the local flux-tube delta-f
 * gyrokinetic solver of arxiv/paper_2604_06085 ("gyaradax"): one Runge-Kutta stage =
 * quasineutrality field solve -> linear terms I,II,IV,V,VII,VIII + dissipation -> dealiased
 * ExB bracket (term III) -> fused RK4 stage update.  Citations are PAPER.md line numbers; R<n>
 * are the readings listed in DESIGN.md.
 *
 * Conventions
 *   - All data pointers are DEVICE pointers unless the name ends in _host.
 *   - f:   [species a][vpar j][mu l][s i][kx p+K][ky m], ky fastest, K=(nkx-1)/2, kx index monotone
 *          from -K to K, ky index m = 0..nky-1 (half spectrum, ky_m = m*ky0).
 *          storage 0: complex64 (float re, float im); 1: complex fp16 (__half2); 2: complex bf16.
 *   - phi: [s i][kx p+K][ky m] complex64, always.
 *   - f, rhs and the host-call device buffers must be 16-byte aligned (slabs move by bulk copies): GK_EINVAL.
 *   - Caller owns f, phi, rhs and the workspace; the context owns only its coefficient tables.
 *   - Hot calls (field_solve, rhs, rk4_step, rk4_steps) are asynchronous on the stream given to
 *     gk_create, never synchronise and never allocate.  The diagnostics calls (gk_fluxes, gk_fluxes_last,
 *     gk_spectra, gk_estimate_dt, gk_rk4_steps_cfl) synchronise the stream; none allocates.
 *   - Every function returns 0 (GK_OK) or a negative error code; no exception crosses the ABI.
 *     After GK_ECUDA the context is poisoned (sticky CUDA error); text in gk_last_error().
 *   - There is no CPU fallback: without a CUDA device gk_create returns GK_ECUDA.
 */
#ifndef GK_H
#define GK_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { GK_OK = 0, GK_EINVAL = -1, GK_ENOMEM = -2, GK_ECUDA = -3, GK_EUNSUPPORTED = -4 };

typedef struct gk_ctx gk_ctx; /* opaque */

/* Phase-space grid (R1, R3, R5). */
typedef struct {
  int nkx, nky, ns, nvpar, nmu; /* nkx odd, ns >= 4, nvpar >= 4, nky >= 1, nmu >= 1               */
  double ky0;                   /* ky_m = m*ky0 in k_theta*rho_ref units                          */
  int ikxspace;                 /* dkx = 2*pi*shat*ky0/ikxspace  */
  double vpar_max;              /* vpar_j = -vpar_max + (j+1/2)*2*vpar_max/nvpar                   */
  int mu_grid;                  /* 0 = Gauss-Laguerre in 2*mu, 1 = uniform in v_perp*/
  double vperp_max;             /* upper end of the uniform v_perp grid                           */
} gk_grid;

/* One kinetic species: charge number, mass, temperature, density (all relative
 * to the reference species) and the gradient drives R/L_T, R/L_n. */
typedef struct { double Z, mass, temp, dens, rlt, rln; } gk_species;

/* Equilibrium scalars of the geometry model chosen by gk_opts.geometry: s-alpha (formulas:
 * reading R2) or circular (R24). */
typedef struct { double q, shat, eps; } gk_salpha;

/* term_mask bits: debugging/test hook that switches individual terms of the RHS. */
enum {
  GK_T_I = 1, GK_T_II = 2, GK_T_IV = 4, GK_T_V = 8, GK_T_VII = 16, GK_T_VIII = 32,
  GK_T_DISS_S = 64, GK_T_DISS_V = 128, GK_T_HYP = 256, GK_T_III = 512, GK_T_ALL = 1023
};

typedef struct {
  int nspecies;            /* number of kinetic species (entries of the gk_species array)         */
  int adiabatic_electrons; /* 1: adiabatic electrons + zonal flux-surface-average correction (R10)*/
                           /* 0: all species kinetic, no correction (R11)           */
  double te, ne;           /* adiabatic-electron temperature and density                          */
  int nonlinear;           /* 1: include term III                                                 */
  double disp_par, disp_vp, disp_x, disp_y; /* nu_s, nu_v, nu_x, nu_y (R9)            */
  int s_closure;           /* 0: upwinded 2nd-order boundary classes; 1: zero ghosts (R7)         */
  int storage;             /* 0 complex64, 1 complex fp16, 2 complex bf16 (BASELINE config 5; R19)*/
  int term_mask;           /* <= 0: all terms                                                     */
  int pad_mx, pad_my;      /* padded real-space grid of the bracket; 0 = automatic (R14).  Must be
                              >= 3K+1 / 3(nky-1)+1 and of the form 2^a * 3^b, b <= 1, <= 256      */
  int geometry;            /* 0: s-alpha (R2); 1: circular concentric (Lapillonne) model from (q, shat, eps),
                              PAPER.md:286-310 eq. 1-4 (R24)                                        */
} gk_opts;

/* Builds all create-time tables (grids, weights, geometry, F_M, J0, Gamma0, Poisson denominators,
 * connectivity classes, stencil table: PAPER.md:65, 336) on the host in double precision, uploads
 * them, and binds the context to `cuda_stream` (a cudaStream_t cast to void*, NULL = default
 * stream).  Errors: GK_EINVAL (bad sizes/null pointers), GK_EUNSUPPORTED (padded grid does not fit
 * the shared-memory strategy), GK_ENOMEM, GK_ECUDA. */
int gk_create(const gk_grid *grid, const gk_species *species, const gk_salpha *geom,
              const gk_opts *opts, void *cuda_stream, gk_ctx **out);
int gk_destroy(gk_ctx *ctx);

/* Bytes of caller-owned device scratch the hot calls need: moment partial sums, two stage states,
 * the RK accumulator, spill space of the bracket kernel.  gk_field_solve and gk_rhs need only the
 * first gk_workspace_bytes_rhs() bytes of it. */
size_t gk_workspace_bytes(const gk_ctx *ctx);
size_t gk_workspace_bytes_rhs(const gk_ctx *ctx);
/* `dev` must be 256-byte aligned and stay valid until replaced or the context is destroyed.
 * GK_EINVAL if too small for gk_workspace_bytes_rhs(); rk4 calls check for the full size. */
int gk_set_workspace(gk_ctx *ctx, void *dev, size_t bytes);

/* Quasineutrality field solve: phi(i,p,m) from f.  phi(kx=0,ky=0) = 0. */
int gk_field_solve(gk_ctx *ctx, const void *f_dev, void *phi_dev);

/* Full right-hand side: solves phi (written to phi_dev), then
 * rhs = I + II + IV + V + VII + VIII + dissipation + III.  rhs_dev has the layout and storage type
 * of f and must not alias it. */
int gk_rhs(gk_ctx *ctx, const void *f_dev, void *phi_dev, void *rhs_dev);

/* One classical RK4 step, phi re-solved at each of the 4 stages; f in-out.
 * gk_rk4_steps does `nsteps` steps (the paper's gksolve/scan) and keeps the
 * velocity-space moments of f_{n+1} from the last stage's epilogue for the next step. */
int gk_rk4_step(gk_ctx *ctx, void *f_dev, double dt);
int gk_rk4_steps(gk_ctx *ctx, void *f_dev, double dt, int nsteps);

/* One RK4 step with HOST buffers (bench.py's end-to-end leg): copies f_host_in -> f_dev, runs gk_rk4_step on
 * f_dev, copies f_dev -> f_host_out, all asynchronous on the context stream in that order (truly asynchronous
 * only for pinned host memory; pageable memory makes the copies synchronous).  f_host_in / f_host_out: host,
 * same layout and storage type as f, may alias; f_dev: device scratch of the size of f, caller-owned.  Does
 * not synchronise at the end: synchronise the stream before reading f_host_out.  GK_EINVAL on null pointers,
 * a misaligned f_dev or a workspace too small for gk_rk4_step, checked before the upload is queued. */
int gk_rk4_step_host(gk_ctx *ctx, const void *f_host_in, void *f_host_out, void *f_dev, double dt);

/* A batch of independent RK4 steps on HOST buffers, software-pipelined over two device buffers: the upload of
 * problem k+1 and the download of problem k-1 run on two copy streams owned by the context while problem k is
 * stepped on the context stream (PCIe is full duplex; one step of the BASELINE grids computes faster than it
 * uploads).  f_host_in[k] / f_host_out[k]: nbatch host pointers (pinned memory, layout and storage type of f; an
 * output must not alias the input of a LATER problem), f_dev0 / f_dev1: two device scratch arrays of the size of
 * f, caller-owned.  Every problem takes exactly the path of gk_rk4_step_host (same kernels, same result).
 * Synchronises all three streams before returning.  Every pointer, the workspace size and the alignment of the
 * device buffers are checked BEFORE anything is enqueued (GK_EINVAL, nothing in flight); a CUDA failure later drains
 * the three streams before it is returned. */
int gk_rk4_batch_host(gk_ctx *ctx, const void *const *f_host_in, void *const *f_host_out, int nbatch,
                      void *f_dev0, void *f_dev1, double dt);

/* Transport fluxes per species (R18): out_host[3*a + {0,1,2}] = particle, heat,
 * parallel-momentum flux of a caller-supplied (f, phi).  One pass over f into per-block partial sums and a
 * fixed-order second pass (deterministic, no atomics, no allocation).  Synchronises the stream. */
int gk_fluxes(gk_ctx *ctx, const void *f_dev, const void *phi_dev, double *out_host);

/* Diagnostics folded into the time step ("computed only at block boundaries").  With
 * diagnostics on, every RK4 step's FIRST stage launch -- which holds f_n and chi = J0 phi(f_n) in registers -- also
 * reduces the flux triple of (f_n, phi(f_n)): no extra pass over f.  gk_fluxes_last returns the fluxes of the state
 * at the START of the most recent step taken by gk_rk4_step(s) (same layout and normalisation as gk_fluxes;
 * deterministic: one writer per partial, fixed-order sum).  Synchronises the stream.  GK_EINVAL if no step has run
 * since diagnostics were switched on. */
int gk_set_diagnostics(gk_ctx *ctx, int on);
int gk_fluxes_last(gk_ctx *ctx, double *out_host);

/* CFL estimate of the time step (PAPER.md:340 estimate_timestep; readings R21-R23).  out_host[4]:
 *   [1] nonlinear bound 2 sqrt2 / max (1/2)(|d_y chi| kx_max + |d_x chi| ky_max), the maximum taken over the padded
 *       real-space grad(chi) of every (species, mu, s) as built by the MOST RECENT stage launch (gk_rhs or the last
 *       stage of gk_rk4_step(s): "one-step lag"; a bare gk_field_solve leaves it as it is); +inf before the first
 *       launch, after gk_reset_cfl, for phi = 0 and with term III off;
 *   [2] von Neumann bound of the streaming and trapping stencils with their dissipation (create-time);
 *   [3] field (omega_H) bound with kinetic electrons, +inf with adiabatic electrons (create-time);
 *   [0] the minimum of the three.
 * Each is the largest step for which classical RK4 is stable on the model problem; no safety factor is applied.
 * Synchronises the stream (reads one word back). */
int gk_estimate_dt(gk_ctx *ctx, double *out_host);

/* CFL-adaptive stepping ("optional CFL-adaptive mode ... updated with one-step lag; the initial step
 * uses a conservative linear-only estimate"): nsteps RK4 steps, step k with dt_k = min(safety * gk_estimate_dt()[0],
 * dt_max) evaluated just before the step (dt_max <= 0: no cap).  dt_used_host (nsteps doubles) and t_advanced_host
 * (one double) may be NULL.  Synchronises once per step. */
int gk_rk4_steps_cfl(gk_ctx *ctx, void *f_dev, int nsteps, double safety, double dt_max, double *dt_used_host,
                     double *t_advanced_host);
/* The nonlinear bound lives in the context and belongs to whatever state the last stage launch saw.  A context that
 * is reused for another state (a new initial condition, or after gk_rhs on some other f) therefore starts
 * gk_rk4_steps_cfl / gk_estimate_dt from that unrelated bound.  gk_reset_cfl puts the context back to "no stage
 * launched yet" ([1] = +inf, so the first step uses the linear-only estimate); asynchronous on the
 * context stream.  gk_field_solve on its own never changes the bound. */
int gk_reset_cfl(gk_ctx *ctx);

/* Spectra of the potential (ky_spec = sum_{s,kx} |phi|^2, kx_spec = sum_{s,ky} |phi|^2, with the
 * Parseval factor P_ky (1 at ky = 0, 2 otherwise) and the weight Delta s = 1/ns applied; R20):
 *   kx_spec_host[p+K] = ds sum_{s,m} P_m |phi|^2   (nkx doubles),
 *   ky_spec_host[m]   = ds P_m sum_{s,p} |phi|^2   (nky doubles).
 * phi_dev: device, [ns][nkx][nky] complex64 (as written by gk_field_solve).  Accumulates in double,
 * deterministic (one block tree per output, no atomics).  Synchronises the stream.  GK_EINVAL on null. */
int gk_spectra(gk_ctx *ctx, const void *phi_dev, double *kx_spec_host, double *ky_spec_host);

/* gk_spectra for callers that cannot allocate device memory.  gk_spectra needs a context, and gk_create builds one
 * out of cudaMalloc'ed tables; that rules it out for a host whose own pool allocator already owns the whole device
 * (every further cudaMalloc fails), for a process under an MPS / MIG memory cap, and for a loop that cannot take
 * cudaMalloc's device-wide synchronisation.  This entry point needs no context and calls no cudaMalloc, cudaFree or
 * allocating library routine: the caller passes the input and the outputs, and the nkx + nky device-side results
 * are staged in a fixed array inside the library image (GK_SPECTRA_STATIC_MAX doubles = 32 KiB, held by every GPU
 * that loads libgk.so until the process exits).
 *   phi_dev:       device, [ns][nkx][nky] complex64, on the CURRENT device;
 *   kx_spec_host:  host, nkx doubles;  ky_spec_host: host, nky doubles -- same definition, normalisation and
 *                  summation order as gk_spectra (the results are bit-identical);
 *   cuda_stream:   a cudaStream_t of the current device cast to void*, NULL = default stream.
 * Limit: nkx + nky <= GK_SPECTRA_STATIC_MAX, else GK_EINVAL (nothing is launched); also GK_EINVAL for null pointers
 * and sizes < 1, GK_ECUDA for CUDA failures.  The text of the last error of the calling thread is returned by
 * gk_spectra_static_error() ("" after a successful call).
 * Set-up: the first call on each device resolves that device's address of the array (cudaGetSymbolAddress); make
 * that first call with the device current and before any stream capture begins.
 * Sharing: all calls on a device use the same array, which keeps the previous call's numbers.  Each call overwrites
 * exactly the entries it reads back, so nothing needs clearing -- but two calls that overlap on the GPU (two
 * streams, or two host threads) race on it: serialise them.  Launches one kernel, then synchronises the stream. */
#define GK_SPECTRA_STATIC_MAX 4096
int gk_spectra_static(const void *phi_dev, int ns, int nkx, int nky, double *kx_spec_host, double *ky_spec_host,
                      void *cuda_stream);
size_t gk_spectra_static_max(void);          /* GK_SPECTRA_STATIC_MAX of the library that was loaded */
const char *gk_spectra_static_error(void);   /* never NULL; thread-local */

/* Test hook: copies a create-time table to host memory as doubles.  `which` is one of
 * "vpar","mu","wmu","kx","ky","B","F","BG","J0","Gamma0","FM","den","zonal","pad","ef","gpz","gzz","sth","cz","R",
 * "kthnorm","dkx".  Returns the
 * number of doubles (also when host_out is NULL), 0 for an unknown name. */
size_t gk_export_table(const gk_ctx *ctx, const char *which, double *host_out, size_t max_doubles);

const char *gk_last_error(const gk_ctx *ctx); /* never NULL; "" if no error */
const char *gk_version(void);  /* "gk-b200 <ver> (sm_100a) src:<16 hex digits>": the digits identify the csrc/ tree the
                                  library was built from (paper_2604_06085_b200/build.py src_hash) */

#ifdef __cplusplus
}
#endif
#endif
