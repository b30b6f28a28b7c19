/* gkref -- the CPU ORACLE for the gk-b200 hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, double-precision restatement of what one Runge-Kutta stage of the local
 * flux-tube delta-f gyrokinetic solver of arxiv/paper_2604_06085 ("gyaradax") computes:
 * quasineutrality field solve, linear terms I,II,IV,V,VII,VIII + dissipation, the dealiased
 * ExB bracket (term III), classical RK4, flux diagnostics.  It shares no code, header, table
 * or constant generator with the CUDA path (paper_2604_06085_b200/csrc); only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Every function cites the PAPER.md passage (or the DESIGN.md reading R<n>, where the paper
 * is silent) it follows.  Parity pins: tests/test_oracle_*.py.  Functions whose coefficients
 * have no pin outside this file say "parity unpinned" here and in DESIGN.md:
 *   - boundary-class stencil coefficients at open chain ends (R7)      parity unpinned
 *   - dissipation defaults and hyper-viscosity form (R9)                parity unpinned
 *   - flux normalisation of gkref_fluxes (R18)                          parity unpinned
 *
 * Layout of f:   [species][vpar j][mu l][s i][kx p+K][ky m]  complex double (re,im), ky fastest.
 * Layout of phi: [s i][kx p+K][ky m] complex double.
 */
#ifndef GKREF_H
#define GKREF_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct gkref gkref;

typedef struct {
  int nkx, nky, ns, nvpar, nmu; /* nkx odd */
  double ky0;                   /* ky_m = m*ky0 (k_theta rho units)                      */
  int ikxspace;                 /* dkx = 2*pi*shat*ky0/ikxspace          */
  double vpar_max;              /* vpar grid uniform on [-vpar_max, vpar_max], midpoints  */
  int mu_grid;                  /* 0 Gauss-Laguerre, 1 uniform in v_perp   */
  double vperp_max;
} gkref_grid;

typedef struct { double Z, mass, temp, dens, rlt, rln; } gkref_species;
typedef struct { double q, shat, eps; } gkref_geom; /* equilibrium scalars of both geometry models */

/* term_mask bits (test hook, "switch terms on one at a time") */
enum {
  GKREF_T_I = 1, GKREF_T_II = 2, GKREF_T_IV = 4, GKREF_T_V = 8, GKREF_T_VII = 16,
  GKREF_T_VIII = 32, GKREF_T_DISS_S = 64, GKREF_T_DISS_V = 128, GKREF_T_HYP = 256,
  GKREF_T_III = 512, GKREF_T_ALL = 1023
};

typedef struct {
  int nspecies;
  int adiabatic_electrons; /* 1: adiabatic electron response with zonal correction (R10)  */
  double te, ne;           /* adiabatic-electron temperature and density                 */
  int nonlinear;           /* 1: include term III                                        */
  double disp_par, disp_vp, disp_x, disp_y; /* nu_s, nu_v, nu_x, nu_y (R9)                */
  int s_closure;           /* 0 upwinded boundary classes, 1 zero ghosts (R7)            */
  int term_mask;           /* <=0: all terms                                             */
  int bracket_method;      /* 0 = padded FFT (own FFT), 1 = direct O(N^2) convolution    */
  int pad_mx, pad_my;      /* 0 = smallest 7-smooth size >= the 3/2-rule minimum (R14)   */
  int geometry;            /* 0 s-alpha (R2), 1 circular (eq. 1-4; R24) */
} gkref_opts;

gkref *gkref_create(const gkref_grid *, const gkref_species *, const gkref_geom *,
                    const gkref_opts *);
void gkref_destroy(gkref *);
int gkref_set_threads(int n); /* OpenMP threads over outer loops only; returns the count used */

/* field solve (R10, R11): phi from f */
void gkref_field_solve(const gkref *, const double *f, double *phi);
/* full RHS: solves phi (written to phi_out), then linear terms + bracket -> rhs */
void gkref_rhs(const gkref *, const double *f, double *phi_out, double *rhs);
/* RHS on ONE (species a, j, l, i) slab only, phi given: out is nkx*nky complex */
void gkref_rhs_slab(const gkref *, const double *f, const double *phi, int a, int j, int l, int i,
                    double *out);
/* classical RK4 step, phi re-solved at each stage (R17); f in-out */
void gkref_rk4_step(const gkref *, double *f, double dt);
/* per-species (particle, heat, momentum) fluxes (R18): out[nspecies*3] */
void gkref_fluxes(const gkref *, const double *f, const double *phi, double *out);
/* kx and ky spectra of |phi|^2 with the Parseval factor and Delta s applied (R20):
 * kx_spec[nkx], ky_spec[nky] */
void gkref_spectra(const gkref *, const double *phi, double *kx_spec, double *ky_spec);

/* CFL estimate of the largest stable RK4 step (readings R21-R23, see gkref.cpp):
 * out[0] = min of out[1] = nonlinear (ExB) bound for this phi, out[2] = von Neumann bound of the streaming and
 * trapping stencils, out[3] = field (omega_H) bound with kinetic electrons (+inf otherwise).  No safety factor. */
void gkref_estimate_dt(const gkref *, const double *phi, double *out4);

/* bracket of two spectral slabs (nkx*nky complex each): 0.5*sum (k'x k''y - k'y k''x) chi f */
void gkref_bracket_slab(const gkref *, const double *chi, const double *fs, int method, int mx,
                        int my, double *out);

/* tables for the pins.  which: see gkref.py TABLES.  Returns number of doubles written
 * (or needed if out == NULL). */
size_t gkref_table(const gkref *, const char *which, double *out);

#ifdef __cplusplus
}
#endif
#endif
