// gk_dev.h -- device-side parameter block of libgk (product path; shares nothing with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define GK_MAX_SPECIES 4
#define GK_SLAB_MAX 8192  // largest nkx*nky a CTA handles (moment accumulators live in registers)

// Per-species scalars, float copies of the host doubles.
struct GkSpeciesDev {
  float Z, T, mass, dens, vR, rlt, rln;
  float ToverZ, ZoverT;
  float momfac;  // Z n 2 pi w_v : species factor of the velocity-space moment (B_i, w_mu applied per point)
};

// Everything the kernels need that is not f itself.  Passed by value (__grid_constant__).
struct GkDev {
  int nsp, nv, nmu, ns, nkx, nky, K, ikx;
  int mx, my;        // padded real-space grid of the bracket (R14)
  int ldx;           // row stride (float2) of the x-transformed half-spectrum arrays  [mx][ldx]
  int ldy;           // row stride (float2) of real-space rows                          [rows][ldy]
  int rc;            // rows per chunk of the y-transform workspace (even, divides mx)
  int adiabatic, mask, storage;
  int jchunk, nchunk;  // vpar chunking of the stage kernel's work items
  int nparts;          // number of moment partial planes = nsp*nmu*nchunk
  int prefetch;        // 1: L2 prefetch of the single-use epilogue operands before the FFT phase
  int gchi_in_smem;    // 1: real-space grad(chi) lives in shared memory, 0: per-CTA global scratch
  float ds_inv, dv_inv;
  float dkx, ky0;      // kx_p = p*dkx, ky_m = m*ky0
  float kxmax, kymax;  // K*dkx, (nky-1)*ky0: largest retained wavenumbers (CFL estimate, R21)
  float invK, invM;    // 1/K, 1/(nky-1) (0 if degenerate)
  float hyp_x, hyp_y;  // nu_x, nu_y of the hyper-viscosity (0 if masked off)
  float nu_s, nu_v;
  float ae;            // ne/Te of the adiabatic electrons
  float fftnorm;       // 1/(mx*my)
  long long slab;      // nkx*nky
  long long nphi;      // ns*nkx*nky
  long long ntot;
  // tables (device pointers, float)
  const float *v, *fmv;             // [nv]  vpar_j, pi^-3/2 exp(-v^2)
  const float *mu, *wmu;            // [nmu]
  const float *fmm;                 // [nmu][ns] exp(-2 mu B)
  const float *B, *F, *BG, *sth, *cz, *Rmaj;  // [ns]  (sth, cz: kappa = -(kx sth + ky cz); Rmaj: R B_t/B)
  const float *ef;                  // [ns] ExB factor of terms III, V and of the fluxes relative to ky/2 (1 in s-alpha)
  const float *kx, *ky;             // [nkx], [nky]
  const float *hypx, *hypy;         // nu_x (kx/kxmax)^4, nu_y (ky/kymax)^4
  const float *J0;                  // [nsp][nmu][ns][nkx][nky]
  const float *dinv;                // [ns][nkx][nky] 1/(A+ae) or 1/A; 0 at (kx,ky)=(0,0)
  const float *zinv;                // [nkx] 1/<A/(A+ae)>_s, 0 at kx=0 (adiabatic only)
  const float2 *twx, *twy;          // [mx], [my] exp(+2 pi i t/N)
  GkSpeciesDev sp[GK_MAX_SPECIES];
  float dcoef[5][2][5];             // s-derivative stencil by (class+2, sign(v)<0, d+2), units 1/ds
  float discoef[5][5];              // s-dissipation stencil (delta^4/12 on class 0)
};

// One stage-kernel launch.
struct GkStageArgs {
  const void *y;     // state the RHS is evaluated on
  const void *fn;    // f_n (modes 2: y_next = f_n + c k)
  void *acc;         // RK accumulator
  void *out;         // y_next / rhs / f_{n+1}
  const float2 *phi; // potential of y
  float2 *mom;       // moment partial planes of `out` (nullptr: skip)
  float2 *gchi;      // per-CTA scratch for real-space grad(chi) when !gchi_in_smem
  float2 *chis;      // per-CTA scratch, 3*slab: chi = J0 phi, D_s chi for v>0, D_s chi for v<0
                     // (warp-specialised kernel: a ring of 3 such triples)
  float2 *nlbuf;     // warp-specialised kernel: per-CTA ring of 2 bracket slabs
  float c, b;        // y_next = base + c*k ; acc (+)= b*k     (dt folded in)
  int mode;          // 0: out = k; 1: acc = y + b k, out = y + c k; 2: acc += b k, out = fn + c k;
                     // 3: out = acc + b k
  int nwork;         // work items = nsp*nmu*ns*nchunk
  // diagnostics folded into the launch (nullptr: off)
  unsigned int *gmax;  // CFL (R21): atomicMax of the bits of max(|d_y chi| kx_max + |d_x chi| ky_max) over the real-space
                     // grad(chi) this launch builds (non-negative floats order like unsigned integers)
  double *fluxp;     // flux partial sums [cta][warp][species][3] of the state `y` (mode 1 only)
};
