// gkref.cpp -- CPU ORACLE (test infrastructure only; see gkref.h).
//
// Plain double-precision restatement of the discretised equations of SURVEY.md 8(c) /
// DESIGN.md "Discrete RHS".  No blocking, no fusion, no reuse across slabs: every point is
// evaluated from the formulas, in the paper's notation.  Citations are PAPER.md line numbers.
//
// Build: g++ -O2 -std=c++17 -fopenmp -shared -fPIC gkref.cpp -o libgkref.so
#include "gkref.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstring>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
static const double PI = 3.14159265358979323846264338327950288;

// ---------------------------------------------------------------------------------------
// Gauss-Laguerre nodes/weights (reading R3, config 1).  Roots of L_n by interlacing: the
// roots of L_k separate the roots of L_{k+1}; bisection in each bracket, then Newton.
// weight w_i = x_i / ((n+1)^2 L_{n+1}(x_i)^2)   (textbook formula).
// ---------------------------------------------------------------------------------------
static double laguerre(int n, double x) {
  double p0 = 1.0, p1 = 1.0 - x;
  if (n == 0) return p0;
  for (int k = 1; k < n; ++k) {
    double p2 = ((2.0 * k + 1.0 - x) * p1 - k * p0) / (k + 1.0);
    p0 = p1;
    p1 = p2;
  }
  return p1;
}

static void gauss_laguerre(int n, std::vector<double> &x, std::vector<double> &w) {
  std::vector<double> prev;  // roots of L_{k-1}
  for (int k = 1; k <= n; ++k) {
    std::vector<double> cur(k);
    for (int r = 0; r < k; ++r) {
      double lo = (r == 0) ? 0.0 : prev[r - 1];
      double hi = (r == k - 1) ? (4.0 * k + 2.0) : prev[r];
      double flo = laguerre(k, lo);
      for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        double fm = laguerre(k, mid);
        if ((fm > 0) == (flo > 0)) { lo = mid; flo = fm; } else { hi = mid; }
      }
      cur[r] = 0.5 * (lo + hi);
    }
    prev = cur;
  }
  x = prev;
  w.resize(n);
  for (int r = 0; r < n; ++r) {
    double l1 = laguerre(n + 1, x[r]);
    w[r] = x[r] / ((n + 1.0) * (n + 1.0) * l1 * l1);
  }
}

// ---------------------------------------------------------------------------------------
// Own complex FFT (any length; recursive Cooley-Tukey on the smallest prime factor, plain
// O(n^2) DFT for prime lengths).  sign = +1: sum x_n e^{+2 pi i nk/N};  -1: e^{-...}.
// Only a faster route to the truncated convolution that defines term III (R13, R14).
// ---------------------------------------------------------------------------------------
static void fft_rec(const cplx *in, cplx *out, int n, int stride, int sign) {
  if (n == 1) { out[0] = in[0]; return; }
  int p = 0;
  for (int d = 2; d * d <= n; ++d)
    if (n % d == 0) { p = d; break; }
  if (p == 0) {  // prime length: direct DFT
    for (int k = 0; k < n; ++k) {
      cplx acc = 0;
      for (int j = 0; j < n; ++j) {
        double ang = sign * 2.0 * PI * ((long long)j * k % n) / n;
        acc += in[(size_t)j * stride] * cplx(std::cos(ang), std::sin(ang));
      }
      out[k] = acc;
    }
    return;
  }
  int m = n / p;
  std::vector<cplx> sub((size_t)n);
  for (int r = 0; r < p; ++r) fft_rec(in + (size_t)r * stride, &sub[(size_t)r * m], m, stride * p, sign);
  for (int k = 0; k < n; ++k) {
    cplx acc = 0;
    for (int r = 0; r < p; ++r) {
      double ang = sign * 2.0 * PI * ((long long)r * k % n) / n;
      acc += sub[(size_t)r * m + (k % m)] * cplx(std::cos(ang), std::sin(ang));
    }
    out[k] = acc;
  }
}

// 2-D transform of a row-major [mx][my] array, in place.
static void fft2d(std::vector<cplx> &a, int mx, int my, int sign) {
  std::vector<cplx> tmp(std::max(mx, my)), col(mx);
  for (int x = 0; x < mx; ++x) {
    fft_rec(&a[(size_t)x * my], tmp.data(), my, 1, sign);
    for (int y = 0; y < my; ++y) a[(size_t)x * my + y] = tmp[y];
  }
  for (int y = 0; y < my; ++y) {
    for (int x = 0; x < mx; ++x) col[x] = a[(size_t)x * my + y];
    fft_rec(col.data(), tmp.data(), mx, 1, sign);
    for (int x = 0; x < mx; ++x) a[(size_t)x * my + y] = tmp[x];
  }
}

static int smooth7(int n) {  // smallest integer >= n with prime factors <= 7
  for (;; ++n) {
    int r = n;
    for (int p : {2, 3, 5, 7})
      while (r % p == 0) r /= p;
    if (r == 1) return n;
  }
}

// ---------------------------------------------------------------------------------------
struct gkref {
  gkref_grid g;
  gkref_geom geo;
  gkref_opts o;
  std::vector<gkref_species> sp;
  int nsp, nv, nmu, ns, nkx, nky, K;
  int mask;
  double dkx, ds, dv, kxmax, kymax;
  // grids and weights (R1, R3)
  std::vector<double> s, theta, v, mu, wmu, kx, ky;
  double wv;
  // s-alpha geometry (R2): B, F=ffun, BG = B*gfun, sin(theta), cz = cos+shat*theta*sin, R
  std::vector<double> B, F, BG, sth, cz, R;
  // metric of k_perp^2 = kx^2 + 2 kx ky gpz + ky^2 gzz (g_psipsi = 1 in both models; ky in k_theta rho units, i.e.
  // g_psizeta / kthnorm and g_zetazeta / kthnorm^2) and the ExB factor ef = 2 E^{psi zeta} / kthnorm
  // (1 in s-alpha: the factor 1/2 of terms III and V, R2)
  std::vector<double> gpz, gzz, ef;
  double kthnorm;
  // species tables
  std::vector<double> vR;                 // sqrt(T/m)
  std::vector<double> J0;                 // [a][l][i][p][m] (R4)
  std::vector<double> G0;                 // [a][i][p][m]
  std::vector<double> FM;                 // [j][l][i]       (R0)
  std::vector<double> Apol;               // [i][p][m] sum_a Z^2 n (1-Gamma0)/T
  // s stencils (R7): dcoef[class+2][sign(0: v>0, 1: v<0)][d+2], discoef[class+2][d+2]
  double dcoef[5][2][5], discoef[5][5];

  size_t nphi() const { return (size_t)ns * nkx * nky; }
  size_t nslab() const { return (size_t)nkx * nky; }
  size_t ntot() const { return (size_t)nsp * nv * nmu * ns * nkx * nky; }
  size_t fidx(int a, int j, int l, int i, int ip, int m) const {
    return ((((((size_t)a * nv + j) * nmu + l) * ns + i) * nkx + ip) * nky + m);
  }
  size_t pidx(int i, int ip, int m) const { return ((size_t)i * nkx + ip) * nky + m; }
  size_t jidx(int a, int l, int i, int ip, int m) const {
    return ((((size_t)a * nmu + l) * ns + i) * nkx + ip) * nky + m;
  }
  double kperp2(int i, int ip, int m) const {  // eq. 2 (s-alpha metric: R2)
    return kx[ip] * kx[ip] + 2.0 * kx[ip] * ky[m] * gpz[i] + ky[m] * ky[m] * gzz[i];
  }
  double kappa(int i, int ip, int m) const {  // kx D^psi + k_zeta D^zeta (R2)
    return -(kx[ip] * sth[i] + ky[m] * cz[i]);
  }
  // Parallel connectivity (R6).  Maps (i+d, ip, m) to an in-grid (i', ip');
  // returns false if the point lies beyond an open chain end.
  bool connect(int i, int d, int ip, int m, int &i2, int &ip2) const {
    i2 = i + d;
    ip2 = ip;
    if (i2 >= ns) {  // leaves at s=+1/2, continues at kx + m*ikxspace*dkx
      i2 -= ns;
      ip2 = ip + m * g.ikxspace;
      if (ip2 > nkx - 1) return false;
    } else if (i2 < 0) {
      i2 += ns;
      ip2 = ip - m * g.ikxspace;
      if (ip2 < 0) return false;
    }
    return true;
  }
  // pos_par_grid_class in {-2..2} (R7)
  int sclass(int i, int ip, int m) const {
    if (m == 0) return 0;  // zonal mode periodic
    if (i < 2 && ip - m * g.ikxspace < 0) return i - 2;
    if (i >= ns - 2 && ip + m * g.ikxspace > nkx - 1) return i - (ns - 3);
    return 0;
  }
  cplx getf(const cplx *f, int a, int j, int l, int i, int d, int ip, int m) const {
    int i2, ip2;
    if (!connect(i, d, ip, m, i2, ip2)) return 0.0;
    return f[fidx(a, j, l, i2, ip2, m)];
  }
  cplx getchi(const cplx *phi, int a, int l, int i, int d, int ip, int m) const {
    int i2, ip2;
    if (!connect(i, d, ip, m, i2, ip2)) return 0.0;
    return J0[jidx(a, l, i2, ip2, m)] * phi[pidx(i2, ip2, m)];
  }
  bool on(int bit) const { return (mask & bit) != 0; }

  void build();
  void field_solve(const cplx *f, cplx *phi) const;
  cplx linear_point(const cplx *f, const cplx *phi, int a, int j, int l, int i, int ip, int m) const;
  void bracket(const cplx *chi, const cplx *fs, int method, int mx, int my, cplx *out) const;
  void rhs_slab(const cplx *f, const cplx *phi, int a, int j, int l, int i, cplx *out) const;
  void rhs(const cplx *f, cplx *phi, cplx *out) const;
};

// ---------------------------------------------------------------------------------------
// create-time tables (step a0 of SURVEY 8(a))
// ---------------------------------------------------------------------------------------
void gkref::build() {
  nsp = o.nspecies; nv = g.nvpar; nmu = g.nmu; ns = g.ns; nkx = g.nkx; nky = g.nky;
  K = (nkx - 1) / 2;
  mask = (o.term_mask <= 0) ? GKREF_T_ALL : o.term_mask;
  if (!o.nonlinear) mask &= ~GKREF_T_III;

  // --- grids (R1) ---
  ds = 1.0 / ns;
  s.resize(ns); theta.resize(ns);
  for (int i = 0; i < ns; ++i) { s[i] = -0.5 + (i + 0.5) * ds; theta[i] = 2.0 * PI * s[i]; }
  dv = 2.0 * g.vpar_max / nv;
  wv = dv;
  v.resize(nv);
  for (int j = 0; j < nv; ++j) v[j] = -g.vpar_max + (j + 0.5) * dv;
  mu.resize(nmu); wmu.resize(nmu);
  if (g.mu_grid == 0) {  // Gauss-Laguerre in x = 2 mu:  int g(mu) dmu = 1/2 sum w e^x g(x/2)
    std::vector<double> x, w;
    gauss_laguerre(nmu, x, w);
    for (int l = 0; l < nmu; ++l) { mu[l] = 0.5 * x[l]; wmu[l] = 0.5 * w[l] * std::exp(x[l]); }
  } else {  // uniform in v_perp: mu = v_perp^2/2, d mu = v_perp d v_perp
    double dvp = g.vperp_max / nmu;
    for (int l = 0; l < nmu; ++l) {
      double vp = (l + 0.5) * dvp;
      mu[l] = 0.5 * vp * vp;
      wmu[l] = vp * dvp;
    }
  }
  // --- geometry ---
  B.resize(ns); F.resize(ns); BG.resize(ns); sth.resize(ns); cz.resize(ns); R.resize(ns);
  gpz.resize(ns); gzz.resize(ns); ef.resize(ns);
  double kxshift = 2.0 * PI * geo.shat;  // kx gained per poloidal turn, per unit ky
  if (o.geometry == 0) {
    // s-alpha (R2)
    kthnorm = geo.q / (2.0 * PI * geo.eps);
    for (int i = 0; i < ns; ++i) {
      double th = theta[i];
      R[i] = 1.0 + geo.eps * std::cos(th);
      B[i] = 1.0 / R[i];
      F[i] = 1.0 / (2.0 * PI * geo.q);                    // ffun  (eps->0 form)
      // gfun = F * d_s B / B;  d_s B = 2 pi eps sin(th) B^2  =>  B*gfun:
      BG[i] = (geo.eps / geo.q) * std::sin(th) * B[i] * B[i];
      sth[i] = std::sin(th);
      cz[i] = std::cos(th) + geo.shat * th * std::sin(th);
      gpz[i] = geo.shat * th;
      gzz[i] = 1.0 + geo.shat * geo.shat * th * th;
      ef[i] = 1.0;
    }
  } else {
    // Circular concentric (Lapillonne) model, reading R24.  Coordinates (R0 = 1): R = 1 + eps cos th,
    // Z = eps sin th, psi = eps, s = (th + eps sin th)/2pi, zeta = -phi/2pi + (q/pi) A,
    // A = atan[ sqrt((1-eps)/(1+eps)) tan(th/2) ] (the "branch-tracked arctan"), q' = shat q/eps.
    // Closed forms of the partial derivatives; gradients: |grad eps| = 1, grad th = e_th/eps, grad phi = e_phi/R.
    const double q = geo.q, eps = geo.eps, sq = std::sqrt(1.0 - eps * eps), dq = geo.shat * q / eps;
    auto point = [&](double th, double *out) {
      const double c = std::cos(th), sn = std::sin(th), Rr = 1.0 + eps * c;
      // B = delta / (1 + eps cos th), delta^2 = 1 + eps^2/(q^2 (1 - eps^2))                         (eq. 1)
      const double w = q * q * (1.0 - eps * eps), dw = 2.0 * q * dq * (1.0 - eps * eps) - 2.0 * eps * q * q;
      const double del = std::sqrt(1.0 + eps * eps / w);
      const double ddel = (2.0 * eps * w - eps * eps * dw) / (w * w) / (2.0 * del);
      const double Bv = del / Rr, B_th = del * eps * sn / (Rr * Rr), B_eps = ddel / Rr - del * c / (Rr * Rr);
      const double B_s = 2.0 * PI / Rr * B_th, B_psi = B_eps - sn / Rr * B_th;                    // eq. 3
      const double A = std::atan(std::sqrt((1.0 - eps) / (1.0 + eps)) * std::tan(0.5 * th));
      const double z_th = (q / PI) * sq / (2.0 * Rr);
      const double z_eps = (dq / PI) * A - (q / PI) * sn / (2.0 * sq * Rr);
      const double g_pz = z_eps, g_zz = 1.0 / (4.0 * PI * PI * Rr * Rr) + z_eps * z_eps + z_th * z_th / (eps * eps);
      const double g_ps = sn / (2.0 * PI), g_zs = z_eps * sn / (2.0 * PI) + z_th * Rr / (2.0 * PI * eps * eps);
      // E tensor: antisymmetric cofactors of the first two metric rows x pi dpf/dpsi / B^2
      const double pref = PI * (eps / (q * sq)) / (Bv * Bv);
      const double Epz = pref * (g_zz - g_pz * g_pz), Eps = pref * (g_zs - g_ps * g_pz), Ezs = pref * (g_pz * g_zs - g_ps * g_zz);
      out[0] = Bv; out[1] = B_s; out[2] = g_pz; out[3] = g_zz;
      out[4] = -2.0 * Eps * B_s / Bv;                                   // D^psi                   (eq. 4)
      out[5] = -2.0 * (-Epz * B_psi + Ezs * B_s) / Bv;                  // D^zeta
      out[6] = Epz; out[7] = Rr; out[8] = 1.0 / del;                    // bt_frac
    };
    double p0[9];
    point(0.0, p0);
    kthnorm = std::sqrt(p0[3]);
    kxshift = dq / kthnorm;   // g_psizeta grows by q' per turn (A -> A + pi): the chain is continuous with this shift
    for (int i = 0; i < ns; ++i) {
      // invert th + eps sin th = 2 pi s (Newton)
      double th = 2.0 * PI * s[i];
      for (int it = 0; it < 50; ++it) th -= (th + eps * std::sin(th) - 2.0 * PI * s[i]) / (1.0 + eps * std::cos(th));
      theta[i] = th;
      double pt[9];
      point(th, pt);
      B[i] = pt[0];
      F[i] = 1.0 / (2.0 * PI * q * sq) / pt[0];                         // ffun = b_ups / B
      BG[i] = F[i] * pt[1];                                             // B gfun = F d_s B
      gpz[i] = pt[2] / kthnorm;
      gzz[i] = pt[3] / (kthnorm * kthnorm);
      sth[i] = -pt[4];                                                  // kappa = kx D^psi + k_zeta D^zeta, k_zeta = ky/kthnorm
      cz[i] = -pt[5] / kthnorm;
      ef[i] = 2.0 * pt[6] / kthnorm;                                    // E^{psi zeta} k_zeta = ef ky / 2
      R[i] = pt[7] * pt[8];                                             // R B_t/B of the momentum flux (R18)
    }
  }
  dkx = kxshift * g.ky0 / g.ikxspace;
  kx.resize(nkx); ky.resize(nky);
  for (int ip = 0; ip < nkx; ++ip) kx[ip] = (ip - K) * dkx;
  for (int m = 0; m < nky; ++m) ky[m] = m * g.ky0;
  kxmax = K * dkx;
  kymax = (nky - 1) * g.ky0;

  // --- species tables ---
  vR.resize(nsp);
  J0.assign((size_t)nsp * nmu * ns * nkx * nky, 0.0);
  G0.assign((size_t)nsp * ns * nkx * nky, 0.0);
  Apol.assign(nphi(), 0.0);
  for (int a = 0; a < nsp; ++a) {
    vR[a] = std::sqrt(sp[a].temp / sp[a].mass);
    double rho = sp[a].mass * vR[a] / std::fabs(sp[a].Z);  // thermal gyroradius / rho_ref
    for (int i = 0; i < ns; ++i)
      for (int ip = 0; ip < nkx; ++ip)
        for (int m = 0; m < nky; ++m) {
          double kp = std::sqrt(kperp2(i, ip, m));
          double b = 0.5 * std::pow(rho * kp / B[i], 2);
          double g0 = std::cyl_bessel_i(0.0, b) * std::exp(-b);        // Gamma0 = I0(b) e^-b
          G0[((size_t)a * ns + i) * nkx * nky + (size_t)ip * nky + m] = g0;
          Apol[pidx(i, ip, m)] += sp[a].Z * sp[a].Z * sp[a].dens * (1.0 - g0) / sp[a].temp;
          for (int l = 0; l < nmu; ++l) {
            double lam = kp * rho * std::sqrt(2.0 * mu[l] / B[i]);     // R4
            J0[jidx(a, l, i, ip, m)] = std::cyl_bessel_j(0.0, lam);
          }
        }
  }
  FM.resize((size_t)nv * nmu * ns);
  for (int j = 0; j < nv; ++j)
    for (int l = 0; l < nmu; ++l)
      for (int i = 0; i < ns; ++i)
        FM[((size_t)j * nmu + l) * ns + i] =
            std::pow(PI, -1.5) * std::exp(-(v[j] * v[j] + 2.0 * mu[l] * B[i]));  // R0

  // --- s stencils (R7).  offsets d = -2..2 stored at d+2; all in units of 1/ds ---
  const double c4[5] = {1.0 / 12, -8.0 / 12, 0.0, 8.0 / 12, -1.0 / 12};  // 4th-order centred
  const double d4[5] = {1.0 / 12, -4.0 / 12, 6.0 / 12, -4.0 / 12, 1.0 / 12};  // delta^4 / 12
  const double upos[5] = {0.5, -2.0, 1.5, 0.0, 0.0};   // 2nd-order upwind, v > 0 (backward)
  const double uneg[5] = {0.0, 0.0, -1.5, 2.0, -0.5};  // 2nd-order upwind, v < 0 (forward)
  for (int c = 0; c < 5; ++c)
    for (int d = 0; d < 5; ++d) {
      bool interior = (c == 2) || (o.s_closure == 1);
      dcoef[c][0][d] = interior ? c4[d] : upos[d];
      dcoef[c][1][d] = interior ? c4[d] : uneg[d];
      discoef[c][d] = interior ? d4[d] : 0.0;
    }
}

// ---------------------------------------------------------------------------------------
// Field solve (R10 adiabatic with zonal correction, R11 kinetic).
//   N(i,p,m) = sum_a Z_a n_a 2 pi B_i sum_{j,l} w_v w_mu,l J0_a f_a
// ---------------------------------------------------------------------------------------
void gkref::field_solve(const cplx *f, cplx *phi) const {
  std::vector<cplx> N(nphi(), 0.0);
#pragma omp parallel for schedule(static)
  for (int i = 0; i < ns; ++i)
    for (int ip = 0; ip < nkx; ++ip)
      for (int m = 0; m < nky; ++m) {
        cplx acc = 0.0;
        for (int a = 0; a < nsp; ++a) {
          cplx mom = 0.0;
          for (int j = 0; j < nv; ++j)
            for (int l = 0; l < nmu; ++l)
              mom += wv * wmu[l] * J0[jidx(a, l, i, ip, m)] * f[fidx(a, j, l, i, ip, m)];
          acc += sp[a].Z * sp[a].dens * 2.0 * PI * B[i] * mom;
        }
        N[pidx(i, ip, m)] = acc;
      }
  if (o.adiabatic_electrons) {
    double ae = o.ne / o.te;  // adiabatic electron response n_e/T_e
    for (int ip = 0; ip < nkx; ++ip)
      for (int m = 0; m < nky; ++m) {
        if (m > 0) {
          for (int i = 0; i < ns; ++i) phi[pidx(i, ip, m)] = N[pidx(i, ip, m)] / (Apol[pidx(i, ip, m)] + ae);
        } else if (ip == K) {
          for (int i = 0; i < ns; ++i) phi[pidx(i, ip, m)] = 0.0;
        } else {
          // zonal: phi_i = (N_i + ae*phibar)/(A_i+ae), phibar = {phi} (flux-surface average,
          // uniform weight in s)  =>  phibar = {N/(A+ae)} / {A/(A+ae)}            (R10)
          cplx num = 0.0;
          double den = 0.0;
          for (int i = 0; i < ns; ++i) {
            double A = Apol[pidx(i, ip, m)];
            num += N[pidx(i, ip, m)] / (A + ae);
            den += A / (A + ae);
          }
          cplx phibar = (num / (double)ns) / (den / (double)ns);
          for (int i = 0; i < ns; ++i)
            phi[pidx(i, ip, m)] = (N[pidx(i, ip, m)] + ae * phibar) / (Apol[pidx(i, ip, m)] + ae);
        }
      }
  } else {
    for (int i = 0; i < ns; ++i)
      for (int ip = 0; ip < nkx; ++ip)
        for (int m = 0; m < nky; ++m) {
          if (ip == K && m == 0) phi[pidx(i, ip, m)] = 0.0;  // denominator := 1, phi := 0 (R11)
          else phi[pidx(i, ip, m)] = N[pidx(i, ip, m)] / Apol[pidx(i, ip, m)];
        }
  }
}

// ---------------------------------------------------------------------------------------
// Linear terms at one grid point (R0, R7-R9).
//   chi = J0_a phi,  kappa = kx D^psi + k_zeta D^zeta,  E = v^2 + 2 mu B,  E_D = v^2 + mu B
// ---------------------------------------------------------------------------------------
cplx gkref::linear_point(const cplx *f, const cplx *phi, int a, int j, int l, int i, int ip,
                         int m) const {
  const cplx I1(0.0, 1.0);
  const gkref_species &S = sp[a];
  const double vj = v[j], mul = mu[l], Bi = B[i];
  const double E = vj * vj + 2.0 * mul * Bi;
  const double ED = vj * vj + mul * Bi;
  const double fm = FM[((size_t)j * nmu + l) * ns + i];
  const double kap = kappa(i, ip, m);
  const int cls = sclass(i, ip, m) + 2;
  const int sg = (vj > 0.0) ? 0 : 1;
  const cplx f0 = f[fidx(a, j, l, i, ip, m)];
  const cplx chi0 = J0[jidx(a, l, i, ip, m)] * phi[pidx(i, ip, m)];
  cplx r = 0.0;

  // parallel derivative of f and of chi, and the 4th difference of f, with the seam gather
  cplx dsf = 0.0, dschi = 0.0, d4f = 0.0;
  for (int d = -2; d <= 2; ++d) {
    cplx fd = getf(f, a, j, l, i, d, ip, m);
    dsf += dcoef[cls][sg][d + 2] * fd;
    d4f += discoef[cls][d + 2] * fd;
    dschi += dcoef[cls][sg][d + 2] * getchi(phi, a, l, i, d, ip, m);
  }
  dsf /= ds; dschi /= ds; d4f /= ds;
  const double cpar = vR[a] * vj * F[i];  // v_R v_par F
  if (on(GKREF_T_I)) r += -cpar * dsf;                                  // I   -v_par grad_par f
  if (on(GKREF_T_DISS_S)) r += -o.disp_par * std::fabs(cpar) * d4f;     // upwinded dissipation
  if (on(GKREF_T_VII)) r += -(S.Z / S.temp) * cpar * fm * dschi;        // VII -Z F_M/T v_par grad_par chi

  // velocity derivative, zero padding outside the grid (R8)
  const double c4[5] = {1.0 / 12, -8.0 / 12, 0.0, 8.0 / 12, -1.0 / 12};
  const double d4[5] = {1.0 / 12, -4.0 / 12, 6.0 / 12, -4.0 / 12, 1.0 / 12};
  cplx dvf = 0.0, d4v = 0.0;
  for (int d = -2; d <= 2; ++d) {
    int j2 = j + d;
    if (j2 < 0 || j2 >= nv) continue;
    cplx fd = f[fidx(a, j2, l, i, ip, m)];
    dvf += c4[d + 2] * fd;
    d4v += d4[d + 2] * fd;
  }
  dvf /= dv; d4v /= dv;
  const double cmir = vR[a] * mul * BG[i];  // v_R mu B G
  if (on(GKREF_T_IV)) r += cmir * dvf;                                  // IV  +mu grad_par B df/dv
  if (on(GKREF_T_DISS_V)) r += -o.disp_vp * std::fabs(cmir) * d4v;

  if (on(GKREF_T_II)) r += -I1 * (S.temp / S.Z) * ED * kap * f0;        // II  -i k.v_D f
  if (on(GKREF_T_V))                                                    // V   -v_E . grad F_M
    r += -I1 * (0.5 * ef[i] * ky[m]) * chi0 * fm * (S.rln + (E - 1.5) * S.rlt);   // E^{psi zeta} k_zeta = ef ky/2
  if (on(GKREF_T_VIII)) r += -I1 * ED * kap * chi0 * fm;                // VIII
  if (on(GKREF_T_HYP)) {                                                // hyper-viscosity (R9)
    double hx = (kxmax > 0) ? std::pow(kx[ip] / kxmax, 4) : 0.0;
    double hy = (kymax > 0) ? std::pow(ky[m] / kymax, 4) : 0.0;
    r += -(o.disp_x * hx + o.disp_y * hy) * f0;
  }
  return r;
}

// ---------------------------------------------------------------------------------------
// Term III on one slab.  Plain definition (R13):
//   III_k = 1/2 sum_{k'+k''=k} (k'_x k''_y - k'_y k''_x) chi_{k'} f_{k''},
// k', k'', k all in the retained set |p|<=K, |m|<=nky-1; the stored half m>=0 is extended by
// g(-p,-m) = conj g(p,m).  Before that, the ky=0 column of each input is replaced by its
// Hermitian average g(p,0) <- (g(p,0)+conj g(-p,0))/2: that is what the paper's
// real-to-complex inverse ("discards the imaginary output by construction") and its packed
// C2C path ("both values are replaced with their Hermitian average") compute.
// method 1 = that sum written out; method 0 = the same through a zero-padded FFT (any
// mx >= 3K+1, my >= 3(nky-1)+1 gives the identical result, R14).
// ---------------------------------------------------------------------------------------
void gkref::bracket(const cplx *chi_in, const cplx *f_in, int method, int mx, int my,
                    cplx *out) const {
  const int M = nky - 1;
  const int nyf = 2 * M + 1;  // full ky range -M..M
  // full-spectrum copies, index [p+K][m+M]
  std::vector<cplx> C((size_t)nkx * nyf), Fq((size_t)nkx * nyf);
  auto fill = [&](const cplx *g, std::vector<cplx> &full) {
    for (int ip = 0; ip < nkx; ++ip) {
      cplx z = 0.5 * (g[(size_t)ip * nky] + std::conj(g[(size_t)(nkx - 1 - ip) * nky]));
      full[(size_t)ip * nyf + M] = z;
      for (int m = 1; m <= M; ++m) {
        full[(size_t)ip * nyf + M + m] = g[(size_t)ip * nky + m];
        full[(size_t)(nkx - 1 - ip) * nyf + M - m] = std::conj(g[(size_t)ip * nky + m]);
      }
    }
  };
  fill(chi_in, C);
  fill(f_in, Fq);
  if (method == 1) {
    for (int ip = 0; ip < nkx; ++ip)
      for (int m = 0; m <= M; ++m) {
        cplx acc = 0.0;
        int p = ip - K;
        for (int p1 = -K; p1 <= K; ++p1) {
          int p2 = p - p1;
          if (p2 < -K || p2 > K) continue;
          for (int m1 = -M; m1 <= M; ++m1) {
            int m2 = m - m1;
            if (m2 < -M || m2 > M) continue;
            double k1x = p1 * dkx, k1y = m1 * g.ky0, k2x = p2 * dkx, k2y = m2 * g.ky0;
            acc += (k1x * k2y - k1y * k2x) * C[(size_t)(p1 + K) * nyf + M + m1] *
                   Fq[(size_t)(p2 + K) * nyf + M + m2];
          }
        }
        out[(size_t)ip * nky + m] = 0.5 * acc;
      }
    return;
  }
  // padded FFT route: g(x,y) = sum g_k e^{i(kx x + ky y)} on an mx x my grid
  if (mx <= 0) mx = smooth7(3 * K + 1);
  if (my <= 0) my = smooth7(3 * M + 1);
  const cplx I1(0.0, 1.0);
  auto grad = [&](const std::vector<cplx> &full, int dir) {
    std::vector<cplx> a((size_t)mx * my, 0.0);
    for (int ip = 0; ip < nkx; ++ip)
      for (int mm = -M; mm <= M; ++mm) {
        int p = ip - K;
        int x = (p % mx + mx) % mx, y = (mm % my + my) % my;
        double k = (dir == 0) ? p * dkx : mm * g.ky0;
        a[(size_t)x * my + y] = I1 * k * full[(size_t)ip * nyf + M + mm];
      }
    fft2d(a, mx, my, +1);
    return a;
  };
  std::vector<cplx> dxc = grad(C, 0), dyc = grad(C, 1), dxf = grad(Fq, 0), dyf = grad(Fq, 1);
  std::vector<cplx> prod((size_t)mx * my);
  for (size_t n = 0; n < prod.size(); ++n)  // -v_E.grad f = 1/2 (d_y chi d_x f - d_x chi d_y f)
    prod[n] = 0.5 * (dyc[n] * dxf[n] - dxc[n] * dyf[n]);
  fft2d(prod, mx, my, -1);
  const double norm = 1.0 / ((double)mx * my);
  for (int ip = 0; ip < nkx; ++ip)
    for (int m = 0; m <= M; ++m) {
      int p = ip - K;
      int x = (p % mx + mx) % mx;
      out[(size_t)ip * nky + m] = norm * prod[(size_t)x * my + m];
    }
}

void gkref::rhs_slab(const cplx *f, const cplx *phi, int a, int j, int l, int i, cplx *out) const {
  for (int ip = 0; ip < nkx; ++ip)
    for (int m = 0; m < nky; ++m) out[(size_t)ip * nky + m] = linear_point(f, phi, a, j, l, i, ip, m);
  if (on(GKREF_T_III)) {
    std::vector<cplx> chi(nslab()), nl(nslab());
    for (int ip = 0; ip < nkx; ++ip)
      for (int m = 0; m < nky; ++m) chi[(size_t)ip * nky + m] = J0[jidx(a, l, i, ip, m)] * phi[pidx(i, ip, m)];
    bracket(chi.data(), &f[fidx(a, j, l, i, 0, 0)], o.bracket_method, o.pad_mx, o.pad_my, nl.data());
    for (size_t n = 0; n < nslab(); ++n) out[n] += ef[i] * nl[n];   // the bracket carries the same ExB factor
  }
}

void gkref::rhs(const cplx *f, cplx *phi, cplx *out) const {
  field_solve(f, phi);
  const long nslabs = (long)nsp * nv * nmu * ns;
#pragma omp parallel for schedule(dynamic, 4)
  for (long t = 0; t < nslabs; ++t) {
    int i = (int)(t % ns);
    int l = (int)((t / ns) % nmu);
    int j = (int)((t / ((long)ns * nmu)) % nv);
    int a = (int)(t / ((long)ns * nmu * nv));
    rhs_slab(f, phi, a, j, l, i, &out[fidx(a, j, l, i, 0, 0)]);
  }
}

// ---------------------------------------------------------------------------------------
// C API
// ---------------------------------------------------------------------------------------
extern "C" {

gkref *gkref_create(const gkref_grid *g, const gkref_species *sp, const gkref_geom *geo,
                    const gkref_opts *o) {
  if (!g || !sp || !geo || !o) return nullptr;
  if (g->nkx % 2 == 0 || g->ns < 4 || g->nvpar < 4 || g->nky < 1 || g->nmu < 1 || o->nspecies < 1)
    return nullptr;
  gkref *h = new gkref();
  h->g = *g; h->geo = *geo; h->o = *o;
  h->sp.assign(sp, sp + o->nspecies);
  h->build();
  return h;
}
void gkref_destroy(gkref *h) { delete h; }

int gkref_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
  return omp_get_max_threads();
#else
  (void)n;
  return 1;
#endif
}

void gkref_field_solve(const gkref *h, const double *f, double *phi) {
  h->field_solve((const cplx *)f, (cplx *)phi);
}
void gkref_rhs(const gkref *h, const double *f, double *phi, double *rhs) {
  h->rhs((const cplx *)f, (cplx *)phi, (cplx *)rhs);
}
void gkref_rhs_slab(const gkref *h, const double *f, const double *phi, int a, int j, int l, int i,
                    double *out) {
  h->rhs_slab((const cplx *)f, (const cplx *)phi, a, j, l, i, (cplx *)out);
}

// Classical RK4 (R17): tableau 1/2, 1/2, 1; weights 1/6, 1/3, 1/3, 1/6.
void gkref_rk4_step(const gkref *h, double *f_io, double dt) {
  const size_t n = h->ntot();
  cplx *f = (cplx *)f_io;
  std::vector<cplx> k1(n), k2(n), k3(n), k4(n), y(n), phi(h->nphi());
  h->rhs(f, phi.data(), k1.data());
  for (size_t q = 0; q < n; ++q) y[q] = f[q] + 0.5 * dt * k1[q];
  h->rhs(y.data(), phi.data(), k2.data());
  for (size_t q = 0; q < n; ++q) y[q] = f[q] + 0.5 * dt * k2[q];
  h->rhs(y.data(), phi.data(), k3.data());
  for (size_t q = 0; q < n; ++q) y[q] = f[q] + dt * k3[q];
  h->rhs(y.data(), phi.data(), k4.data());
  for (size_t q = 0; q < n; ++q) f[q] += dt / 6.0 * (k1[q] + 2.0 * k2[q] + 2.0 * k3[q] + k4[q]);
}

// Fluxes (R18 -- parity unpinned):
//  flux_a[q] = - sum_i (1/ns) sum_{p,m} P_m (ky_m/2) 2 pi B_i sum_{j,l} w_v w_mu Im[conj(chi) f] M_q
//  M = {1, E*T_a, v_j * m_a v_R * R_i B_t/B}, B_t/B = 1 in s-alpha, P_m = 1 (m=0) or 2.
void gkref_fluxes(const gkref *h, const double *f_in, const double *phi_in, double *out) {
  const cplx *f = (const cplx *)f_in, *phi = (const cplx *)phi_in;
  for (int a = 0; a < h->nsp; ++a) {
    double acc[3] = {0, 0, 0};
    for (int j = 0; j < h->nv; ++j)
      for (int l = 0; l < h->nmu; ++l)
        for (int i = 0; i < h->ns; ++i)
          for (int ip = 0; ip < h->nkx; ++ip)
            for (int m = 0; m < h->nky; ++m) {
              cplx chi = h->J0[h->jidx(a, l, i, ip, m)] * phi[h->pidx(i, ip, m)];
              double im = std::imag(std::conj(chi) * f[h->fidx(a, j, l, i, ip, m)]);
              double P = (m == 0) ? 1.0 : 2.0;
              double w = -(1.0 / h->ns) * P * 0.5 * h->ef[i] * h->ky[m] * 2.0 * PI * h->B[i] * h->wv * h->wmu[l] * im;
              double E = h->v[j] * h->v[j] + 2.0 * h->mu[l] * h->B[i];
              acc[0] += w;
              acc[1] += w * E * h->sp[a].temp;
              acc[2] += w * h->v[j] * h->sp[a].mass * h->vR[a] * h->R[i];
            }
    for (int q = 0; q < 3; ++q) out[a * 3 + q] = acc[q];
  }
}

// Spectra of the potential (ky_spec = sum_{s,kx} |phi|^2, kx_spec = sum_{s,ky} |phi|^2;
// "the Parseval factor P_ky and parallel integration weight Delta s are applied"; R20:
// both factors in both spectra, Delta s = 1/ns, P_m = 1 (m=0) or 2):
//   kx_spec[p] = ds sum_i sum_m P_m |phi(i,p,m)|^2 ,   ky_spec[m] = ds P_m sum_i sum_p |phi(i,p,m)|^2
void gkref_spectra(const gkref *h, const double *phi_in, double *kx_spec, double *ky_spec) {
  const cplx *phi = (const cplx *)phi_in;
  const double ds = 1.0 / h->ns;
  for (int ip = 0; ip < h->nkx; ++ip) kx_spec[ip] = 0.0;
  for (int m = 0; m < h->nky; ++m) ky_spec[m] = 0.0;
  for (int i = 0; i < h->ns; ++i)
    for (int ip = 0; ip < h->nkx; ++ip)
      for (int m = 0; m < h->nky; ++m) {
        const double P = (m == 0) ? 1.0 : 2.0;
        const double a2 = std::norm(phi[h->pidx(i, ip, m)]);
        kx_spec[ip] += ds * P * a2;
        ky_spec[m] += ds * P * a2;
      }
}

// ---------------------------------------------------------------------------------------
// CFL estimate of the time step ("estimate_timestep": "the minimum of (i) the
// nonlinear CFL from the maximum real-space ExB velocity gradient, (ii) a von Neumann stability analysis
// of the streaming and trapping stencils, and (iii) for kinetic electrons, a field CFL based on the
// electrostatic Alfven frequency").  The paper prints no formula for (i) and (ii) and a dimensionally
// garbled one for (iii); readings R21-R23 of DESIGN.md:
//
//  every bound is the LARGEST step for which classical RK4 is stable on the model problem, no safety
//  factor (the caller applies one).  RK4: R(z) = 1 + z + z^2/2 + z^3/6 + z^4/24; on the imaginary axis
//  |R(iy)| <= 1  <=>  |y| <= 2 sqrt 2.
//
//  R21 (i)   term III advects f with v_E = (1/2)(-d_y chi, d_x chi); a uniform velocity u acts on the
//            retained spectrum with eigenvalues i(u_x kx + u_y ky), so
//              lambda_NL = max over (a, l, i) and the points (x, y) of the padded real-space grid of
//                          (1/2) ( |d_y chi| kx_max + |d_x chi| ky_max ),   dt_NL = 2 sqrt2 / lambda_NL.
//            chi = J0_a phi with the ky = 0 column Hermitian-averaged exactly as in the bracket (R15);
//            the real-space grid is the bracket's (pad_mx x pad_my).
//  R22 (ii)  frozen-coefficient von Neumann analysis of terms I + IV with their dissipation on the interior
//            stencils: symbols sigma(t) = (8 sin t - sin 2t)/6 of the centred 4th-order first derivative
//            and d(t) = (2 - 2 cos t)^2 / 12 of delta^4/12,
//              z(t, t') = c_s [ -i sigma(t) - nu_s d(t) ] + c_v [ +i sigma(t') - nu_v d(t') ],
//              c_s = max_{a,j,i} |v_R v_j F_i| / ds,   c_v = max_{a,l,i} |v_R mu_l B_i G_i| / dv,
//            dt_lin = min over the 64 x 64 angles t, t' = 2 pi k/64 of the first exit of the ray {tau z}
//            from the RK4 stability region (located by 4096 uniform steps to 4/|z|, then bisection).
//  R23 (iii) kinetic electrons: the cold-fluid response of every species to the parallel electric field
//            closes with the polarisation A = sum_a Z_a^2 n_a (1 - Gamma0_a)/T_a into the electrostatic
//            shear-Alfven (omega_H) oscillation
//              omega_H^2(i,p,m) = sum_a (v_R,a F_i k_s)^2 Z_a^2 n_a <v_par^2> / (T_a A(i,p,m)),
//            <v_par^2> = int v_par^2 F_M d^3v = 1/2, k_s = max_t sigma(t) / ds = 1.372 / ds the largest
//            parallel wavenumber the stencil represents;  dt_field = 2 sqrt2 / max_{(i,p,m) != zonal (0,0)} omega_H.
//            (PAPER.md:356 prints "omega ~ k_perp sqrt(me/mi) v_th,i/(q ds B)", the reciprocal of this
//            dependence on k_perp, mass ratio and B: taken as a garbled statement of the same mode, whose
//            frequency the operator's eigen-solve shows to scale as 1/k_perp, tests/test_oracle_cfl.py.)
//            +infinity with adiabatic electrons.
//  out[0] = min(out[1], out[2], out[3]); out[1] = dt_NL (+inf if phi = 0 or term III is off),
//  out[2] = dt_lin, out[3] = dt_field.
// ---------------------------------------------------------------------------------------
static double rk4_amp2(std::complex<double> z) {
  std::complex<double> R = 1.0 + z * (1.0 + z * (0.5 + z * (1.0 / 6.0 + z / 24.0)));
  return std::norm(R);
}
// first exit of the ray {tau z, tau > 0} from |R| <= 1
static double rk4_ray_limit(std::complex<double> z) {
  const double az = std::abs(z);
  if (az == 0.0) return HUGE_VAL;
  const int NSTEP = 4096;
  const double tmax = 4.0 / az;
  double lo = 0.0, hi = -1.0;
  for (int k = 1; k <= NSTEP; ++k) {
    double t = tmax * k / NSTEP;
    if (rk4_amp2(t * z) > 1.0 + 1e-13) { hi = t; break; }
    lo = t;
  }
  if (hi < 0.0) return tmax;
  for (int it = 0; it < 80; ++it) {
    double mid = 0.5 * (lo + hi);
    if (rk4_amp2(mid * z) > 1.0 + 1e-13) hi = mid; else lo = mid;
  }
  return lo;
}

void gkref_estimate_dt(const gkref *h, const double *phi_in, double *out) {
  const cplx *phi = (const cplx *)phi_in;
  const cplx I1(0.0, 1.0);
  const double lim = 2.0 * std::sqrt(2.0);
  // ---- (i) nonlinear ----
  double lamnl = 0.0;
  if (h->on(GKREF_T_III)) {
    const int nkx = h->nkx, nky = h->nky, K = h->K, M = nky - 1;
    int mx = h->o.pad_mx > 0 ? h->o.pad_mx : smooth7(3 * K + 1);
    int my = h->o.pad_my > 0 ? h->o.pad_my : smooth7(3 * M + 1);
    for (int a = 0; a < h->nsp; ++a)
      for (int l = 0; l < h->nmu; ++l)
        for (int i = 0; i < h->ns; ++i) {
          std::vector<cplx> gx((size_t)mx * my, 0.0), gy((size_t)mx * my, 0.0);
          for (int ip = 0; ip < nkx; ++ip)
            for (int m = 0; m <= M; ++m) {
              cplx c = h->J0[h->jidx(a, l, i, ip, m)] * phi[h->pidx(i, ip, m)];
              int p = ip - K;
              if (m == 0) {  // Hermitian average of the ky = 0 column (R15)
                int iq = nkx - 1 - ip;
                c = 0.5 * (c + std::conj(h->J0[h->jidx(a, l, i, iq, 0)] * phi[h->pidx(i, iq, 0)]));
              }
              int x = (p % mx + mx) % mx;
              gx[(size_t)x * my + m] = I1 * (p * h->dkx) * c;
              gy[(size_t)x * my + m] = I1 * (m * h->g.ky0) * c;
              if (m > 0) {  // g(-p, -m) = conj g(p, m)
                int x2 = ((-p) % mx + mx) % mx, y2 = my - m;
                gx[(size_t)x2 * my + y2] = I1 * (-p * h->dkx) * std::conj(c);
                gy[(size_t)x2 * my + y2] = I1 * (-m * h->g.ky0) * std::conj(c);
              }
            }
          fft2d(gx, mx, my, +1);
          fft2d(gy, mx, my, +1);
          for (size_t n = 0; n < gx.size(); ++n) {
            double lam = 0.5 * h->ef[i] * (std::fabs(gy[n].real()) * h->kxmax + std::fabs(gx[n].real()) * h->kymax);
            lamnl = std::max(lamnl, lam);
          }
        }
  }
  out[1] = lamnl > 0.0 ? lim / lamnl : HUGE_VAL;
  // ---- (ii) von Neumann, streaming + trapping ----
  double cs = 0.0, cv = 0.0;
  for (int a = 0; a < h->nsp; ++a)
    for (int i = 0; i < h->ns; ++i) {
      for (int j = 0; j < h->nv; ++j) cs = std::max(cs, std::fabs(h->vR[a] * h->v[j] * h->F[i]) / h->ds);
      for (int l = 0; l < h->nmu; ++l) cv = std::max(cv, std::fabs(h->vR[a] * h->mu[l] * h->BG[i]) / h->dv);
    }
  if (!h->on(GKREF_T_I)) cs = 0.0;
  if (!h->on(GKREF_T_IV)) cv = 0.0;
  const double nus = h->on(GKREF_T_DISS_S) ? h->o.disp_par : 0.0, nuv = h->on(GKREF_T_DISS_V) ? h->o.disp_vp : 0.0;
  const int NA = 64;
  double dtlin = HUGE_VAL;
  for (int k1 = 0; k1 < NA; ++k1)
    for (int k2 = 0; k2 < NA; ++k2) {
      double t1 = 2.0 * PI * k1 / NA, t2 = 2.0 * PI * k2 / NA;
      double s1 = (8.0 * std::sin(t1) - std::sin(2.0 * t1)) / 6.0, d1 = std::pow(2.0 - 2.0 * std::cos(t1), 2) / 12.0;
      double s2 = (8.0 * std::sin(t2) - std::sin(2.0 * t2)) / 6.0, d2 = std::pow(2.0 - 2.0 * std::cos(t2), 2) / 12.0;
      cplx z = cs * cplx(-nus * d1, -s1) + cv * cplx(-nuv * d2, s2);
      dtlin = std::min(dtlin, rk4_ray_limit(z));
    }
  out[2] = dtlin;
  // ---- (iii) field CFL, kinetic electrons only ----
  out[3] = HUGE_VAL;
  if (!h->o.adiabatic_electrons && h->on(GKREF_T_I) && h->on(GKREF_T_VII)) {
    double smax = 0.0;  // max_t sigma(t), located on a fine grid (the maximum is flat: 1.3722)
    for (int k = 0; k <= 100000; ++k) {
      double t = PI * k / 100000.0;
      smax = std::max(smax, (8.0 * std::sin(t) - std::sin(2.0 * t)) / 6.0);
    }
    double om2 = 0.0;
    for (int i = 0; i < h->ns; ++i)
      for (int ip = 0; ip < h->nkx; ++ip)
        for (int m = 0; m < h->nky; ++m) {
          if (ip == h->K && m == 0) continue;
          double num = 0.0;
          for (int a = 0; a < h->nsp; ++a) {
            double c = h->vR[a] * h->F[i] * smax / h->ds;
            num += c * c * h->sp[a].Z * h->sp[a].Z * h->sp[a].dens * 0.5 / h->sp[a].temp;
          }
          om2 = std::max(om2, num / h->Apol[h->pidx(i, ip, m)]);
        }
    if (om2 > 0.0) out[3] = lim / std::sqrt(om2);
  }
  out[0] = std::min(out[1], std::min(out[2], out[3]));
}

void gkref_bracket_slab(const gkref *h, const double *chi, const double *fs, int method, int mx,
                        int my, double *out) {
  h->bracket((const cplx *)chi, (const cplx *)fs, method, mx, my, (cplx *)out);
}

size_t gkref_table(const gkref *h, const char *which, double *out) {
  std::string w(which);
  const std::vector<double> *src = nullptr;
  std::vector<double> tmp;
  if (w == "s") src = &h->s;
  else if (w == "theta") src = &h->theta;
  else if (w == "vpar") src = &h->v;
  else if (w == "mu") src = &h->mu;
  else if (w == "wmu") src = &h->wmu;
  else if (w == "kx") src = &h->kx;
  else if (w == "ky") src = &h->ky;
  else if (w == "B") src = &h->B;
  else if (w == "F") src = &h->F;
  else if (w == "BG") src = &h->BG;
  else if (w == "R") src = &h->R;
  else if (w == "vR") src = &h->vR;
  else if (w == "J0") src = &h->J0;
  else if (w == "Gamma0") src = &h->G0;
  else if (w == "FM") src = &h->FM;
  else if (w == "Apol") src = &h->Apol;
  else if (w == "ef") src = &h->ef;
  else if (w == "gpz") src = &h->gpz;
  else if (w == "gzz") src = &h->gzz;
  else if (w == "sth") src = &h->sth;
  else if (w == "cz") src = &h->cz;
  else if (w == "kthnorm") { tmp = {h->kthnorm}; src = &tmp; }
  else if (w == "dkx") { tmp = {h->dkx}; src = &tmp; }
  else if (w == "wv") { tmp = {h->wv}; src = &tmp; }
  else if (w == "kperp2" || w == "kappa" || w == "sclass") {
    tmp.resize(h->nphi());
    for (int i = 0; i < h->ns; ++i)
      for (int ip = 0; ip < h->nkx; ++ip)
        for (int m = 0; m < h->nky; ++m)
          tmp[h->pidx(i, ip, m)] = (w == "kperp2") ? h->kperp2(i, ip, m)
                                   : (w == "kappa") ? h->kappa(i, ip, m)
                                                    : (double)h->sclass(i, ip, m);
    src = &tmp;
  } else if (w == "dcoef") {
    tmp.assign(&h->dcoef[0][0][0], &h->dcoef[0][0][0] + 50);
    src = &tmp;
  } else if (w == "pad") {
    tmp = {(double)(h->o.pad_mx > 0 ? h->o.pad_mx : smooth7(3 * h->K + 1)),
           (double)(h->o.pad_my > 0 ? h->o.pad_my : smooth7(3 * (h->nky - 1) + 1))};
    src = &tmp;
  } else return 0;
  if (out) std::memcpy(out, src->data(), src->size() * sizeof(double));
  return src->size();
}

}  // extern "C"
