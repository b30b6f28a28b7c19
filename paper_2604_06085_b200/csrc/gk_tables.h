// gk_tables.h -- create-time tables of libgk, computed on the host in double precision
// (step a0: PAPER.md:65, 336).  Product path: its own quadrature / Bessel / geometry code,
// nothing shared with oracle/.
#pragma once
#include <cmath>
#include <vector>

#include "../../include/gk.h"

namespace gkt {

constexpr double kPi = 3.14159265358979323846264338327950288;

// J0(x) = (1/pi) int_0^pi cos(x sin t) dt and I0(b) e^-b = (1/pi) int_0^pi exp(b (cos t - 1)) dt by the
// periodic trapezoid rule (spectrally accurate: the error is ~ J_{2M}(x), I_{2M}(b) e^-b).
inline double bessel_j0(double x) {
  const int M = 64 + (int)(1.5 * std::fabs(x));
  double s = 0.0;
  for (int k = 0; k < M; ++k) {
    double t = kPi * (k + 0.5) / M;  // midpoint rule on [0, pi]
    s += std::cos(x * std::sin(t));
  }
  return s / M;
}
inline double bessel_i0e(double b) {
  const int M = 64 + (int)(1.5 * std::fabs(b));
  double s = 0.0;
  for (int k = 0; k < M; ++k) {
    double t = kPi * (k + 0.5) / M;
    s += std::exp(b * (std::cos(t) - 1.0));
  }
  return s / M;
}

// Gauss-Laguerre by Golub-Welsch: nodes = eigenvalues of the Jacobi matrix (diag 2k+1, off-diag k),
// found by Sturm-sequence bisection; weights from the Christoffel function 1 / sum_k L_k(x)^2.
inline int sturm_count(int n, double x) {  // number of eigenvalues < x
  int cnt = 0;
  double d = 1.0;
  for (int k = 0; k < n; ++k) {
    double a = 2.0 * k + 1.0, b2 = (k == 0) ? 0.0 : (double)k * k;
    d = (a - x) - (k == 0 ? 0.0 : b2 / d);
    if (d == 0.0) d = 1e-300;
    if (d < 0) ++cnt;
  }
  return cnt;
}
inline void gauss_laguerre(int n, std::vector<double> &x, std::vector<double> &w) {
  x.resize(n);
  w.resize(n);
  for (int r = 0; r < n; ++r) {
    double lo = 0.0, hi = 4.0 * n + 3.0;
    for (int it = 0; it < 200; ++it) {
      double mid = 0.5 * (lo + hi);
      if (sturm_count(n, mid) > r) hi = mid; else lo = mid;
    }
    x[r] = 0.5 * (lo + hi);
    double p0 = 1.0, p1 = 1.0 - x[r], sum = 1.0;
    if (n > 1) sum += p1 * p1;
    for (int k = 1; k + 1 < n; ++k) {
      double p2 = ((2.0 * k + 1.0 - x[r]) * p1 - k * p0) / (k + 1.0);
      p0 = p1;
      p1 = p2;
      sum += p1 * p1;
    }
    w[r] = 1.0 / sum;
  }
}

struct Tables {
  int nsp, nv, nmu, ns, nkx, nky, K;
  double dkx, ds, dv, wv;
  std::vector<double> v, fmv, mu, wmu, fmm, B, F, BG, sth, cz, Rmaj, kx, ky, hypx, hypy;
  std::vector<double> J0, G0, den, dinv, zinv;
  std::vector<double> vR;
  double dcoef[5][2][5], discoef[5][5];
};

inline void build_tables(const gk_grid &g, const gk_species *sp, const gk_salpha &geo, const gk_opts &o,
                         Tables &T) {
  T.nsp = o.nspecies; T.nv = g.nvpar; T.nmu = g.nmu; T.ns = g.ns; T.nkx = g.nkx; T.nky = g.nky;
  T.K = (g.nkx - 1) / 2;
  const int nsp = T.nsp, nv = T.nv, nmu = T.nmu, ns = T.ns, nkx = T.nkx, nky = T.nky, K = T.K;
  T.ds = 1.0 / ns;
  T.dv = 2.0 * g.vpar_max / nv;
  T.wv = T.dv;
  T.dkx = 2.0 * kPi * geo.shat * g.ky0 / g.ikxspace;
  T.v.resize(nv); T.fmv.resize(nv);
  for (int j = 0; j < nv; ++j) {
    T.v[j] = -g.vpar_max + (j + 0.5) * T.dv;
    T.fmv[j] = std::exp(-T.v[j] * T.v[j]) / (kPi * std::sqrt(kPi));
  }
  T.mu.resize(nmu); T.wmu.resize(nmu);
  if (g.mu_grid == 0) {
    std::vector<double> x, w;
    gauss_laguerre(nmu, x, w);
    for (int l = 0; l < nmu; ++l) { T.mu[l] = 0.5 * x[l]; T.wmu[l] = 0.5 * w[l] * std::exp(x[l]); }
  } else {
    const double h = g.vperp_max / nmu;
    for (int l = 0; l < nmu; ++l) {
      const double vp = (l + 0.5) * h;
      T.mu[l] = 0.5 * vp * vp;
      T.wmu[l] = vp * h;
    }
  }
  T.kx.resize(nkx); T.ky.resize(nky); T.hypx.resize(nkx); T.hypy.resize(nky);
  for (int ip = 0; ip < nkx; ++ip) {
    T.kx[ip] = (ip - K) * T.dkx;
    T.hypx[ip] = (K > 0) ? o.disp_x * std::pow((double)(ip - K) / K, 4) : 0.0;
  }
  for (int m = 0; m < nky; ++m) {
    T.ky[m] = m * g.ky0;
    T.hypy[m] = (nky > 1) ? o.disp_y * std::pow((double)m / (nky - 1), 4) : 0.0;
  }
  // s-alpha geometry (R2)
  T.B.resize(ns); T.F.resize(ns); T.BG.resize(ns); T.sth.resize(ns); T.cz.resize(ns); T.Rmaj.resize(ns);
  T.fmm.resize((size_t)nmu * ns);
  std::vector<double> theta(ns);
  for (int i = 0; i < ns; ++i) {
    theta[i] = 2.0 * kPi * (-0.5 + (i + 0.5) * T.ds);
    const double ct = std::cos(theta[i]), st = std::sin(theta[i]);
    T.Rmaj[i] = 1.0 + geo.eps * ct;
    T.B[i] = 1.0 / T.Rmaj[i];
    T.F[i] = 0.5 / (kPi * geo.q);
    T.BG[i] = geo.eps * st / (geo.q * T.Rmaj[i] * T.Rmaj[i]);
    T.sth[i] = st;
    T.cz[i] = ct + geo.shat * theta[i] * st;
    for (int l = 0; l < nmu; ++l) T.fmm[(size_t)l * ns + i] = std::exp(-2.0 * T.mu[l] * T.B[i]);
  }
  // FLR kernels and Poisson denominators
  const size_t nphi = (size_t)ns * nkx * nky;
  T.vR.resize(nsp);
  T.J0.assign((size_t)nsp * nmu * nphi, 0.0);
  T.G0.assign((size_t)nsp * nphi, 0.0);
  T.den.assign(nphi, 0.0);
  for (int a = 0; a < nsp; ++a) {
    T.vR[a] = std::sqrt(sp[a].temp / sp[a].mass);
    const double rho = sp[a].mass * T.vR[a] / std::fabs(sp[a].Z);
    for (int i = 0; i < ns; ++i)
      for (int ip = 0; ip < nkx; ++ip)
        for (int m = 0; m < nky; ++m) {
          const size_t e = ((size_t)i * nkx + ip) * nky + m;
          const double kxl = T.kx[ip] + geo.shat * theta[i] * T.ky[m];
          const double kperp = std::sqrt(kxl * kxl + T.ky[m] * T.ky[m]);
          const double arg = rho * kperp / T.B[i];
          const double g0 = bessel_i0e(0.5 * arg * arg);
          T.G0[(size_t)a * nphi + e] = g0;
          T.den[e] += sp[a].Z * sp[a].Z * sp[a].dens * (1.0 - g0) / sp[a].temp;
          for (int l = 0; l < nmu; ++l)
            T.J0[((size_t)a * nmu + l) * nphi + e] =
                bessel_j0(kperp * rho * std::sqrt(2.0 * T.mu[l] / T.B[i]));
        }
  }
  T.dinv.assign(nphi, 0.0);
  T.zinv.assign(nkx, 0.0);
  const double ae = o.adiabatic_electrons ? o.ne / o.te : 0.0;
  for (size_t e = 0; e < nphi; ++e) {
    const int m = (int)(e % nky), ip = (int)((e / nky) % nkx);
    T.den[e] += ae;
    T.dinv[e] = (ip == K && m == 0) ? 0.0 : 1.0 / T.den[e];
  }
  if (o.adiabatic_electrons)
    for (int ip = 0; ip < nkx; ++ip) {
      if (ip == K) continue;
      double zs = 0.0;  // <A/(A+ae)>_s in double: it is O(kx^2) (R10)
      for (int i = 0; i < ns; ++i) {
        const double d = T.den[((size_t)i * nkx + ip) * nky];
        zs += (d - ae) / d;
      }
      T.zinv[ip] = (double)ns / zs;
    }
  // s stencils by class and streaming direction (R7)
  const double c4[5] = {1.0 / 12, -8.0 / 12, 0.0, 8.0 / 12, -1.0 / 12};
  const double d4[5] = {1.0 / 12, -4.0 / 12, 6.0 / 12, -4.0 / 12, 1.0 / 12};
  const double up[2][5] = {{0.5, -2.0, 1.5, 0.0, 0.0}, {0.0, 0.0, -1.5, 2.0, -0.5}};
  for (int c = 0; c < 5; ++c)
    for (int d = 0; d < 5; ++d) {
      const bool centred = (c == 2) || (o.s_closure == 1);
      for (int sg = 0; sg < 2; ++sg) T.dcoef[c][sg][d] = centred ? c4[d] : up[sg][d];
      T.discoef[c][d] = centred ? d4[d] : 0.0;
    }
}

}  // namespace gkt
