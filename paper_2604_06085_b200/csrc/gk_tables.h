// gk_tables.h -- create-time tables of libgk, computed on the host in double precision
// (step a0: PAPER.md:65, 336).  Product path: its own quadrature / Bessel / geometry code,
// nothing shared with oracle/.
#pragma once
#include <algorithm>
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

// ---------------------------------------------------------------------------------------------------------------
// Create-time part of the CFL estimate (readings R22, R23 of DESIGN.md): the largest RK4-stable
// step of (ii) the streaming and trapping stencils by a frozen-coefficient von Neumann analysis and (iii), with
// kinetic electrons, of the electrostatic shear-Alfven (omega_H) oscillation.  No safety factor.
// ---------------------------------------------------------------------------------------------------------------
// |R(z)|^2 of classical RK4, R(z) = 1 + z + z^2/2 + z^3/6 + z^4/24
inline double rk4_gain2(double zr, double zi) {
  // Horner in complex arithmetic written out
  double ar = 1.0 / 24.0, ai = 0.0;
  const double c[4] = {1.0 / 6.0, 0.5, 1.0, 1.0};
  for (int k = 0; k < 4; ++k) {
    const double tr = ar * zr - ai * zi + c[k], ti = ar * zi + ai * zr;
    ar = tr; ai = ti;
  }
  return ar * ar + ai * ai;
}
// first tau > 0 at which the ray {tau z} leaves the stability region |R| <= 1
inline double rk4_first_exit(double zr, double zi) {
  const double az = std::hypot(zr, zi);
  if (az == 0.0) return HUGE_VAL;
  const double tmax = 4.0 / az;
  const int n = 4096;
  double lo = 0.0, hi = -1.0;
  for (int k = 1; k <= n; ++k) {
    const double t = tmax * k / n;
    if (rk4_gain2(t * zr, t * zi) > 1.0 + 1e-13) { hi = t; break; }
    lo = t;
  }
  if (hi < 0.0) return tmax;
  for (int it = 0; it < 100; ++it) {
    const double mid = 0.5 * (lo + hi);
    (rk4_gain2(mid * zr, mid * zi) > 1.0 + 1e-13 ? hi : lo) = mid;
  }
  return lo;
}
inline void cfl_static(const Tables &T, const gk_species *sp, const gk_opts &o, int mask, double *dt_lin,
                       double *dt_field) {
  // (ii) z(t, t') = c_s [-i sigma(t) - nu_s d(t)] + c_v [+i sigma(t') - nu_v d(t')], 64 x 64 angles
  double cs = 0.0, cv = 0.0;
  for (int a = 0; a < T.nsp; ++a)
    for (int i = 0; i < T.ns; ++i) {
      cs = std::max(cs, std::fabs(T.vR[a] * T.F[i]) * std::max(std::fabs(T.v.front()), std::fabs(T.v.back())) / T.ds);
      cv = std::max(cv, std::fabs(T.vR[a] * T.BG[i]) * T.mu.back() / T.dv);
    }
  for (int l = 0; l < T.nmu; ++l)   // the mu grid is increasing for both grid types; keep the scan honest anyway
    for (int a = 0; a < T.nsp; ++a)
      for (int i = 0; i < T.ns; ++i) cv = std::max(cv, std::fabs(T.vR[a] * T.mu[l] * T.BG[i]) / T.dv);
  if (!(mask & GK_T_I)) cs = 0.0;
  if (!(mask & GK_T_IV)) cv = 0.0;
  const double nus = (mask & GK_T_DISS_S) ? o.disp_par : 0.0, nuv = (mask & GK_T_DISS_V) ? o.disp_vp : 0.0;
  double best = HUGE_VAL;
  const int NA = 64;
  double sg[NA], d4[NA];
  for (int k = 0; k < NA; ++k) {
    const double t = 2.0 * kPi * k / NA;
    sg[k] = (8.0 * std::sin(t) - std::sin(2.0 * t)) / 6.0;
    d4[k] = (2.0 - 2.0 * std::cos(t)) * (2.0 - 2.0 * std::cos(t)) / 12.0;
  }
  for (int k1 = 0; k1 < NA; ++k1)
    for (int k2 = 0; k2 < NA; ++k2)
      best = std::min(best, rk4_first_exit(-cs * nus * d4[k1] - cv * nuv * d4[k2], -cs * sg[k1] + cv * sg[k2]));
  *dt_lin = best;
  // (iii) omega_H^2 = sum_a (v_R F k_s)^2 Z^2 n <v_par^2> / (T A), <v_par^2> = 1/2, k_s = max sigma / ds;
  // max sigma in closed form: cos t = 1 - sqrt(6)/2
  *dt_field = HUGE_VAL;
  if (!o.adiabatic_electrons && (mask & GK_T_I) && (mask & GK_T_VII)) {
    const double ct = 1.0 - std::sqrt(6.0) / 2.0, st = std::sqrt(1.0 - ct * ct);
    const double ks = (8.0 * st - 2.0 * st * ct) / 6.0 / T.ds;
    double om2 = 0.0;
    for (int i = 0; i < T.ns; ++i) {
      double num = 0.0;
      for (int a = 0; a < T.nsp; ++a) {
        const double c = T.vR[a] * T.F[i] * ks;
        num += c * c * sp[a].Z * sp[a].Z * sp[a].dens * 0.5 / sp[a].temp;
      }
      for (int ip = 0; ip < T.nkx; ++ip)
        for (int m = 0; m < T.nky; ++m) {
          if (ip == T.K && m == 0) continue;
          om2 = std::max(om2, num / T.den[((size_t)i * T.nkx + ip) * T.nky + m]);
        }
    }
    if (om2 > 0.0) *dt_field = 2.0 * std::sqrt(2.0) / std::sqrt(om2);
  }
}

}  // namespace gkt
