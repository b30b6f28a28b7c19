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

// One point of the circular concentric (Lapillonne) model, PAPER.md:286-310 (reading R24), from gradient VECTORS in
// the orthonormal frame (e_r, e_theta, e_phi) of the poloidal plane (R0 = 1: R = 1 + eps cos th, Z = eps sin th):
// psi = eps, s = (th + eps sin th)/2pi, zeta = -phi/2pi + (q/pi) atan[sqrt((1-eps)/(1+eps)) tan(th/2)], q' = shat q/eps.
struct CircPoint { double B, dBds, gpz, gzz, Dpsi, Dzeta, Epz, R, btfrac; };
inline CircPoint circ_point(double q, double shat, double eps, double th) {
  const double ct = std::cos(th), st = std::sin(th), R = 1.0 + eps * ct;
  // zeta: chain rule through a = sqrt((1-eps)/(1+eps)), t = tan(th/2)
  const double a = std::sqrt((1.0 - eps) / (1.0 + eps)), t = std::tan(0.5 * th), den = 1.0 + a * a * t * t;
  const double A = std::atan(a * t);
  const double dA_dth = a * 0.5 * (1.0 + t * t) / den;
  const double dA_deps = t * (-1.0 / ((1.0 + eps) * (1.0 + eps) * a)) / den;
  const double z_eps = (shat * q / eps) / kPi * A + q / kPi * dA_deps, z_th = q / kPi * dA_dth;
  const double gpsi[3] = {1.0, 0.0, 0.0};
  const double gs[3] = {st / (2.0 * kPi), R / (2.0 * kPi * eps), 0.0};
  const double gz[3] = {z_eps, z_th / eps, -1.0 / (2.0 * kPi * R)};
  auto dot = [](const double *x, const double *y) { return x[0] * y[0] + x[1] * y[1] + x[2] * y[2]; };
  // B = delta / R (eq. 1) through its logarithmic derivatives; x = eps^2 / (q^2 (1 - eps^2))
  const double x = eps * eps / (q * q * (1.0 - eps * eps));
  const double dx = x * (2.0 / eps - 2.0 * shat / eps + 2.0 * eps / (1.0 - eps * eps));
  const double delta = std::sqrt(1.0 + x), B = delta / R;
  const double B_eps = B * (0.5 * dx / (1.0 + x) - ct / R), B_th = B * eps * st / R;
  // derivatives at fixed (psi, s): the Jacobian of (eps, th) -> (psi, s) is [[1, 0], [s_eps, s_th]] (eq. 3)
  const double s_eps = st / (2.0 * kPi), s_th = R / (2.0 * kPi);
  const double dBds = B_th / s_th, dBdpsi = B_eps - s_eps * dBds;
  const double gpp = dot(gpsi, gpsi), gpz = dot(gpsi, gz), gzz = dot(gz, gz), gps = dot(gpsi, gs), gzs = dot(gz, gs);
  // E tensor: cofactors of the first two metric rows x pi dpf/dpsi / B^2; D from eq. 4
  const double pref = kPi * (eps / (q * std::sqrt(1.0 - eps * eps))) / (B * B);
  const double Epz = pref * (gpp * gzz - gpz * gpz), Eps = pref * (gpp * gzs - gps * gpz), Ezs = pref * (gpz * gzs - gps * gzz);
  CircPoint c;
  c.B = B; c.dBds = dBds; c.gpz = gpz; c.gzz = gzz;
  c.Dpsi = -2.0 * Eps * dBds / B;
  c.Dzeta = -2.0 * (-Epz * dBdpsi + Ezs * dBds) / B;
  c.Epz = Epz; c.R = R; c.btfrac = 1.0 / delta;
  return c;
}

struct Tables {
  int nsp, nv, nmu, ns, nkx, nky, K;
  double dkx, ds, dv, wv;
  std::vector<double> v, fmv, mu, wmu, fmm, B, F, BG, sth, cz, Rmaj, kx, ky, hypx, hypy;
  std::vector<double> gpz, gzz, ef;   // k_perp^2 = kx^2 + 2 kx ky gpz + ky^2 gzz; ExB factor relative to ky/2
  double kthnorm;
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
  // geometry: s-alpha (R2) or circular (R24)
  T.B.resize(ns); T.F.resize(ns); T.BG.resize(ns); T.sth.resize(ns); T.cz.resize(ns); T.Rmaj.resize(ns);
  T.gpz.resize(ns); T.gzz.resize(ns); T.ef.resize(ns);
  T.fmm.resize((size_t)nmu * ns);
  double kx_per_turn = 2.0 * kPi * geo.shat;      // kx gained per poloidal turn and unit ky
  if (o.geometry == 0) {
    T.kthnorm = geo.q / (2.0 * kPi * geo.eps);
    for (int i = 0; i < ns; ++i) {
      const double th = 2.0 * kPi * (-0.5 + (i + 0.5) * T.ds);
      const double ct = std::cos(th), st = std::sin(th);
      T.Rmaj[i] = 1.0 + geo.eps * ct;
      T.B[i] = 1.0 / T.Rmaj[i];
      T.F[i] = 0.5 / (kPi * geo.q);
      T.BG[i] = geo.eps * st / (geo.q * T.Rmaj[i] * T.Rmaj[i]);
      T.sth[i] = st;
      T.cz[i] = ct + geo.shat * th * st;
      T.gpz[i] = geo.shat * th;
      T.gzz[i] = 1.0 + geo.shat * geo.shat * th * th;
      T.ef[i] = 1.0;
    }
  } else {
    T.kthnorm = std::sqrt(circ_point(geo.q, geo.shat, geo.eps, 0.0).gzz);
    kx_per_turn = (geo.shat * geo.q / geo.eps) / T.kthnorm;   // g_psizeta grows by q' per turn of the branch-tracked arctan
    const double b_ups = 1.0 / (2.0 * kPi * geo.q * std::sqrt(1.0 - geo.eps * geo.eps));
    for (int i = 0; i < ns; ++i) {
      const double sv = -0.5 + (i + 0.5) * T.ds;
      double lo = 2.0 * kPi * sv - 1.0, hi = 2.0 * kPi * sv + 1.0;   // th + eps sin th = 2 pi s by bisection (monotone)
      for (int it = 0; it < 200; ++it) {
        const double mid = 0.5 * (lo + hi);
        (mid + geo.eps * std::sin(mid) < 2.0 * kPi * sv ? lo : hi) = mid;
      }
      const CircPoint c = circ_point(geo.q, geo.shat, geo.eps, 0.5 * (lo + hi));
      T.B[i] = c.B;
      T.F[i] = b_ups / c.B;                                  // ffun
      T.BG[i] = T.F[i] * c.dBds;                             // B gfun = F d_s B
      T.sth[i] = -c.Dpsi;                                    // kappa = kx D^psi + (ky / kthnorm) D^zeta = -(kx sth + ky cz)
      T.cz[i] = -c.Dzeta / T.kthnorm;
      T.gpz[i] = c.gpz / T.kthnorm;
      T.gzz[i] = c.gzz / (T.kthnorm * T.kthnorm);
      T.ef[i] = 2.0 * c.Epz / T.kthnorm;                     // E^{psi zeta} k_zeta = ef ky / 2
      T.Rmaj[i] = c.R * c.btfrac;                            // R B_t / B of the momentum flux (R18)
    }
  }
  for (int i = 0; i < ns; ++i)
    for (int l = 0; l < nmu; ++l) T.fmm[(size_t)l * ns + i] = std::exp(-2.0 * T.mu[l] * T.B[i]);
  T.dkx = kx_per_turn * g.ky0 / g.ikxspace;
  T.kx.resize(nkx); T.ky.resize(nky); T.hypx.resize(nkx); T.hypy.resize(nky);
  for (int ip = 0; ip < nkx; ++ip) {
    T.kx[ip] = (ip - K) * T.dkx;
    T.hypx[ip] = (K > 0) ? o.disp_x * std::pow((double)(ip - K) / K, 4) : 0.0;
  }
  for (int m = 0; m < nky; ++m) {
    T.ky[m] = m * g.ky0;
    T.hypy[m] = (nky > 1) ? o.disp_y * std::pow((double)m / (nky - 1), 4) : 0.0;
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
          const double kperp = std::sqrt(T.kx[ip] * T.kx[ip] + 2.0 * T.kx[ip] * T.ky[m] * T.gpz[i] +
                                         T.ky[m] * T.ky[m] * T.gzz[i]);                                    // eq. 2
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
