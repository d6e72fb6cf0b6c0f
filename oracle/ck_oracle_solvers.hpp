// ORACLE -- TEST INFRASTRUCTURE ONLY (see ck_oracle_chem.hpp).  Jacobians, dense LU, the two
// OneStep functions and the adaptive driver of arXiv 1608.05794, step by step in the paper's
// order: Algorithm 1, ROS4 Eqs. 6-7 with Table C.3
// (PAPER.md:455-481), RKF45 Eqs. 2-3 with Table B.2.
//
// Readings:
//   G3  Table B.2 repaired: a42=-7200/2197, a54=-845/4104, a64=1859/4104 (pinned by exact-rational
//       order conditions and row sums, tests/test_oracle_tableaus.py)
//   G4  gamma = 0.57282 (table), not 0.572816 (text)      G5  printed "b_i" are the m_i of Eq. 7
//   G6  a43 = 0, alpha_i / gamma_i unused (autonomous)     G7  weighted RMS error, accept iff err < 1
//   G8  EstimateH0 / AdjustStepSize: NOT specified by the paper -> "parity unpinned"; the rule below
//       (textbook starting step of ref. [47]; safety 0.9, factor in [0.2,5], no growth after a reject)
//       is a shared free choice.   G11 loop is while t < t_f.   G12 CVODE-style FD increment.
#pragma once
#include "ck_oracle_chem.hpp"
#include <algorithm>

namespace cko {

// ---- Jacobians (O3) ------------------------------------------------------------------------
// complex step: J[:,j] = Im f(y + i*1e-30 e_j)/1e-30.  Row-major J[i*N+j] = d f_i / d y_j.
inline void jac_complex_step(const Mech& m, const double* y, double p, double* J) {
  const int N = m.K + 1;
  std::vector<std::complex<double>> yc(N), fc(N);
  for (int j = 0; j < N; ++j) {
    for (int i = 0; i < N; ++i) yc[i] = y[i];
    yc[j] = std::complex<double>(y[j], 1e-30);
    rhs(m, yc.data(), p, fc.data());
    for (int i = 0; i < N; ++i) J[i * N + j] = fc[i].imag() / 1e-30;
  }
}

// forward-mode derivative with cancellation-aware magnitude (scale of the Jacobian parity bound)
inline void jac_magdual(const Mech& m, const double* y, double p, double* J, double* Jmag) {
  const int N = m.K + 1;
  std::vector<MagDual> yd(N), fd(N);
  for (int j = 0; j < N; ++j) {
    for (int i = 0; i < N; ++i) yd[i] = MagDual(y[i]);
    yd[j] = MagDual(y[j], 1.0, 1.0);
    rhs(m, yd.data(), p, fd.data());
    for (int i = 0; i < N; ++i) { J[i * N + j] = fd[i].d; Jmag[i * N + j] = fd[i].a; }
  }
}

inline double wrms(const double* v, const double* y, int N, double rtol, double atol) {
  double s = 0;
  for (int i = 0; i < N; ++i) { double w = v[i] / (rtol * std::fabs(y[i]) + atol); s += w * w; }
  return std::sqrt(s / N);
}

// first-order forward differences "following the approach used in CVODE", G12
inline void jac_fd(const Mech& m, const double* y, double p, const double* f0, double h, double rtol, double atol,
                   double* J) {
  const int N = m.K + 1;
  const double eps = std::ldexp(1.0, -52);
  double fn = wrms(f0, y, N, rtol, atol);
  double s0 = (fn != 0.0) ? 1000.0 * N * eps * std::fabs(h) * fn : 1.0;
  std::vector<double> yp(y, y + N), fp(N);
  for (int j = 0; j < N; ++j) {
    double sig = std::max(std::sqrt(eps) * std::fabs(y[j]), s0 * (rtol * std::fabs(y[j]) + atol));
    yp[j] = y[j] + sig;
    rhs(m, yp.data(), p, fp.data());
    for (int i = 0; i < N; ++i) J[i * N + j] = (fp[i] - f0[i]) / sig;
    yp[j] = y[j];
  }
}

// ---- dense LU with partial pivoting (first maximal |a| on ties), O4 ---------------------------
inline bool lu_factor(double* A, int* piv, int N) {
  for (int k = 0; k < N; ++k) {
    int p = k;
    double best = std::fabs(A[k * N + k]);
    for (int i = k + 1; i < N; ++i)
      if (std::fabs(A[i * N + k]) > best) { best = std::fabs(A[i * N + k]); p = i; }
    piv[k] = p;
    if (!(best > 0.0)) return false;
    if (p != k)
      for (int j = 0; j < N; ++j) std::swap(A[k * N + j], A[p * N + j]);
    for (int i = k + 1; i < N; ++i) {
      double l = A[i * N + k] / A[k * N + k];
      A[i * N + k] = l;
      for (int j = k + 1; j < N; ++j) A[i * N + j] -= l * A[k * N + j];
    }
  }
  return true;
}
inline void lu_solve(const double* A, const int* piv, int N, double* b) {
  // P A = L U with whole rows swapped in lu_factor, so L belongs to the FINAL row order: apply all of P first
  for (int k = 0; k < N; ++k) std::swap(b[k], b[piv[k]]);
  for (int k = 0; k < N; ++k)
    for (int i = k + 1; i < N; ++i) b[i] -= A[i * N + k] * b[k];
  for (int k = N - 1; k >= 0; --k) {
    b[k] /= A[k * N + k];
    for (int i = 0; i < k; ++i) b[i] -= A[i * N + k] * b[k];
  }
}

// ---- coefficients ------------------------------------------------------------------------------
namespace ros4 {  // Table C.3, read per G4-G6
constexpr double gam = 0.57282;
constexpr double a21 = 2.0, a31 = 1.867943637803922, a32 = 0.2344449711399156;
constexpr double c21 = -7.137615036412310, c31 = 2.580708087951457, c32 = 0.6515950076447975;
constexpr double c41 = -2.137148994382534, c42 = -0.3214669691237626, c43 = -0.6949742501781779;
constexpr double m1 = 2.255570073418735, m2 = 0.2870493262186792, m3 = 0.4353179431840180, m4 = 1.093502252409163;
constexpr double e1 = -0.2815431932141155, e2 = -0.07276199124938920, e3 = -0.1082196201495311, e4 = -1.093502252409163;
}  // namespace ros4
namespace rkf {  // Table B.2, repaired per G3
constexpr double a21 = 1.0 / 4;
constexpr double a31 = 3.0 / 32, a32 = 9.0 / 32;
constexpr double a41 = 1932.0 / 2197, a42 = -7200.0 / 2197, a43 = 7296.0 / 2197;
constexpr double a51 = 439.0 / 216, a52 = -8.0, a53 = 3680.0 / 513, a54 = -845.0 / 4104;
constexpr double a61 = -8.0 / 27, a62 = 2.0, a63 = -3544.0 / 2565, a64 = 1859.0 / 4104, a65 = -11.0 / 40;
constexpr double b1 = 25.0 / 216, b3 = 1408.0 / 2565, b4 = 2197.0 / 4104, b5 = -1.0 / 5;
constexpr double h1 = 16.0 / 135, h3 = 6656.0 / 12825, h4 = 28561.0 / 56430, h5 = -9.0 / 50, h6 = 2.0 / 55;
}  // namespace rkf

struct Counters { long long rhs = 0, jac = 0, lu = 0; };

// generic f so that the OneStep functions can be order-tested on toy ODEs (tests/test_oracle_tableaus.py)
struct Problem {
  virtual int dim() const = 0;
  virtual void f(const double* y, double* out) const = 0;
  virtual void jac(const double* y, const double* f0, double h, double* J) const = 0;
  virtual int jac_rhs_evals() const { return 0; }  // RHS evaluations one jac() call costs (N for FD)
  virtual ~Problem() {}
};

struct Reactor : Problem {
  const Mech& m; double p; int jac_mode; double rtol, atol;
  Reactor(const Mech& m_, double p_, int jm, double rt, double at) : m(m_), p(p_), jac_mode(jm), rtol(rt), atol(at) {}
  int dim() const override { return m.K + 1; }
  void f(const double* y, double* out) const override { rhs(m, y, p, out); }
  void jac(const double* y, const double* f0, double h, double* J) const override {
    if (jac_mode == 0) jac_complex_step(m, y, p, J); else jac_fd(m, y, p, f0, h, rtol, atol, J);
  }
  int jac_rhs_evals() const override { return jac_mode == 0 ? 0 : m.K + 1; }
};

// ---- ROS4 attempt (O4): Eq. 6-7 ------------------------------------------------------------------
// returns false on zero pivot.  ynew = y + sum m_i u_i ; err = sum E_i u_i
inline bool ros4_step(const Problem& pr, const double* y, double h, double* ynew, double* err, Counters& c) {
  using namespace ros4;
  const int N = pr.dim();
  std::vector<double> f0(N), J(N * N), A(N * N), u1(N), u2(N), u3(N), u4(N), yt(N), ft(N);
  std::vector<int> piv(N);
  pr.f(y, f0.data()); c.rhs++;
  pr.jac(y, f0.data(), h, J.data()); c.jac++; c.rhs += pr.jac_rhs_evals();
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j) A[i * N + j] = (i == j ? 1.0 / (h * gam) : 0.0) - J[i * N + j];
  c.lu++;
  if (!lu_factor(A.data(), piv.data(), N)) return false;
  for (int i = 0; i < N; ++i) u1[i] = f0[i];
  lu_solve(A.data(), piv.data(), N, u1.data());
  for (int i = 0; i < N; ++i) yt[i] = y[i] + a21 * u1[i];
  pr.f(yt.data(), ft.data()); c.rhs++;
  for (int i = 0; i < N; ++i) u2[i] = ft[i] + (c21 / h) * u1[i];
  lu_solve(A.data(), piv.data(), N, u2.data());
  for (int i = 0; i < N; ++i) yt[i] = y[i] + a31 * u1[i] + a32 * u2[i];
  pr.f(yt.data(), ft.data()); c.rhs++;
  for (int i = 0; i < N; ++i) u3[i] = ft[i] + (c31 * u1[i] + c32 * u2[i]) / h;
  lu_solve(A.data(), piv.data(), N, u3.data());
  for (int i = 0; i < N; ++i) u4[i] = ft[i] + (c41 * u1[i] + c42 * u2[i] + c43 * u3[i]) / h;  // a4j=a3j, a43=0
  lu_solve(A.data(), piv.data(), N, u4.data());
  for (int i = 0; i < N; ++i) {
    ynew[i] = y[i] + m1 * u1[i] + m2 * u2[i] + m3 * u3[i] + m4 * u4[i];
    err[i] = e1 * u1[i] + e2 * u2[i] + e3 * u3[i] + e4 * u4[i];
  }
  return true;
}

// ---- RKF45 attempt (O5): Eq. 2-3; 4th-order solution advanced, err = 5th - 4th -------------------
inline bool rkf45_step(const Problem& pr, const double* y, double h, double* ynew, double* err, Counters& c) {
  using namespace rkf;
  const int N = pr.dim();
  std::vector<double> k1(N), k2(N), k3(N), k4(N), k5(N), k6(N), yt(N);
  auto ev = [&](const double* yy, std::vector<double>& k) { pr.f(yy, k.data()); c.rhs++; for (int i = 0; i < N; ++i) k[i] *= h; };
  ev(y, k1);
  for (int i = 0; i < N; ++i) yt[i] = y[i] + a21 * k1[i];
  ev(yt.data(), k2);
  for (int i = 0; i < N; ++i) yt[i] = y[i] + a31 * k1[i] + a32 * k2[i];
  ev(yt.data(), k3);
  for (int i = 0; i < N; ++i) yt[i] = y[i] + a41 * k1[i] + a42 * k2[i] + a43 * k3[i];
  ev(yt.data(), k4);
  for (int i = 0; i < N; ++i) yt[i] = y[i] + a51 * k1[i] + a52 * k2[i] + a53 * k3[i] + a54 * k4[i];
  ev(yt.data(), k5);
  for (int i = 0; i < N; ++i) yt[i] = y[i] + a61 * k1[i] + a62 * k2[i] + a63 * k3[i] + a64 * k4[i] + a65 * k5[i];
  ev(yt.data(), k6);
  for (int i = 0; i < N; ++i) {
    ynew[i] = y[i] + b1 * k1[i] + b3 * k3[i] + b4 * k4[i] + b5 * k5[i];
    err[i] = (h1 - b1) * k1[i] + (h3 - b3) * k3[i] + (h4 - b4) * k4[i] + (h5 - b5) * k5[i] + h6 * k6[i];
  }
  return true;
}

// ---- EstimateH0 (G8; starting-step rule of the paper's ref. [47]) --------------------------------
inline double estimate_h0(const Problem& pr, const double* y, double dt, double rtol, double atol, Counters& c) {
  const int N = pr.dim();
  std::vector<double> f0(N), y1(N), f1(N), df(N);
  pr.f(y, f0.data()); c.rhs++;
  double d0 = wrms(y, y, N, rtol, atol), d1 = wrms(f0.data(), y, N, rtol, atol);
  double ha = (d0 < 1e-5 || d1 < 1e-5) ? 1e-6 * dt : 0.01 * d0 / d1;
  for (int i = 0; i < N; ++i) y1[i] = y[i] + ha * f0[i];
  pr.f(y1.data(), f1.data()); c.rhs++;
  for (int i = 0; i < N; ++i) df[i] = f1[i] - f0[i];
  double d2 = wrms(df.data(), y, N, rtol, atol) / ha;
  double dm = std::max(d1, d2);
  double hb = (dm <= 1e-15) ? std::max(1e-6 * dt, 1e-3 * ha) : std::pow(0.01 / dm, 1.0 / 5.0);
  return std::min(std::min(100.0 * ha, hb), dt);
}

struct Result { int n_accept = 0, n_reject = 0, status = 0; double h_last = 0; Counters c; };

// ---- adaptive driver, Algorithm 1 (O6) ------------------------------------------------------------
// solver: 0 ROS4 (q=4), 1 RKF45 (q=5).  status: 0 ok, 1 max_steps, 2 h underflow, 3 non-finite, 4 zero pivot
inline Result integrate(const Problem& pr, int solver, double* y, double dt, double rtol, double atol, double h0,
                        int max_steps) {
  const int N = pr.dim();
  Result r;
  std::vector<double> yn(N), e(N);
  double t = 0;
  double h = (h0 > 0) ? h0 : estimate_h0(pr, y, dt, rtol, atol, r.c);
  const double q = (solver == 0) ? 4.0 : 5.0;
  double fac_max = 5.0;
  while (t < dt) {
    if (r.n_accept + r.n_reject >= max_steps) { r.status = 1; break; }
    if (!std::isfinite(h)) { r.status = 3; break; }
    if (h < 1e-12 * dt) { r.status = 2; break; }
    bool last = false;
    if (h >= dt - t) { h = dt - t; last = true; }
    bool ok = (solver == 0) ? ros4_step(pr, y, h, yn.data(), e.data(), r.c) : rkf45_step(pr, y, h, yn.data(), e.data(), r.c);
    if (!ok) { r.status = 4; break; }
    double s = 0;
    for (int i = 0; i < N; ++i) {
      double sc = atol + rtol * std::max(std::fabs(y[i]), std::fabs(yn[i]));
      double w = e[i] / sc;
      s += w * w;
    }
    double err = std::sqrt(s / N);
    r.h_last = h;
    if (std::isfinite(err) && err < 1.0) {
      for (int i = 0; i < N; ++i) y[i] = yn[i];
      t = last ? dt : t + h;
      r.n_accept++;
      h *= std::min(fac_max, std::max(0.2, 0.9 * std::pow(std::max(err, 1e-10), -1.0 / q)));
      fac_max = 5.0;
    } else {
      r.n_reject++;
      if (std::isfinite(err)) h *= std::min(1.0, std::max(0.2, 0.9 * std::pow(std::max(err, 1e-10), -1.0 / q)));
      else h *= 0.2;
      fac_max = 1.0;
    }
  }
  return r;
}

}  // namespace cko
