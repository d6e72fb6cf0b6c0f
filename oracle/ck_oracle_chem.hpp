// ORACLE -- TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded CPU restatement of the
// chemistry right-hand side of arXiv 1608.05794 (Eqs. 12-19), written from the
// paper in its order and notation.  Shares no code with the CUDA path (paper_1608_05794_b200/csrc).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference may use it.
//
// The scalar type S is a template parameter: double (parity + timing), long double ("truth" for
// the RHS parity bound P1), std::complex<double> (complex-step Jacobian, O3) and MagDual
// (forward derivative + cancellation-aware magnitude, the scale of the Jacobian parity bound).
//
// Readings of garbled / silent passages:
//   G1  Eq. 19 is read as the standard NASA-7 forms of ref. [29]
//   G2  Eq. 13 is read as  Tdot = - sum_k H_k(molar) wdot_k / (rho * c_p(mass))
//   G9  c_i: three-body [M]_i; falloff Pr/(1+Pr) F with Lindemann F=1 or Troe F (CHEMKIN convention)
//   G10 Eq. 17 exponent is sum_k (nu''-nu'), K_p = exp(-sum nu g), g = H/RT - S/R
// Pins: tests/test_oracle_chem.py (thermo identities, invariants, equilibrium fixed point, falloff
// limits, brute-force Jacobian) -- see DESIGN.md "Oracle pins".
#pragma once
#include <cmath>
#include <complex>
#include <cstdint>
#include <vector>

namespace cko {

constexpr double R_U = 8.31446261815324e7;    // erg/(mol K)          (O1)
constexpr double R_CAL = 1.98720425864083;    // cal/(mol K), for E/R (O1)
constexpr double P_0 = 1.01325e6;             // dyn/cm^2, "one atmosphere" PAPER.md:130
constexpr double TINY = 1e-300;               // log guard (O2.3)

struct Mech {
  int K = 0, R = 0, E = 0;
  std::vector<double> W;                 // [K] g/mol
  std::vector<int> elem;                 // [K*E]
  std::vector<double> lo, hi, tmid;      // [K*7],[K*7],[K]
  std::vector<int> rptr, rspec, rnu;     // CSR nu'
  std::vector<int> pptr, pspec, pnu;     // CSR nu''
  std::vector<double> A, beta, Ea;       // [R]
  std::vector<uint8_t> rev, type;        // [R]; type 0 plain 1 three-body 2 Lindemann 3 Troe
  std::vector<double> A0, beta0, Ea0;    // [R]
  std::vector<double> troe;              // [R*4] a, T***, T*, T** (T**<0: absent)
  std::vector<int> eptr, espec;          // CSR non-unit efficiencies
  std::vector<double> eval;
  // 0: constant pressure (Eq. 12-13; the argument `p` of rhs is the pressure).  1: constant volume ("rho is
  // constant ... replacing c_p with c_v and h_k with u_k in Eq. (13)"); the argument `p` of rhs is then the mass density.
  int const_volume = 0;
};

// ---- scalar helpers -----------------------------------------------------------------------
inline double re(double x) { return x; }
inline double re(long double x) { return (double)x; }
inline double re(const std::complex<double>& x) { return x.real(); }
inline long double lre(long double x) { return x; }

// forward-mode value/derivative/magnitude triple: a >= |d| with sums taken in absolute value,
// so a is the size a derivative would have had without cancellation (parity bound scale for J).
struct MagDual {
  double v = 0, d = 0, a = 0;
  MagDual() {}
  MagDual(double v_) : v(v_) {}
  MagDual(double v_, double d_, double a_) : v(v_), d(d_), a(a_) {}
};
inline double re(const MagDual& x) { return x.v; }
inline MagDual operator+(const MagDual& x, const MagDual& y) { return {x.v + y.v, x.d + y.d, x.a + y.a}; }
inline MagDual operator-(const MagDual& x, const MagDual& y) { return {x.v - y.v, x.d - y.d, x.a + y.a}; }
inline MagDual operator-(const MagDual& x) { return {-x.v, -x.d, x.a}; }
inline MagDual operator*(const MagDual& x, const MagDual& y) {
  return {x.v * y.v, x.d * y.v + x.v * y.d, x.a * std::fabs(y.v) + std::fabs(x.v) * y.a};
}
inline MagDual operator/(const MagDual& x, const MagDual& y) {
  double q = x.v / y.v;
  return {q, (x.d - q * y.d) / y.v, (x.a + std::fabs(q) * y.a) / std::fabs(y.v)};
}
inline MagDual& operator+=(MagDual& x, const MagDual& y) { x = x + y; return x; }
inline MagDual& operator-=(MagDual& x, const MagDual& y) { x = x - y; return x; }
inline MagDual& operator*=(MagDual& x, const MagDual& y) { x = x * y; return x; }
inline MagDual exp(const MagDual& x) { double e = std::exp(x.v); return {e, e * x.d, e * x.a}; }
inline MagDual log(const MagDual& x) { return {std::log(x.v), x.d / x.v, x.a / std::fabs(x.v)}; }
inline MagDual log10(const MagDual& x) {
  const double il = 1.0 / std::log(10.0);
  return {std::log10(x.v), il * x.d / x.v, il * x.a / std::fabs(x.v)};
}

using std::exp;
using std::log;
using std::log10;

template <class S> inline S guard(const S& x) { return re(x) < TINY ? S(TINY) : x; }  // max(x,1e-300) on the real part
template <class S> inline S ipow(const S& x, int n) { S r(1.0); for (int i = 0; i < n; ++i) r = r * x; return r; }

// Optional by-products of one RHS evaluation (double, real parts)
struct RhsAux {
  std::vector<double> D;      // [N] cancellation-aware scale of f
  std::vector<double> qf, qr; // [R] forward / reverse rates of progress incl. c_i
  double rho = 0, cp = 0;
};

// f = RHS(y; p).  y[0]=T, y[1+k]=Y_k.  PAPER.md:99-137; step numbers are SURVEY.md 8(c) O2.
template <class S>
void rhs(const Mech& m, const S* y, double p, S* f, RhsAux* aux = nullptr) {
  const int K = m.K, R = m.R;
  const S T = y[0];
  const S lnT = log(T);
  std::vector<S> cpR(K), hRT(K), sR(K), g(K), C(K), w(K, S(0.0));
  // (1) thermo, Eq. 19 read per G1: range high iff T > T_mid,k
  for (int k = 0; k < K; ++k) {
    const double* a = (re(T) > m.tmid[k]) ? &m.hi[7 * k] : &m.lo[7 * k];
    S T2 = T * T, T3 = T2 * T, T4 = T3 * T;
    cpR[k] = S(a[0]) + S(a[1]) * T + S(a[2]) * T2 + S(a[3]) * T3 + S(a[4]) * T4;
    hRT[k] = S(a[0]) + S(a[1] / 2) * T + S(a[2] / 3) * T2 + S(a[3] / 4) * T3 + S(a[4] / 5) * T4 + S(a[5]) / T;
    sR[k] = S(a[0]) * lnT + S(a[1]) * T + S(a[2] / 2) * T2 + S(a[3] / 3) * T3 + S(a[4] / 4) * T4 + S(a[6]);
    g[k] = hRT[k] - sR[k];
  }
  // (2) ideal gas: rho = p / (R_u T sum Y_k/W_k); C_k = rho Y_k / W_k
  S Ssum(0.0);
  for (int k = 0; k < K; ++k) Ssum = Ssum + y[1 + k] / S(m.W[k]);
  // constant volume: rho is the given constant and the pressure follows from the same equation of state
  const S rho = m.const_volume ? S(p) : S(p) / (S(R_U) * T * Ssum);
  for (int k = 0; k < K; ++k) C[k] = rho * y[1 + k] / S(m.W[k]);
  if (aux) { aux->qf.assign(R, 0.0); aux->qr.assign(R, 0.0); }
  // (3) reactions in index order
  for (int i = 0; i < R; ++i) {
    S kf = exp(S(std::log(m.A[i])) + S(m.beta[i]) * lnT - S(m.Ea[i] / R_CAL) / T);  // Eq. 15
    S ci(1.0);
    if (m.type[i] != 0) {
      S M(0.0);
      for (int k = 0; k < K; ++k) M = M + C[k];
      for (int e = m.eptr[i]; e < m.eptr[i + 1]; ++e) M = M + S(m.eval[e] - 1.0) * C[m.espec[e]];
      if (m.type[i] == 1) {
        ci = M;
      } else {
        S k0 = exp(S(std::log(m.A0[i])) + S(m.beta0[i]) * lnT - S(m.Ea0[i] / R_CAL) / T);
        S Pr = k0 * M / kf;
        S F(1.0);
        if (m.type[i] == 3) {
          const double* t = &m.troe[4 * i];
          S Fc = S(1.0 - t[0]) * exp(-T / S(t[1])) + S(t[0]) * exp(-T / S(t[2]));
          if (t[3] >= 0) Fc = Fc + exp(-S(t[3]) / T);
          S lF = log10(guard(Fc)), lP = log10(guard(Pr));
          S c = S(-0.4) - S(0.67) * lF, n = S(0.75) - S(1.27) * lF;
          S f1 = (lP + c) / (n - S(0.14) * (lP + c));
          F = exp(S(std::log(10.0)) * lF / (S(1.0) + f1 * f1));
        }
        ci = Pr / (S(1.0) + Pr) * F;
      }
    }
    S kr(0.0);
    if (m.rev[i]) {  // Eqs. 16-18 read per G10
      int dnu = 0;
      S dg(0.0);
      for (int e = m.pptr[i]; e < m.pptr[i + 1]; ++e) { dnu += m.pnu[e]; dg = dg + S((double)m.pnu[e]) * g[m.pspec[e]]; }
      for (int e = m.rptr[i]; e < m.rptr[i + 1]; ++e) { dnu -= m.rnu[e]; dg = dg - S((double)m.rnu[e]) * g[m.rspec[e]]; }
      S base = S(P_0) / (S(R_U) * T);
      S Kc = exp(-dg);
      if (dnu > 0) Kc = Kc * ipow(base, dnu);
      if (dnu < 0) Kc = Kc / ipow(base, -dnu);
      kr = kf / Kc;
    }
    S pf(1.0), pr(1.0);  // Eq. 14, integer nu by repeated multiplication
    for (int e = m.rptr[i]; e < m.rptr[i + 1]; ++e) pf = pf * ipow(C[m.rspec[e]], m.rnu[e]);
    for (int e = m.pptr[i]; e < m.pptr[i + 1]; ++e) pr = pr * ipow(C[m.pspec[e]], m.pnu[e]);
    S qf = ci * kf * pf, qr = ci * kr * pr;
    S q = ci * (kf * pf - kr * pr);
    if (aux) { aux->qf[i] = std::fabs(re(qf)); aux->qr[i] = std::fabs(re(qr)); }
    for (int e = m.pptr[i]; e < m.pptr[i + 1]; ++e) w[m.pspec[e]] = w[m.pspec[e]] + S((double)m.pnu[e]) * q;
    for (int e = m.rptr[i]; e < m.rptr[i + 1]; ++e) w[m.rspec[e]] = w[m.rspec[e]] - S((double)m.rnu[e]) * q;
  }
  // (4) Eqs. 12-13 (13 read per G2)
  S cp(0.0), hw(0.0);
  for (int k = 0; k < K; ++k) {
    f[1 + k] = w[k] * S(m.W[k]) / rho;
    cp = cp + y[1 + k] * cpR[k] / S(m.W[k]);
    hw = hw + hRT[k] * w[k];
  }
  cp = S(R_U) * cp;
  if (m.const_volume) {
    // u_k = h_k - R_u T / W_k (molar: U_k/(R_u T) = H_k/(R_u T) - 1);  c_v = c_p - R_u sum_k Y_k / W_k
    S uw(0.0);
    for (int k = 0; k < K; ++k) uw = uw + (hRT[k] - S(1.0)) * w[k];
    const S cv = cp - S(R_U) * Ssum;
    f[0] = -(S(R_U) * T * uw) / (rho * cv);
  } else {
    f[0] = -(S(R_U) * T * hw) / (rho * cp);
  }
  if (aux) {
    aux->rho = re(rho); aux->cp = re(cp);
    std::vector<double> Dw(K, 0.0);
    for (int i = 0; i < R; ++i) {
      double s = aux->qf[i] + aux->qr[i];
      std::vector<int> net(K, 0);  // |net nu_ki|
      for (int e = m.pptr[i]; e < m.pptr[i + 1]; ++e) net[m.pspec[e]] += m.pnu[e];
      for (int e = m.rptr[i]; e < m.rptr[i + 1]; ++e) net[m.rspec[e]] -= m.rnu[e];
      for (int k = 0; k < K; ++k) Dw[k] += std::abs(net[k]) * s;
    }
    aux->D.assign(K + 1, 0.0);
    double dT = 0;
    for (int k = 0; k < K; ++k) {
      aux->D[1 + k] = m.W[k] / re(rho) * Dw[k];
      dT += std::fabs(R_U * re(T) * (re(hRT[k]) - (m.const_volume ? 1.0 : 0.0))) * Dw[k];
    }
    aux->D[0] = dT / (re(rho) * (m.const_volume ? re(cp) - R_U * re(Ssum) : re(cp)));
  }
}

// Thermo only (for the identity pins): cp/R, H/RT, S/R of species k at T
template <class S>
void thermo(const Mech& m, int k, S T, S* cpR, S* hRT, S* sR) {
  const double* a = (re(T) > m.tmid[k]) ? &m.hi[7 * k] : &m.lo[7 * k];
  S T2 = T * T, T3 = T2 * T, T4 = T3 * T;
  *cpR = S(a[0]) + S(a[1]) * T + S(a[2]) * T2 + S(a[3]) * T3 + S(a[4]) * T4;
  *hRT = S(a[0]) + S(a[1] / 2) * T + S(a[2] / 3) * T2 + S(a[3] / 4) * T3 + S(a[4] / 5) * T4 + S(a[5]) / T;
  *sR = S(a[0]) * log(T) + S(a[1]) * T + S(a[2] / 2) * T2 + S(a[3] / 3) * T3 + S(a[4] / 4) * T4 + S(a[6]);
}

}  // namespace cko
