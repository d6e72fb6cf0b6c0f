// ORACLE -- TEST INFRASTRUCTURE ONLY.  extern "C" entry points of the CPU oracle, called through
// ctypes by oracle/ck_oracle.py.  Batch layout is component-major y[c*ld + r] (same as include/ck.h).
// The outer loop over reactors may run under OpenMP `schedule(dynamic,1)` -- the structure of the
// paper's own multithreaded baseline; nthreads=1 gives the plain serial oracle.
#include "ck_oracle_solvers.hpp"
#include <cstring>
#ifdef _OPENMP
#include <omp.h>
#endif

using namespace cko;

namespace {
struct Toy : Problem {  // y1' = -y1 y2 ; y2' = y1 y2 - y2/2   (order test of the OneStep functions)
  int dim() const override { return 2; }
  void f(const double* y, double* o) const override { o[0] = -y[0] * y[1]; o[1] = y[0] * y[1] - 0.5 * y[1]; }
  void jac(const double* y, const double*, double, double* J) const override {
    J[0] = -y[1]; J[1] = -y[0]; J[2] = y[1]; J[3] = y[0] - 0.5;
  }
};
struct Lin : Problem {  // y' = lambda y  (linear test equation)
  double lam;
  explicit Lin(double l) : lam(l) {}
  int dim() const override { return 1; }
  void f(const double* y, double* o) const override { o[0] = lam * y[0]; }
  void jac(const double*, const double*, double, double* J) const override { J[0] = lam; }
};
}  // namespace

extern "C" {

void* cko_mech_create(int K, int R, int E, const double* W, const int* elem, const double* lo, const double* hi,
                      const double* tmid, const int* rptr, const int* rspec, const int* rnu, const int* pptr,
                      const int* pspec, const int* pnu, const double* A, const double* beta, const double* Ea,
                      const uint8_t* rev, const uint8_t* type, const double* A0, const double* beta0,
                      const double* Ea0, const double* troe, const int* eptr, const int* espec, const double* eval) {
  Mech* m = new Mech;
  m->K = K; m->R = R; m->E = E;
  m->W.assign(W, W + K);
  m->elem.assign(elem, elem + (size_t)K * E);
  m->lo.assign(lo, lo + 7 * K); m->hi.assign(hi, hi + 7 * K); m->tmid.assign(tmid, tmid + K);
  m->rptr.assign(rptr, rptr + R + 1); m->rspec.assign(rspec, rspec + rptr[R]); m->rnu.assign(rnu, rnu + rptr[R]);
  m->pptr.assign(pptr, pptr + R + 1); m->pspec.assign(pspec, pspec + pptr[R]); m->pnu.assign(pnu, pnu + pptr[R]);
  m->A.assign(A, A + R); m->beta.assign(beta, beta + R); m->Ea.assign(Ea, Ea + R);
  m->rev.assign(rev, rev + R); m->type.assign(type, type + R);
  m->A0.assign(A0, A0 + R); m->beta0.assign(beta0, beta0 + R); m->Ea0.assign(Ea0, Ea0 + R);
  m->troe.assign(troe, troe + 4 * R);
  m->eptr.assign(eptr, eptr + R + 1); m->espec.assign(espec, espec + eptr[R]); m->eval.assign(eval, eval + eptr[R]);
  return m;
}
void cko_mech_free(void* h) { delete (Mech*)h; }
void cko_set_const_volume(void* h, int on) { ((Mech*)h)->const_volume = on ? 1 : 0; }

// prec 0: double, 1: long double (result rounded to double).  D (optional) = cancellation-aware scale.
void cko_rhs(void* h, long long n, const double* y, long long ld, const double* p, double* f, long long ldf,
             double* D, int prec, int nthreads) {
  const Mech& m = *(Mech*)h;
  const int N = m.K + 1;
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads > 0 ? nthreads : 1)
  for (long long r = 0; r < n; ++r) {
    RhsAux aux;
    if (prec == 0) {
      std::vector<double> yy(N), ff(N);
      for (int c = 0; c < N; ++c) yy[c] = y[c * ld + r];
      rhs<double>(m, yy.data(), p[r], ff.data(), D ? &aux : nullptr);
      for (int c = 0; c < N; ++c) f[c * ldf + r] = ff[c];
    } else {
      std::vector<long double> yy(N), ff(N);
      for (int c = 0; c < N; ++c) yy[c] = y[c * ld + r];
      rhs<long double>(m, yy.data(), p[r], ff.data(), D ? &aux : nullptr);
      for (int c = 0; c < N; ++c) f[c * ldf + r] = (double)ff[c];
    }
    if (D) for (int c = 0; c < N; ++c) D[c * ldf + r] = aux.D[c];
  }
}

// rates of progress of one state: qf[R], qr[R] (absolute values, including c_i), rho, cp
void cko_rates(void* h, const double* y, double p, double* qf, double* qr, double* rho_cp) {
  const Mech& m = *(Mech*)h;
  std::vector<double> f(m.K + 1);
  RhsAux aux;
  rhs<double>(m, y, p, f.data(), &aux);
  std::memcpy(qf, aux.qf.data(), sizeof(double) * m.R);
  std::memcpy(qr, aux.qr.data(), sizeof(double) * m.R);
  rho_cp[0] = aux.rho; rho_cp[1] = aux.cp;
}

void cko_thermo(void* h, int k, double T, double* out3) {
  thermo<double>(*(Mech*)h, k, T, &out3[0], &out3[1], &out3[2]);
}

// one state (contiguous y[N]); J row-major [N*N].  mode 0 complex step, 1 CVODE-style FD, 2 MagDual (+Jmag)
void cko_jac(void* h, const double* y, double p, int mode, double hstep, double rtol, double atol, double* J,
             double* Jmag) {
  const Mech& m = *(Mech*)h;
  const int N = m.K + 1;
  if (mode == 0) jac_complex_step(m, y, p, J);
  else if (mode == 1) {
    std::vector<double> f0(N);
    rhs<double>(m, y, p, f0.data());
    jac_fd(m, y, p, f0.data(), hstep, rtol, atol, J);
  } else jac_magdual(m, y, p, J, Jmag);
}

int cko_lu_factor(double* A, int* piv, int N) { return lu_factor(A, piv, N) ? 0 : 1; }
void cko_lu_solve(const double* A, const int* piv, int N, double* b) { lu_solve(A, piv, N, b); }

// solver 0 ROS4, 1 RKF45.  counters[3] = total rhs, jac, lu (summed over reactors)
void cko_integrate(void* h, int solver, long long n, double* y, long long ld, const double* p, double dt, double rtol,
                   double atol, int jac_mode, double h0, int max_steps, int* n_accept, int* n_reject, int* status,
                   double* h_last, long long* counters, int nthreads) {
  const Mech& m = *(Mech*)h;
  const int N = m.K + 1;
  long long c_rhs = 0, c_jac = 0, c_lu = 0;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads > 0 ? nthreads : 1) reduction(+ : c_rhs, c_jac, c_lu)
  for (long long r = 0; r < n; ++r) {
    std::vector<double> yy(N);
    for (int c = 0; c < N; ++c) yy[c] = y[c * ld + r];
    Reactor pr(m, p[r], jac_mode, rtol, atol);
    Result res = integrate(pr, solver, yy.data(), dt, rtol, atol, h0, max_steps);
    for (int c = 0; c < N; ++c) y[c * ld + r] = yy[c];
    if (n_accept) n_accept[r] = res.n_accept;
    if (n_reject) n_reject[r] = res.n_reject;
    if (status) status[r] = res.status;
    if (h_last) h_last[r] = res.h_last;
    c_rhs += res.c.rhs; c_jac += res.c.jac; c_lu += res.c.lu;
  }
  if (counters) { counters[0] = c_rhs; counters[1] = c_jac; counters[2] = c_lu; }
}

double cko_estimate_h0(void* h, const double* y, double p, double dt, double rtol, double atol) {
  Counters c;
  Reactor pr(*(Mech*)h, p, 0, rtol, atol);
  return estimate_h0(pr, y, dt, rtol, atol, c);
}

// brute force: classical RK4, fixed step, on one reactor (pin 5).  Independent of OneStep/driver.
void cko_rk4(void* h, double* y, double p, double dt, long long nsteps) {
  const Mech& m = *(Mech*)h;
  const int N = m.K + 1;
  std::vector<double> k1(N), k2(N), k3(N), k4(N), yt(N);
  const double hs = dt / (double)nsteps;
  for (long long s = 0; s < nsteps; ++s) {
    rhs<double>(m, y, p, k1.data());
    for (int i = 0; i < N; ++i) yt[i] = y[i] + 0.5 * hs * k1[i];
    rhs<double>(m, yt.data(), p, k2.data());
    for (int i = 0; i < N; ++i) yt[i] = y[i] + 0.5 * hs * k2[i];
    rhs<double>(m, yt.data(), p, k3.data());
    for (int i = 0; i < N; ++i) yt[i] = y[i] + hs * k3[i];
    rhs<double>(m, yt.data(), p, k4.data());
    for (int i = 0; i < N; ++i) y[i] += hs / 6.0 * (k1[i] + 2 * k2[i] + 2 * k3[i] + k4[i]);
  }
}

// fixed-step runs of the OneStep functions on toy problems (order pins).
// problem 0: 2-D nonlinear toy on [0,1] from (1,1) wait see Toy; problem 1: y'=lam*y, y(0)=1 on [0,tend]
// out: y[dim] at the end, then |err estimate| of the LAST step per component.
void cko_onestep_fixed(int solver, int problem, double lam, double tend, int nsteps, const double* y0, double* out) {
  Toy toy; Lin lin(lam);
  const Problem& pr = (problem == 0) ? (const Problem&)toy : (const Problem&)lin;
  const int N = pr.dim();
  std::vector<double> y(y0, y0 + N), yn(N), e(N);
  Counters c;
  const double hs = tend / nsteps;
  for (int s = 0; s < nsteps; ++s) {
    if (solver == 0) ros4_step(pr, y.data(), hs, yn.data(), e.data(), c);
    else rkf45_step(pr, y.data(), hs, yn.data(), e.data(), c);
    y = yn;
  }
  for (int i = 0; i < N; ++i) { out[i] = y[i]; out[N + i] = e[i]; }
  out[2 * N] = (double)c.rhs;
}

// adaptive driver on the toy problem (controller sanity: error scales with tolerance)
void cko_toy_adaptive(int solver, double tend, double rtol, double atol, const double* y0, double* out, int* steps) {
  Toy toy;
  std::vector<double> y(y0, y0 + 2);
  Result r = integrate(toy, solver, y.data(), tend, rtol, atol, 0.0, 1000000);
  out[0] = y[0]; out[1] = y[1];
  steps[0] = r.n_accept; steps[1] = r.n_reject; steps[2] = r.status;
}

// the coefficient tables the oracle actually uses (for exact-rational order-condition pins)
void cko_tableaus(double* rkf_a /*6x6*/, double* rkf_b /*6*/, double* rkf_bh /*6*/, double* ros /*gam,a21,a31,a32,c21,c31,c32,c41,c42,c43,m1..4,e1..4*/) {
  std::memset(rkf_a, 0, 36 * sizeof(double));
  using namespace rkf;
  rkf_a[1 * 6 + 0] = a21;
  rkf_a[2 * 6 + 0] = a31; rkf_a[2 * 6 + 1] = a32;
  rkf_a[3 * 6 + 0] = a41; rkf_a[3 * 6 + 1] = a42; rkf_a[3 * 6 + 2] = a43;
  rkf_a[4 * 6 + 0] = a51; rkf_a[4 * 6 + 1] = a52; rkf_a[4 * 6 + 2] = a53; rkf_a[4 * 6 + 3] = a54;
  rkf_a[5 * 6 + 0] = a61; rkf_a[5 * 6 + 1] = a62; rkf_a[5 * 6 + 2] = a63; rkf_a[5 * 6 + 3] = a64; rkf_a[5 * 6 + 4] = a65;
  double b[6] = {b1, 0, b3, b4, b5, 0}, bh[6] = {h1, 0, h3, h4, h5, h6};
  std::memcpy(rkf_b, b, sizeof b); std::memcpy(rkf_bh, bh, sizeof bh);
  double r[18] = {ros4::gam, ros4::a21, ros4::a31, ros4::a32, ros4::c21, ros4::c31, ros4::c32, ros4::c41, ros4::c42,
                  ros4::c43, ros4::m1, ros4::m2, ros4::m3, ros4::m4, ros4::e1, ros4::e2, ros4::e3, ros4::e4};
  std::memcpy(ros, r, sizeof r);
}

int cko_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
