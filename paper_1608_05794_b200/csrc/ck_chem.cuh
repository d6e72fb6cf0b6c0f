// Device-side chemistry shared by the kernels: temperature state, NASA-7 thermo, and the rate of
// progress of one reaction (Eq. 14-19), written once and instantiated for the two
// data mappings used by the library:
//   CS = BLOCK : thread-per-reactor, concentrations of reactor `tid` at C[s*BLOCK] (conflict-free columns)
//   CS = 1     : group-per-reactor (warp / CTA cooperative), concentrations of the reactor at C[s]
#pragma once
#include "ck_internal.h"

namespace ck {

struct TState {
  double T, lnT, invT;
  int tint;  // temperature interval of the k_r table
};

__device__ __forceinline__ TState make_tstate(const MechDev& m, double T) {
  TState t;
  t.T = T;
  t.lnT = log(T);
  t.invT = 1.0 / T;
  int ti = 0;
#pragma unroll
  for (int e = 0; e < MAX_TINT - 1; ++e) ti += (e < m.nT - 1 && T > m.tedge[e]) ? 1 : 0;
  t.tint = ti;
  return t;
}

// cp_k/R and H_k/(R T) of species k (Eq. 19 in the NASA-7 reading G1); range high iff T > t_mid[k]
__device__ __forceinline__ void thermo_cp_h(const MechDev& m, int k, const TState& t, double& cpR, double& hRT) {
  const double* a = (t.T > __ldg(m.tmid + k)) ? m.nhi : m.nlo;
  const int K = m.K;
  const double a1 = __ldg(a + k), a2 = __ldg(a + K + k), a3 = __ldg(a + 2 * K + k), a4 = __ldg(a + 3 * K + k),
               a5 = __ldg(a + 4 * K + k), a6 = __ldg(a + 5 * K + k);
  const double T = t.T;
  cpR = fma(fma(fma(fma(a5, T, a4), T, a3), T, a2), T, a1);
  hRT = fma(fma(fma(fma(a5 * 0.2, T, a4 * 0.25), T, a3 * (1.0 / 3.0)), T, a2 * 0.5), T, a1) + a6 * t.invT;
}
// d(cp_k/R)/dT (for the analytic Jacobian)
__device__ __forceinline__ double thermo_dcp(const MechDev& m, int k, const TState& t) {
  const double* a = (t.T > __ldg(m.tmid + k)) ? m.nhi : m.nlo;
  const int K = m.K;
  const double a2 = __ldg(a + K + k), a3 = __ldg(a + 2 * K + k), a4 = __ldg(a + 3 * K + k), a5 = __ldg(a + 4 * K + k);
  const double T = t.T;
  return fma(fma(fma(4.0 * a5, T, 3.0 * a4), T, 2.0 * a3), T, a2);
}

__device__ __forceinline__ double ipow_small(double x, int n) {
  double r = x;
  for (int i = 1; i < n; ++i) r *= x;
  return r;
}

// Everything the Jacobian needs about one reaction besides q itself.
struct RateAux {
  double kf, kr, ci, pf, pr;   // q = ci (kf pf - kr pr)
  double dlnkf_dT, dlnkr_dT;   // temperature derivatives of the rate constants
  double dci_dM;               // d c_i / d [M]_i at constant T   (0 for plain rows)
  double dci_dT;               // d c_i / d T at constant concentrations (falloff rows)
};

// Rate of progress q_i of regrouped reaction r.  WANT_AUX also fills the derivative pieces.
template <int CS, bool WANT_AUX>
__device__ __forceinline__ double reaction_q(const MechDev& m, int r, const TState& t, const double* __restrict__ C,
                                             double Ctot, RateAux* aux) {
  const int R = m.R;
  const double beta = __ldg(m.beta + r), Ta = __ldg(m.Ta + r);
  const double kf = exp(fma(beta, t.lnT, __ldg(m.lnA + r)) - Ta * t.invT);  // Eq. 15
  const double* c = m.krc + (size_t)t.tint * 7 * R + r;
  const double c1 = __ldg(c + R), c2 = __ldg(c + 2 * (size_t)R), c3 = __ldg(c + 3 * (size_t)R),
               c4 = __ldg(c + 4 * (size_t)R), c5 = __ldg(c + 5 * (size_t)R), c6 = __ldg(c + 6 * (size_t)R);
  const double T = t.T;
  const double poly = fma(fma(fma(c6, T, c5), T, c4), T, c3) * T;
  const double kr = exp(fma(c1, t.lnT, __ldg(c)) + fma(c2, t.invT, poly));  // Eq. 16-18 folded (ck_mech.cu)
  double ci = 1.0, dci_dM = 0.0, dci_dT = 0.0;
  if (r >= m.r_tb) {  // third-body / falloff factor c_i (reading G9)
    const int j = r - m.r_tb;
    double M = Ctot;
    for (int e = __ldg(m.eptr + j), e1 = __ldg(m.eptr + j + 1); e < e1; ++e)
      M = fma(__ldg(m.eval1 + e), C[(size_t)__ldg(m.espec + e) * CS], M);
    if (r < m.r_lind) {
      ci = M;
      if (WANT_AUX) dci_dM = 1.0;
    } else {
      const int jl = r - m.r_lind;
      const double beta0 = __ldg(m.beta0 + jl), Ta0 = __ldg(m.Ta0 + jl);
      const double k0 = exp(fma(beta0, t.lnT, __ldg(m.lnA0 + jl)) - Ta0 * t.invT);
      const double k0_kf = k0 / kf;
      const double Pr = k0_kf * M;
      const double inv1p = 1.0 / (1.0 + Pr);
      const double L = Pr * inv1p;  // Lindemann
      double F = 1.0, dlnF_dlP = 0.0, dlnF_dT = 0.0;
      if (r >= m.r_troe) {
        const int jt = r - m.r_troe, nt = R - m.r_troe;
        const double a = __ldg(m.troe + jt), i3 = __ldg(m.troe + nt + jt), i1 = __ldg(m.troe + 2 * nt + jt),
                     T2 = __ldg(m.troe + 3 * nt + jt);
        const double e3 = exp(-T * i3), e1 = exp(-T * i1);
        double Fc = fma(1.0 - a, e3, a * e1);
        double e2 = 0.0;
        if (T2 >= 0.0) { e2 = exp(-T2 * t.invT); Fc += e2; }
        const double il10 = 0.43429448190325182765;  // 1/ln 10
        const double ln10 = 2.30258509299404568402;
        const double Fcg = fmax(Fc, 1e-300), Prg = fmax(Pr, 1e-300);
        const double lF = log(Fcg) * il10, lP = log(Prg) * il10;
        const double cc = fma(-0.67, lF, -0.4), nn = fma(-1.27, lF, 0.75);
        const double x = lP + cc;
        const double den = fma(-0.14, x, nn);
        const double f1 = x / den;
        const double g = 1.0 / fma(f1, f1, 1.0);
        F = exp(ln10 * lF * g);
        if (WANT_AUX) {
          // ln F = ln10 * lF / (1 + f1^2);  f1 = x/den, x = lP + cc(lF), den = nn(lF) - 0.14 x
          const double df1_dx = nn / (den * den);              // (den + 0.14 x)/den^2 = nn/den^2
          const double dlnF_df1 = -ln10 * lF * g * g * 2.0 * f1;
          dlnF_dlP = (Pr > 1e-300) ? dlnF_df1 * df1_dx : 0.0;  // d lnF / d log10 Pr
          // T dependence through lF (F_cent):  d lF/dT = il10 * Fc'/Fc
          double dFc = -(1.0 - a) * i3 * e3 - a * i1 * e1 + e2 * T2 * t.invT * t.invT;
          const double dlF_dT = (Fc > 1e-300) ? il10 * dFc / Fc : 0.0;
          // f1 depends on lF via cc = -0.4 - 0.67 lF and nn = 0.75 - 1.27 lF: d f1/d lF = (-0.67 den - x(-1.27 + 0.14*0.67))/den^2
          const double df1_dlF = (-0.67 * den - x * (-1.27 + 0.14 * 0.67)) / (den * den);
          const double dlnF_dlF = ln10 * g + dlnF_df1 * df1_dlF;
          dlnF_dT = dlnF_dlF * dlF_dT;
        }
      }
      ci = L * F;
      if (WANT_AUX) {
        // Pr = (k0/kf) M:  dPr/dM = k0/kf ;  dlnPr/dT = (beta0 - beta)/T + (Ta0 - Ta)/T^2
        const double dlnPr_dT = ((beta0 - beta) + (Ta0 - Ta) * t.invT) * t.invT;
        const double il10 = 0.43429448190325182765;
        // d ci / d Pr = F/(1+Pr)^2 + L F dlnF/dPr,  dlnF/dPr = dlnF_dlP * il10 / Pr
        const double dci_dPr = F * inv1p * inv1p + ((Pr > 0.0) ? ci * dlnF_dlP * il10 / Pr : 0.0);
        dci_dM = dci_dPr * k0_kf;
        dci_dT = dci_dPr * Pr * dlnPr_dT + ci * dlnF_dT;
      }
    }
  }
  double pf = 1.0, pr = 1.0;  // Eq. 14, integer nu by repeated multiplication
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    const int e = __ldg(m.part + (size_t)s * R + r);
    if (e) pf *= ipow_small(C[(size_t)(e >> 8) * CS], e & 255);
  }
#pragma unroll
  for (int s = 3; s < 6; ++s) {
    const int e = __ldg(m.part + (size_t)s * R + r);
    if (e) pr *= ipow_small(C[(size_t)(e >> 8) * CS], e & 255);
  }
  if (WANT_AUX) {
    aux->kf = kf; aux->kr = kr; aux->ci = ci; aux->pf = pf; aux->pr = pr;
    aux->dlnkf_dT = (beta + Ta * t.invT) * t.invT;
    aux->dlnkr_dT = (kr > 0.0) ? fma(fma(fma(4.0 * c6, T, 3.0 * c5), T, 2.0 * c4), T, c3) + (c1 - c2 * t.invT) * t.invT : 0.0;
    aux->dci_dM = dci_dM; aux->dci_dT = dci_dT;
  }
  return ci * (kf * pf - kr * pr);
}

}  // namespace ck
