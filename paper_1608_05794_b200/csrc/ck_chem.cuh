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

// Coefficients of the exponential's polynomial (and its reduction constants) in the constant bank: a DFMA takes a
// constant-bank operand directly, whereas a 64-bit literal costs two UMOV per use inside the hot loops.
static __constant__ double ck_expc[16] = {
    0x1.af632a0f7e2cep-26, 0x1.28b4101c77212p-22, 0x1.71ddf56d8deb5p-19, 0x1.a01991a10d9aep-16,
    0x1.a01a01b1461c5p-13, 0x1.6c16c1880029fp-10, 0x1.111111110f21ep-7,  0x1.555555554f0bap-5,
    0x1.555555555555ap-3,  0x1.0000000000011p-1,  1.0,                    1.0,
    1.4426950408889634074, 6755399441055744.0,   -6.93147180369123816490e-01, -1.90821492927058770002e-10};

// exp(x) for the rate constants: x = n ln2 + r, |r| <= ln2/2, degree-11 polynomial (Chebyshev-node interpolation
// of e^r on [-ln2/2, ln2/2], max relative error 1.6e-17 before rounding), 2^n applied to the exponent field.
// 15 FP64-pipe instructions; no branches: the argument is CLAMPED to [-708, 708], so an
// irreversible reaction (c0 = -inf) gets k_r = 3e-308 instead of 0 (absolute effect < 1e-300 on any rate) and
// an overflowing argument saturates at 8e307.  With 16 warps per SM the Horner chain is hidden by other warps
// (an Estrin form, 4 more instructions, was faster only at 8 warps per SM).
__device__ __forceinline__ double ck_exp(double x) {
  const double MAGIC = 6755399441055744.0;  // 1.5 * 2^52
  {  // clamp |x| to 708 with integer operations on the high word (FP64 min/max is a DSETP + two selects each, on
     // the contended FP64 pipe); NaN and infinities land on +-708 as well
    const int hx = __double2hiint(x);
    const bool big = (hx & 0x7fffffff) >= 0x40862000;
    x = big ? __hiloint2double((hx & 0x80000000) | 0x40862000, 0) : x;
  }
  const double t = fma(x, 1.4426950408889634074, MAGIC);
  const int n = __double2loint(t);
  const double nf = t - MAGIC;
  double r = fma(nf, -6.93147180369123816490e-01, x);
  r = fma(nf, -1.90821492927058770002e-10, r);
  double p = 0x1.af632a0f7e2cep-26;
  p = fma(p, r, 0x1.28b4101c77212p-22);
  p = fma(p, r, 0x1.71ddf56d8deb5p-19);
  p = fma(p, r, 0x1.a01991a10d9aep-16);
  p = fma(p, r, 0x1.a01a01b1461c5p-13);
  p = fma(p, r, 0x1.6c16c1880029fp-10);
  p = fma(p, r, 0x1.111111110f21ep-7);
  p = fma(p, r, 0x1.555555554f0bap-5);
  p = fma(p, r, 0x1.555555555555ap-3);
  p = fma(p, r, 0x1.0000000000011p-1);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);
  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
}

// The same polynomial without the clamp: ONLY for rows whose arguments the packer has bounded (|x| < 680 over
// [T_SAFE_LO, T_SAFE_HI]) and temperatures inside that window.  15 FP64-pipe instructions, 3 integer ones.
__device__ __forceinline__ double ck_exp_nc(double x) {
  const double MAGIC = ck_expc[13];
  const double t = fma(x, ck_expc[12], MAGIC);
  const int n = __double2loint(t);
  const double nf = t - MAGIC;
  double r = fma(nf, ck_expc[14], x);
  r = fma(nf, ck_expc[15], r);
  double p = ck_expc[0];
#pragma unroll
  for (int i = 1; i < 12; ++i) p = fma(p, r, ck_expc[i]);
  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
}

// 1/y and ln(x) for the falloff rows: branch-free, a few ulp (the library versions are correctly rounded but cost
// ~22 and ~65 instructions with a slow-path branch each; a Troe row needs two logarithms and two divisions).
__device__ __forceinline__ double ck_rcp(double y) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(y));   // ~20 good bits
  double e = fma(-y, r, 1.0);
  r = fma(r, e, r);
  e = fma(-y, r, 1.0);
  r = fma(r, e, r);
  e = fma(-y, r, 1.0);
  return fma(r, e, r);
}
// x must be a positive NORMAL number (callers guard with fmax(x, 1e-300))
__device__ __forceinline__ double ck_log(double x) {
  int hi = __double2hiint(x);
  int e = (hi >> 20) - 1023;
  hi = (hi & 0x000fffff) | 0x3ff00000;                    // mantissa in [1, 2)
  double mnt = __hiloint2double(hi, __double2loint(x));
  const bool big = mnt > 1.4142135623730951;
  mnt = big ? mnt * 0.5 : mnt;                            // [sqrt(1/2), sqrt(2)]
  e += big ? 1 : 0;
  const double f = mnt - 1.0;
  const double s = f * ck_rcp(2.0 + f);                   // ln(m) = 2 atanh(s), |s| <= 0.1716
  const double z = s * s;
  double p = 1.0 / 21.0;
  p = fma(p, z, 1.0 / 19.0);
  p = fma(p, z, 1.0 / 17.0);
  p = fma(p, z, 1.0 / 15.0);
  p = fma(p, z, 1.0 / 13.0);
  p = fma(p, z, 1.0 / 11.0);
  p = fma(p, z, 1.0 / 9.0);
  p = fma(p, z, 1.0 / 7.0);
  p = fma(p, z, 1.0 / 5.0);
  p = fma(p, z, 1.0 / 3.0);
  const double lm = fma(2.0 * s * z, p, 2.0 * s);
  const double ed = (double)e;
  return fma(ed, 6.93147180369123816490e-01, fma(ed, 1.90821492927058770002e-10, lm));
}

// Constants of one reaction gathered into registers (from the SoA arrays or from a staged rpack row).
struct RxnConst {
  double lnA, beta, Ta, c0, c1, c2, c3, c4, c5, c6;
  int slot[6];  // species index (or the dummy K) of the three reactant and three product slots
  int dup;      // nonzero: a species sits in two slots (scatter slot by slot)
};
__device__ __forceinline__ RxnConst load_rxn_global(const MechDev& m, int r, int tint) {
  RxnConst k;
  const int R = m.R;
  k.lnA = __ldg(m.lnA + r); k.beta = __ldg(m.beta + r); k.Ta = __ldg(m.Ta + r);
  const double* c = m.krc + (size_t)tint * 7 * R + r;
  k.c0 = __ldg(c); k.c1 = __ldg(c + R); k.c2 = __ldg(c + 2 * (size_t)R); k.c3 = __ldg(c + 3 * (size_t)R);
  k.c4 = __ldg(c + 4 * (size_t)R); k.c5 = __ldg(c + 5 * (size_t)R); k.c6 = __ldg(c + 6 * (size_t)R);
#pragma unroll
  for (int s = 0; s < 6; ++s) k.slot[s] = __ldg(m.slot + (size_t)s * R + r);
  k.dup = 1;
  return k;
}
// row = pointer to the reaction's rpack row (shared or global memory, 16-byte aligned).  With two temperature
// intervals (the common case) BOTH coefficient sets are read with warp-uniform addresses and selected per lane:
// lanes of one warp sit in different intervals almost always (independent reactors), and a per-lane address
// would split every 16-byte broadcast into several shared-memory wavefronts.
// PRE: slots 0, 1, 3, 4 come back as the pre-shifted words (slot << 12) of the row header, slots 2 and 5 are not decoded
template <bool PRE = false>
__device__ __forceinline__ RxnConst load_rxn_row(const double* row, int tint, int nT = 0) {
  RxnConst k;
  const double2 a = *reinterpret_cast<const double2*>(row);
  const double2 b = *reinterpret_cast<const double2*>(row + 2);
  k.lnA = a.x; k.beta = a.y; k.Ta = b.x;
  const unsigned lo = (unsigned)__double2loint(b.y), hi = (unsigned)__double2hiint(b.y);
  if (PRE) {
    const uint4 w = *reinterpret_cast<const uint4*>(row + 4);
    k.slot[0] = (int)w.x; k.slot[1] = (int)w.y; k.slot[3] = (int)w.z; k.slot[4] = (int)w.w;
    k.slot[2] = k.slot[5] = 0;
  } else {
    k.slot[0] = lo & 1023u; k.slot[1] = (lo >> 10) & 1023u; k.slot[2] = (lo >> 20) & 1023u;
    k.slot[3] = hi & 1023u; k.slot[4] = (hi >> 10) & 1023u; k.slot[5] = (hi >> 20) & 1023u;
  }
  k.dup = (int)(hi >> 31);
  if (nT == 2) {
    const double2* c = reinterpret_cast<const double2*>(row + RPH);
    const double2 l01 = c[0], l23 = c[1], l45 = c[2], l67 = c[3], h01 = c[4], h23 = c[5], h45 = c[6], h67 = c[7];
    const bool h = tint != 0;
    k.c0 = h ? h01.x : l01.x; k.c1 = h ? h01.y : l01.y; k.c2 = h ? h23.x : l23.x; k.c3 = h ? h23.y : l23.y;
    k.c4 = h ? h45.x : l45.x; k.c5 = h ? h45.y : l45.y; k.c6 = h ? h67.x : l67.x;
    return k;
  }
  const double2* c = reinterpret_cast<const double2*>(row + RPH + 8 * tint);
  const double2 c01 = c[0], c23 = c[1], c45 = c[2], c67 = c[3];
  k.c0 = c01.x; k.c1 = c01.y; k.c2 = c23.x; k.c3 = c23.y; k.c4 = c45.x; k.c5 = c45.y; k.c6 = c67.x;
  return k;
}

// Rate constants of Eq. 15 and of Eq. 16-18 folded into one polynomial (ck_mech.cu)
template <bool NC = false>
__device__ __forceinline__ void rate_constants(const RxnConst& k, const TState& t, double& kf, double& kr) {
  const double xf = fma(k.beta, t.lnT, k.lnA) - k.Ta * t.invT;
  const double T = t.T;
  const double poly = fma(fma(fma(k.c6, T, k.c5), T, k.c4), T, k.c3) * T;
  const double xr = fma(k.c1, t.lnT, k.c0) + fma(k.c2, t.invT, poly);
  kf = NC ? ck_exp_nc(xf) : ck_exp(xf);
  kr = NC ? ck_exp_nc(xr) : ck_exp(xr);
}

// Everything the Jacobian needs about one reaction besides q itself.
struct RateAux {
  double kf, kr, ci, pf, pr;   // q = ci (kf pf - kr pr)
  double dlnkf_dT, dlnkr_dT;   // temperature derivatives of the rate constants
  double dci_dM;               // d c_i / d [M]_i at constant T   (0 for plain rows)
  double dci_dT;               // d c_i / d T at constant concentrations (falloff rows)
  double M;                    // [M]_i of a third-body / falloff row (0 for plain rows)
};

// Rate of progress q_i of regrouped reaction r.  WANT_AUX also fills the derivative pieces.
// TYPE >= 0 fixes the row kind at compile time (0 plain, 1 three-body, 2 Lindemann, 3 Troe) and promises a staged
// xrow; TYPE < 0 reads the kind off the group boundaries.
template <int CS, bool WANT_AUX, int TYPE = -1>
__device__ __forceinline__ double reaction_q(const MechDev& m, int r, const RxnConst& k, const TState& t,
                                             const double* __restrict__ C, double Ctot, RateAux* aux,
                                             const double* __restrict__ xrow = nullptr) {
  const double beta = k.beta, Ta = k.Ta;
  const double c1 = k.c1, c2 = k.c2, c3 = k.c3, c4 = k.c4, c5 = k.c5, c6 = k.c6;
  const double T = t.T;
  double kf, kr;
  rate_constants(k, t, kf, kr);
  double ci = 1.0, dci_dM = 0.0, dci_dT = 0.0, Mi = 0.0;
  if (TYPE < 0 ? (r >= m.r_tb) : (TYPE >= 1)) {  // third-body / falloff factor c_i (reading G9)
    const int j = r - m.r_tb;
    double M = Ctot;
    // constants of this row: from the staged xpack row (shared memory) when given, else from global memory
    const double* xr = (TYPE >= 0 || xrow) ? xrow : m.xpack + (size_t)j * 16;
    const unsigned long long xw = (unsigned long long)__double_as_longlong(xr[7]);
    const int ne = (int)(xw & 15ull);
    if (ne != 15) {
      for (int e = 0; e < ne; ++e) M = fma(xr[8 + e], C[(size_t)((xw >> (4 + 10 * e)) & 1023ull) * CS], M);
    } else {
      for (int e = __ldg(m.eptr + j), e1 = __ldg(m.eptr + j + 1); e < e1; ++e)
        M = fma(__ldg(m.eval1 + e), C[(size_t)__ldg(m.espec + e) * CS], M);
    }
    Mi = M;
    if (TYPE < 0 ? (r < m.r_lind) : (TYPE == 1)) {
      ci = M;
      if (WANT_AUX) dci_dM = 1.0;
    } else {
      const double beta0 = xr[1], Ta0 = xr[2];
      // k_0 / k_inf from the DIFFERENCE of the two Arrhenius arguments: one exponential, no division
      const double k0_kf = ck_exp(fma(beta0 - beta, t.lnT, xr[0] - k.lnA) - (Ta0 - Ta) * t.invT);
      const double Pr = k0_kf * M;
      const double inv1p = ck_rcp(1.0 + Pr);
      const double L = Pr * inv1p;  // Lindemann
      double F = 1.0, dlnF_dlP = 0.0, dlnF_dT = 0.0;
      if (TYPE < 0 ? (r >= m.r_troe) : (TYPE == 3)) {
        const double a = xr[3], i3 = xr[4], i1 = xr[5], T2 = xr[6];
        const double e3 = ck_exp(-T * i3), e1 = ck_exp(-T * i1);
        double Fc = fma(1.0 - a, e3, a * e1);
        double e2 = 0.0;
        if (T2 >= 0.0) { e2 = ck_exp(-T2 * t.invT); Fc += e2; }
        const double il10 = 0.43429448190325182765;  // 1/ln 10
        const double ln10 = 2.30258509299404568402;
        const double Fcg = fmax(Fc, 1e-300), Prg = fmax(Pr, 1e-300);
        const double lF = ck_log(Fcg) * il10, lP = ck_log(Prg) * il10;
        const double cc = fma(-0.67, lF, -0.4), nn = fma(-1.27, lF, 0.75);
        const double x = lP + cc;
        const double den = fma(-0.14, x, nn);
        const double den2 = den * den;
        const double g = den2 * ck_rcp(fma(x, x, den2));  // 1 / (1 + f1^2), f1 = x / den: one reciprocal instead of two divisions
        F = ck_exp(ln10 * lF * g);
        if (WANT_AUX) {
          // ln F = ln10 * lF / (1 + f1^2);  f1 = x/den, x = lP + cc(lF), den = nn(lF) - 0.14 x
          const double f1 = x / den;
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
  // Eq. 14: products over the slots (nu copies of each species; the dummy slot holds C = 1)
  const double pf = C[(size_t)k.slot[0] * CS] * C[(size_t)k.slot[1] * CS] * C[(size_t)k.slot[2] * CS];
  const double pr = C[(size_t)k.slot[3] * CS] * C[(size_t)k.slot[4] * CS] * C[(size_t)k.slot[5] * CS];
  if (WANT_AUX) {
    aux->kf = kf; aux->kr = kr; aux->ci = ci; aux->pf = pf; aux->pr = pr;
    aux->dlnkf_dT = (beta + Ta * t.invT) * t.invT;
    aux->dlnkr_dT = (kr > 0.0) ? fma(fma(fma(4.0 * c6, T, 3.0 * c5), T, 2.0 * c4), T, c3) + (c1 - c2 * t.invT) * t.invT : 0.0;
    aux->dci_dM = dci_dM; aux->dci_dT = dci_dT; aux->M = Mi;
  }
  return ci * (kf * pf - kr * pr);
}

}  // namespace ck
