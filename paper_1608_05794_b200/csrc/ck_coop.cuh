// Group-per-reactor (CTA-cooperative) chemistry: one CTA of G threads evaluates the RHS and the analytic
// Jacobian of ONE reactor whose state lives in shared memory.  Used by ck_jac and the ROS4 step kernel,
// where the dense N x N matrix must stay on chip.
//   threads over species  : thermo, concentrations, species sums (gather form, no atomics)
//   threads over reactions: rates of progress q_i (and their derivatives)
#pragma once
#include "ck_chem.cuh"

namespace ck {

// Deterministic CTA-wide sum; `red` is a shared scratch of >= 33 doubles.  All threads get the result.
template <int G>
__device__ __forceinline__ double block_sum(double v, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if (G == 32) return v;
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) red[w] = v;
  __syncthreads();
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < G / 32; ++i) s += red[i];
  return s;
}

// two sums with one barrier pair; red: >= 2 * (G / 32) doubles
template <int G>
__device__ __forceinline__ void block_sum2(double& a, double& b, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
  if (G == 32) return;
  constexpr int W = G / 32;
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) { red[w] = a; red[W + w] = b; }
  __syncthreads();
  double sa = 0.0, sb = 0.0;
#pragma unroll
  for (int i = 0; i < W; ++i) { sa += red[i]; sb += red[W + i]; }
  a = sa; b = sb;
}

// Shared-memory working set of the cooperative chemistry (pointers into the CTA's dynamic smem)
struct CoopChem {
  double* C;     // [K+1] concentrations, C[K] = 1
  double* cpR;   // [K]
  double* hRT;   // [K]
  double* yw;    // [K] Y_k / W_k
  double* q;     // [R] rates of progress
  double* w;     // [K] production rates omega_k
  double* red;   // [40] reduction scratch
  // Jacobian only:
  double* dqs;   // [6][R] d q_i / d C_slot (0 for dummy slots)
  double* dqT;   // [R]    d q_i / d T at constant concentrations
  double* dqM;   // [R]    d q_i / d [M]_i
  double* si;    // [R]    sum_m (d q_i/d C_m) C_m
  double* dns;   // [K]    dense third-body coefficient of row k: sum_i nu_ki dq_i/d[M]_i
  double* sig;   // [K]    sum_i nu_ki s_i
  double* tau;   // [K]    sum_i nu_ki dq_i/dT|_C
  int* dsl;      // [6][R] slot species of every reaction (shared-memory copy: the row assembly would otherwise
                 //        wait on a global load per reaction)
};
struct CoopScalars { double rho, S, cps, Ctot, hw; };

// jc > 0: the per-reaction derivative arrays hold one CHUNK of jc reactions (rhs_jac_coop); jc = 0: all R reactions
__host__ __device__ inline int coop_chem_doubles(int K, int R, bool jac, int jc = 0) {
  const int L = jc > 0 ? jc : R;
  return (K + 1) + 4 * K + R + 40 + (jac ? 12 * L + 3 * K : 0) + 8;
}
__device__ __forceinline__ CoopChem coop_carve(double* base, int K, int R, bool jac, int jc = 0) {
  const int L = jc > 0 ? jc : R;
  CoopChem c;
  c.C = base; base += K + 1;
  c.cpR = base; base += K;
  c.hRT = base; base += K;
  c.yw = base; base += K;
  c.w = base; base += K;
  c.q = base; base += R;
  c.red = base; base += 40;
  c.dqs = base; base += jac ? 6 * L : 0;
  c.dqT = base; base += jac ? L : 0;
  c.dqM = base; base += jac ? L : 0;
  c.si = base; base += jac ? L : 0;
  c.dns = base; base += jac ? K : 0;
  c.sig = base; base += jac ? K : 0;
  c.tau = base; base += jac ? K : 0;
  c.dsl = reinterpret_cast<int*>(base);
  return c;
}

// f = RHS(y; p) for the reactor whose state is y[0..N) in shared memory; result to fout[0..N) (shared).
// JAC additionally fills the per-reaction derivative arrays.  Ends with a __syncthreads().
template <int G, bool JAC>
__device__ __forceinline__ CoopScalars rhs_coop(const MechDev& m, const double* __restrict__ y, double p,
                                                double* __restrict__ fout, const CoopChem& c, TState& t) {
  const int K = m.K, R = m.R, tid = threadIdx.x;
  t = make_tstate(m, y[0]);
  double Sp = 0.0, cp = 0.0;
  const double sub = m.cv ? 1.0 : 0.0;
  for (int k = tid; k < K; k += G) {
    double cpR, hRT;
    thermo_cp_h(m, k, t, cpR, hRT);
    cpR -= sub; hRT -= sub;   // constant volume: c_v,k / R = c_p,k / R - 1, U_k / (R T) = H_k / (R T) - 1
    const double yw = y[1 + k] * __ldg(m.invW + k);
    c.cpR[k] = cpR; c.hRT[k] = hRT; c.yw[k] = yw;
    Sp += yw;
    cp = fma(yw, cpR, cp);
  }
  CoopScalars s;
  s.S = block_sum<G>(Sp, c.red);
  s.cps = block_sum<G>(cp, c.red);
  s.rho = m.cv ? p : (p / (R_U * t.T)) / s.S;   // constant volume: `p` is the density
  s.Ctot = m.cv ? s.rho * s.S : p / (R_U * t.T);
  for (int k = tid; k < K; k += G) c.C[k] = s.rho * c.yw[k];
  if (tid == 0) c.C[K] = 1.0;
  __syncthreads();
  for (int r = tid; r < R; r += G) {
    const RxnConst kc = load_rxn_global(m, r, t.tint);
    RateAux a;
    const double q = reaction_q<1, JAC>(m, r, kc, t, c.C, s.Ctot, JAC ? &a : nullptr);
    c.q[r] = q;
    if (JAC) {
      const double c0 = c.C[kc.slot[0]], c1 = c.C[kc.slot[1]], c2 = c.C[kc.slot[2]];
      const double c3 = c.C[kc.slot[3]], c4 = c.C[kc.slot[4]], c5 = c.C[kc.slot[5]];
      const double gf = a.ci * a.kf, gr = -a.ci * a.kr;
      double d[6] = {gf * c1 * c2, gf * c0 * c2, gf * c0 * c1, gr * c4 * c5, gr * c3 * c5, gr * c3 * c4};
      double sum = 0.0;
#pragma unroll
      for (int x = 0; x < 6; ++x) {
        if (kc.slot[x] == K) d[x] = 0.0;
        c.dqs[(size_t)x * R + r] = d[x];
        c.dsl[(size_t)x * R + r] = kc.slot[x];
        sum = fma(d[x], c.C[kc.slot[x]], sum);
      }
      const double net = a.kf * a.pf - a.kr * a.pr;
      const double dM = a.dci_dM * net;
      c.dqM[r] = dM;
      c.dqT[r] = a.ci * (a.kf * a.pf * a.dlnkf_dT - a.kr * a.pr * a.dlnkr_dT) + a.dci_dT * net;
      // [M]_i = sum_m alpha_im C_m (Ctot = sum C), so sum_m dq/dC_m C_m gains dM * [M]_i
      double M = 0.0;
      if (r >= m.r_tb) {
        const int j = r - m.r_tb;
        M = s.Ctot;
        for (int e = __ldg(m.eptr + j), e1 = __ldg(m.eptr + j + 1); e < e1; ++e)
          M = fma(__ldg(m.eval1 + e), c.C[__ldg(m.espec + e)], M);
      }
      c.si[r] = fma(dM, M, sum);
    }
  }
  __syncthreads();
  const double irho = 1.0 / s.rho;
  double hwp = 0.0;
  for (int k = tid; k < K; k += G) {
    double w = 0.0;
    for (int e = __ldg(m.tptr + k), e1 = __ldg(m.tptr + k + 1); e < e1; ++e) {
      const int en = __ldg(m.tent + e);
      w = fma((double)((en & 255) - 128), c.q[en >> 8], w);
    }
    c.w[k] = w;
    hwp = fma(c.hRT[k], w, hwp);
    fout[1 + k] = w * __ldg(m.W + k) * irho;
  }
  s.hw = block_sum<G>(hwp, c.red);
  if (tid == 0) fout[0] = -(t.T * s.hw) / (s.rho * s.cps);
  __syncthreads();
  return s;
}

// f(y) AND the species rows G_kj of the analytic Jacobian in one pass over the reactions, G reactions at a time:
// the per-reaction derivative arrays then hold a single chunk (12 G doubles instead of 12 R), which is what lets
// more reactors share an SM.  Requires K <= G (thread k owns species row k and walks its reaction list, sorted by
// reaction index, with a private cursor).  Leaves q, omega, f, dns / sig / tau as rhs_coop<.,true> + the row phase
// of jac_coop would; the caller finishes with jac_coop_finish.  A is zeroed here.
template <int G>
__device__ __forceinline__ CoopScalars rhs_jac_coop(const MechDev& m, const double* __restrict__ y, double p,
                                                    double* __restrict__ fout, const CoopChem& c, TState& t,
                                                    double* __restrict__ A, int lda) {
  const int K = m.K, R = m.R, N = K + 1, tid = threadIdx.x;
  t = make_tstate(m, y[0]);
  double Sp = 0.0, cp = 0.0;
  const double sub = m.cv ? 1.0 : 0.0;
  for (int k = tid; k < K; k += G) {
    double cpR, hRT;
    thermo_cp_h(m, k, t, cpR, hRT);
    cpR -= sub; hRT -= sub;   // constant volume: c_v,k / R = c_p,k / R - 1, U_k / (R T) = H_k / (R T) - 1
    const double yw = y[1 + k] * __ldg(m.invW + k);
    c.cpR[k] = cpR; c.hRT[k] = hRT; c.yw[k] = yw;
    Sp += yw;
    cp = fma(yw, cpR, cp);
  }
  for (int idx = tid; idx < N * lda; idx += G) A[idx] = 0.0;
  CoopScalars s;
  s.S = block_sum<G>(Sp, c.red);
  s.cps = block_sum<G>(cp, c.red);
  s.rho = m.cv ? p : (p / (R_U * t.T)) / s.S;   // constant volume: `p` is the density
  s.Ctot = m.cv ? s.rho * s.S : p / (R_U * t.T);
  for (int k = tid; k < K; k += G) c.C[k] = s.rho * c.yw[k];
  if (tid == 0) c.C[K] = 1.0;
  __syncthreads();
  const bool has_row = tid < K;
  double* row = A + (size_t)(1 + (has_row ? tid : 0)) * lda + 1;
  int e = has_row ? __ldg(m.tptr + tid) : 0;
  const int e1 = has_row ? __ldg(m.tptr + tid + 1) : 0;
  double dns = 0.0, sig = 0.0, tau = 0.0;
  for (int c0 = 0; c0 < R; c0 += G) {
    const int r = c0 + tid;
    if (r < R) {
      const RxnConst kc = load_rxn_global(m, r, t.tint);
      RateAux a;
      const double q = reaction_q<1, true>(m, r, kc, t, c.C, s.Ctot, &a);
      c.q[r] = q;
      const double x0 = c.C[kc.slot[0]], x1 = c.C[kc.slot[1]], x2 = c.C[kc.slot[2]];
      const double x3 = c.C[kc.slot[3]], x4 = c.C[kc.slot[4]], x5 = c.C[kc.slot[5]];
      const double gf = a.ci * a.kf, gr = -a.ci * a.kr;
      double d[6] = {gf * x1 * x2, gf * x0 * x2, gf * x0 * x1, gr * x4 * x5, gr * x3 * x5, gr * x3 * x4};
      double sum = 0.0;
      int sl[6];
#pragma unroll
      for (int x = 0; x < 6; ++x) {
        sl[x] = kc.slot[x];
        if (sl[x] == K) d[x] = 0.0;
        sum = fma(d[x], c.C[sl[x]], sum);
      }
      // a species may sit in two slots (nu = 2, or on both sides): fold the later slot into the earlier one HERE,
      // once per reaction, so that the row assembly can load, update and store a reaction's entries together
      if (__ldg(m.rflag + r)) {
#pragma unroll
        for (int x = 1; x < 6; ++x)
#pragma unroll
          for (int y2 = 0; y2 < x; ++y2)
            if (sl[x] == sl[y2] && sl[x] != K) { d[y2] += d[x]; d[x] = 0.0; sl[x] = K; }
      }
#pragma unroll
      for (int x = 0; x < 6; ++x) { c.dqs[x * G + tid] = d[x]; c.dsl[x * G + tid] = sl[x]; }
      const double net = a.kf * a.pf - a.kr * a.pr;
      const double dM = a.dci_dM * net;
      c.dqM[tid] = dM;
      c.dqT[tid] = a.ci * (a.kf * a.pf * a.dlnkf_dT - a.kr * a.pr * a.dlnkr_dT) + a.dci_dT * net;
      double M = 0.0;
      if (r >= m.r_tb) {
        const int j = r - m.r_tb;
        M = s.Ctot;
        for (int z = __ldg(m.eptr + j), z1 = __ldg(m.eptr + j + 1); z < z1; ++z)
          M = fma(__ldg(m.eval1 + z), c.C[__ldg(m.espec + z)], M);
      }
      c.si[tid] = fma(dM, M, sum);
    }
    __syncthreads();
    // species rows: entries of this chunk (the reaction list of a row is sorted by reaction index)
    while (e < e1) {
      const int en = __ldg(m.tent + e);
      const int i = en >> 8;
      if (i >= c0 + G) break;
      const int j = i - c0;
      const double nu = (double)((en & 255) - 128);
      int sl[6];
      double d[6], rv[6];
#pragma unroll
      for (int x = 0; x < 6; ++x) { sl[x] = c.dsl[x * G + j]; d[x] = c.dqs[x * G + j]; }
#pragma unroll
      for (int x = 0; x < 6; ++x)
        if (sl[x] != K) rv[x] = row[sl[x]];
#pragma unroll
      for (int x = 0; x < 6; ++x)
        if (sl[x] != K) row[sl[x]] = fma(nu, d[x], rv[x]);
      sig = fma(nu, c.si[j], sig);
      tau = fma(nu, c.dqT[j], tau);
      if (i >= m.r_tb) {
        const double dM = nu * c.dqM[j];
        dns += dM;
        const int jj = i - m.r_tb;
        for (int z = __ldg(m.eptr + jj), z1 = __ldg(m.eptr + jj + 1); z < z1; ++z) {
          const int sp = __ldg(m.espec + z);
          row[sp] = fma(dM, __ldg(m.eval1 + z), row[sp]);
        }
      }
      ++e;
    }
    __syncthreads();
  }
  if (has_row) { c.dns[tid] = dns; c.sig[tid] = sig; c.tau[tid] = tau; }
  const double irho = 1.0 / s.rho;
  double hwp = 0.0;
  for (int k = tid; k < K; k += G) {
    double w = 0.0;
    for (int z = __ldg(m.tptr + k), z1 = __ldg(m.tptr + k + 1); z < z1; ++z) {
      const int en = __ldg(m.tent + z);
      w = fma((double)((en & 255) - 128), c.q[en >> 8], w);
    }
    c.w[k] = w;
    hwp = fma(c.hRT[k], w, hwp);
    fout[1 + k] = w * __ldg(m.W + k) * irho;
  }
  s.hw = block_sum<G>(hwp, c.red);
  if (tid == 0) fout[0] = -(t.T * s.hw) / (s.rho * s.cps);
  __syncthreads();
  return s;
}

// Analytic Jacobian A[i*lda + j] = d f_i / d y_j (i, j = 0 is T) from the pieces left in shared memory by
// rhs_coop<G,true>; `f` is that call's output.  Chain rule at constant p:
//   C_m = rho Y_m / W_m, rho = p/(R_u T S):  dC_m/dT = -C_m/T,  dC_m/dY_j = delta_mj rho/W_j - C_m/(S W_j)
//   G_kj = sum_i nu_ki dq_i/dC_j,  sigma_k = sum_i nu_ki sum_m dq_i/dC_m C_m,  tau_k = sum_i nu_ki dq_i/dT|_C
//   d omega_k/dY_j = (rho/W_j) G_kj - sigma_k/(S W_j),   d omega_k/dT = tau_k - sigma_k/T
// Ends with a __syncthreads().
// temperature row, temperature column and the in-place transform of the species block (see jac_coop)
template <int G>
__device__ __forceinline__ void jac_coop_finish(const MechDev& m, const CoopChem& c, const CoopScalars& s, const TState& t,
                                         const double* __restrict__ f, double* __restrict__ A, int lda) {
  const int K = m.K, tid = threadIdx.x;
  // scalars of the temperature row
  // constant volume: rho does not depend on y, so every term that came from d rho / d y (the sigma terms, f_k / T,
  // f_k / (S W_j), one of the two f_T / T) drops out: sg = 0; c.cpR / c.hRT / s.cps already hold c_v and u (rhs_coop)
  const double sg = m.cv ? 0.0 : 1.0;
  double hs = 0.0, ht = 0.0, hcw = 0.0, dcp = 0.0;
  for (int k = tid; k < K; k += G) {
    hs = fma(c.hRT[k], sg * c.sig[k], hs);
    ht = fma(c.hRT[k], c.tau[k] - sg * c.sig[k] * t.invT, ht);
    hcw = fma((c.cpR[k] - c.hRT[k]) * t.invT, c.w[k], hcw);
    dcp = fma(c.yw[k], thermo_dcp(m, k, t), dcp);
  }
  hs = block_sum<G>(hs, c.red);
  ht = block_sum<G>(ht, c.red);
  hcw = block_sum<G>(hcw, c.red);
  dcp = block_sum<G>(dcp, c.red);
  const double phi = t.T / (s.rho * s.cps);
  const double fT = f[0];
  const double iS = 1.0 / s.S;
  for (int j = tid; j < K; j += G) {
    double col = 0.0;
    for (int k = 0; k < K; ++k) col = fma(c.hRT[k], A[(size_t)(1 + k) * lda + 1 + j] + c.dns[k], col);
    const double iWj = __ldg(m.invW + j);
    A[1 + j] = -phi * (s.rho * iWj * col - hs * iS * iWj) + fT * (sg * iS * iWj - c.cpR[j] * iWj / s.cps);
  }
  if (tid == 0) A[0] = -phi * (hcw + ht) + fT * ((1.0 + sg) * t.invT - dcp / s.cps);
  __syncthreads();
  // species rows: in-place transform of G into d f_k / d Y_j, and the temperature column
  const double irho = 1.0 / s.rho;
  for (int idx = tid; idx < K * K; idx += G) {
    const int k = idx / K, j = idx - k * K;
    const double Wk = __ldg(m.W + k), iWj = __ldg(m.invW + j);
    double* a = A + (size_t)(1 + k) * lda + 1 + j;
    *a = Wk * iWj * (*a + c.dns[k]) + sg * (f[1 + k] - Wk * irho * c.sig[k]) * iS * iWj;
  }
  for (int k = tid; k < K; k += G)
    A[(size_t)(1 + k) * lda] = __ldg(m.W + k) * irho * (c.tau[k] - sg * c.sig[k] * t.invT) + sg * f[1 + k] * t.invT;
  __syncthreads();
}

template <int G>
__device__ __forceinline__ void jac_coop(const MechDev& m, const CoopChem& c, const CoopScalars& s, const TState& t,
                                         const double* __restrict__ f, double* __restrict__ A, int lda) {
  const int K = m.K, R = m.R, N = K + 1, tid = threadIdx.x;
  for (int idx = tid; idx < N * lda; idx += G) A[idx] = 0.0;
  __syncthreads();
  // rows of G, one thread per species row (no two threads touch the same row)
  for (int k = tid; k < K; k += G) {
    double* row = A + (size_t)(1 + k) * lda + 1;
    double dns = 0.0, sig = 0.0, tau = 0.0;
    for (int e = __ldg(m.tptr + k), e1 = __ldg(m.tptr + k + 1); e < e1; ++e) {
      const int en = __ldg(m.tent + e);
      const int i = en >> 8;
      const double nu = (double)((en & 255) - 128);
      int sl[6];
      double d[6], rv[6];
#pragma unroll
      for (int x = 0; x < 6; ++x) { sl[x] = c.dsl[(size_t)x * R + i]; d[x] = c.dqs[(size_t)x * R + i]; }
      // a species may sit in two slots (nu = 2, or on both sides): fold the later slot into the earlier one so
      // that the six row entries can be loaded, updated and stored together (one shared-memory round trip)
#pragma unroll
      for (int x = 1; x < 6; ++x)
#pragma unroll
        for (int y = 0; y < x; ++y)
          if (sl[x] == sl[y] && sl[x] != K) { d[y] += d[x]; sl[x] = K; }
#pragma unroll
      for (int x = 0; x < 6; ++x)
        if (sl[x] != K) rv[x] = row[sl[x]];
#pragma unroll
      for (int x = 0; x < 6; ++x)
        if (sl[x] != K) row[sl[x]] = fma(nu, d[x], rv[x]);
      sig = fma(nu, c.si[i], sig);
      tau = fma(nu, c.dqT[i], tau);
      if (i >= m.r_tb) {
        const double dM = nu * c.dqM[i];
        dns += dM;
        const int j = i - m.r_tb;
        for (int z = __ldg(m.eptr + j), z1 = __ldg(m.eptr + j + 1); z < z1; ++z) {
          const int sp = __ldg(m.espec + z);
          row[sp] = fma(dM, __ldg(m.eval1 + z), row[sp]);
        }
      }
    }
    c.dns[k] = dns; c.sig[k] = sig; c.tau[k] = tau;
  }
  __syncthreads();
  jac_coop_finish<G>(m, c, s, t, f, A, lda);
}

}  // namespace ck
