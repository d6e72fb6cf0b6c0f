// Latency-optimised RKF45 finisher: ONE reactor per 384-thread CTA, every attempt of Algorithm 1
// with its six evaluations of f (Eq. 8-19) laid out for the shortest dependent chain, because the
// stragglers of the step-count distribution (tens of thousands of attempts where the median is ~130)
// are a SERIAL chain of attempts whose length sets the run time of the whole batch.
//
// Included by ck_rkf.cu after RkfArgs / RKF_T.  What differs from the cooperative evaluation of ck_coop.cuh:
//  * roles instead of loops: warp 0 owns the species (lane l: species l, l + 32, ...), threads 32.. own the reactions,
//    so the thermodynamic sums S = sum Y_k / W_k and c_p are ONE warp's shuffle reduction (no block reduction), and
//    while warp 0 does thermo -> density -> concentrations the reaction threads compute everything that depends on T
//    only: k_f, k_r (Eq. 15-18 through the packed polynomial), k_0 / k_inf and the Troe centre F_cent with its logarithm;
//  * after ONE barrier the reaction threads finish with what depends on concentrations ([M], P_r, the Troe blend, the
//    concentration products), three barriers per evaluation instead of five; the species thermo coefficients, the
//    falloff rows and each lane's share of the transposed stoichiometry are staged once per CTA (shared memory /
//    registers), and every short loop has a compile-time trip count with predicated entries so that its loads are
//    independent;
//  * the temperature equation needs sum_k h_k omega_k = sum_i q_i (sum_k nu_ki h_k): each reaction thread forms its own
//    enthalpy of reaction from the species enthalpies and the sum over reactions rides on the barrier that publishes q,
//    so no reduction follows the production-rate gather;
//  * the stage argument y + h sum_j a_sj k_j is formed by its consumers (every thread for T, warp 0 for its species):
//    no stage-combination phase and no barrier between evaluations;
//  * error norm and accept / reject are warp 0's; the NEW STEP SIZE is computed lazily, by warp 0 while the reaction
//    threads are busy with the first evaluation of the next attempt (f(y_n) does not depend on h), so the power
//    function of the controller is off the critical path; h reaches the other warps through shared memory.
// Arithmetic per reaction is rate_constants / the falloff blend of ck_chem.cuh operation by operation; ln T and 1 / T
// come from the branch-free ck_log / ck_rcp (a few ulp), sums run in a different order: results agree with the other
// RKF45 kernels to rounding, and every path is tested against the oracle.
#pragma once

namespace ck {

constexpr int WIDE_G = 384;
constexpr int WIDE_GE = 12;   // transposed-stoichiometry entries a lane keeps in registers

// shared memory of one CTA, in doubles
__host__ __device__ inline size_t rkf_wide_smem_doubles(int K, int R, int r_tb, int n_tent) {
  const size_t N = K + 1;
  return 7 * N + 2 * N + (size_t)R + 16 + 8 + 14 * (size_t)K + 17 * (size_t)(R - r_tb) + (size_t)((n_tent + K + 2 + 1) >> 1);
}

template <int G>
__global__ void __launch_bounds__(G, 1) rkf45_wide_kernel(const MechDev m, const RkfArgs a, const int cls) {
  extern __shared__ double sm[];
  __shared__ long long s_next;
  const int K = m.K, R = m.R, N = K + 1, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = G / 32, RT = G - 32;     // warps; reaction threads
  double* Y = sm;                  // y_n
  double* F = Y + N;               // six evaluations, F[j * N + c]
  double* C = F + 6 * N;           // [K+1] concentrations, C[K] = 1 (dummy slot)
  double* H = C + N;               // [K+1] H_k / (R T) (constant volume: U_k / (R T)), H[K] = 0
  double* q = H + N;               // [R]
  double* red = q + R;             // [16] per-warp partial sums of q_i * (enthalpy of reaction i) / (R T)
  double* sc = red + 16;           // scalars: 0 coefficient of the temperature equation, 1 C_tot, 2 1 / rho, 3 h, 4 go, 5 go_pre
  double* th = sc + 8;             // [14][K]: NASA-7 a1..a6 low range, a1..a6 high range, t_mid, 1 / W
  double* xp = th + 14 * K;        // [R - r_tb][17]: falloff / third-body rows (odd stride: conflict-free)
  int* s_tptr = reinterpret_cast<int*>(xp + 17 * (size_t)(R - m.r_tb));
  int* s_tent = s_tptr + K + 1;
  for (int i = tid; i <= K; i += G) s_tptr[i] = __ldg(m.tptr + i);
  for (int i = tid; i < m.n_tent; i += G) s_tent[i] = __ldg(m.tent + i);
  for (int i = tid; i < 6 * K; i += G) { th[i] = __ldg(m.nlo + i); th[6 * K + i] = __ldg(m.nhi + i); }
  for (int i = tid; i < K; i += G) { th[12 * K + i] = __ldg(m.tmid + i); th[13 * K + i] = __ldg(m.invW + i); }
  for (int i = tid; i < (R - m.r_tb) * 16; i += G) xp[(size_t)(i >> 4) * 17 + (i & 15)] = __ldg(m.xpack + i);
  if (tid == 0) { C[K] = 1.0; H[K] = 0.0; }
  // ---- production-rate gather: QS adjacent lanes share species gk; this lane's entries live in registers ------------
  const int QS = (4 * K <= G) ? 4 : ((2 * K <= G) ? 2 : 1);
  const int gk = tid / QS, gpart = tid % QS;
  const double gW = (gk < K) ? __ldg(m.W + gk) : 0.0;
  int gi[WIDE_GE];        // reaction index
  double gn[WIDE_GE];     // nu (0 for padding entries)
  bool fits_l = true;
  {
    const int e0 = (gk < K) ? __ldg(m.tptr + gk) : 0, e1 = (gk < K) ? __ldg(m.tptr + gk + 1) : 0;
    fits_l = (e1 - e0) <= QS * WIDE_GE;
#pragma unroll
    for (int x = 0; x < WIDE_GE; ++x) {
      const int e = e0 + gpart + x * QS;
      const int en = (e < e1) ? __ldg(m.tent + e) : 128;   // (reaction 0, nu = 0)
      gi[x] = en >> 8;
      gn[x] = (double)((en & 255) - 128);
    }
  }
  const bool gfit = __syncthreads_and(fits_l ? 1 : 0) != 0;
  // ---- this thread's reaction (one each when R <= RT): what never changes ----------------------------------------------
  // Rows are sorted by kind (plain, three-body, Lindemann, Troe); each kind starts on a warp boundary when the threads
  // suffice, so that a warp runs ONE kind's code (a mixed warp would run the kinds one after the other).
  const int r0 = tid - 32;
  const bool one = R <= RT;
  int rr = 0;
  bool on = false;
  if (one && warp != 0) {
    const int nTr = R - m.r_troe, nLi = m.r_troe - m.r_lind, nTb = m.r_lind - m.r_tb;
    const int pTr = (nTr + 31) & ~31, pLi = (nLi + 31) & ~31, pTb = (nTb + 31) & ~31;
    if (pTr + pLi + pTb + m.r_tb <= RT) {
      if (r0 < pTr) { rr = m.r_troe + r0; on = r0 < nTr; }
      else if (r0 < pTr + pLi) { rr = m.r_lind + (r0 - pTr); on = r0 - pTr < nLi; }
      else if (r0 < pTr + pLi + pTb) { rr = m.r_tb + (r0 - pTr - pLi); on = r0 - pTr - pLi < nTb; }
      else { rr = r0 - pTr - pLi - pTb; on = rr < m.r_tb; }
    } else {
      rr = r0; on = r0 < R;
    }
    if (!on) rr = 0;
  }
  const bool tb = on && rr >= m.r_tb, fo = on && rr >= m.r_lind, troe = on && rr >= m.r_troe;
  const double* xs = xp + (size_t)(tb ? rr - m.r_tb : 0) * 17;
  const double k_lnA = __ldg(m.lnA + rr), k_beta = __ldg(m.beta + rr), k_Ta = __ldg(m.Ta + rr);
  int sl[6];
#pragma unroll
  for (int x = 0; x < 6; ++x) sl[x] = __ldg(m.slot + (size_t)x * R + rr);
  const long long n_ev = fin_count(a, cls);
  unsigned long long c_rhs = 0, c_att = 0, c_acc = 0, c_rej = 0, c_fail = 0;
  for (;;) {
    __syncthreads();
    if (tid == 0) s_next = (long long)atomicAdd(fin_queue(a, cls), 1ULL);
    __syncthreads();
    if (s_next >= n_ev) break;
    const long long r = *fin_entry(a, cls, s_next);
    const double p = a.p[r], ip = 1.0 / p;
    for (int i = tid; i < N; i += G) Y[i] = a.y[(size_t)i * a.ld + r];
    for (int i = tid; i < 6 * N; i += G) F[i] = 0.0;   // the stage sums read all rows (zero coefficients for the later ones)
    // controller state: carried identically by every lane of warp 0
    double t = a.rec_t[r], hn = a.rec_h[r], fac_max = a.rec_fac[r], h_used = 0.0;
    int nacc = a.rec_acc[r], nrej = a.rec_rej[r], status = CK_ST_OK;
    double err_prev = 0.0;     // sum of squares of the attempt whose step-size update is still pending
    bool pend = false, acc_prev = false, last = false;
    if (tid == 0) {
      int go = t < a.dt;
      if (go && nacc + nrej >= a.max_steps) go = 0;
      sc[5] = (double)go;
    }
    if (warp == 0 && t < a.dt && nacc + nrej >= a.max_steps) status = CK_ST_MAX_STEPS;
    for (;;) {
      __syncthreads();   // A: y_n and the continue flag of the previous attempt
      if (sc[5] == 0.0) break;
      double h = 0.0;
      bool stop = false;
#pragma unroll 1
      for (int s = 0; s < 6; ++s) {
        // ---- stage argument, formed by its consumers: T by every thread --------------------------------------------
        const int srow = s > 0 ? s - 1 : 0;
        double cj[5];
#pragma unroll
        for (int j = 0; j < 5; ++j) cj[j] = (j < s) ? RKF_T[srow][j] : 0.0;
        double T;
        {
          double acc = 0.0;
#pragma unroll
          for (int j = 0; j < 5; ++j) acc = fma(cj[j], F[j * N], acc);   // rows >= s: stale but finite, times zero
          T = fma(h, acc, Y[0]);
        }
        TState ts;
        ts.T = T;
        ts.invT = ck_rcp(T);
        double kf = 0.0, kr = 0.0, k0kf = 0.0, lF = 0.0, cc = 0.0, nn = 0.0;
        if (warp == 0) {
          // ---- species warp: thermo, S, c_p, density, concentrations (needs T and 1 / T only) ----------------------
          const double sub = m.cv ? 1.0 : 0.0;   // constant volume: c_v,k and u_k
          double S = 0.0, cp = 0.0;
          double yw[4];
#pragma unroll
          for (int x = 0; x < 4; ++x) {   // no branches: lanes past K work on species K - 1 with weight zero
            const int k0 = lane + 32 * x;
            if (32 * x < K) {             // warp-uniform
              const int k = min(k0, K - 1);
              double acc = 0.0;
#pragma unroll
              for (int j = 0; j < 5; ++j) acc = fma(cj[j], F[j * N + 1 + k], acc);
              const double yk = fma(h, acc, Y[1 + k]);
              const double* c = th + ((T > th[12 * K + k]) ? 6 * K : 0) + k;
              const double a1 = c[0], a2 = c[K], a3 = c[2 * K], a4 = c[3 * K], a5 = c[4 * K], a6 = c[5 * K];
              const double cpR = fma(fma(fma(fma(a5, T, a4), T, a3), T, a2), T, a1);
              const double hRT = fma(fma(fma(fma(a5 * 0.2, T, a4 * 0.25), T, a3 * (1.0 / 3.0)), T, a2 * 0.5), T, a1) + a6 * ts.invT;
              yw[x] = (k0 < K) ? yk * th[13 * K + k] : 0.0;
              H[k] = hRT - sub;
              S += yw[x];
              cp = fma(yw[x], cpR - sub, cp);
            } else {
              yw[x] = 0.0;
            }
          }
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) { S += __shfl_xor_sync(0xffffffffu, S, o); cp += __shfl_xor_sync(0xffffffffu, cp, o); }
          // constant pressure: rho = p / (R T S); both rho and 1 / rho from ONE reciprocal
          const double iS = ck_rcp(S);
          const double rho = m.cv ? p : (p * ts.invT * (1.0 / R_U)) * iS;
          const double irho = m.cv ? ip : (T * R_U * ip) * S;
#pragma unroll
          for (int x = 0; x < 4; ++x) { const int k = lane + 32 * x; if (k < K) C[k] = rho * yw[x]; }
          if (lane == 0) {
            sc[0] = -T * irho * ck_rcp(cp);
            sc[1] = m.cv ? rho * S : p * ts.invT * (1.0 / R_U);
            sc[2] = irho;
          }
        } else if (one) {
          // ---- reaction threads: everything that depends on T only ---------------------------------------------------
          {
            int ti = 0;
#pragma unroll
            for (int e = 0; e < MAX_TINT - 1; ++e) ti += (e < m.nT - 1 && T > m.tedge[e]) ? 1 : 0;
            ts.tint = ti;
          }
          const double* c = m.krc + (size_t)ts.tint * 7 * R + rr;
          RxnConst kc;
          kc.lnA = k_lnA; kc.beta = k_beta; kc.Ta = k_Ta;
          kc.c0 = __ldg(c); kc.c1 = __ldg(c + R); kc.c2 = __ldg(c + 2 * (size_t)R); kc.c3 = __ldg(c + 3 * (size_t)R);
          kc.c4 = __ldg(c + 4 * (size_t)R); kc.c5 = __ldg(c + 5 * (size_t)R); kc.c6 = __ldg(c + 6 * (size_t)R);
          // one straight-line block per row kind: the independent exponentials / logarithms of a block interleave
          if (troe) {
            const double a3 = -T * xs[4], a1 = -T * xs[5], T2 = xs[6], a2 = -fabs(T2) * ts.invT;
            ts.lnT = ck_log(T);
            const double x0 = fma(xs[1] - k_beta, ts.lnT, xs[0] - k_lnA) - (xs[2] - k_Ta) * ts.invT;
            rate_constants(kc, ts, kf, kr);
            k0kf = ck_exp(x0);
            const double e3 = ck_exp(a3), e1 = ck_exp(a1), e2x = ck_exp(a2);
            const double aa = xs[3];
            double Fc = fma(1.0 - aa, e3, aa * e1);
            Fc = (T2 >= 0.0) ? Fc + e2x : Fc;
            lF = ck_log(fmax(Fc, 1e-300)) * 0.43429448190325182765;
            cc = fma(-0.67, lF, -0.4);
            nn = fma(-1.27, lF, 0.75);
          } else if (fo) {
            ts.lnT = ck_log(T);
            const double x0 = fma(xs[1] - k_beta, ts.lnT, xs[0] - k_lnA) - (xs[2] - k_Ta) * ts.invT;
            rate_constants(kc, ts, kf, kr);
            k0kf = ck_exp(x0);
          } else {
            ts.lnT = ck_log(T);
            rate_constants(kc, ts, kf, kr);
          }
        } else {
          int ti = 0;
#pragma unroll
          for (int e = 0; e < MAX_TINT - 1; ++e) ti += (e < m.nT - 1 && T > m.tedge[e]) ? 1 : 0;
          ts.tint = ti;
          ts.lnT = ck_log(T);
        }
        __syncthreads();   // #1: C, H, scalars
        if (warp != 0) {
          double hq = 0.0;
          if (on) {
            double ci = 1.0;
            if (tb) {
              double M = sc[1];
              const unsigned long long xw = (unsigned long long)__double_as_longlong(xs[7]);
              const int ne = (int)(xw & 15ull);
              if (ne != 15) {
#pragma unroll
                for (int e = 0; e < 6; ++e) {
                  const bool in = e < ne;
                  M = fma(in ? xs[8 + e] : 0.0, C[in ? (int)((xw >> (4 + 10 * e)) & 1023ull) : K], M);
                }
              } else {
                const int j = rr - m.r_tb;
                for (int e = __ldg(m.eptr + j), e1 = __ldg(m.eptr + j + 1); e < e1; ++e)
                  M = fma(__ldg(m.eval1 + e), C[__ldg(m.espec + e)], M);
              }
              if (troe) {
                const double Pr = k0kf * M;
                const double L = Pr * ck_rcp(1.0 + Pr);
                const double lP = ck_log(fmax(Pr, 1e-300)) * 0.43429448190325182765;
                const double x = lP + cc;
                const double den = fma(-0.14, x, nn);
                const double den2 = den * den;
                const double g = den2 * ck_rcp(fma(x, x, den2));
                ci = L * ck_exp(2.30258509299404568402 * lF * g);
              } else if (fo) {
                const double Pr = k0kf * M;
                ci = Pr * ck_rcp(1.0 + Pr);
              } else {
                ci = M;
              }
            }
            const double pf = C[sl[0]] * C[sl[1]] * C[sl[2]];
            const double pr = C[sl[3]] * C[sl[4]] * C[sl[5]];
            const double qi = ci * (kf * pf - kr * pr);
            q[rr] = qi;
            const double dH = (H[sl[3]] + H[sl[4]] + H[sl[5]]) - (H[sl[0]] + H[sl[1]] + H[sl[2]]);
            hq = qi * dH;
          } else if (!one) {   // larger models: every reaction thread walks its share with the common evaluation
            for (int r2 = r0; r2 < R; r2 += RT) {
              const RxnConst k2 = load_rxn_global(m, r2, ts.tint);
              const double qi = reaction_q<1, false>(m, r2, k2, ts, C, sc[1], nullptr);
              q[r2] = qi;
              const double dH = (H[k2.slot[3]] + H[k2.slot[4]] + H[k2.slot[5]]) - (H[k2.slot[0]] + H[k2.slot[1]] + H[k2.slot[2]]);
              hq = fma(qi, dH, hq);
            }
          }
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) hq += __shfl_xor_sync(0xffffffffu, hq, o);
          if (lane == 0) red[warp] = hq;
        } else if (s == 0) {
          // ---- warp 0 is idle here: the pending step-size update and the guards of Algorithm 1 ----
          if (pend) {
            // err = sqrt(es / N); 0.9 err^(-1/5) = 0.9 exp(-0.1 ln(es / N)), clamped below at err = 1e-10
            const double fac = isfinite(err_prev) ? 0.9 * ck_exp(-0.1 * ck_log(fmax(err_prev / N, 1e-20))) : 0.2;
            hn = hn * (acc_prev ? fmin(fac_max, fmax(0.2, fac)) : fmin(1.0, fmax(0.2, fac)));
            fac_max = acc_prev ? 5.0 : 1.0;
            pend = false;
          }
          int go = 1;
          if (!isfinite(hn)) { status = CK_ST_NONFINITE; go = 0; }
          else if (hn < 1e-12 * a.dt) { status = CK_ST_H_UNDERFLOW; go = 0; }
          last = false;
          if (go && hn >= a.dt - t) { hn = a.dt - t; last = true; }
          if (lane == 0) { sc[3] = hn; sc[4] = (double)go; }
        }
        __syncthreads();   // #2: q, red (and, in evaluation 0, h)
        // ---- production rates ----------------------------------------------------------------------------------------
        double* Fs = F + s * N;
        {
          double w0 = 0.0, w1 = 0.0, w2 = 0.0;
          if (gfit) {
#pragma unroll
            for (int x = 0; x < WIDE_GE; x += 3) {
              w0 = fma(gn[x], q[gi[x]], w0);
              if (x + 1 < WIDE_GE) w1 = fma(gn[x + 1], q[gi[x + 1]], w1);
              if (x + 2 < WIDE_GE) w2 = fma(gn[x + 2], q[gi[x + 2]], w2);
            }
          } else if (gk < K) {
            int e = s_tptr[gk] + gpart;
            const int e1 = s_tptr[gk + 1];
            for (; e + QS < e1; e += 2 * QS) {   // two independent chains
              const int en0 = s_tent[e], en1 = s_tent[e + QS];
              w0 = fma((double)((en0 & 255) - 128), q[en0 >> 8], w0);
              w1 = fma((double)((en1 & 255) - 128), q[en1 >> 8], w1);
            }
            if (e < e1) { const int en0 = s_tent[e]; w0 = fma((double)((en0 & 255) - 128), q[en0 >> 8], w0); }
          }
          double w = (w0 + w1) + w2;
          if (QS >= 2) w += __shfl_xor_sync(0xffffffffu, w, 1);
          if (QS >= 4) w += __shfl_xor_sync(0xffffffffu, w, 2);
          if (gk < K && gpart == 0) Fs[1 + gk] = w * gW * sc[2];
        }
        if (tid == G - 1) {   // the temperature equation (Eq. 9): -T sum_k h_k omega_k / (rho c_p)
          double hw = 0.0;
#pragma unroll
          for (int x = 1; x < NW; ++x) hw += red[x];
          Fs[0] = sc[0] * hw;
        }
        if (s == 0) { h = sc[3]; stop = sc[4] == 0.0; }
        __syncthreads();   // #3: F[s]
        if (stop) break;
      }
      if (stop) break;
      // ---- candidate, error norm, accept / reject: warp 0 (Algorithm 1) -----------------------------
      if (warp == 0) {
        double es = 0.0, yn[4];
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          const int i0 = lane + 32 * x;
          yn[x] = 0.0;
          if (32 * x < N) {   // warp-uniform
            const int i = min(i0, N - 1);
            double yb = 0.0, eb = 0.0;
#pragma unroll
            for (int j = 0; j < 6; ++j) { const double k = F[j * N + i]; yb = fma(RKF_T[5][j], k, yb); eb = fma(RKF_T[6][j], k, eb); }
            const double y0 = Y[i];
            yn[x] = fma(h, yb, y0);
            const double w = (h * eb) * ck_rcp(fma(a.rtol, fmax(fabs(y0), fabs(yn[x])), a.atol));
            es = (i0 < N) ? fma(w, w, es) : es;
          }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) es += __shfl_xor_sync(0xffffffffu, es, o);
        // err = sqrt(es / N) < 1 decides; the square root itself waits for the step-size update
        h_used = h;
        err_prev = es; pend = true;
        acc_prev = isfinite(es) && es < (double)N;
        if (acc_prev) {
#pragma unroll
          for (int x = 0; x < 4; ++x) { const int i = lane + 32 * x; if (i < N) Y[i] = yn[x]; }
          t = last ? a.dt : t + h;
          nacc++;
        } else {
          nrej++;
          if (!isfinite(es))   // some evaluation was not finite: it must not meet a zero coefficient in the next attempt
            for (int i = lane; i < 6 * N; i += 32) F[i] = 0.0;
        }
        int go = t < a.dt;
        if (go && nacc + nrej >= a.max_steps) { status = CK_ST_MAX_STEPS; go = 0; }
        if (lane == 0) sc[5] = (double)go;
      }
      c_rhs += 6;
    }
    __syncthreads();
    for (int i = tid; i < N; i += G) a.y[(size_t)i * a.ld + r] = Y[i];
    if (tid == 0) {
      if (a.n_accept) a.n_accept[r] = nacc;
      if (a.n_reject) a.n_reject[r] = nrej;
      if (a.status) a.status[r] = status;
      if (a.h_last) a.h_last[r] = h_used;
      a.att[r] = nacc + nrej;
      c_att += nacc + nrej; c_acc += nacc; c_rej += nrej; c_fail += (status != CK_ST_OK);
    }
  }
  if (tid == 0) {
    atomicAdd(&a.stats->rhs_evals, c_rhs); atomicAdd(&a.stats->attempts, c_att);
    atomicAdd(&a.stats->accepted, c_acc); atomicAdd(&a.stats->rejected, c_rej);
    atomicAdd(&a.stats->failed, c_fail);
  }
}

}  // namespace ck
