// Thread-per-reactor analytic Jacobian (rows of the species equations), the Jacobian of the batched ROS4 rounds
// (ck_ros_rounds.cu) and of ck_jac on large batches.
//
// The paper only cites an analytic Jacobian; the formulas are derived from Eq. 12-19 in
// DESIGN.md "Analytic Jacobian" (same ones as ck_coop.cuh).  Mapping: one thread owns one reactor, like ck_rhs, so the
// reaction constants are warp-uniform and every HBM access of the batch arrays is coalesced.  Two per-thread arrays
// with data-dependent (warp-uniform) indices are needed: the concentrations C_k (shared-memory columns) and ONE row of
// the matrix at a time (tensor memory, 2 x 32-bit columns per entry -- the same tcgen05.ld/st pattern as the production
// rate accumulators of ck_rhs_tmem.cuh, whose columns this kernel reuses).
//
//   phase A  f(y) as in ck_rhs, with the derivative pieces of every reaction written to a scratch array G2 that is
//            component-major over the slots (coalesced):  g_f = c_i k_f, g_r = c_i k_r, s_i = sum_m dq_i/dC_m C_m,
//            theta_i = dq_i/dT|_C - s_i / T (the total temperature derivative at constant p and Y), and for
//            third-body / falloff rows dq_i/d[M]_i.
//   phase B  gather form, one species row k at a time (the transposed stoichiometry tptr/tent lists the reactions of
//            species k): row_k[j] += nu_ki dq_i/dC_j with dq_i/dC_slot = g_f prod(other reactant C) resp.
//            -g_r prod(other product C) rebuilt from G2 and the C columns; the scalars sigma_k, tau_k and the dense
//            third-body coefficient ride along; then the chain rule at constant p turns the row into d f_k / d y and
//            the row leaves the chip once.  No atomics, no global read-modify-write.
//   The temperature ROW is a linear combination of the species rows (differentiate sum_k h_k f_k + c_p f_T = 0, the
//   identity that pins reading G2 of Eq. 13):
//       d f_T/d y_j = - sum_k hh_k J_kj - f_T cc_j            hh_k = h_k / c_p,  cc_j = c_p,j / c_p  (mass units)
//       d f_T/d T   = - sum_k hh_k J_kT - sum_k f_k cc_k - f_T (sum_k Y_k c_p,k') / c_p
//   so this kernel emits hh, cc and the last two terms (HC array) and whoever holds all rows finishes row 0: the LU
//   kernel of the ROS4 rounds while it loads the matrix, or jac_trow_kernel for ck_jac.
#pragma once
#include "ck_rhs_tmem.cuh"

namespace ck {

// positions of one matrix row in tensor memory: 0 = temperature column, 1 + j = species j, 1 + K = sink of the dummy
// species; padded to a multiple of four so that rows leave in 32-byte pieces
__host__ __device__ inline int jac_npt(int K) { return (K + 2 + 3) & ~3; }
// leading dimension of a reactor-major row (N entries padded to a multiple of four doubles)
__host__ __device__ inline int jac_np(int N) { return (N + 3) & ~3; }
// doubles per slot of the scratch array G2 / of the HC array
__host__ __device__ inline int jac_g2_rows(int R, int r_tb) { return 4 * R + (R - r_tb); }
__host__ __device__ inline int jac_hc_rows(int K) { return 2 * K + 1; }
// shared memory: C columns | staging buffer of phase A, aliased in phase B by its tables: W, 1/W, one packed slot word
// per reaction, the transposed stoichiometry tent[] and its row pointers (reloaded per batch of reactors: a few KB)
__host__ __device__ inline size_t jac_tables_doubles(int K, int R, int n_tent) {
  return (size_t)2 * K + (size_t)R + (((size_t)n_tent + K + 2 + 1) >> 1);
}
__host__ __device__ inline size_t jac_tpr_smem_bytes(int K, int R, int n_tent, int rstride, int block) {
  const size_t st = (size_t)rhs_stage_doubles(rstride), tb = jac_tables_doubles(K, R, n_tent);
  return ((size_t)(K + 1) * block + (st > tb ? st : tb)) * sizeof(double);
}
// CTA width for which both the C columns (shared memory) and the row buffer (tensor memory, one column set per group
// of four warps) fit; 0 if the mechanism is too large for this kernel
inline int jac_tpr_block(const MechDev& m) {
  const int npt = jac_npt(m.K);
  if (4 * 2 * npt <= 512 && jac_tpr_smem_bytes(m.K, m.R, m.n_tent, m.rstride, 512) <= 227 * 1024) return 512;
  if (2 * 2 * npt <= 512 && jac_tpr_smem_bytes(m.K, m.R, m.n_tent, m.rstride, 224) <= 227 * 1024) return 224;
  return 0;
}

__device__ __forceinline__ void tm_ld8(uint32_t taddr, double (&v)[4]) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr));
  tm_wait_ld();
#pragma unroll
  for (int x = 0; x < 4; ++x) v[x] = __hiloint2double((int)r[2 * x + 1], (int)r[2 * x]);
}
__device__ __forceinline__ void tm_zero8(uint32_t taddr) {
  const uint32_t z = 0u;
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %1, %1, %1, %1, %1, %1, %1};" ::"r"(taddr), "r"(z));
}

__device__ __forceinline__ double thermo_row_dcp(const double* __restrict__ row, const TState& t) {
  const double* a = row + ((t.T > row[2]) ? 9 : 4);
  const double T = t.T;
  return fma(fma(fma(4.0 * a[4], T, 3.0 * a[3]), T, 2.0 * a[2]), T, a[1]);
}

// phase-B tables in shared memory (filled once per CTA)
struct JacTables {
  const unsigned long long* slotw;  // [R] six 10-bit slots; bit 63: a species in two slots; bit 62: A + B <=> C + D shaped
  const int* tptr;                  // [K + 1]
  const int* tent;                  // [n_tent]
};

struct JacOut {
  double* f;        // [N][ldf]  f(y)
  long long ldf;
  double* J;        // reactor-major: J[slot * sstride + i * ldr + j]; component-major: J[(i * N + j) * ldJ + slot]; rows 1..K
  long long ldJ;
  int ldr;          // reactor-major only: row stride (>= N rounded up to a multiple of four) ...
  long long sstride;  // ... and doubles per slot
  double* hc;       // [2K + 1][ldh]  hh_k, cc_k, and the constant of d f_T / d T
  long long ldh;
  double* g2;       // [jac_g2_rows][ldg] scratch (indexed by thread)
  long long ldg;
  const int* list;  // null: thread i works on column i; else on column list[i] of y / p / f / hc / J
};

// phase A for one row of kind TYPE: rate of progress with derivative pieces, omega scatter, G2 stores
template <int BLOCK, int TYPE>
__device__ __forceinline__ void jac_phaseA_row(const MechDev& m, int r, const double* __restrict__ row, const double* __restrict__ xrow,
                                               const TState& t, const double* __restrict__ Cs, double Ctot, uint32_t wt,
                                               double* __restrict__ g2, long long ldg, bool store) {
  const RxnConst kc = load_rxn_row(row, t.tint);
  RateAux a;
  const double q = reaction_q<BLOCK, true, TYPE>(m, r, kc, t, Cs, Ctot, &a, xrow);
  slow_scatter_tmem(kc, q, m.K, wt);
  const double ff = a.kf * a.pf, rr = a.kr * a.pr, net = ff - rr;
  const int K = m.K;
  const int nf = (kc.slot[0] != K) + (kc.slot[1] != K) + (kc.slot[2] != K);
  const int nr = (kc.slot[3] != K) + (kc.slot[4] != K) + (kc.slot[5] != K);
  // s_i = sum_m dq_i/dC_m C_m: every real reactant slot contributes c_i k_f prod_f, every product slot -c_i k_r prod_r
  double si = a.ci * ((double)nf * ff - (double)nr * rr);
  double dqT = a.ci * (ff * a.dlnkf_dT - rr * a.dlnkr_dT) + a.dci_dT * net;
  if (TYPE >= 1) {
    const double dM = a.dci_dM * net;
    si = fma(dM, a.M, si);
    if (store) g2[(size_t)(4 * m.R + (r - m.r_tb)) * ldg] = dM;
  }
  if (store) {
    g2[(size_t)(4 * r) * ldg] = a.ci * a.kf;
    g2[(size_t)(4 * r + 1) * ldg] = a.ci * a.kr;
    g2[(size_t)(4 * r + 2) * ldg] = si;
    g2[(size_t)(4 * r + 3) * ldg] = m.cv ? dqT : fma(-si, t.invT, dqT);   // d C_m / d T = 0 at constant volume
  }
}

// RM: reactor-major output of the NEGATED species rows (row stride o.ldr, o.sstride doubles per slot), else component-major J.  MUST be called by every thread of the CTA.
// yin / out pointers are pre-offset to this thread's slot (component-major arrays) resp. reactor (Jrm).
template <int BLOCK, bool RM>
__device__ __forceinline__ void jac_thread_tmem(const MechDev& m, const double* __restrict__ yin, long long ldin, double p,
                                                const JacOut& o, long long slot, long long gslot, double* __restrict__ Cs, uint32_t wt,
                                                double* __restrict__ stage, bool store, int part = 0, int nsub = 1) {
  const int K = m.K, R = m.R, rs = m.rstride, N = K + 1;
  const int tid = threadIdx.x;
  const TState t = make_tstate(m, yin[0]);
  double* const fout = o.f + slot;
  double* const g2 = o.g2 + gslot;   // the scratch is indexed by thread, the outputs by column
  double* const hc = o.hc + slot;
  // ---- phase A: f(y) (as rhs_thread_tmem) ----------------------------------------------------------------------
  double S = 0.0, cps = 0.0, dcp = 0.0;
  for (int k0 = 0; k0 < K; k0 += RHS_CHUNK) {
    const int nk = min(RHS_CHUNK, K - k0);
    __syncthreads();
    for (int idx = tid; idx < nk * SPS; idx += BLOCK) stage[idx] = __ldg(m.spack + (size_t)k0 * SPS + idx);
    __syncthreads();
#pragma unroll 4
    for (int j = 0; j < nk; ++j) {
      const double* row = stage + j * SPS;
      const double yw = yin[(size_t)(k0 + j + 1) * ldin] * row[1];
      S += yw;
      cps = fma(yw, thermo_row_cp(row, t), cps);
      dcp = fma(yw, thermo_row_dcp(row, t), dcp);
      Cs[(k0 + j) * BLOCK] = yw;
      tm_st2(wt + 2 * (k0 + j), 0.0);
    }
  }
  const double rho = m.cv ? p : (p / (R_U * t.T)) / S;   // constant volume (m.cv): `p` is the density
  const double Ctot = m.cv ? rho * S : p / (R_U * t.T);
  const double sub = m.cv ? 1.0 : 0.0, sg = m.cv ? 0.0 : 1.0;   // see jac_coop_finish (ck_coop.cuh)
#pragma unroll 4
  for (int k = 0; k < K; ++k) Cs[k * BLOCK] *= rho;
  Cs[K * BLOCK] = 1.0;
  tm_st2(wt + 2 * K, 0.0);
  tm_wait_st();
  double* xstage = stage + RHS_CHUNK * (rs > 16 ? rs : 16);
  for (int r0 = 0; r0 < R; r0 += RHS_CHUNK) {
    const int nr = min(RHS_CHUNK, R - r0);
    const double* src = m.rpack + (size_t)r0 * rs;
    const int x0 = max(r0, m.r_tb);
    const int nx = max(0, r0 + nr - x0);
    __syncthreads();
    for (int idx = tid; idx < nr * rs; idx += BLOCK) stage[idx] = __ldg(src + idx);
    for (int idx = tid; idx < nx * 16; idx += BLOCK) xstage[idx] = __ldg(m.xpack + (size_t)(x0 - m.r_tb) * 16 + idx);
    __syncthreads();
    const int j1 = min(nr, max(0, m.r_tb - r0)), j2 = min(nr, max(0, m.r_lind - r0)), j3 = min(nr, max(0, m.r_troe - r0));
    const double* xs = xstage - (size_t)(x0 - r0) * 16;
    int j = 0;
    for (; j < j1; ++j) jac_phaseA_row<BLOCK, 0>(m, r0 + j, stage + j * rs, xs, t, Cs, Ctot, wt, g2, o.ldg, store);
    for (; j < j2; ++j) jac_phaseA_row<BLOCK, 1>(m, r0 + j, stage + j * rs, xs + 16 * j, t, Cs, Ctot, wt, g2, o.ldg, store);
    for (; j < j3; ++j) jac_phaseA_row<BLOCK, 2>(m, r0 + j, stage + j * rs, xs + 16 * j, t, Cs, Ctot, wt, g2, o.ldg, store);
    for (; j < nr; ++j) jac_phaseA_row<BLOCK, 3>(m, r0 + j, stage + j * rs, xs + 16 * j, t, Cs, Ctot, wt, g2, o.ldg, store);
  }
  const double irho = 1.0 / rho, icps = 1.0 / (cps - sub * S);   // c_v / R = c_p / R - S at constant volume
  double hw = 0.0;
  for (int k0 = 0; k0 < K; k0 += RHS_CHUNK) {
    const int nk = min(RHS_CHUNK, K - k0);
    __syncthreads();
    for (int idx = tid; idx < nk * SPS; idx += BLOCK) stage[idx] = __ldg(m.spack + (size_t)k0 * SPS + idx);
    __syncthreads();
    for (int j = 0; j < nk; ++j) {
      const double* row = stage + j * SPS;
      double w;
      tm_ld2(wt + 2 * (k0 + j), w);
      tm_wait_ld();
      const double hrt = thermo_row_h(row, t) - sub;
      hw = fma(hrt, w, hw);
      if (store) {
        fout[(size_t)(k0 + j + 1) * o.ldf] = w * row[0] * irho;
        hc[(size_t)(k0 + j) * o.ldh] = t.T * hrt * row[1] * icps;            // hh_k = T (H_k/RT) / (W_k cps)
        hc[(size_t)(K + k0 + j) * o.ldh] = (thermo_row_cp(row, t) - sub) * row[1] * icps;  // cc_k = (cp_k/R) / (W_k cps)
      }
    }
  }
  const double fT = -(t.T * hw) * irho * icps;
  if (store) fout[0] = fT;
  // ---- phase B: species rows ------------------------------------------------------------------------------------
  __syncthreads();
  double* sW = stage;        // [K] W_k
  double* siW = stage + K;   // [K] 1 / W_k
  for (int k = tid; k < K; k += BLOCK) { sW[k] = __ldg(m.W + k); siW[k] = __ldg(m.invW + k); }
  JacTables tb;
  {
    unsigned long long* slotw = reinterpret_cast<unsigned long long*>(stage + 2 * K);
    int* tptr = reinterpret_cast<int*>(slotw + R);
    int* tent = tptr + K + 1;
    for (int i = tid; i < R; i += BLOCK) {
      unsigned long long w = (unsigned long long)__double_as_longlong(__ldg(m.rpack + (size_t)i * rs + 3));
      const unsigned s2 = (unsigned)(w >> 20) & 1023u, s5 = (unsigned)(w >> 52) & 1023u;
      w &= ~(1ull << 62);
      if (i < m.r_tb && s2 == (unsigned)K && s5 == (unsigned)K && !(w >> 63)) w |= 1ull << 62;   // plain rows only
      slotw[i] = w;
    }
    for (int i = tid; i <= K; i += BLOCK) tptr[i] = __ldg(m.tptr + i);
    for (int i = tid; i < m.n_tent; i += BLOCK) tent[i] = __ldg(m.tent + i);
    tb.slotw = slotw; tb.tptr = tptr; tb.tent = tent;
  }
  const int npt = jac_npt(K);
  for (int c = 0; c < npt; c += 4) tm_zero8(wt + 2 * c);
  tm_wait_st();
  __syncthreads();
  const double iS = 1.0 / S;
  const int NP = jac_np(N);
  double sfc = 0.0;  // sum_k f_k cc_k
  constexpr int CB = BLOCK * 8;  // bytes between C columns
  const char* Cb = reinterpret_cast<const char*>(Cs);
  // nsub > 1: this thread is one of nsub that work on the SAME reactor (each ran phase A in full, on its own columns and
  // scratch, and wrote the same f / hc values); the species rows are dealt out round-robin
  for (int k = part; k < K; k += nsub) {
    double sig = 0.0, tht = 0.0, dns = 0.0;
    const int e0 = tb.tptr[k], e1 = tb.tptr[k + 1];
    // software pipeline: the scratch values of entry e + 1 are in flight while entry e is processed
    int en = (e0 < e1) ? tb.tent[e0] : 0;
    double gf = 0.0, gr = 0.0, si = 0.0, th = 0.0;
    if (e0 < e1) {
      const size_t og = (size_t)(4 * (en >> 8)) * o.ldg;
      gf = g2[og]; gr = g2[og + o.ldg]; si = g2[og + 2 * o.ldg]; th = g2[og + 3 * o.ldg];
    }
    for (int e = e0; e < e1; ++e) {
      const int i = en >> 8;
      const double nu = (double)((en & 255) - 128);
      const double cgf = gf, ngr = -gr;
      sig = fma(nu, si, sig);
      tht = fma(nu, th, tht);
      if (e + 1 < e1) {
        en = tb.tent[e + 1];
        const size_t og = (size_t)(4 * (en >> 8)) * o.ldg;
        gf = g2[og]; gr = g2[og + o.ldg]; si = g2[og + 2 * o.ldg]; th = g2[og + 3 * o.ldg];
      }
      const unsigned long long sw = tb.slotw[i];
      const unsigned lo = (unsigned)sw, hi = (unsigned)(sw >> 32);
      const unsigned s0 = lo & 1023u, s1 = (lo >> 10) & 1023u, s3 = hi & 1023u, s4 = (hi >> 10) & 1023u;
      if (hi & 0x40000000u) {  // A + B <=> C + D shaped row (third slots empty, species distinct): four entries
        const double c0 = *reinterpret_cast<const double*>(Cb + s0 * CB), c1 = *reinterpret_cast<const double*>(Cb + s1 * CB);
        const double c3 = *reinterpret_cast<const double*>(Cb + s3 * CB), c4 = *reinterpret_cast<const double*>(Cb + s4 * CB);
        uint32_t rl[4], rh[4];
        const uint32_t t0 = wt + 2 + 2 * s0, t1 = wt + 2 + 2 * s1, t3 = wt + 2 + 2 * s3, t4 = wt + 2 + 2 * s4;
        tm_ld2_raw(t0, rl[0], rh[0]); tm_ld2_raw(t1, rl[1], rh[1]); tm_ld2_raw(t3, rl[2], rh[2]); tm_ld2_raw(t4, rl[3], rh[3]);
        const double d0 = nu * (cgf * c1), d1 = nu * (cgf * c0), d3 = nu * (ngr * c4), d4 = nu * (ngr * c3);
        tm_wait_ld();
        tm_st2(t0, d0 + __hiloint2double((int)rh[0], (int)rl[0]));
        tm_st2(t1, d1 + __hiloint2double((int)rh[1], (int)rl[1]));
        tm_st2(t3, d3 + __hiloint2double((int)rh[2], (int)rl[2]));
        tm_st2(t4, d4 + __hiloint2double((int)rh[3], (int)rl[3]));
        tm_wait_st();
        continue;
      }
      const unsigned s2 = (lo >> 20) & 1023u, s5 = (hi >> 20) & 1023u;
      const unsigned sl[6] = {s0, s1, s2, s3, s4, s5};
      double c[6];
#pragma unroll
      for (int x = 0; x < 6; ++x) c[x] = *reinterpret_cast<const double*>(Cb + sl[x] * CB);
      const double d[6] = {cgf * (c[1] * c[2]), cgf * (c[0] * c[2]), cgf * (c[0] * c[1]),
                           ngr * (c[4] * c[5]), ngr * (c[3] * c[5]), ngr * (c[3] * c[4])};
      if (i >= m.r_tb) {  // third-body / falloff row: dense coefficient + the listed efficiencies
        const int jx = i - m.r_tb;
        const double ndM = nu * g2[(size_t)(4 * R + jx) * o.ldg];
        dns += ndM;
        const double* xr = m.xpack + (size_t)jx * 16;
        const unsigned long long xw = (unsigned long long)__double_as_longlong(__ldg(xr + 7));
        const int ne = (int)(xw & 15ull);
        if (ne != 15) {
          for (int z = 0; z < ne; ++z) {
            const uint32_t col = wt + 2 * (1 + (int)((xw >> (4 + 10 * z)) & 1023ull));
            double w;
            tm_ld2(col, w);
            tm_wait_ld();
            tm_st2(col, fma(ndM, __ldg(xr + 8 + z), w));
            tm_wait_st();
          }
        } else {
          for (int z = __ldg(m.eptr + jx), z1 = __ldg(m.eptr + jx + 1); z < z1; ++z) {
            const uint32_t col = wt + 2 * (1 + __ldg(m.espec + z));
            double w;
            tm_ld2(col, w);
            tm_wait_ld();
            tm_st2(col, fma(ndM, __ldg(m.eval1 + z), w));
            tm_wait_st();
          }
        }
      }
      if (!(hi >> 31)) {
        uint32_t rl[6], rh[6];
#pragma unroll
        for (int x = 0; x < 6; ++x) tm_ld2_raw(wt + 2 * (1 + sl[x]), rl[x], rh[x]);
        tm_wait_ld();
#pragma unroll
        for (int x = 0; x < 6; ++x) tm_st2(wt + 2 * (1 + sl[x]), fma(nu, d[x], __hiloint2double((int)rh[x], (int)rl[x])));
        tm_wait_st();
      } else {
#pragma unroll
        for (int x = 0; x < 6; ++x) {
          double w;
          tm_ld2(wt + 2 * (1 + sl[x]), w);
          tm_wait_ld();
          tm_st2(wt + 2 * (1 + sl[x]), fma(nu, d[x], w));
          tm_wait_st();
        }
      }
    }
    // chain rule at constant p: J_kj = (W_k / W_j)(G_kj + dns_k) + (f_k - W_k sig_k / rho) / (S W_j)
    //                           J_kT = (W_k / rho) Theta_k + f_k / T,  Theta_k = sum_i nu_ki theta_i
    const double Wk = sW[k];
    const double fk = store ? fout[(size_t)(1 + k) * o.ldf] : 0.0;
    const double beta = fma(Wk, dns, sg * (fk - Wk * irho * sig) * iS);
    const double JkT = fma(Wk * irho, tht, sg * fk * t.invT);
    if (store) sfc = fma(fk, hc[(size_t)(K + k) * o.ldh], sfc);
    double* const rowbase = RM ? o.J + (size_t)(1 + k) * o.ldr : nullptr;
    // odd row stride (the LU's shared-memory image): every other row starts 8 bytes off a 16-byte boundary
    const bool odd_row = RM && (o.ldr & 1) && ((1 + k) & 1);
    double carry = 0.0;
    for (int c0 = 0; c0 < NP; c0 += 4) {
      double v[4];
      tm_ld8(wt + 2 * c0, v);
      tm_zero8(wt + 2 * c0);
#pragma unroll
      for (int x = 0; x < 4; ++x) {
        const int cidx = c0 + x;  // position: 0 = T column, 1 + j = species j
        const int j = min(max(cidx - 1, 0), K - 1);
        v[x] = (cidx == 0) ? JkT : ((cidx <= K) ? siW[j] * fma(Wk, v[x], beta) : 0.0);
      }
      if (store) {
        if (RM) {  // rows of -J (what the factorisation of I/(h gamma) - J starts from), in the row stride of the LU's image
          double* dst = rowbase + c0;
          if (!odd_row) {
            reinterpret_cast<double2*>(dst)[0] = make_double2(-v[0], -v[1]);
            reinterpret_cast<double2*>(dst)[1] = make_double2(-v[2], -v[3]);
          } else {  // row starts 8 bytes off a 16-byte boundary: pair the last element of a piece with the first of the next
            if (c0 == 0) dst[0] = -v[0];
            else *reinterpret_cast<double2*>(dst - 1) = make_double2(carry, -v[0]);
            *reinterpret_cast<double2*>(dst + 1) = make_double2(-v[1], -v[2]);
          }
          carry = -v[3];
        } else {
#pragma unroll
          for (int x = 0; x < 4; ++x)
            if (c0 + x < N) o.J[((size_t)(1 + k) * N + c0 + x) * o.ldJ] = v[x];
        }
      }
    }
    if (store && odd_row) rowbase[NP - 1] = carry;
    tm_wait_st();
  }
  if (nsub > 1) {   // the sum runs over ALL rows: redo it from this thread's own phase-A outputs
    sfc = 0.0;
    if (store && part == 0)
      for (int k = 0; k < K; ++k) sfc = fma(fout[(size_t)(1 + k) * o.ldf], hc[(size_t)(K + k) * o.ldh], sfc);
  }
  if (store && part == 0) hc[(size_t)(2 * K) * o.ldh] = -sfc - fT * dcp * icps;
}

// One CTA per SM, persistent over batches of BLOCK slots (as rhs_kernel_tmem).  n_dev (optional) overrides n with a
// device-side count (the active-list length of the ROS4 rounds).
template <int BLOCK, bool RM>
__global__ void __launch_bounds__(BLOCK, 1) jac_rows_kernel(const MechDev m, long long n, const int* __restrict__ n_dev,
                                                            const double* __restrict__ y, long long ld,
                                                            const double* __restrict__ p, JacOut o, const int nsub = 1) {
  extern __shared__ double sm[];
  __shared__ uint32_t s_tmem;
  if (n_dev) n = *n_dev;
  const int tid = threadIdx.x, warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  if (warp == 0) {
    const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&s_tmem);
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(dst));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tbase = s_tmem;
  const uint32_t wt = tbase + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 2 * jac_npt(m.K));
  double* Cs = sm + tid;
  double* stage = sm + (size_t)(m.K + 1) * BLOCK;
  // nsub threads per reactor (the caller picks nsub > 1 when the batch leaves lanes idle: the kernel's duration is one
  // thread's latency, most of it the K species rows, whatever the count).  The parts are dealt out by WARP (threads
  // [g BLOCK / nsub, (g + 1) BLOCK / nsub) take part g): the tensor-memory accesses are warp-collective, so the lanes of a
  // warp must walk the same rows.  nsub must divide BLOCK / 32.
  const int per = BLOCK / nsub;                 // reactors per CTA pass
  const int part = tid / per, local = tid - part * per;
  for (long long b = blockIdx.x; b * per < n; b += gridDim.x) {
    const long long r = b * per + local;
    const bool act = r < n;
    const long long rr = act ? r : n - 1;
    const long long gs = (long long)part * n + rr;   // scratch column of this thread: dense per part, < nsub * n
    const long long col = o.list ? (long long)o.list[rr] : rr;   // which column of y / p / f / hc / J this thread works on
    JacOut oo = o;
    if (RM) oo.J = o.J + (size_t)col * o.sstride;
    else oo.J = o.J + col;
    jac_thread_tmem<BLOCK, RM>(m, y + col, ld, p[col], oo, col, gs, Cs, wt, stage, act, part, nsub);
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tbase));
}

// Row 0 of a component-major Jacobian from its species rows (see the header): one thread per reactor.
static __global__ void __launch_bounds__(128) jac_trow_kernel(int K, long long n, const double* __restrict__ f, long long ldf,
                                                       const double* __restrict__ hc, long long ldh, double* __restrict__ J,
                                                       long long ldJ) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  const int N = K + 1;
  const double fT = f[r];
  for (int c = 0; c < N; ++c) {
    double acc = 0.0;
    for (int k = 0; k < K; ++k) acc = fma(hc[(size_t)k * ldh + r], J[((size_t)(1 + k) * N + c) * ldJ + r], acc);
    J[(size_t)c * ldJ + r] = (c == 0) ? (hc[(size_t)(2 * K) * ldh + r] - acc) : -acc - fT * hc[(size_t)(K + c - 1) * ldh + r];
  }
}

}  // namespace ck
