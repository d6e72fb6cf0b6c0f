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
//            component-major over the slots (coalesced):  g_f = c_i k_f, g_r = c_i k_r, dq_i/dT|_C, and for third-body /
//            falloff rows dq_i/d[M]_i and dq_i/d[M]_i [M]_i.
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
__host__ __device__ inline int jac_g2_rows(int R, int r_tb) { return 3 * R + 2 * (R - r_tb); }
__host__ __device__ inline int jac_hc_rows(int K) { return 2 * K + 1; }
__host__ __device__ inline size_t jac_tpr_smem_bytes(int K, int rstride, int block) {
  const size_t st = (size_t)rhs_stage_doubles(rstride);
  return ((size_t)(K + 1) * block + (st > (size_t)2 * K ? st : (size_t)2 * K)) * sizeof(double);
}
// CTA width for which both the C columns (shared memory) and the row buffer (tensor memory, one column set per group
// of four warps) fit; 0 if the mechanism is too large for this kernel
inline int jac_tpr_block(int K, int rstride) {
  const int npt = jac_npt(K);
  if (4 * 2 * npt <= 512 && jac_tpr_smem_bytes(K, rstride, 512) <= 227 * 1024) return 512;
  if (2 * 2 * npt <= 512 && jac_tpr_smem_bytes(K, rstride, 224) <= 227 * 1024) return 224;
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

struct JacOut {
  double* f;        // [N][ldf]  f(y)
  long long ldf;
  double* J;        // reactor-major: J[slot * N * NP + i * NP + j]; component-major: J[(i * N + j) * ldJ + slot]; rows 1..K
  long long ldJ;
  double* hc;       // [2K + 1][ldh]  hh_k, cc_k, and the constant of d f_T / d T
  long long ldh;
  double* g2;       // [jac_g2_rows][ldg] scratch
  long long ldg;
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
  if (store) {
    g2[(size_t)(3 * r) * ldg] = a.ci * a.kf;
    g2[(size_t)(3 * r + 1) * ldg] = a.ci * a.kr;
    g2[(size_t)(3 * r + 2) * ldg] = a.ci * (ff * a.dlnkf_dT - rr * a.dlnkr_dT) + a.dci_dT * net;
    if (TYPE >= 1) {
      const double dM = a.dci_dM * net;
      const size_t o = (size_t)(3 * m.R + 2 * (r - m.r_tb)) * ldg;
      g2[o] = dM;
      g2[o + ldg] = dM * a.M;
    }
  }
}

// RM: reactor-major output (rows padded to NP), else component-major.  MUST be called by every thread of the CTA.
// yin / out pointers are pre-offset to this thread's slot (component-major arrays) resp. reactor (Jrm).
template <int BLOCK, bool RM>
__device__ __forceinline__ void jac_thread_tmem(const MechDev& m, const double* __restrict__ yin, long long ldin, double p,
                                                const JacOut& o, long long slot, double* __restrict__ Cs, uint32_t wt,
                                                double* __restrict__ stage, bool store) {
  const int K = m.K, R = m.R, rs = m.rstride, N = K + 1;
  const int tid = threadIdx.x;
  const TState t = make_tstate(m, yin[0]);
  double* const fout = o.f + slot;
  double* const g2 = o.g2 + slot;
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
  const double Ctot = p / (R_U * t.T);
  const double rho = Ctot / S;
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
  const double irho = 1.0 / rho, icps = 1.0 / cps;
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
      const double hrt = thermo_row_h(row, t);
      hw = fma(hrt, w, hw);
      if (store) {
        fout[(size_t)(k0 + j + 1) * o.ldf] = w * row[0] * irho;
        hc[(size_t)(k0 + j) * o.ldh] = t.T * hrt * row[1] * icps;            // hh_k = T (H_k/RT) / (W_k cps)
        hc[(size_t)(K + k0 + j) * o.ldh] = thermo_row_cp(row, t) * row[1] * icps;  // cc_k = (cp_k/R) / (W_k cps)
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
  const int npt = jac_npt(K);
  for (int c = 0; c < npt; c += 4) tm_zero8(wt + 2 * c);
  tm_wait_st();
  __syncthreads();
  const double iS = 1.0 / S;
  const int NP = jac_np(N);
  double sfc = 0.0;  // sum_k f_k cc_k
  for (int k = 0; k < K; ++k) {
    double sig = 0.0, tau = 0.0, dns = 0.0;
    const int e1 = __ldg(m.tptr + k + 1);
    for (int e = __ldg(m.tptr + k); e < e1; ++e) {
      const int en = __ldg(m.tent + e);
      const int i = en >> 8;
      const double nu = (double)((en & 255) - 128);
      const double swd = __ldg(m.rpack + (size_t)i * rs + 3);
      const unsigned lo = (unsigned)__double2loint(swd), hi = (unsigned)__double2hiint(swd);
      int sl[6] = {(int)(lo & 1023u), (int)((lo >> 10) & 1023u), (int)((lo >> 20) & 1023u),
                   (int)(hi & 1023u), (int)((hi >> 10) & 1023u), (int)((hi >> 20) & 1023u)};
      const bool dup = (hi >> 31) != 0;
      const double gf = g2[(size_t)(3 * i) * o.ldg], gr = g2[(size_t)(3 * i + 1) * o.ldg], dqT = g2[(size_t)(3 * i + 2) * o.ldg];
      double c[6];
#pragma unroll
      for (int x = 0; x < 6; ++x) c[x] = Cs[sl[x] * BLOCK];
      const double ngr = -gr;
      double d[6] = {gf * (c[1] * c[2]), gf * (c[0] * c[2]), gf * (c[0] * c[1]),
                     ngr * (c[4] * c[5]), ngr * (c[3] * c[5]), ngr * (c[3] * c[4])};
      const int nf = (sl[0] != K) + (sl[1] != K) + (sl[2] != K), nrv = (sl[3] != K) + (sl[4] != K) + (sl[5] != K);
      double si = (double)nf * (d[0] * c[0]) + (double)nrv * (d[3] * c[3]);
      if (i >= m.r_tb) {  // third-body / falloff row: dense coefficient + the listed efficiencies
        const int jx = i - m.r_tb;
        const size_t og = (size_t)(3 * R + 2 * jx) * o.ldg;
        const double dM = g2[og];
        si += g2[og + o.ldg];
        const double ndM = nu * dM;
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
      sig = fma(nu, si, sig);
      tau = fma(nu, dqT, tau);
      if (!dup) {
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
    //                           J_kT = (W_k / rho)(tau_k - sig_k / T) + f_k / T
    const double Wk = sW[k];
    const double fk = store ? fout[(size_t)(1 + k) * o.ldf] : 0.0;
    const double beta = fma(Wk, dns, (fk - Wk * irho * sig) * iS);
    const double JkT = Wk * irho * (tau - sig * t.invT) + fk * t.invT;
    if (store) sfc = fma(fk, hc[(size_t)(K + k) * o.ldh], sfc);
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
        if (RM) {
          double2* dst = reinterpret_cast<double2*>(o.J + (size_t)(1 + k) * NP + c0);
          dst[0] = make_double2(v[0], v[1]);
          dst[1] = make_double2(v[2], v[3]);
        } else {
#pragma unroll
          for (int x = 0; x < 4; ++x)
            if (c0 + x < N) o.J[((size_t)(1 + k) * N + c0 + x) * o.ldJ] = v[x];
        }
      }
    }
    tm_wait_st();
  }
  if (store) hc[(size_t)(2 * K) * o.ldh] = -sfc - fT * dcp * icps;
}

// One CTA per SM, persistent over batches of BLOCK slots (as rhs_kernel_tmem).  n_dev (optional) overrides n with a
// device-side count (the active-list length of the ROS4 rounds).
template <int BLOCK, bool RM>
__global__ void __launch_bounds__(BLOCK, 1) jac_rows_kernel(const MechDev m, long long n, const int* __restrict__ n_dev,
                                                            const double* __restrict__ y, long long ld,
                                                            const double* __restrict__ p, JacOut o) {
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
  const int N = m.K + 1;
  for (long long b = blockIdx.x; b * BLOCK < n; b += gridDim.x) {
    const long long r = b * BLOCK + tid;
    const bool act = r < n;
    const long long rr = act ? r : n - 1;
    JacOut oo = o;
    if (RM) oo.J = o.J + (size_t)rr * N * jac_np(N);
    else oo.J = o.J + rr;
    jac_thread_tmem<BLOCK, RM>(m, y + rr, ld, p[rr], oo, rr, Cs, wt, stage, act);
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tbase));
}

// Row 0 of a component-major Jacobian from its species rows (see the header): one thread per reactor.
__global__ void __launch_bounds__(128) jac_trow_kernel(int K, long long n, const double* __restrict__ f, long long ldf,
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
