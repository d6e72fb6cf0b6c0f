// Thread-per-reactor RHS evaluation shared by ck_rhs and the RKF45 step kernel (see ck_rhs.cu for the mapping).
#pragma once
#include "ck_chem.cuh"

namespace ck {

constexpr int RHS_CHUNK = 32;  // reactions (or species) staged per shared-memory chunk

__host__ __device__ inline int rhs_stage_doubles(int rstride) { return RHS_CHUNK * (rstride > 16 ? rstride : 16); }
__host__ __device__ inline size_t rhs_smem_bytes(int K, int rstride, int block) {
  return ((size_t)2 * (K + 1) * block + (size_t)rhs_stage_doubles(rstride)) * sizeof(double);
}

// cp/R and H/(RT) from a staged species row (spack layout: W, 1/W, t_mid, 0, lo a1..a6, hi a1..a6)
__device__ __forceinline__ void thermo_row(const double* __restrict__ row, const TState& t, double& cpR, double& hRT) {
  const double* a = row + ((t.T > row[2]) ? 10 : 4);
  const double T = t.T;
  const double a1 = a[0], a2 = a[1], a3 = a[2], a4 = a[3], a5 = a[4], a6 = a[5];
  cpR = fma(fma(fma(fma(a5, T, a4), T, a3), T, a2), T, a1);
  hRT = fma(fma(fma(fma(a5 * 0.2, T, a4 * 0.25), T, a3 * (1.0 / 3.0)), T, a2 * 0.5), T, a1) + a6 * t.invT;
}

// One RHS evaluation for the reactor of this thread; MUST be called by every thread of the CTA (species
// and reaction constants are staged cooperatively through `stage`, RHS_CHUNK rows at a time, so that the
// inner loops read them as shared-memory broadcasts instead of L2 round trips).
// yin / fout are pre-offset to the reactor's column.  Cs, ws: shared-memory columns of this thread
// (pre-offset by tid), stride BLOCK, K+1 entries each (entry K: dummy concentration 1 / sink accumulator).
template <int BLOCK>
__device__ __forceinline__ void rhs_thread(const MechDev& m, const double* __restrict__ yin, long long ldin, double p,
                                           double* __restrict__ fout, long long ldout, double* __restrict__ Cs,
                                           double* __restrict__ ws, double* __restrict__ stage, bool store) {
  const int K = m.K, R = m.R, rs = m.rstride;
  const int tid = threadIdx.x;
  const TState t = make_tstate(m, yin[0]);
  // (2) ideal gas: S = sum Y_k/W_k, rho = p/(R_u T S), C_k = rho Y_k/W_k; cp sum on the way
  double S = 0.0, cps = 0.0;
  for (int k0 = 0; k0 < K; k0 += RHS_CHUNK) {
    const int nk = min(RHS_CHUNK, K - k0);
    __syncthreads();
    for (int idx = tid; idx < nk * 16; idx += BLOCK) stage[idx] = __ldg(m.spack + (size_t)k0 * 16 + idx);
    __syncthreads();
#pragma unroll 4
    for (int j = 0; j < nk; ++j) {
      const double* row = stage + j * 16;
      const double yw = yin[(size_t)(k0 + j + 1) * ldin] * row[1];
      double cpR, hRT;
      thermo_row(row, t, cpR, hRT);
      S += yw;
      cps = fma(yw, cpR, cps);
      Cs[(k0 + j) * BLOCK] = yw;
      ws[(k0 + j) * BLOCK] = 0.0;
    }
  }
  const double Ctot = p / (R_U * t.T);  // = rho * S
  const double rho = Ctot / S;
#pragma unroll 4
  for (int k = 0; k < K; ++k) Cs[k * BLOCK] *= rho;
  Cs[K * BLOCK] = 1.0;
  ws[K * BLOCK] = 0.0;
  // (3) reactions, chunk by chunk
  for (int r0 = 0; r0 < R; r0 += RHS_CHUNK) {
    const int nr = min(RHS_CHUNK, R - r0);
    const double* src = m.rpack + (size_t)r0 * rs;
    __syncthreads();  // previous chunk fully consumed
    for (int idx = tid; idx < nr * rs; idx += BLOCK) stage[idx] = __ldg(src + idx);
    __syncthreads();
    // rows [r0, r0+nfast) have six distinct slot species: two reactions in flight, loads before stores
    const int nfast = max(0, min(nr, m.r_dup - r0)) & ~1;
    for (int j = 0; j < nfast; j += 2) {
      const RxnConst ka = load_rxn_row(stage + j * rs, t.tint);
      const RxnConst kb = load_rxn_row(stage + (j + 1) * rs, t.tint);
      double kfa, kra, kfb, krb;
      rate_constants(ka, t, kfa, kra);
      rate_constants(kb, t, kfb, krb);
      const double pfa = Cs[ka.slot[0] * BLOCK] * Cs[ka.slot[1] * BLOCK] * Cs[ka.slot[2] * BLOCK];
      const double pra = Cs[ka.slot[3] * BLOCK] * Cs[ka.slot[4] * BLOCK] * Cs[ka.slot[5] * BLOCK];
      const double pfb = Cs[kb.slot[0] * BLOCK] * Cs[kb.slot[1] * BLOCK] * Cs[kb.slot[2] * BLOCK];
      const double prb = Cs[kb.slot[3] * BLOCK] * Cs[kb.slot[4] * BLOCK] * Cs[kb.slot[5] * BLOCK];
      const double qa = fma(kfa, pfa, -kra * pra);
      const double qb = fma(kfb, pfb, -krb * prb);
      double w[6];
#pragma unroll
      for (int s = 0; s < 6; ++s) w[s] = ws[ka.slot[s] * BLOCK];
#pragma unroll
      for (int s = 0; s < 6; ++s) ws[ka.slot[s] * BLOCK] = (s < 3) ? w[s] - qa : w[s] + qa;
#pragma unroll
      for (int s = 0; s < 6; ++s) w[s] = ws[kb.slot[s] * BLOCK];
#pragma unroll
      for (int s = 0; s < 6; ++s) ws[kb.slot[s] * BLOCK] = (s < 3) ? w[s] - qb : w[s] + qb;
    }
    // remaining rows (repeated species, third-body, falloff): one at a time, sequential scatter
    for (int j = nfast; j < nr; ++j) {
      const RxnConst kc = load_rxn_row(stage + j * rs, t.tint);
      const double q = reaction_q<BLOCK, false>(m, r0 + j, kc, t, Cs, Ctot, nullptr);
#pragma unroll
      for (int s = 0; s < 6; ++s) {
        double* w = ws + kc.slot[s] * BLOCK;
        *w = (s < 3) ? *w - q : *w + q;
      }
    }
  }
  // (4) Eq. 12-13 (13 in reading G2)
  const double irho = 1.0 / rho;
  double hw = 0.0;
  for (int k0 = 0; k0 < K; k0 += RHS_CHUNK) {
    const int nk = min(RHS_CHUNK, K - k0);
    __syncthreads();
    for (int idx = tid; idx < nk * 16; idx += BLOCK) stage[idx] = __ldg(m.spack + (size_t)k0 * 16 + idx);
    __syncthreads();
#pragma unroll 4
    for (int j = 0; j < nk; ++j) {
      const double* row = stage + j * 16;
      double cpR, hRT;
      thermo_row(row, t, cpR, hRT);
      const double w = ws[(k0 + j) * BLOCK];
      hw = fma(hRT, w, hw);
      if (store) fout[(size_t)(k0 + j + 1) * ldout] = w * row[0] * irho;
    }
  }
  if (store) fout[0] = -(t.T * hw) / (rho * cps);  // R_u cancels: -R_u T hw / (rho R_u cps)
}

// largest block whose columns fit in shared memory, halved while the grid would leave most SMs idle
inline int rhs_pick_block(int K, int rstride, long long n) {
  const size_t cap = 227 * 1024;
  int block = 256;
  while (block >= 32 && rhs_smem_bytes(K, rstride, block) > cap) block >>= 1;
  if (block < 32) return 0;
  while (block > 32 && (n + block - 1) / block < 148) block >>= 1;
  return block;
}

}  // namespace ck
