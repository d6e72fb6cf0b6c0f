// Thread-per-reactor RHS evaluation shared by ck_rhs and the RKF45 step kernel (see ck_rhs.cu for the mapping).
#pragma once
#include "ck_chem.cuh"

namespace ck {

constexpr int RHS_CHUNK = 32;  // reactions (or species) staged per shared-memory chunk

// staging buffer: RHS_CHUNK reaction rows (or species rows of 16) + RHS_CHUNK special rows of 16
__host__ __device__ inline int rhs_stage_doubles(int rstride) { return RHS_CHUNK * ((rstride > 16 ? rstride : 16) + 16); }
__host__ __device__ inline size_t rhs_smem_bytes(int K, int rstride, int block) {
  return ((size_t)2 * (K + 1) * block + (size_t)rhs_stage_doubles(rstride)) * sizeof(double);
}

// cp/R resp. H/(RT) from a staged species row (spack layout, ck_internal.h): the H/RT coefficients are stored
// pre-divided (a2/2, a3/3, ...), and each of the two species loops evaluates only the polynomial it needs
__device__ __forceinline__ double thermo_row_cp(const double* __restrict__ row, const TState& t) {
  const double* a = row + ((t.T > row[2]) ? 9 : 4);
  const double T = t.T;
  return fma(fma(fma(fma(a[4], T, a[3]), T, a[2]), T, a[1]), T, a[0]);
}
__device__ __forceinline__ double thermo_row_h(const double* __restrict__ row, const TState& t) {
  const double* a = row + ((t.T > row[2]) ? 20 : 14);
  const double T = t.T;
  return fma(fma(fma(fma(a[4], T, a[3]), T, a[2]), T, a[1]), T, a[0]) + a[5] * t.invT;
}

// Four reactions with six distinct slot species each, all in flight: rate constants, products, then the
// omega scatter with every load issued before the stores.  Slots 1, 2, 4, 5 may hold the dummy index K
// (warp-uniform): those accesses are predicated off and cost no shared-memory wavefronts.
template <int BLOCK>
__device__ __forceinline__ void fast_group(const RxnConst (&kc)[4], const TState& t, int K, const double* __restrict__ Cs,
                                           double* __restrict__ ws) {
  double q[4];
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    double kf, kr;
    rate_constants(kc[u], t, kf, kr);
    double pf = Cs[kc[u].slot[0] * BLOCK], pr = Cs[kc[u].slot[3] * BLOCK];
    if (kc[u].slot[1] != K) pf *= Cs[kc[u].slot[1] * BLOCK];
    if (kc[u].slot[2] != K) pf *= Cs[kc[u].slot[2] * BLOCK];
    if (kc[u].slot[4] != K) pr *= Cs[kc[u].slot[4] * BLOCK];
    if (kc[u].slot[5] != K) pr *= Cs[kc[u].slot[5] * BLOCK];
    q[u] = fma(kf, pf, -kr * pr);
  }
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    double w[6];
#pragma unroll
    for (int s = 0; s < 6; ++s)
      if (s == 0 || s == 3 || kc[u].slot[s] != K) w[s] = ws[kc[u].slot[s] * BLOCK];
#pragma unroll
    for (int s = 0; s < 6; ++s)
      if (s == 0 || s == 3 || kc[u].slot[s] != K) ws[kc[u].slot[s] * BLOCK] = (s < 3) ? w[s] - q[u] : w[s] + q[u];
  }
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
    for (int idx = tid; idx < nk * SPS; idx += BLOCK) stage[idx] = __ldg(m.spack + (size_t)k0 * SPS + idx);
    __syncthreads();
#pragma unroll 8
    for (int j = 0; j < nk; ++j) {
      const double* row = stage + j * SPS;
      const double yw = yin[(size_t)(k0 + j + 1) * ldin] * row[1];
      S += yw;
      cps = fma(yw, thermo_row_cp(row, t), cps);
      Cs[(k0 + j) * BLOCK] = yw;
      ws[(k0 + j) * BLOCK] = 0.0;
    }
  }
  // constant pressure: rho = p / (R_u T S); constant volume (m.cv): `p` IS rho; Ctot = sum_k C_k = rho S either way
  const double rho = m.cv ? p : (p / (R_U * t.T)) / S;
  const double Ctot = m.cv ? rho * S : p / (R_U * t.T);
#pragma unroll 4
  for (int k = 0; k < K; ++k) Cs[k * BLOCK] *= rho;
  Cs[K * BLOCK] = 1.0;
  ws[K * BLOCK] = 0.0;
  // (3) reactions, chunk by chunk
  double* xstage = stage + RHS_CHUNK * (rs > 16 ? rs : 16);
  for (int r0 = 0; r0 < R; r0 += RHS_CHUNK) {
    const int nr = min(RHS_CHUNK, R - r0);
    const double* src = m.rpack + (size_t)r0 * rs;
    const int x0 = max(r0, m.r_tb);                 // first special row of this chunk
    const int nx = max(0, r0 + nr - x0);
    __syncthreads();  // previous chunk fully consumed
    for (int idx = tid; idx < nr * rs; idx += BLOCK) stage[idx] = __ldg(src + idx);
    for (int idx = tid; idx < nx * 16; idx += BLOCK) xstage[idx] = __ldg(m.xpack + (size_t)(x0 - m.r_tb) * 16 + idx);
    __syncthreads();
    // rows [r0, r0+nfast) have six distinct slot species: four reactions in flight, loads before stores
    const int nfast = max(0, min(nr, m.r_dup - r0)) & ~3;
    for (int j = 0; j < nfast; j += 4) {
      RxnConst kc[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) kc[u] = load_rxn_row(stage + (j + u) * rs, t.tint);  // (uniform both-interval loads + select measured 4 % slower)
      fast_group<BLOCK>(kc, t, K, Cs, ws);
    }
    // remaining rows (repeated species, third-body, falloff): one at a time, sequential scatter
    for (int j = nfast; j < nr; ++j) {
      const RxnConst kc = load_rxn_row(stage + j * rs, t.tint);
      const int r = r0 + j;
      const double q = reaction_q<BLOCK, false>(m, r, kc, t, Cs, Ctot, nullptr, xstage + (r >= x0 ? (r - x0) * 16 : 0));
      if (!kc.dup) {  // six distinct slot species: one round trip
        double w[6];
#pragma unroll
        for (int s = 0; s < 6; ++s)
          if (s == 0 || s == 3 || kc.slot[s] != K) w[s] = ws[kc.slot[s] * BLOCK];
#pragma unroll
        for (int s = 0; s < 6; ++s)
          if (s == 0 || s == 3 || kc.slot[s] != K) ws[kc.slot[s] * BLOCK] = (s < 3) ? w[s] - q : w[s] + q;
      } else {
#pragma unroll
        for (int s = 0; s < 6; ++s) {
          double* w = ws + kc.slot[s] * BLOCK;
          *w = (s < 3) ? *w - q : *w + q;
        }
      }
    }
  }
  // (4) Eq. 12-13 (13 in reading G2)
  const double irho = 1.0 / rho;
  const double sub = m.cv ? 1.0 : 0.0;   // constant volume: u_k / (R_u T) = H_k / (R_u T) - 1 and c_v / R_u = c_p / R_u - S
  double hw = 0.0;
  for (int k0 = 0; k0 < K; k0 += RHS_CHUNK) {
    const int nk = min(RHS_CHUNK, K - k0);
    __syncthreads();
    for (int idx = tid; idx < nk * SPS; idx += BLOCK) stage[idx] = __ldg(m.spack + (size_t)k0 * SPS + idx);
    __syncthreads();
#pragma unroll 4
    for (int j = 0; j < nk; ++j) {
      const double* row = stage + j * SPS;
      const double w = ws[(k0 + j) * BLOCK];
      hw = fma(thermo_row_h(row, t) - sub, w, hw);
      if (store) fout[(size_t)(k0 + j + 1) * ldout] = w * row[0] * irho;
    }
  }
  if (store) fout[0] = -(t.T * hw) / (rho * (cps - sub * S));  // R_u cancels: -R_u T hw / (rho R_u cps)
}

// largest block whose columns fit in shared memory, halved while the grid would leave most SMs idle
inline int rhs_pick_block(int K, int rstride, long long n, int sms) {
  const size_t cap = 227 * 1024;
  int block = 256;
  while (block >= 32 && rhs_smem_bytes(K, rstride, block) > cap) block >>= 1;
  if (block < 32) return 0;
  while (block > 32 && (n + block - 1) / block < sms) block >>= 1;
  return block;
}

}  // namespace ck
