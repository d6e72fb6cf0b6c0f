// ck_rhs variant with the production-rate accumulators in TENSOR MEMORY (Blackwell TMEM).
//
// The thread-per-reactor RHS needs two per-thread arrays with warp-uniform, data-dependent indices: the
// concentrations C_k (read-only in the reaction loop) and the accumulators omega_k (read-modify-write).  In
// shared memory the two columns cost 2 (K+1) 8 B per thread and pin the occupancy at 8 warps per SM.  TMEM is
// 128 lanes x 512 32-bit columns per SM, and tcgen05.ld/st address it exactly the way these columns are used:
// one column address for the whole warp, each thread touching its own lane.  Warp w of the CTA owns lane quadrant
// w & 3 and the column range (w >> 2) * 2 (K+1); with the accumulators there, shared memory holds only C and the
// CTA can be 512 threads: 16 warps per SM, and the accumulator traffic leaves the shared-memory pipe.
// Limits: 2 (K+1) columns per warp and four warps per quadrant => K + 1 <= 64.
#pragma once
#include "ck_rhs_thread.cuh"

namespace ck {

__device__ __forceinline__ void tm_ld2(uint32_t taddr, double& v) {
  uint32_t a, b;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "r"(taddr));
  v = __hiloint2double((int)b, (int)a);
}
// issue the load only; the two halves are combined after tm_wait_ld()
__device__ __forceinline__ void tm_ld2_raw(uint32_t taddr, uint32_t& a, uint32_t& b) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "r"(taddr));
}
__device__ __forceinline__ void tm_st2(uint32_t taddr, double v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"((uint32_t)__double2loint(v)),
               "r"((uint32_t)__double2hiint(v)));
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__host__ __device__ inline size_t rhs_tmem_smem_bytes(int K, int rstride, int block) {
  return ((size_t)(K + 1) * block + (size_t)rhs_stage_doubles(rstride)) * sizeof(double);
}

// NG reactions with six distinct slot species in flight; accumulators in TMEM at column base `wt`
// B22: every reaction of the group is A + B <=> C + D (slots 0, 1, 3, 4 live, 2 and 5 dummy): no predicates at all
template <int BLOCK, int NG, bool B22, bool NC>
__device__ __forceinline__ void fast_group_tmem(const RxnConst (&kc)[NG], const TState& t, int K,
                                                const double* __restrict__ Cs, uint32_t wt) {
  // the packed rows carry slot << 12 (byte offset of a C column of 512 reactors); narrower power-of-two CTAs shift it down
  static_assert(!B22 || BLOCK == 512 || BLOCK == 256 || BLOCK == 128, "pre-shifted slot words need a power-of-two CTA width");
  constexpr int SH = (BLOCK == 512) ? 0 : (BLOCK == 256 ? 1 : 2);
  double q[NG];
#pragma unroll
  for (int u = 0; u < NG; ++u) {
    double kf, kr;
    rate_constants<NC>(kc[u], t, kf, kr);
    double pf, pr;
    if (B22) {  // slot words are byte offsets of the C columns
      const char* Cb = reinterpret_cast<const char*>(Cs);
      pf = *reinterpret_cast<const double*>(Cb + ((unsigned)kc[u].slot[0] >> SH)) *
           *reinterpret_cast<const double*>(Cb + ((unsigned)kc[u].slot[1] >> SH));
      pr = *reinterpret_cast<const double*>(Cb + ((unsigned)kc[u].slot[3] >> SH)) *
           *reinterpret_cast<const double*>(Cb + ((unsigned)kc[u].slot[4] >> SH));
    } else {
      pf = Cs[kc[u].slot[0] * BLOCK]; pr = Cs[kc[u].slot[3] * BLOCK];
      if (kc[u].slot[1] != K) pf *= Cs[kc[u].slot[1] * BLOCK];
      if (kc[u].slot[2] != K) pf *= Cs[kc[u].slot[2] * BLOCK];
      if (kc[u].slot[4] != K) pr *= Cs[kc[u].slot[4] * BLOCK];
      if (kc[u].slot[5] != K) pr *= Cs[kc[u].slot[5] * BLOCK];
    }
    q[u] = fma(kf, pf, -kr * pr);
  }
#pragma unroll
  for (int u = 0; u < NG; ++u) {
    uint32_t lo[6], hi[6];
#pragma unroll
    for (int s = 0; s < 6; ++s)
      if (B22 ? (s != 2 && s != 5) : (s == 0 || s == 3 || kc[u].slot[s] != K))
        tm_ld2_raw(wt + (B22 ? (unsigned)kc[u].slot[s] >> 11 : 2u * kc[u].slot[s]), lo[s], hi[s]);
    tm_wait_ld();
#pragma unroll
    for (int s = 0; s < 6; ++s)
      if (B22 ? (s != 2 && s != 5) : (s == 0 || s == 3 || kc[u].slot[s] != K)) {
        const double w = __hiloint2double((int)hi[s], (int)lo[s]);
        tm_st2(wt + (B22 ? (unsigned)kc[u].slot[s] >> 11 : 2u * kc[u].slot[s]), (s < 3) ? w - q[u] : w + q[u]);
      }
    tm_wait_st();
  }
}

// fast rows of one staged chunk: [0, n22) four A+B<=>C+D rows at a time, [n22, nfast) two generic rows at a time
template <int BLOCK, bool NC>
__device__ __forceinline__ void fast_rows_tmem(const double* __restrict__ stage, int rs, int n22, int nfast, const TState& t,
                                               int K, const double* __restrict__ Cs, uint32_t wt) {
  constexpr bool PRE = (BLOCK == 512 || BLOCK == 256 || BLOCK == 128);
  for (int j = 0; j < n22; j += 4) {
    RxnConst kc[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) kc[u] = load_rxn_row<PRE>(stage + (j + u) * rs, t.tint);
    fast_group_tmem<BLOCK, 4, PRE, NC>(kc, t, K, Cs, wt);
  }
  for (int j = n22; j < nfast; j += 2) {
    RxnConst kc[2];
#pragma unroll
    for (int u = 0; u < 2; ++u) kc[u] = load_rxn_row(stage + (j + u) * rs, t.tint);
    fast_group_tmem<BLOCK, 2, false, NC>(kc, t, K, Cs, wt);
  }
}

// omega scatter of one row outside the fast groups
__device__ __forceinline__ void slow_scatter_tmem(const RxnConst& kc, double q, int K, uint32_t wt) {
  if (!kc.dup) {  // six distinct slot species: one tensor-memory round trip
    uint32_t lo[6], hi[6];
#pragma unroll
    for (int s = 0; s < 6; ++s)
      if (s == 0 || s == 3 || kc.slot[s] != K) tm_ld2_raw(wt + 2 * kc.slot[s], lo[s], hi[s]);
    tm_wait_ld();
#pragma unroll
    for (int s = 0; s < 6; ++s)
      if (s == 0 || s == 3 || kc.slot[s] != K) {
        const double w = __hiloint2double((int)hi[s], (int)lo[s]);
        tm_st2(wt + 2 * kc.slot[s], (s < 3) ? w - q : w + q);
      }
    tm_wait_st();
  } else {
#pragma unroll
    for (int s = 0; s < 6; ++s) {  // slot by slot: a species sits in two slots
      double w;
      tm_ld2(wt + 2 * kc.slot[s], w);
      tm_wait_ld();
      tm_st2(wt + 2 * kc.slot[s], (s < 3) ? w - q : w + q);
      tm_wait_st();
    }
  }
}

// NP consecutive rows of kind TYPE outside the fast groups (reaction_q): rates of progress first (independent chains
// the scheduler can interleave), then the scatters in row order
template <int BLOCK, int TYPE, int NP>
__device__ __forceinline__ void slow_rows_tmem(const MechDev& m, int r, const double* __restrict__ row, int rs,
                                               const double* __restrict__ xrow, const TState& t,
                                               const double* __restrict__ Cs, double Ctot, uint32_t wt) {
  RxnConst kc[NP];
  double q[NP];
#pragma unroll
  for (int u = 0; u < NP; ++u) {
    kc[u] = load_rxn_row(row + u * rs, t.tint);
    q[u] = reaction_q<BLOCK, false, TYPE>(m, r + u, kc[u], t, Cs, Ctot, nullptr, xrow + u * 16);
  }
#pragma unroll
  for (int u = 0; u < NP; ++u) slow_scatter_tmem(kc[u], q[u], m.K, wt);
}

// CVM: reactor kind at compile time (0 constant pressure, 1 constant volume) or -1 = read m.cv at run time.  ck_rhs
// dispatches on the kind (the run-time switch costs the headline kernel 1.9 %: 2.512 vs 2.466 ms per pass of config 2).
template <int BLOCK, int CVM = -1>
__device__ __forceinline__ void rhs_thread_tmem(const MechDev& m, const double* __restrict__ yin, long long ldin, double p,
                                                double* __restrict__ fout, long long ldout, double* __restrict__ Cs,
                                                uint32_t wt, double* __restrict__ stage, bool store) {
  const int K = m.K, R = m.R, rs = m.rstride;
  const int tid = threadIdx.x;
  const bool cv = (CVM < 0) ? (m.cv != 0) : (CVM == 1);
  const TState t = make_tstate(m, yin[0]);
  // every reactor of the warp inside the window for which the packer bounded the fast rows' exp arguments?
  const bool allsafe = __all_sync(0xffffffffu, t.T >= m.t_safe_lo && t.T <= m.t_safe_hi);
  double S = 0.0, cps = 0.0;
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
      Cs[(k0 + j) * BLOCK] = yw;
      tm_st2(wt + 2 * (k0 + j), 0.0);
    }
  }
  // constant pressure: rho = p / (R_u T S); constant volume (m.cv): `p` IS rho; Ctot = sum_k C_k = rho S either way
  const double Ctot = cv ? p * S : p / (R_U * t.T);
  const double rho = cv ? p : Ctot / S;
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
    const int n22 = max(0, min(nr, m.r_22 - r0)) & ~3;
    const int nfast = n22 + (max(0, min(nr, m.r_dup - r0) - n22) & ~1);
    if (allsafe) fast_rows_tmem<BLOCK, true>(stage, rs, n22, nfast, t, K, Cs, wt);
    else fast_rows_tmem<BLOCK, false>(stage, rs, n22, nfast, t, K, Cs, wt);
    // the rest of the chunk one row at a time, one loop per row kind (the groups are contiguous)
    const int j1 = min(nr, max(nfast, m.r_tb - r0)), j2 = min(nr, max(nfast, m.r_lind - r0)),
              j3 = min(nr, max(nfast, m.r_troe - r0));
    const double* xs = xstage - (size_t)(x0 - r0) * 16;  // xs + 16 j: falloff row of chunk row j
    int j = nfast;
    for (; j < j1; ++j) slow_rows_tmem<BLOCK, 0, 1>(m, r0 + j, stage + j * rs, rs, xs, t, Cs, Ctot, wt);
    for (; j + 1 < j2; j += 2) slow_rows_tmem<BLOCK, 1, 2>(m, r0 + j, stage + j * rs, rs, xs + 16 * j, t, Cs, Ctot, wt);
    for (; j < j2; ++j) slow_rows_tmem<BLOCK, 1, 1>(m, r0 + j, stage + j * rs, rs, xs + 16 * j, t, Cs, Ctot, wt);
    for (; j < j3; ++j) slow_rows_tmem<BLOCK, 2, 1>(m, r0 + j, stage + j * rs, rs, xs + 16 * j, t, Cs, Ctot, wt);
    for (; j < nr; ++j) slow_rows_tmem<BLOCK, 3, 1>(m, r0 + j, stage + j * rs, rs, xs + 16 * j, t, Cs, Ctot, wt);
  }
  const double irho = 1.0 / rho;
  const double sub = cv ? 1.0 : 0.0;   // constant volume: u_k / (R_u T) = H_k / (R_u T) - 1 and c_v / R_u = c_p / R_u - S
  double hw = 0.0;
  for (int k0 = 0; k0 < K; k0 += RHS_CHUNK) {
    const int nk = min(RHS_CHUNK, K - k0);
    __syncthreads();
    for (int idx = tid; idx < nk * SPS; idx += BLOCK) stage[idx] = __ldg(m.spack + (size_t)k0 * SPS + idx);
    __syncthreads();
    for (int j0 = 0; j0 < nk; j0 += 4) {  // four accumulators per tensor-memory round trip
      uint32_t lo[4], hi[4];
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (j0 + u < nk) tm_ld2_raw(wt + 2 * (k0 + j0 + u), lo[u], hi[u]);
      tm_wait_ld();
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (j0 + u < nk) {
          const double* row = stage + (j0 + u) * SPS;
          const double w = __hiloint2double((int)hi[u], (int)lo[u]);
          hw = fma((CVM == 0) ? thermo_row_h(row, t) : thermo_row_h(row, t) - sub, w, hw);
          if (store) fout[(size_t)(k0 + j0 + u + 1) * ldout] = w * row[0] * irho;
        }
    }
  }
  if (store) fout[0] = -(t.T * hw) / (rho * ((CVM == 0) ? cps : cps - sub * S));
}

// tensor-memory columns a CTA of `block` threads allocates: one set of 2 (K+1) per group of four warps, rounded up to
// a power of two >= 32 (0: does not fit)
__host__ __device__ inline int rhs_tmem_cols(int K, int block) {
  const int need = ((block + 127) / 128) * 2 * (K + 1);
  if (need > 512) return 0;
  int c = 32;
  while (c < need) c <<= 1;
  return c;
}

template <int BLOCK, int CVM>
__global__ void __launch_bounds__(BLOCK, 1) rhs_kernel_tmem(const MechDev m, long long n, const double* __restrict__ y,
                                                            long long ld, const double* __restrict__ p,
                                                            double* __restrict__ f, long long ldf) {
  extern __shared__ double sm[];
  __shared__ uint32_t s_tmem;
  // warp index broadcast from lane 0: tells the compiler it is warp-uniform, so the tensor-memory addresses below stay
  // in uniform registers
  const int tid = threadIdx.x, warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  const uint32_t ncols = (uint32_t)rhs_tmem_cols(m.K, BLOCK);
  if (warp == 0) {  // one warp allocates the CTA's columns
    const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&s_tmem);
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst), "r"(ncols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tbase = s_tmem;
  // lane quadrant of this warp in bits 31..16, its column range in bits 15..0
  const uint32_t wt = tbase + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 2 * (m.K + 1));
  double* Cs = sm + tid;
  double* stage = sm + (size_t)(m.K + 1) * BLOCK;
  for (long long b = blockIdx.x; b * BLOCK < n; b += gridDim.x) {
    const long long r = b * BLOCK + tid;
    const bool act = r < n;
    const long long rr = act ? r : n - 1;
    rhs_thread_tmem<BLOCK, CVM>(m, y + rr, ld, p[rr], f + rr, ldf, Cs, wt, stage, act);
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tbase), "r"(ncols));
}

}  // namespace ck
