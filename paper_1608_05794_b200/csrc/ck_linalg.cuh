// Per-reactor dense linear algebra in shared memory (factorisation of
// (1/(h gamma)) I - J and the four stage solves of Eq. 6).  A is row-major with an ODD leading dimension
// so that a column walk (stride lda) is shared-memory bank-conflict free for 8-byte elements.
#pragma once
#include "ck_internal.h"

namespace ck {

// CTA-wide argmax of |v| over candidates (val, idx); ties go to the smaller index (first maximal
// element, the same rule as the reference definition of partial pivoting).  red: >= 2*(G/32) doubles.
template <int G>
__device__ __forceinline__ int block_argmax(double val, int idx, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const double v2 = __shfl_xor_sync(0xffffffffu, val, o);
    const int i2 = __shfl_xor_sync(0xffffffffu, idx, o);
    if (v2 > val || (v2 == val && i2 < idx)) { val = v2; idx = i2; }
  }
  if (G == 32) return idx;
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  int* ired = reinterpret_cast<int*>(red + G / 32);
  __syncthreads();
  if (l == 0) { red[w] = val; ired[w] = idx; }
  __syncthreads();
  double bv = red[0];
  int bi = ired[0];
#pragma unroll
  for (int i = 1; i < G / 32; ++i) {
    const double v2 = red[i];
    const int i2 = ired[i];
    if (v2 > bv || (v2 == bv && i2 < bi)) { bv = v2; bi = i2; }
  }
  return bi;
}

// In-place LU with partial pivoting, P A = L U (unit lower L below the diagonal, whole rows swapped).
// piv[k] = row exchanged with row k at step k.  Returns false on a zero / non-finite pivot column.
// One thread per trailing row; the pivot row is read as a shared-memory broadcast.
template <int G>
__device__ __forceinline__ bool lu_factor_block(double* __restrict__ A, int lda, int N, int* __restrict__ piv,
                                                double* red) {
  const int tid = threadIdx.x;
  for (int k = 0; k < N; ++k) {
    double best = -1.0;
    int bi = 0x7fffffff;
    for (int i = k + tid; i < N; i += G) {
      const double v = fabs(A[(size_t)i * lda + k]);
      if (v > best) { best = v; bi = i; }  // ascending i: the first maximal element wins
    }
    const int p = block_argmax<G>(best, bi, red);
    if (p == 0x7fffffff) return false;
    const double pv = A[(size_t)p * lda + k];
    if (!(fabs(pv) > 0.0) || !isfinite(pv)) return false;  // uniform: every thread reads the same value
    __syncthreads();
    if (tid == 0) piv[k] = p;
    if (p != k)
      for (int j = tid; j < N; j += G) {
        const double a = A[(size_t)k * lda + j];
        A[(size_t)k * lda + j] = A[(size_t)p * lda + j];
        A[(size_t)p * lda + j] = a;
      }
    __syncthreads();
    const double ipv = 1.0 / pv;
    for (int i = k + 1 + tid; i < N; i += G) {
      double* row = A + (size_t)i * lda;
      const double l = row[k] * ipv;
      row[k] = l;
      const double* prow = A + (size_t)k * lda;
      for (int j = k + 1; j < N; ++j) row[j] = fma(-l, prow[j], row[j]);
    }
    __syncthreads();
  }
  return true;
}

// Solve (P A = L U) x = b by ONE warp with the right-hand side in registers: lane l owns rows l, l+32, ...
// (NR = ceil(N/32) of them); b[k] travels by shuffle, so there is no shared-memory traffic for b and no
// barrier.  b_in / x_out are shared arrays; must be called by all 32 lanes of the warp.
template <int NR>
__device__ __forceinline__ void lu_solve_warp(const double* __restrict__ A, int lda, int N, const int* __restrict__ piv,
                                              const double* __restrict__ b_in, double* __restrict__ x_out) {
  const int lane = threadIdx.x & 31;
  // apply the row exchanges to b in shared memory order: x_out <- P b (sequential, lane 0)
  if (lane == 0) {
    for (int i = 0; i < N; ++i) x_out[i] = b_in[i];
    for (int k = 0; k < N; ++k) {
      const int p = piv[k];
      if (p != k) { const double t = x_out[k]; x_out[k] = x_out[p]; x_out[p] = t; }
    }
  }
  __syncwarp();
  double b[NR];
#pragma unroll
  for (int r = 0; r < NR; ++r) b[r] = (lane + 32 * r < N) ? x_out[lane + 32 * r] : 0.0;
  // forward substitution with unit L
#pragma unroll
  for (int kk = 0; kk < NR; ++kk) {
    for (int l = 0; l < 32; ++l) {
      const int k = kk * 32 + l;
      if (k >= N) break;
      const double bk = __shfl_sync(0xffffffffu, b[kk], l);
#pragma unroll
      for (int r = 0; r < NR; ++r) {
        const int i = lane + 32 * r;
        if (r >= kk && i > k && i < N) b[r] = fma(-A[(size_t)i * lda + k], bk, b[r]);
      }
    }
  }
  // back substitution with U
#pragma unroll
  for (int kk = NR - 1; kk >= 0; --kk) {
    for (int l = 31; l >= 0; --l) {
      const int k = kk * 32 + l;
      if (k >= N) continue;
      if (lane == l) b[kk] = b[kk] / A[(size_t)k * lda + k];
      const double bk = __shfl_sync(0xffffffffu, b[kk], l);
#pragma unroll
      for (int r = 0; r < NR; ++r) {
        const int i = lane + 32 * r;
        if (r <= kk && i < k) b[r] = fma(-A[(size_t)i * lda + k], bk, b[r]);
      }
    }
  }
#pragma unroll
  for (int r = 0; r < NR; ++r)
    if (lane + 32 * r < N) x_out[lane + 32 * r] = b[r];
  __syncwarp();
}

}  // namespace ck

// ---------------------------------------------------------------------------------------------------------
// Register-resident variant for compile-time N <= G (one thread per matrix row, the row in registers):
// the rank-1 update of step k is N-k register FMAs per thread against the pivot row, which every thread reads
// as a shared-memory broadcast -- 8 bytes of shared-memory traffic per 32 FMAs instead of 24 bytes per FMA in
// the shared-memory version above.  Pivoting is IMPLICIT: rows never move; the thread whose row is chosen at
// step k records pstep = k and drops out of the elimination, so P A = L U holds with P given by pstep.
// One barrier per step for the broadcast (double-buffered) plus one for the cross-warp argmax.
namespace ck {

template <int G>
__device__ __forceinline__ int block_argmax1(double val, int idx, double* red2, int parity) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const double v2 = __shfl_xor_sync(0xffffffffu, val, o);
    const int i2 = __shfl_xor_sync(0xffffffffu, idx, o);
    if (v2 > val || (v2 == val && i2 < idx)) { val = v2; idx = i2; }
  }
  if (G == 32) return idx;
  constexpr int W = G / 32;
  double* rv = red2 + parity * 2 * W;
  int* ri = reinterpret_cast<int*>(rv + W);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { rv[w] = val; ri[w] = idx; }
  __syncthreads();
  double bv = rv[0];
  int bi = ri[0];
#pragma unroll
  for (int i = 1; i < W; ++i) {
    const double v2 = rv[i];
    const int i2 = ri[i];
    if (v2 > bv || (v2 == bv && i2 < bi)) { bv = v2; bi = i2; }
  }
  return bi;
}

// Steps are instantiated by template recursion (compile-time k): nvcc does not fully unroll a 54-trip loop whose
// body holds another unrolled loop, and a partially unrolled loop would index the row dynamically (local memory).
template <int N, int G, int K>
__device__ __forceinline__ void lu_factor_step(double (&a)[N], int& pstep, double* __restrict__ bc, double* red2, bool& ok) {
  if constexpr (K < N) {
    const int tid = threadIdx.x;
    const double v = (pstep == -1) ? fabs(a[K]) : -1.0;
    const int p = block_argmax1<G>(v, tid, red2, K & 1);
    double* b = bc + (K & 1) * N;
    if (tid == p) {
      pstep = K;
#pragma unroll
      for (int j = K; j < N; ++j) b[j] = a[j];
    }
    __syncthreads();
    const double pv = b[K];
    if (!(fabs(pv) > 0.0) || !isfinite(pv)) ok = false;  // uniform; keep going so that barriers stay aligned
    const double ipv = 1.0 / pv;
    if (pstep == -1) {
      const double l = a[K] * ipv;
      a[K] = l;
#pragma unroll
      for (int j = K + 1; j < N; ++j) a[j] = fma(-l, b[j], a[j]);
    } else if (pstep == K) {
      a[K] = ipv;
    }
    lu_factor_step<N, G, K + 1>(a, pstep, bc, red2, ok);
  }
}
template <int N, int G, int K>
__device__ __forceinline__ void lu_fwd_step(const double (&a)[N], int pstep, double& b, double* __restrict__ bs) {
  if constexpr (K < N) {
    if (pstep == K) bs[K & 1] = b;
    __syncthreads();
    if (pstep > K) b = fma(-a[K], bs[K & 1], b);
    lu_fwd_step<N, G, K + 1>(a, pstep, b, bs);
  }
}
template <int N, int G, int K>
__device__ __forceinline__ void lu_bwd_step(const double (&a)[N], int pstep, double& b, double* __restrict__ bs) {
  if constexpr (K >= 0) {
    if (pstep == K) { b *= a[K]; bs[K & 1] = b; }
    __syncthreads();
    if (pstep >= 0 && pstep < K) b = fma(-a[K], bs[K & 1], b);
    lu_bwd_step<N, G, K - 1>(a, pstep, b, bs);
  }
}

// a: this thread's row (thread tid < N owns row tid).  bc: shared scratch of 2*N doubles; red2: 4*(G/32)+8 doubles.
// On return a holds L (multipliers, columns < pstep), 1/U_kk at column pstep, U beyond it.  false: zero pivot.
template <int N, int G>
__device__ __forceinline__ bool lu_factor_rows(double (&a)[N], int& pstep, double* __restrict__ bc, double* red2) {
  pstep = (threadIdx.x < N) ? -1 : -2;
  bool ok = true;
  lu_factor_step<N, G, 0>(a, pstep, bc, red2, ok);
  __syncthreads();
  return ok;
}

// Solve with the factors left by lu_factor_rows.  b: this thread's right-hand-side entry (row tid) on entry, the
// solution component x[pstep] on return.  bs: shared scratch of 2 doubles.
template <int N, int G>
__device__ __forceinline__ void lu_solve_rows(const double (&a)[N], int pstep, double& b, double* __restrict__ bs) {
  lu_fwd_step<N, G, 0>(a, pstep, b, bs);       // forward: L y = P b
  lu_bwd_step<N, G, N - 1>(a, pstep, b, bs);   // backward: U x = y
  __syncthreads();
}

}  // namespace ck

// ---------------------------------------------------------------------------------------------------------
// Generic-N variant of the same scheme with the rows in shared memory (thread tid < N owns row tid, implicit
// pivoting, runtime N <= G): small code (no unrolling over k), and the rank-1 update is register-blocked eight
// columns at a time -- all loads issued before the FMAs and stores -- because a one-column-per-trip loop is bound
// by the shared-memory round trip of each iteration (measured: 100 cycles per FMA).
// dinv[k] receives 1/U_kk.  The barrier inside block_argmax1 of step k+1 orders step k's row updates before any
// read of the next pivot row, so there is one barrier per step (G > 32) or a __syncwarp (G == 32).
namespace ck {

// Pivot search with the pivot's reciprocal riding along: `v` = |candidate| (or -1 for rows that are out), `inv` =
// 1/candidate computed by the caller OFF the critical path.  Warp stage: two REDUX.MAX over the 64-bit pattern of
// |x| (monotone as an unsigned integer; +1 on the high word so that a live zero still beats a dead row) and a
// ballot for the first lane holding the maximum; CTA stage: one shared-memory exchange and one barrier.
// red2: 2 parities x 4 x (G/32) doubles.  Returns the pivot row; *ipv = its reciprocal.
template <int G>
__device__ __forceinline__ int block_argmax2(double v, double inv, int idx, double* red2, int parity, double* ipv) {
  const unsigned hi = (v >= 0.0 || v != v) ? (unsigned)__double2hiint(fabs(v)) + 1u : 0u;
  const unsigned lo = (unsigned)__double2loint(v);
  const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
  const unsigned lo2 = (hi == mh) ? lo : 0u;
  const unsigned ml = __reduce_max_sync(0xffffffffu, lo2);
  const unsigned win = __ballot_sync(0xffffffffu, hi == mh && lo2 == ml);
  const int wl = __ffs(win) - 1;
  int bi = __shfl_sync(0xffffffffu, idx, wl);
  double binv = __shfl_sync(0xffffffffu, inv, wl);
  if (G == 32) { *ipv = binv; return bi; }
  constexpr int W = G / 32;
  double* base = red2 + parity * 4 * W;
  unsigned* rk = reinterpret_cast<unsigned*>(base);           // [W][2] keys
  int* ri = reinterpret_cast<int*>(base + W);                 // [W] rows
  double* rinv = base + 2 * W;                                // [W] reciprocals
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { rk[2 * w] = mh; rk[2 * w + 1] = ml; ri[w] = bi; rinv[w] = binv; }
  __syncthreads();
  unsigned bh = rk[0], bl = rk[1];
  bi = ri[0]; binv = rinv[0];
#pragma unroll
  for (int i = 1; i < W; ++i) {
    const unsigned h2 = rk[2 * i], l2 = rk[2 * i + 1];
    if (h2 > bh || (h2 == bh && l2 > bl)) { bh = h2; bl = l2; bi = ri[i]; binv = rinv[i]; }
  }
  *ipv = binv;
  return bi;
}

template <int G>
__device__ __forceinline__ bool lu_factor_rows_smem(double* __restrict__ A, int lda, int N, int& pstep,
                                                    double* __restrict__ dinv, double* red2) {
  const int tid = threadIdx.x;
  pstep = (tid < N) ? -1 : -2;
  bool ok = true;
  double* row = A + (size_t)(tid < N ? tid : 0) * lda;
  double cand = row[0];
  double cinv = 1.0 / cand;
  for (int k = 0; k < N; ++k) {
    double ipv;
    const int p = block_argmax2<G>((pstep == -1) ? fabs(cand) : -1.0, cinv, tid, red2, k & 1, &ipv);
    if (G == 32) __syncwarp();
    if (!isfinite(ipv) || ipv == 0.0) ok = false;  // zero / non-finite pivot (uniform)
    const double* prow = A + (size_t)p * lda;
    if (tid == p) { pstep = k; dinv[k] = ipv; }
    else if (pstep == -1) {
      const double l = cand * ipv;
      row[k] = l;
      int j = k + 1;
      if (j < N) {  // next step's candidate and its reciprocal first: they head the next step's critical path
        cand = fma(-l, prow[j], row[j]);
        row[j] = cand;
        cinv = 1.0 / cand;
        ++j;
      }
      for (; j + 8 <= N; j += 8) {
        double r[8], u[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) { r[x] = row[j + x]; u[x] = prow[j + x]; }
#pragma unroll
        for (int x = 0; x < 8; ++x) row[j + x] = fma(-l, u[x], r[x]);
      }
      if (j < N) {  // ragged tail as ONE predicated block: a scalar loop pays a shared-memory round trip per column
        double r[8], u[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) { r[x] = (j + x < N) ? row[j + x] : 0.0; u[x] = (j + x < N) ? prow[j + x] : 0.0; }
#pragma unroll
        for (int x = 0; x < 8; ++x) if (j + x < N) row[j + x] = fma(-l, u[x], r[x]);
      }
    }
  }
  __syncthreads();
  return ok;
}

// b: entry `tid` of the right-hand side on entry, x[pstep] on return.  bs: 2 doubles of shared scratch.
template <int G>
__device__ __forceinline__ void lu_solve_rows_smem(const double* __restrict__ A, int lda, int N, int pstep,
                                                   const double* __restrict__ dinv, double& b, double* __restrict__ bs) {
  const double* row = A + (size_t)(threadIdx.x < N ? threadIdx.x : 0) * lda;
  for (int k0 = 0; k0 < N; k0 += 4) {  // forward: L y = P b ; multipliers prefetched four steps ahead
    double l[4];
#pragma unroll
    for (int x = 0; x < 4; ++x) l[x] = (k0 + x < N) ? row[k0 + x] : 0.0;
#pragma unroll
    for (int x = 0; x < 4; ++x) {
      const int k = k0 + x;
      if (k < N) {
        if (pstep == k) bs[k & 1] = b;
        __syncthreads();
        if (pstep > k) b = fma(-l[x], bs[k & 1], b);
      }
    }
  }
  for (int k0 = N - 1; k0 >= 0; k0 -= 4) {  // backward: U x = y
    double u[4];
#pragma unroll
    for (int x = 0; x < 4; ++x) u[x] = (k0 - x >= 0) ? row[k0 - x] : 0.0;
#pragma unroll
    for (int x = 0; x < 4; ++x) {
      const int k = k0 - x;
      if (k >= 0) {
        if (pstep == k) { b *= dinv[k]; bs[k & 1] = b; }
        __syncthreads();
        if (pstep >= 0 && pstep < k) b = fma(-u[x], bs[k & 1], b);
      }
    }
  }
  __syncthreads();
}

}  // namespace ck

// ---------------------------------------------------------------------------------------------------------
// Stage solves, four elimination steps per barrier.  lu_solve_rows_smem spends one barrier round trip per step
// (2N per solve, ~100 cycles each, nothing to overlap it with); here the owners of four consecutive steps publish
// their entries of b together, and every thread solves the 4 x 4 triangular diagonal block redundantly from a
// compact copy of it (Lb / Ub, filled once per factorisation by lu_compact4) before updating its own entry with four
// FMAs.  The operation order per entry is that of the step-by-step solve, so the results are bit-identical.
namespace ck {

// Lb[3k + x] = L[p_k][k0 + x] for k0 + x < k,  Ub[3k + x] = U[p_k][k + 1 + x] for k + 1 + x <= k0 + 3  (k0 = k & ~3,
// p_k the row chosen at step k); zero elsewhere.  Lb, Ub: 3N doubles each.
template <int G>
__device__ __forceinline__ void lu_compact4(const double* __restrict__ A, int lda, int N, int pstep, double* __restrict__ Lb,
                                            double* __restrict__ Ub) {
  if (pstep >= 0) {
    const int k = pstep, k0 = k & ~3;
    const double* row = A + (size_t)threadIdx.x * lda;
#pragma unroll
    for (int x = 0; x < 3; ++x) {
      Lb[3 * k + x] = (k0 + x < k) ? row[k0 + x] : 0.0;
      const int j = k + 1 + x;
      Ub[3 * k + x] = (j <= k0 + 3 && j < N) ? row[j] : 0.0;
    }
  }
  __syncthreads();
}

// One block of NB <= 4 steps of the forward (FWD) or backward substitution; straight-line code (selects, no
// branches: with two warps per CTA a taken branch costs more than the arithmetic it skips).
template <int NB, bool FWD>
__device__ __forceinline__ void lu_solve_block4(const double* __restrict__ row, int k0, int pstep, const double* __restrict__ dinv,
                                                const double* __restrict__ Lb, const double* __restrict__ Ub, double& b,
                                                double* __restrict__ bsp) {
  double l[NB];
#pragma unroll
  for (int x = 0; x < NB; ++x) l[x] = row[k0 + x];
  const int o = pstep - k0;
  if (o >= 0 && o < NB) bsp[o] = b;
  __syncthreads();
  double v[4] = {0.0, 0.0, 0.0, 0.0};
  if constexpr (FWD) {
    const double* L = Lb + 3 * k0;
    v[0] = bsp[0];
    if constexpr (NB > 1) v[1] = fma(-L[3], v[0], bsp[1]);
    if constexpr (NB > 2) v[2] = fma(-L[7], v[1], fma(-L[6], v[0], bsp[2]));
    if constexpr (NB > 3) v[3] = fma(-L[11], v[2], fma(-L[10], v[1], fma(-L[9], v[0], bsp[3])));
    double upd = b;
#pragma unroll
    for (int x = 0; x < NB; ++x) upd = fma(-l[x], v[x], upd);
    b = (o >= NB) ? upd : b;
  } else {
    const double* U = Ub + 3 * k0;
    if constexpr (NB > 3) v[3] = bsp[3] * dinv[k0 + 3];
    if constexpr (NB > 2) v[2] = (NB > 3 ? fma(-U[6], v[3], bsp[2]) : bsp[2]) * dinv[k0 + 2];
    if constexpr (NB > 1) {
      double t = bsp[1];
      if constexpr (NB > 3) t = fma(-U[4], v[3], t);
      if constexpr (NB > 2) t = fma(-U[3], v[2], t);
      v[1] = t * dinv[k0 + 1];
    }
    {
      double t = bsp[0];
      if constexpr (NB > 3) t = fma(-U[2], v[3], t);
      if constexpr (NB > 2) t = fma(-U[1], v[2], t);
      if constexpr (NB > 1) t = fma(-U[0], v[1], t);
      v[0] = t * dinv[k0];
    }
    double upd = b;
#pragma unroll
    for (int x = NB - 1; x >= 0; --x) upd = fma(-l[x], v[x], upd);
    b = (pstep >= 0 && o < 0) ? upd : b;
  }
  b = (o == 0) ? v[0] : b;
  b = (o == 1) ? v[1] : b;
  b = (o == 2) ? v[2] : b;
  b = (o == 3) ? v[3] : b;
}

// b: entry `tid` of the right-hand side on entry, x[pstep] on return.  bs: 8 doubles of shared scratch.
template <int G>
__device__ __forceinline__ void lu_solve_rows_blk(const double* __restrict__ A, int lda, int N, int pstep,
                                                  const double* __restrict__ dinv, const double* __restrict__ Lb,
                                                  const double* __restrict__ Ub, double& b, double* __restrict__ bs) {
  const double* row = A + (size_t)(threadIdx.x < N ? threadIdx.x : 0) * lda;
  const int Nf = N & ~3, tail = N & 3;
  int par = 0;
#pragma unroll 2
  for (int k0 = 0; k0 < Nf; k0 += 4, par ^= 4) lu_solve_block4<4, true>(row, k0, pstep, dinv, Lb, Ub, b, bs + par);
  if (tail) {  // the ragged last block, forward then backward (uniform branch, once per solve)
    if (tail == 1) { lu_solve_block4<1, true>(row, Nf, pstep, dinv, Lb, Ub, b, bs + par); par ^= 4; lu_solve_block4<1, false>(row, Nf, pstep, dinv, Lb, Ub, b, bs + par); }
    else if (tail == 2) { lu_solve_block4<2, true>(row, Nf, pstep, dinv, Lb, Ub, b, bs + par); par ^= 4; lu_solve_block4<2, false>(row, Nf, pstep, dinv, Lb, Ub, b, bs + par); }
    else { lu_solve_block4<3, true>(row, Nf, pstep, dinv, Lb, Ub, b, bs + par); par ^= 4; lu_solve_block4<3, false>(row, Nf, pstep, dinv, Lb, Ub, b, bs + par); }
    par ^= 4;
  }
#pragma unroll 2
  for (int k0 = Nf - 4; k0 >= 0; k0 -= 4, par ^= 4) lu_solve_block4<4, false>(row, k0, pstep, dinv, Lb, Ub, b, bs + par);
  __syncthreads();
}

}  // namespace ck
