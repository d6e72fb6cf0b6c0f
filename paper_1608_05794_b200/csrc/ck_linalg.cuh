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
