// ck_integrate_ros, batched rounds: every step ATTEMPT of every active reactor is one pass through a short pipeline
// of kernels over the compacted active list (the divergence-control layer of SURVEY.md 8(a) a14: active-reactor
// compaction and re-batching between step attempts).
//
// Why: in the fused CTA-per-reactor kernel (ck_ros.cu) the chemistry -- f(y), the analytic Jacobian and two stage
// evaluations per attempt -- runs CTA-cooperatively at ~4 k SM-cycles per evaluation, against ~0.7 k for the
// thread-per-reactor tensor-memory kernel of ck_rhs.  Here the chemistry runs thread-per-reactor over the whole active
// list (ck_rhs itself and jac_rows_kernel, ck_jac_tpr.cuh); only what is genuinely per-reactor dense linear algebra --
// the LU factorisation of I/(h gamma) - J and the four stage solves of Eq. 6 -- stays cooperative
// (ck_lu_warp.cuh: blocked, trailing update on the FP64 tensor cores, right-hand sides by shuffle), with the matrix
// streamed in from HBM once per attempt.  One attempt round:
//
//   gather     Yw[:, s] = y[:, act[s]]                                              (thread per slot)
//   jac_rows   f0 = f(y), species rows of J, pieces of row 0 -> F0, JB, HC, all indexed by REACTOR; only for the
//              reactors whose state changed since their last Jacobian -- after a REJECTED attempt y_n, hence f(y_n)
//              and J(y_n), are what they were (a third of config 3's attempts), only h changes          (thread per reactor)
//   lu         row 0, A = I/(h gamma) - J, P A = L U (-> LU, per slot), u1 = A^-1 f0, YT = y + a21 u1   (2-4 warps per slot)
//   ck_rhs     FT = f(YT)                                                                     (thread per slot)
//   solve2     u2 = A^-1 (FT + c21/h u1), YT = y + a31 u1 + a32 u2                            (2-4 warps per slot)
//   ck_rhs     FT = f(YT)
//   solve34    u3, u4, y*, error, accept / reject, new h (Algorithm 1), re-queue   (2-4 warps per slot)
//
// Reactors that reached t_f or failed leave the list; the next round runs on the survivors, compacted.  When few
// are left the round's fixed latency (one thread-per-reactor wave) dominates, so the tail is re-batched once more:
// the survivors finish in the fused CTA-per-reactor kernel in resume mode.  Arithmetic per reactor does not depend
// on its slot or on which driver finishes it beyond rounding order, so both drivers are tested against the oracle.
#include <algorithm>
#include <cstdlib>
#include <vector>

#include "ck_bulk.cuh"
#include "ck_jac_tpr.cuh"
#include "ck_lu_warp.cuh"
#include "ck_ros_common.cuh"

namespace ck {

struct RoundArgs {
  long long n, ld, cap;
  double* y;
  const double* p;
  double dt, rtol, atol, h0;
  int max_steps;
  int *n_accept, *n_reject, *status;
  double* h_last;
  int* att;
  // per-reactor controller state
  double *t, *h, *fac;
  int *nacc, *nrej;
  // active lists and counters: cnt[0] = active now, cnt[1] = appended for the next round
  int *act, *act2, *cnt;
  // need[r]: bit 0 = active in the next round, bit 1 = needs a fresh Jacobian; compacted IN REACTOR ORDER into act2 / jl2
  // (cnt[1] / cnt[3]) -- an atomic append would scatter neighbouring threads over the whole matrix array (measured: +60 %
  // on the Jacobian kernel)
  int *jl, *jl2, *need;
  int always_jac;   // measurement (flags bit 6): a fresh Jacobian for every attempt, as the fused kernel does
  // per-slot arrays
  double *Yw, *Pw, *YT, *FT;       // component-major [N][cap] ([cap] for Pw)
  double* F0;                      // [N][cap] f(y_n), indexed by REACTOR (kept across a rejected attempt)
  double *U1, *U2;                 // reactor-major [cap][N]
  double* HC;                      // [2K+1][cap], indexed by REACTOR
  double* G2;                      // [g2rows][cap]
  double* JB;                      // [cap][lu_stride]: species rows of -J in the layout of the factorisation, by REACTOR
  double* LU;                      // [cap][lu_stride]: L\U of this attempt, by slot (row stride lu_ldr)
  long long lu_stride;
  int lu_ldr;
  double* dinv;                    // [cap][N]
  int* pst;                        // [cap][N] row permutation of the factorisation
  double* hs;                      // [cap] step size of this attempt
  int* flg;                        // [cap] bit 0: clipped to t_f, bit 1: zero pivot
  DevStats* stats;
};

__global__ void ros_init_kernel(RoundArgs a) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (r == 0) { a.cnt[0] = (int)a.n; a.cnt[1] = 0; a.cnt[2] = 0; a.cnt[3] = 0; }
  if (r >= a.n) return;
  a.act[r] = (int)r;
  a.t[r] = 0.0; a.h[r] = a.h0; a.fac[r] = 5.0;
  a.nacc[r] = 0; a.nrej[r] = 0;
  a.need[r] = 0;
}

__global__ void ros_gather_kernel(RoundArgs a, int N) {
  const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= a.cnt[0]) return;
  const int r = a.act[s];
  a.Pw[s] = a.p[r];
  for (int c = 0; c < N; ++c) a.Yw[(size_t)c * a.cap + s] = a.y[(size_t)c * a.ld + r];
}

// EstimateH0 (reading G8), thread per slot.  Part a: d0, d1, h_a, YT = y + h_a f0.  Part b: d2, h0.
__global__ void ros_h0a_kernel(RoundArgs a, int N) {
  const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= a.cnt[0]) return;
  double s0 = 0.0, s1 = 0.0;
  for (int c = 0; c < N; ++c) {
    const double y = a.Yw[(size_t)c * a.cap + s], f = a.F0[(size_t)c * a.cap + s];
    const double w = 1.0 / fma(a.rtol, fabs(y), a.atol);
    s0 = fma(y * w, y * w, s0);
    s1 = fma(f * w, f * w, s1);
  }
  const double d0 = sqrt(s0 / N), d1 = sqrt(s1 / N);
  const double ha = (d0 < 1e-5 || d1 < 1e-5) ? 1e-6 * a.dt : 0.01 * d0 / d1;
  for (int c = 0; c < N; ++c) a.YT[(size_t)c * a.cap + s] = fma(ha, a.F0[(size_t)c * a.cap + s], a.Yw[(size_t)c * a.cap + s]);
  a.hs[s] = ha;
  a.dinv[s] = d1;  // scratch until the first factorisation
}
__global__ void ros_h0b_kernel(RoundArgs a, int N) {
  const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= a.cnt[0]) return;
  const double ha = a.hs[s], d1 = a.dinv[s];
  double s2 = 0.0;
  for (int c = 0; c < N; ++c) {
    const double y = a.Yw[(size_t)c * a.cap + s];
    const double w = (a.FT[(size_t)c * a.cap + s] - a.F0[(size_t)c * a.cap + s]) / fma(a.rtol, fabs(y), a.atol);
    s2 = fma(w, w, s2);
  }
  const double d2 = sqrt(s2 / N) / ha;
  const double dm = fmax(d1, d2);
  const double hb = (dm <= 1e-15) ? fmax(1e-6 * a.dt, 1e-3 * ha) : pow(0.01 / dm, 0.2);
  a.h[a.act[s]] = fmin(fmin(100.0 * ha, hb), a.dt);
}

// reactors whose first step size already fails the guards of Algorithm 1 leave before the first round
__global__ void ros_guard_kernel(RoundArgs a) {
  const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= a.cnt[0]) return;
  const int r = a.act[s];
  const double h = a.h[r];
  int st = CK_ST_OK;
  if (a.max_steps <= 0) st = CK_ST_MAX_STEPS;
  else if (!isfinite(h)) st = CK_ST_NONFINITE;
  else if (h < 1e-12 * a.dt) st = CK_ST_H_UNDERFLOW;
  if (st == CK_ST_OK) { a.need[r] = 3; return; }
  if (a.n_accept) a.n_accept[r] = 0;
  if (a.n_reject) a.n_reject[r] = 0;
  if (a.status) a.status[r] = st;
  if (a.h_last) a.h_last[r] = 0.0;
  a.att[r] = 0;
  atomicAdd(&a.stats->failed, 1ULL);
}
// need[] -> act2 (bit 0: active in the next round) and jl2 (bit 1: needs a fresh Jacobian), both ascending inside a block of
// 1024 reactors (blocks land in the order of their atomics): slots and matrix blocks stay in reactor order
__global__ void __launch_bounds__(1024) ros_lists_kernel(RoundArgs a) {
  __shared__ int wsum[2][32];
  __shared__ int base[2];
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int flg = r < a.n ? a.need[r] : 0;
  const unsigned b0 = __ballot_sync(0xffffffffu, flg & 1), b1 = __ballot_sync(0xffffffffu, flg & 2);
  if (lane == 0) { wsum[0][warp] = __popc(b0); wsum[1][warp] = __popc(b1); }
  __syncthreads();
  if (warp < 2) {
    const int v = wsum[warp][lane];
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    wsum[warp][lane] = x - v;
    if (lane == 31) base[warp] = x > 0 ? atomicAdd(&a.cnt[warp == 0 ? 1 : 3], x) : 0;
  }
  __syncthreads();
  const unsigned below = (1u << lane) - 1u;
  if (flg & 1) a.act2[base[0] + wsum[0][warp] + __popc(b0 & below)] = (int)r;
  if (flg & 2) a.jl2[base[1] + wsum[1][warp] + __popc(b1 & below)] = (int)r;
}
__global__ void ros_swap_kernel(RoundArgs a) { a.cnt[0] = a.cnt[1]; a.cnt[1] = 0; a.cnt[2] = a.cnt[3]; a.cnt[3] = 0; }

// ---- warp-per-reactor kernels: blocked DMMA LU and shuffle solves (ck_lu_warp.cuh); CTA = one warp = one slot ------
// The slot's block in HBM is the shared-memory image of the matrix (luw_np(N) rows of stride luw_lda(N)): it moves
// as a flat vector copy.  pst[] holds the row permutation.
__host__ __device__ inline size_t rw_smem_bytes(int N) {
  const int NP = luw_np(N);
  return ((size_t)luw_block_doubles(N) + 5 * (size_t)NP) * sizeof(double) + (size_t)NP * sizeof(int);
}
struct RwShared { double *A, *dinv, *v0, *v1, *v2, *v3; int* perm; };
__device__ __forceinline__ RwShared rw_carve(double* sm, int N) {
  const int NP = luw_np(N);
  RwShared s;
  s.A = sm; sm += luw_block_doubles(N);
  s.dinv = sm; sm += NP; s.v0 = sm; sm += NP; s.v1 = sm; sm += NP; s.v2 = sm; sm += NP; s.v3 = sm; sm += NP;
  s.perm = reinterpret_cast<int*>(sm);
  return s;
}
// RW warps per CTA: warp 0 runs the serial chains (panel steps, solves), all warps the parallel phases
template <int RWT>
__device__ __forceinline__ void rw_copy_block(double* __restrict__ dst, const double* __restrict__ src, int doubles) {
  const int tid = threadIdx.x;
  const double2* s2 = reinterpret_cast<const double2*>(src);
  double2* d2 = reinterpret_cast<double2*>(dst);
  const int n2 = doubles >> 1;
#pragma unroll 8
  for (int i = tid; i < n2; i += RWT) d2[i] = s2[i];
}
// the slot's matrix block -> shared memory as ONE bulk copy (the caller has made sure that nobody still uses sh.A and waits
// on `bar` with the current parity before reading it)
__device__ __forceinline__ void rw_issue_block_load(const double* __restrict__ src, int N, const RwShared& sh, uint64_t* bar) {
  if (threadIdx.x == 0) {
    fence_async_smem();
    bulk_load(sh.A, src, (uint32_t)(luw_block_doubles(N) * sizeof(double)), bar);
  }
}
template <int RWT>
__device__ __forceinline__ void rw_load_factors(const RoundArgs& a, long long s, int N, const RwShared& sh, uint64_t* bar, uint32_t parity) {
  const int tid = threadIdx.x;
  rw_issue_block_load(a.LU + (size_t)s * a.lu_stride, N, sh, bar);
  for (int i = tid; i < N; i += RWT) { sh.dinv[i] = a.dinv[(size_t)s * N + i]; sh.perm[i] = a.pst[(size_t)s * N + i]; }
  mbar_wait(bar, parity);
}

template <int NR, int RW>
__global__ void __launch_bounds__(32 * RW) ros_lu_w_kernel(RoundArgs a, int K) {
  using namespace ros4c;
  constexpr int RWT = 32 * RW;
  extern __shared__ double sm[];
  __shared__ int s_ok;
  __shared__ __align__(8) uint64_t s_bar;
  const int N = K + 1, lda = luw_lda(N), NP = luw_np(N), tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const RwShared sh = rw_carve(sm, N);
  const long long na = a.cnt[0];
  if (tid == 0) mbar_init(&s_bar, 1);
  uint32_t parity = 0;
  for (long long s = blockIdx.x; s < na; s += gridDim.x) {
    const int r = a.act[s];
    if (tid == 0) bulk_store_wait_read();   // the previous slot's factors have left shared memory
    __syncthreads();
    double* blk = a.LU + (size_t)s * a.lu_stride;
    // the reactor's block (rows 1..K of -J, written by jac_rows_kernel in the image's layout) arrives as one bulk copy
    rw_issue_block_load(a.JB + (size_t)r * a.lu_stride, N, sh, &s_bar);
    for (int k = tid; k < K; k += RWT) { sh.v0[k] = a.HC[(size_t)k * a.cap + r]; sh.v1[k] = a.HC[(size_t)(K + k) * a.cap + r]; }
    for (int i = tid; i < N; i += RWT) sh.v2[i] = a.F0[(size_t)i * a.cap + r];
    double h = a.h[r];
    const double trem = a.dt - a.t[r];
    int flg = 0;
    if (h >= trem) { h = trem; flg = 1; }
    const double ihg = 1.0 / (h * gam);
    mbar_wait(&s_bar, parity);
    parity ^= 1u;
    // padding rows / columns of the image: stale (factors of an earlier round, or never written)
    for (int idx = tid; idx < (NP - N) * lda; idx += RWT) sh.A[(size_t)N * lda + idx] = 0.0;
    for (int i = tid; i < NP; i += RWT)
      for (int j = jac_np(N); j < lda; ++j) sh.A[(size_t)i * lda + j] = 0.0;
    __syncthreads();
    // row 0 of A = I/(h gamma) - J from the (negated) species rows (ck_jac_tpr.cuh): -J_0j = -sum_k hh_k M_kj + f_T cc_j
    const double fT = sh.v2[0];
    const double jtt = a.HC[(size_t)(2 * K) * a.cap + r];
    for (int j = tid; j < NP; j += RWT) {
      double acc0 = 0.0, acc1 = 0.0;
      int k = 0;
      for (; k + 1 < K; k += 2) {
        acc0 = fma(sh.v0[k], sh.A[(size_t)(1 + k) * lda + j], acc0);
        acc1 = fma(sh.v0[k + 1], sh.A[(size_t)(2 + k) * lda + j], acc1);
      }
      if (k < K) acc0 = fma(sh.v0[k], sh.A[(size_t)(1 + k) * lda + j], acc0);
      const double acc = acc0 + acc1;
      sh.A[j] = (j >= N) ? 0.0 : ((j == 0) ? (-jtt - acc) : (fT * sh.v1[j - 1] - acc));
    }
    __syncthreads();
    for (int i = tid; i < N; i += RWT) sh.A[(size_t)i * lda + i] += ihg;
    __syncthreads();
    const bool ok = lu_factor_warp_dmma<NR, RW>(sh.A, lda, N, sh.perm, sh.dinv);
    if (tid == 0) s_ok = ok ? 1 : 0;
    __syncthreads();
    if (!s_ok) flg |= 2;
    fence_async_smem();      // the factors, written through the generic proxy, become visible to the bulk store
    __syncthreads();
    if (tid == 0) bulk_store(blk, sh.A, (uint32_t)(luw_block_doubles(N) * sizeof(double)));
    for (int i = tid; i < N; i += RWT) { a.dinv[(size_t)s * N + i] = sh.dinv[i]; a.pst[(size_t)s * N + i] = sh.perm[i]; }
    if (warp == 0) {
      double bb[NR];
#pragma unroll
      for (int q = 0; q < NR; ++q) { const int i = lane + 32 * q; bb[q] = (i < N) ? sh.v2[sh.perm[i]] : 0.0; }
      lu_solve_warp_regs<NR>(sh.A, lda, N, sh.dinv, bb);   // u1 = A^-1 f0
#pragma unroll
      for (int q = 0; q < NR; ++q) {
        const int i = lane + 32 * q;
        if (i < N) {
          a.U1[(size_t)s * N + i] = bb[q];
          a.YT[(size_t)i * a.cap + s] = fma(a21, bb[q], a.Yw[(size_t)i * a.cap + s]);
        }
      }
      if (lane == 0) { a.hs[s] = h; a.flg[s] = flg; }
    }
  }
  if (tid == 0) bulk_store_wait_read();
}

template <int NR, int RW>
__global__ void __launch_bounds__(32 * RW) ros_solve2_w_kernel(RoundArgs a, int K) {
  using namespace ros4c;
  constexpr int RWT = 32 * RW;
  extern __shared__ double sm[];
  const int N = K + 1, lda = luw_lda(N), tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const RwShared sh = rw_carve(sm, N);
  __shared__ __align__(8) uint64_t s_bar;
  if (threadIdx.x == 0) mbar_init(&s_bar, 1);
  uint32_t parity = 0;
  const long long na = a.cnt[0];
  for (long long s = blockIdx.x; s < na; s += gridDim.x) {
    __syncthreads();
    rw_load_factors<RWT>(a, s, N, sh, &s_bar, parity);
    parity ^= 1u;
    const double ih = 1.0 / a.hs[s];
    for (int i = tid; i < N; i += RWT) {
      const double u1 = a.U1[(size_t)s * N + i];
      sh.v0[i] = u1;
      sh.v2[i] = fma(c21 * ih, u1, a.FT[(size_t)i * a.cap + s]);
    }
    __syncthreads();
    if (warp == 0) {
      double bb[NR];
#pragma unroll
      for (int q = 0; q < NR; ++q) { const int i = lane + 32 * q; bb[q] = (i < N) ? sh.v2[sh.perm[i]] : 0.0; }
      lu_solve_warp_regs<NR>(sh.A, lda, N, sh.dinv, bb);   // u2
#pragma unroll
      for (int q = 0; q < NR; ++q) {
        const int i = lane + 32 * q;
        if (i < N) {
          a.U2[(size_t)s * N + i] = bb[q];
          a.YT[(size_t)i * a.cap + s] = a.Yw[(size_t)i * a.cap + s] + a31 * sh.v0[i] + a32 * bb[q];
        }
      }
    }
  }
}

template <int NR, int RW>
__global__ void __launch_bounds__(32 * RW) ros_solve34_w_kernel(RoundArgs a, int K) {
  using namespace ros4c;
  constexpr int RWT = 32 * RW;
  extern __shared__ double sm[];
  const int N = K + 1, lda = luw_lda(N), tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const RwShared sh = rw_carve(sm, N);
  __shared__ __align__(8) uint64_t s_bar;
  if (threadIdx.x == 0) mbar_init(&s_bar, 1);
  uint32_t parity = 0;
  const long long na = a.cnt[0];
  unsigned long long c_acc = 0, c_rej = 0, c_fail = 0;
  for (long long s = blockIdx.x; s < na; s += gridDim.x) {
    const int r = a.act[s];
    __syncthreads();
    rw_load_factors<RWT>(a, s, N, sh, &s_bar, parity);
    parity ^= 1u;
    const double h = a.hs[s], ih = 1.0 / h;
    const int flg = a.flg[s];
    double u1[NR], u2[NR], ft[NR], y0[NR];
#pragma unroll
    for (int q = 0; q < NR; ++q) {
      const int i = lane + 32 * q;
      const bool in = warp == 0 && i < N;
      u1[q] = in ? a.U1[(size_t)s * N + i] : 0.0;
      u2[q] = in ? a.U2[(size_t)s * N + i] : 0.0;
      ft[q] = in ? a.FT[(size_t)i * a.cap + s] : 0.0;
      y0[q] = in ? a.Yw[(size_t)i * a.cap + s] : 0.0;
      if (in) sh.v2[i] = ft[q] + (c31 * u1[q] + c32 * u2[q]) * ih;
    }
    __syncthreads();
    if (warp != 0) continue;
    double u3[NR], u4[NR];
#pragma unroll
    for (int q = 0; q < NR; ++q) { const int i = lane + 32 * q; u3[q] = (i < N) ? sh.v2[sh.perm[i]] : 0.0; }
    lu_solve_warp_regs<NR>(sh.A, lda, N, sh.dinv, u3);
#pragma unroll
    for (int q = 0; q < NR; ++q) {
      const int i = lane + 32 * q;
      if (i < N) sh.v3[i] = ft[q] + (c41 * u1[q] + c42 * u2[q] + c43 * u3[q]) * ih;
    }
    __syncwarp();
#pragma unroll
    for (int q = 0; q < NR; ++q) { const int i = lane + 32 * q; u4[q] = (i < N) ? sh.v3[sh.perm[i]] : 0.0; }
    lu_solve_warp_regs<NR>(sh.A, lda, N, sh.dinv, u4);
    double es = 0.0, yn[NR];
#pragma unroll
    for (int q = 0; q < NR; ++q) {
      const int i = lane + 32 * q;
      yn[q] = 0.0;
      if (i < N) {
        yn[q] = y0[q] + m1 * u1[q] + m2 * u2[q] + m3 * u3[q] + m4 * u4[q];
        const double e = e1 * u1[q] + e2 * u2[q] + e3 * u3[q] + e4 * u4[q];
        const double w = e / fma(a.rtol, fmax(fabs(y0[q]), fabs(yn[q])), a.atol);
        es = fma(w, w, es);
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) es += __shfl_xor_sync(0xffffffffu, es, o);
    const double err = sqrt(es / N);
    double tcur = a.t[r], hn = h, fac_max = a.fac[r];
    int nacc = a.nacc[r], nrej = a.nrej[r], status = CK_ST_OK;
    bool done = false, accepted = false;
    if (flg & 2) { status = CK_ST_ZERO_PIVOT; done = true; }
    else if (isfinite(err) && err < 1.0) {
#pragma unroll
      for (int q = 0; q < NR; ++q) { const int i = lane + 32 * q; if (i < N) a.y[(size_t)i * a.ld + r] = yn[q]; }
      tcur = (flg & 1) ? a.dt : tcur + h;
      nacc++;
      accepted = true;
      hn = h * fmin(fac_max, fmax(0.2, 0.9 * pow(fmax(err, 1e-10), -0.25)));
      fac_max = 5.0;
      c_acc++;
    } else {
      nrej++;
      hn = h * (isfinite(err) ? fmin(1.0, fmax(0.2, 0.9 * pow(fmax(err, 1e-10), -0.25))) : 0.2);
      fac_max = 1.0;
      c_rej++;
    }
    if (!done) {
      if (!(tcur < a.dt)) done = true;
      else if (nacc + nrej >= a.max_steps) { status = CK_ST_MAX_STEPS; done = true; }
      else if (!isfinite(hn)) { status = CK_ST_NONFINITE; done = true; }
      else if (hn < 1e-12 * a.dt) { status = CK_ST_H_UNDERFLOW; done = true; }
    }
    if (lane == 0) {
      a.t[r] = tcur; a.h[r] = hn; a.fac[r] = fac_max; a.nacc[r] = nacc; a.nrej[r] = nrej;
      if (done) {
        if (a.n_accept) a.n_accept[r] = nacc;
        if (a.n_reject) a.n_reject[r] = nrej;
        if (a.status) a.status[r] = status;
        if (a.h_last) a.h_last[r] = (flg & 2) ? 0.0 : h;
        a.att[r] = nacc + nrej;
        a.need[r] = 0;
        c_fail += (status != CK_ST_OK);
      } else {
        a.need[r] = (accepted || a.always_jac) ? 3 : 1;   // still active; y_n moved: f(y_n) and J(y_n) are due again
      }
    }
  }
  if (tid == 0) {
    atomicAdd(&a.stats->attempts, c_acc + c_rej);
    atomicAdd(&a.stats->accepted, c_acc);
    atomicAdd(&a.stats->rejected, c_rej);
    atomicAdd(&a.stats->failed, c_fail);
  }
}

}  // namespace ck

using namespace ck;

extern "C" int32_t ck_rhs(const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double* dydt,
                          int64_t ld_out, void* stream);

namespace {
inline size_t al256(size_t x) { return (x + 255) & ~size_t(255); }
inline int rr_lu_ldr(const ck_mech* m) { return luw_lda(m->K + 1); }   // the slot's block is the shared-memory image of the matrix
inline long long rr_lu_stride(const ck_mech* m) {
  const int N = m->K + 1;
  return (long long)luw_block_doubles(N);
}

struct RrLayout {
  size_t att, t, h, fac, nacc, nrej, act, act2, jl, jl2, need, cnt, Yw, Pw, F0, YT, FT, U1, U2, HC, G2, JB, LU, dinv, pst, hs, flg, total;
};
RrLayout rr_layout(const ck_mech* m, int64_t n) {
  const size_t N = m->K + 1, cap = (size_t)n;
  RrLayout L;
  size_t o = sizeof(DevStats);
  auto put = [&](size_t bytes) { const size_t at = o; o += al256(bytes); return at; };
  L.att = put(cap * 4);   // must follow the header: integrate_report reads it there
  L.t = put(cap * 8); L.h = put(cap * 8); L.fac = put(cap * 8);
  L.nacc = put(cap * 4); L.nrej = put(cap * 4);
  L.act = put(cap * 4); L.act2 = put(cap * 4); L.jl = put(cap * 4); L.jl2 = put(cap * 4); L.need = put(cap * 4); L.cnt = put(64);
  L.Yw = put(N * cap * 8); L.Pw = put(cap * 8); L.F0 = put(N * cap * 8); L.YT = put(N * cap * 8); L.FT = put(N * cap * 8);
  L.U1 = put(N * cap * 8); L.U2 = put(N * cap * 8);
  L.HC = put((size_t)jac_hc_rows(m->K) * cap * 8);
  L.G2 = put((size_t)jac_g2_rows(m->R, m->dev.r_tb) * cap * 8);
  L.JB = put(cap * (size_t)rr_lu_stride(m) * 8);
  L.LU = put(cap * (size_t)rr_lu_stride(m) * 8);
  L.dinv = put(cap * N * 8); L.pst = put(cap * N * 4);
  L.hs = put(cap * 8); L.flg = put(cap * 4);
  L.total = o;
  return L;
}

template <int BLOCK>
int32_t launch_jac_rows_rm(const ck_mech* m, const RoundArgs& a, long long na, int sms, cudaStream_t st) {
  const size_t smem = jac_tpr_smem_bytes(m->K, m->R, m->dev.n_tent, m->dev.rstride, BLOCK);
  CK_CUDA(cudaFuncSetAttribute(jac_rows_kernel<BLOCK, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  JacOut o{};
  o.f = a.F0; o.ldf = a.cap; o.J = a.JB; o.ldJ = 0; o.ldr = a.lu_ldr; o.sstride = a.lu_stride;
  o.hc = a.HC; o.ldh = a.cap; o.g2 = a.G2; o.ldg = a.cap;
  o.list = a.jl;   // thread i works on reactor jl[i]: state straight from y, outputs by reactor
  // several threads per reactor while the list leaves lanes (and scratch columns) idle; nsub divides BLOCK / 32
  int nsub = 1;
  const long long lanes = std::min<long long>((long long)sms * BLOCK, a.cap);   // a.cap: columns of the scratch array
  if (BLOCK == 512) { while (nsub < 8 && na * nsub * 2 <= lanes) nsub *= 2; }
  else if (BLOCK == 224 && na * 7 <= lanes) nsub = 7;
  const long long per = BLOCK / nsub;
  const long long grid = std::max<long long>(1, std::min<long long>((na + per - 1) / per, sms));
  jac_rows_kernel<BLOCK, true><<<(unsigned)grid, BLOCK, smem, st>>>(m->dev, na, a.cnt + 2, a.y, a.ld, a.p, o, nsub);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}

template <int NR, int RW>
int32_t launch_warp(const ck_mech* m, const RoundArgs& a, long long na, int sms, int which, cudaStream_t st) {
  constexpr int RWT = 32 * RW;
  const int N = m->K + 1;
  const size_t smem = rw_smem_bytes(N);
  int per_sm = 0;
  auto go = [&](auto kern) -> int32_t {
    CK_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CK_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, RWT, smem));
    const long long grid = std::max<long long>(1, std::min<long long>(na, (long long)std::max(per_sm, 1) * sms));
    kern<<<(unsigned)grid, RWT, smem, st>>>(a, m->K);
    CK_CUDA(cudaGetLastError());
    return CK_OK;
  };
  if (which == 0) return go(ros_lu_w_kernel<NR, RW>);
  if (which == 1) return go(ros_solve2_w_kernel<NR, RW>);
  return go(ros_solve34_w_kernel<NR, RW>);
}

int32_t coop_dispatch(const ck_mech* m, const RoundArgs& a, long long na, int sms, int which, cudaStream_t st) {
  const int N = m->K + 1;
  if (N <= 32) return launch_warp<1, 2>(m, a, na, sms, which, st);
  if (N <= 64) return launch_warp<2, 2>(m, a, na, sms, which, st);
  if (N <= 96) return launch_warp<3, 4>(m, a, na, sms, which, st);
  return launch_warp<4, 4>(m, a, na, sms, which, st);
}
}  // namespace

namespace ck {

bool ros_rounds_supported(const ck_mech* m) {
  const int N = m->K + 1;
  return N <= 128 && jac_tpr_block(m->dev) != 0 && m->dev.rstride <= 64 &&
         rw_smem_bytes(N) <= 227 * 1024;
}
size_t ros_rounds_workspace(const ck_mech* m, int64_t n) { return n > 0 ? rr_layout(m, n).total : sizeof(DevStats); }

int32_t ros_rounds_run(const ck_mech* m, int64_t n, double* y, int64_t ld, const double* p, double dt, const ck_opts* o,
                       int32_t* n_accept, int32_t* n_reject, int32_t* status, double* h_last, void* ws, size_t ws_bytes,
                       int* rounds_out, double* lane_util, cudaStream_t st) {
  const RrLayout L = rr_layout(m, n);
  if (ws_bytes < L.total) { set_error("ck_integrate_ros: workspace of %zu bytes needed, %zu given", L.total, ws_bytes); return CK_EWORKSPACE; }
  const int N = m->K + 1;
  char* w = (char*)ws;
  RoundArgs a{};
  a.n = n; a.ld = ld; a.cap = n; a.y = y; a.p = p; a.dt = dt; a.rtol = o->rtol; a.atol = o->atol; a.h0 = o->h0;
  a.max_steps = o->max_steps > 0 ? o->max_steps : 100000;
  a.always_jac = (o->flags & 64) ? 1 : 0;
  a.n_accept = n_accept; a.n_reject = n_reject; a.status = status; a.h_last = h_last;
  a.stats = (DevStats*)ws;
  a.att = (int*)(w + L.att); a.t = (double*)(w + L.t); a.h = (double*)(w + L.h); a.fac = (double*)(w + L.fac);
  a.nacc = (int*)(w + L.nacc); a.nrej = (int*)(w + L.nrej); a.act = (int*)(w + L.act); a.act2 = (int*)(w + L.act2);
  a.jl = (int*)(w + L.jl); a.jl2 = (int*)(w + L.jl2); a.need = (int*)(w + L.need);
  a.cnt = (int*)(w + L.cnt);
  a.Yw = (double*)(w + L.Yw); a.Pw = (double*)(w + L.Pw); a.F0 = (double*)(w + L.F0); a.YT = (double*)(w + L.YT);
  a.FT = (double*)(w + L.FT); a.U1 = (double*)(w + L.U1); a.U2 = (double*)(w + L.U2); a.HC = (double*)(w + L.HC);
  a.G2 = (double*)(w + L.G2); a.JB = (double*)(w + L.JB); a.LU = (double*)(w + L.LU); a.lu_stride = rr_lu_stride(m); a.lu_ldr = rr_lu_ldr(m); a.dinv = (double*)(w + L.dinv); a.pst = (int*)(w + L.pst);
  a.hs = (double*)(w + L.hs); a.flg = (int*)(w + L.flg);
  int sms = 0;
  CK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, m->device));
  const unsigned tb = 256, gn = (unsigned)((n + tb - 1) / tb);
  int* h_cnt = nullptr;  // pinned: the active count comes back once per round
  CK_CUDA(cudaHostAlloc((void**)&h_cnt, 4 * sizeof(int), cudaHostAllocDefault));
  auto fail = [&](int32_t rc) { cudaFreeHost(h_cnt); return rc; };
  long long nj = 0;   // reactors that need a fresh Jacobian in the coming round
  auto read_count = [&](long long* na) -> int32_t {
    CK_CUDA(cudaMemcpyAsync(h_cnt, a.cnt, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
    CK_CUDA(cudaStreamSynchronize(st));
    *na = h_cnt[0];
    nj = h_cnt[2];
    return CK_OK;
  };
  int32_t rc;
  unsigned long long rhs_evals = 0, jac_evals = 0;
  double slots_act = 0, slots_tot = 0;   // lane utilisation: active slots / lanes issued, summed over the launches
  const int jblock = jac_tpr_block(m->dev), G = 32 * ((N + 31) / 32);
  auto count_tpr = [&](long long na, int block) { slots_act += (double)na; slots_tot += (double)((na + block - 1) / block) * block; };
  ros_init_kernel<<<gn, tb, 0, st>>>(a);
  ros_gather_kernel<<<gn, tb, 0, st>>>(a, N);
  long long na = n;
  if (!(o->h0 > 0.0)) {  // EstimateH0: two evaluations
    if ((rc = ck_rhs(m, na, a.Yw, a.cap, a.Pw, a.F0, a.cap, st))) return fail(rc);
    ros_h0a_kernel<<<gn, tb, 0, st>>>(a, N);
    if ((rc = ck_rhs(m, na, a.YT, a.cap, a.Pw, a.FT, a.cap, st))) return fail(rc);
    ros_h0b_kernel<<<gn, tb, 0, st>>>(a, N);
    rhs_evals += 2 * (unsigned long long)na;
  }
  ros_guard_kernel<<<gn, tb, 0, st>>>(a);
  ros_lists_kernel<<<(unsigned)((n + 1023) / 1024), 1024, 0, st>>>(a);
  ros_swap_kernel<<<1, 1, 0, st>>>(a);
  std::swap(a.act, a.act2);
  std::swap(a.jl, a.jl2);
  if ((rc = read_count(&na))) return fail(rc);
  // the tail (few survivors: a round costs one thread-per-reactor wave whatever the count) goes to the fused kernel
  // A round costs a fixed latency whatever the count (the thread-per-reactor Jacobian alone takes ~2 ms for N = 54, ~3.7 ms
  // for N = 112), the fused kernel a cost per reactor and attempt that grows like N^2..3 (0.19 us for N = 54, 1.4 us for
  // N = 112, measured): the break-even is ~16 k reactors for N = 54 and ~4 k for N = 112.
  const double bq = 54.0 / (double)N;
  const long long tail = std::max<long long>(1, std::min<long long>(n / 4, std::max<long long>(2048, (long long)(16384.0 * bq * bq))));
  int rounds = 0;
  while (na >= tail && na > 0) {
    const unsigned ga = (unsigned)((na + tb - 1) / tb);
    ros_gather_kernel<<<ga, tb, 0, st>>>(a, N);
    if (nj > 0) {
      rc = (jblock == 512) ? launch_jac_rows_rm<512>(m, a, nj, sms, st) : launch_jac_rows_rm<224>(m, a, nj, sms, st);
      if (rc) return fail(rc);
    }
    if ((rc = coop_dispatch(m, a, na, sms, 0, st))) return fail(rc);
    if ((rc = ck_rhs(m, na, a.YT, a.cap, a.Pw, a.FT, a.cap, st))) return fail(rc);
    if ((rc = coop_dispatch(m, a, na, sms, 1, st))) return fail(rc);
    if ((rc = ck_rhs(m, na, a.YT, a.cap, a.Pw, a.FT, a.cap, st))) return fail(rc);
    if ((rc = coop_dispatch(m, a, na, sms, 2, st))) return fail(rc);
    ros_lists_kernel<<<(unsigned)((n + 1023) / 1024), 1024, 0, st>>>(a);
    ros_swap_kernel<<<1, 1, 0, st>>>(a);
    std::swap(a.act, a.act2);
    std::swap(a.jl, a.jl2);
    rhs_evals += 2 * (unsigned long long)na + (unsigned long long)nj; jac_evals += (unsigned long long)nj;
    if (nj > 0) count_tpr(nj, jblock);
    count_tpr(na, 512); count_tpr(na, 512);
    slots_act += 3.0 * na * N; slots_tot += 3.0 * na * G;
    rounds++;
    if ((rc = read_count(&na))) return fail(rc);
  }
  CK_CUDA(cudaGetLastError());
  // counters of the rounds (the fused kernel adds its own below)
  unsigned long long add[2] = {rhs_evals, jac_evals};
  DevStats* ds = a.stats;
  CK_CUDA(cudaMemcpyAsync(h_cnt, a.cnt, sizeof(int), cudaMemcpyDeviceToHost, st));   // keep ordering simple
  CK_CUDA(cudaStreamSynchronize(st));
  {
    DevStats hs;
    CK_CUDA(cudaMemcpy(&hs, ds, sizeof hs, cudaMemcpyDeviceToHost));
    hs.rhs_evals += add[0]; hs.jac_evals += add[1];
    hs.lane_active = (unsigned long long)slots_act; hs.lane_total = (unsigned long long)slots_tot;
    hs.queue = 0;
    CK_CUDA(cudaMemcpy(ds, &hs, sizeof hs, cudaMemcpyHostToDevice));
  }
  if (na > 0) {
    RosArgs f{};
    f.n = n; f.ld = ld; f.y = y; f.p = p; f.dt = dt; f.rtol = o->rtol; f.atol = o->atol; f.h0 = o->h0;
    f.jac_mode = CK_JAC_ANALYTIC; f.max_steps = a.max_steps; f.use_queue = 1;
    f.n_accept = n_accept; f.n_reject = n_reject; f.status = status; f.h_last = h_last;
    f.att = a.att; f.stats = a.stats;
    f.list = a.act; f.list_n = a.cnt; f.rt = a.t; f.rh = a.h; f.rfac = a.fac; f.racc = a.nacc; f.rrej = a.nrej;
    if ((rc = ros_fused_launch(m, f, na, nullptr, st))) return fail(rc);
    rounds++;
  }
  cudaFreeHost(h_cnt);
  *rounds_out = rounds;
  *lane_util = slots_tot > 0 ? slots_act / slots_tot : 1.0;
  return CK_OK;
}

}  // namespace ck

// ---- ck_jac_batched: the thread-per-reactor analytic Jacobian through the C ABI ---------------------------------------
// workspace: f [N][n], HC [2K+1][n], G2 [g2rows][n]
size_t ck_jac_workspace(const ck_mech* m, int64_t n) {
  if (n <= 0) return 256;
  const size_t N = m->K + 1;
  return al256(N * (size_t)n * 8) + al256((size_t)jac_hc_rows(m->K) * n * 8) + al256((size_t)jac_g2_rows(m->R, m->dev.r_tb) * n * 8);
}

namespace {
template <int BLOCK>
int32_t launch_jac_rows_cm(const ck_mech* m, long long n, const double* y, long long ld, const double* p, const JacOut& o,
                           cudaStream_t st) {
  const size_t smem = jac_tpr_smem_bytes(m->K, m->R, m->dev.n_tent, m->dev.rstride, BLOCK);
  CK_CUDA(cudaFuncSetAttribute(jac_rows_kernel<BLOCK, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int sms = 0;
  CK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, m->device));
  const long long grid = std::max<long long>(1, std::min<long long>((n + BLOCK - 1) / BLOCK, sms));
  jac_rows_kernel<BLOCK, false><<<(unsigned)grid, BLOCK, smem, st>>>(m->dev, n, nullptr, y, ld, p, o);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}
}  // namespace

extern "C" int32_t ck_jac_batched(const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double* J,
                                  int64_t ldJ, void* ws, size_t ws_bytes, void* stream) {
  if (!m) { set_error("ck_jac_batched: null mechanism"); return CK_EINVAL; }
  if (n < 0 || ld < n || ldJ < n) { set_error("ck_jac_batched: bad n/ld"); return CK_EINVAL; }
  if (n == 0) return CK_OK;
  if (!y || !p || !J) { set_error("ck_jac_batched: null batch pointer"); return CK_EINVAL; }
  const int block = jac_tpr_block(m->dev);
  if (block == 0 || m->dev.rstride > 64) { set_error("ck_jac_batched: %d species do not fit the thread-per-reactor kernel (use ck_jac)", m->K); return CK_EUNSUPPORTED; }
  if (!ws || ws_bytes < ck_jac_workspace(m, n)) { set_error("ck_jac_batched: workspace of %zu bytes needed", ck_jac_workspace(m, n)); return CK_EWORKSPACE; }
  CK_CUDA(cudaSetDevice(m->device));
  cudaStream_t st = (cudaStream_t)stream;
  const size_t N = m->K + 1;
  char* w = (char*)ws;
  JacOut o{};
  o.f = (double*)w; o.ldf = n; w += al256(N * (size_t)n * 8);
  o.hc = (double*)w; o.ldh = n; w += al256((size_t)jac_hc_rows(m->K) * n * 8);
  o.g2 = (double*)w; o.ldg = n;
  o.J = J; o.ldJ = ldJ;
  int32_t rc = (block == 512) ? launch_jac_rows_cm<512>(m, n, y, ld, p, o, st) : launch_jac_rows_cm<224>(m, n, y, ld, p, o, st);
  if (rc) return rc;
  jac_trow_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(m->K, n, o.f, o.ldf, o.hc, o.ldh, J, ldJ);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}
