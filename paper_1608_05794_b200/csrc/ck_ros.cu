// ck_jac and ck_integrate_ros: CTA-per-reactor kernels with the dense N x N matrix in shared memory.
//
// ROS4 attempt (Eq. 6-7; Table C.3, PAPER.md:455-481 with gamma = 0.57282, a43 = 0, the
// printed "b_i" used as m_i -- DESIGN.md readings G4-G6):
//   f0 = f(y); J = df/dy(y); factor A = I/(h gamma) - J;
//   A u1 = f0;                      f2 = f(y + a21 u1);           A u2 = f2 + (c21/h) u1
//   f3 = f(y + a31 u1 + a32 u2);    A u3 = f3 + (c31 u1 + c32 u2)/h
//   A u4 = f3 + (c41 u1 + c42 u2 + c43 u3)/h;   y* = y + sum m_i u_i;   e = sum E_i u_i
// Driver: Algorithm 1 per reactor, weighted-RMS error, accept iff err < 1,
// controller of DESIGN.md reading G8.  Reactors are handed to CTAs through a device-side work queue (one
// atomic fetch per reactor), so reactors that need many attempts never hold other reactors' lanes idle.
#include <algorithm>
#include <cstdlib>
#include <vector>

#include "ck_coop.cuh"
#include "ck_linalg.cuh"
#include "ck_stats.h"
#include "ck_ros_common.cuh"

namespace ck {


__host__ __device__ inline int ros_lda(int N) { return N | 1; }
// doubles of dynamic shared memory of the ROS4 / jac kernels
// chunk length of the per-reaction derivative arrays: G when thread k can own species row k, else all reactions
__host__ __device__ inline int ros_jc(int K, int G) { return K <= G ? G : 0; }
__host__ __device__ inline size_t ros_smem_doubles(int K, int R, int G) {
  const int N = K + 1;
  return (size_t)N * ros_lda(N) + 12 * (size_t)N + (size_t)(N + 1) / 2 + 8 + coop_chem_doubles(K, R, true, ros_jc(K, G));
}

struct RosShared {
  double *A, *y, *yn, *f0, *ft, *u1, *u2, *u3, *u4, *yt, *rhs, *tmp, *e;
  int* piv;
  CoopChem c;
};
__device__ __forceinline__ RosShared ros_carve(double* sm, int K, int R, int G) {
  const int N = K + 1;
  RosShared s;
  s.A = sm; sm += (size_t)N * ros_lda(N);
  s.y = sm; sm += N; s.yn = sm; sm += N; s.f0 = sm; sm += N; s.ft = sm; sm += N;
  s.u1 = sm; sm += N; s.u2 = sm; sm += N; s.u3 = sm; sm += N; s.u4 = sm; sm += N;
  s.yt = sm; sm += N; s.rhs = sm; sm += N; s.tmp = sm; sm += N; s.e = sm; sm += N;
  s.piv = reinterpret_cast<int*>(sm); sm += (N + 1) / 2 + 8;
  s.c = coop_carve(sm, K, R, true, ros_jc(K, G));
  return s;
}

// weighted RMS norm sqrt(sum (v_i / (rtol |y_i| + atol))^2 / N)
template <int G>
__device__ __forceinline__ double wrms_coop(const double* v, const double* y, int N, double rtol, double atol, double* red) {
  double s = 0.0;
  for (int i = threadIdx.x; i < N; i += G) { const double w = v[i] / fma(rtol, fabs(y[i]), atol); s = fma(w, w, s); }
  return sqrt(block_sum<G>(s, red) / N);
}

// ONE out-of-line copy of the plain evaluation f(y) -> f for the integrator's six call sites (EstimateH0 x 2, two
// stages, FD Jacobian x 2).  Inlined six times it made ros4_kernel ~24 k instructions, and with five CTAs per SM in
// different phases the kernel ran out of instruction cache (every phase slowed down when any phase's code grew).
// Arguments are offsets into the CTA's dynamic shared memory so that the callee still sees shared-memory pointers
// (LDS/STS, not generic accesses); the mechanism is read through the kernel's __grid_constant__ parameter.
template <int G>
__device__ __noinline__ void rhs_stage(const MechDev* __restrict__ mp, int y_off, double p, int f_off) {
  extern __shared__ double sm[];
  const RosShared s = ros_carve(sm, mp->K, mp->R, G);
  TState t;
  rhs_coop<G, false>(*mp, sm + y_off, p, sm + f_off, s.c, t);
}

// Jacobian of the reactor in s.y into s.A: analytic, or CVODE-style forward differences (PAPER.md:281,
// reading G12): sigma_j = max(sqrt(eps)|y_j|, sigma_0 (rtol|y_j| + atol)), sigma_0 = 1000 N eps |h| ||f||_wrms.
// Leaves f(y) in s.f0.  Returns the number of RHS evaluations spent.
template <int G>
__device__ __forceinline__ int jacobian_coop(const MechDev& m, RosShared& s, double p, int mode, double h, double rtol,
                                             double atol) {
  const int N = m.K + 1, lda = ros_lda(N), tid = threadIdx.x;
  TState t;
  if (mode == CK_JAC_ANALYTIC) {
    if (m.K <= G) {  // one pass over the reactions, derivative arrays one chunk long
      const CoopScalars sc = rhs_jac_coop<G>(m, s.y, p, s.f0, s.c, t, s.A, lda);
      jac_coop_finish<G>(m, s.c, sc, t, s.f0, s.A, lda);
    } else {
      const CoopScalars sc = rhs_coop<G, true>(m, s.y, p, s.f0, s.c, t);
      jac_coop<G>(m, s.c, sc, t, s.f0, s.A, lda);
    }
    return 1;
  }
  rhs_stage<G>(&m, (int)(s.y - s.A), p, (int)(s.f0 - s.A));
  const double eps = 2.220446049250313e-16;
  const double fn = wrms_coop<G>(s.f0, s.y, N, rtol, atol, s.c.red);
  const double s0 = (fn != 0.0) ? 1000.0 * N * eps * fabs(h) * fn : 1.0;
  for (int i = tid; i < N; i += G) s.yt[i] = s.y[i];
  __syncthreads();
  for (int j = 0; j < N; ++j) {
    const double yj = s.y[j];
    const double sig = fmax(sqrt(eps) * fabs(yj), s0 * fma(rtol, fabs(yj), atol));
    __syncthreads();
    if (tid == 0) s.yt[j] = yj + sig;
    __syncthreads();
    rhs_stage<G>(&m, (int)(s.yt - s.A), p, (int)(s.ft - s.A));
    for (int i = tid; i < N; i += G) s.A[(size_t)i * lda + j] = (s.ft[i] - s.f0[i]) / sig;
    if (tid == 0) s.yt[j] = yj;
  }
  __syncthreads();
  return N + 1;
}

template <int G>
__global__ void __launch_bounds__(G) jac_kernel(const __grid_constant__ MechDev m, long long n, const double* __restrict__ y, long long ld,
                                                const double* __restrict__ p, int mode, double h, double rtol, double atol,
                                                double* __restrict__ J, long long ldJ) {
  extern __shared__ double sm[];
  RosShared s = ros_carve(sm, m.K, m.R, G);
  const int N = m.K + 1, lda = ros_lda(N), tid = threadIdx.x;
  for (long long r = blockIdx.x; r < n; r += gridDim.x) {
    __syncthreads();
    for (int i = tid; i < N; i += G) s.y[i] = y[(size_t)i * ld + r];
    __syncthreads();
    jacobian_coop<G>(m, s, p[r], mode, h, rtol, atol);
    for (int idx = tid; idx < N * N; idx += G) {
      const int i = idx / N, j = idx - i * N;
      J[(size_t)idx * ldJ + r] = s.A[(size_t)i * lda + j];
    }
  }
}


// EstimateH0 (reading G8; the starting-step rule of the paper's ref. [47]); 2 RHS evaluations
template <int G>
__device__ __forceinline__ double estimate_h0_coop(const MechDev& m, RosShared& s, double p, double dt, double rtol,
                                                   double atol) {
  const int N = m.K + 1, tid = threadIdx.x;
  rhs_stage<G>(&m, (int)(s.y - s.A), p, (int)(s.f0 - s.A));
  const double d0 = wrms_coop<G>(s.y, s.y, N, rtol, atol, s.c.red);
  const double d1 = wrms_coop<G>(s.f0, s.y, N, rtol, atol, s.c.red);
  const double ha = (d0 < 1e-5 || d1 < 1e-5) ? 1e-6 * dt : 0.01 * d0 / d1;
  __syncthreads();
  for (int i = tid; i < N; i += G) s.yt[i] = fma(ha, s.f0[i], s.y[i]);
  __syncthreads();
  rhs_stage<G>(&m, (int)(s.yt - s.A), p, (int)(s.ft - s.A));
  for (int i = tid; i < N; i += G) s.tmp[i] = s.ft[i] - s.f0[i];
  __syncthreads();
  const double d2 = wrms_coop<G>(s.tmp, s.y, N, rtol, atol, s.c.red) / ha;
  const double dm = fmax(d1, d2);
  const double hb = (dm <= 1e-15) ? fmax(1e-6 * dt, 1e-3 * ha) : pow(0.01 / dm, 0.2);
  return fmin(fmin(100.0 * ha, hb), dt);
}

// one stage solve with the register-resident factors: reload this thread's row of L\U from shared memory
template <int NS, int G>
__device__ __forceinline__ void solve_rows_smem(const double* __restrict__ A, int lda, int pstep, const double* __restrict__ b_in,
                                                double* __restrict__ x_out, double* bs) {
  const int tid = threadIdx.x;
  double a[NS];
  if (tid < NS) {
#pragma unroll
    for (int j = 0; j < NS; ++j) a[j] = A[(size_t)tid * lda + j];
  } else {
#pragma unroll
    for (int j = 0; j < NS; ++j) a[j] = 0.0;
  }
  double b = (tid < NS) ? b_in[tid] : 0.0;
  lu_solve_rows<NS, G>(a, pstep, b, bs);
  if (pstep >= 0) x_out[pstep] = b;
  __syncthreads();
}

// minimum resident CTAs per SM the register allocation must allow (shared memory sets the real limit:
// 5 at N = 54; without the bound the kernel takes 254 registers and only 4 CTAs of 64 threads fit)
constexpr int ros_min_ctas(int G) { return G == 32 ? 12 : (G == 64 ? 5 : 1); }

template <int G, int NR, int NS>
__global__ void __launch_bounds__(G, ros_min_ctas(G)) ros4_kernel(const __grid_constant__ MechDev m, const RosArgs a) {
  using namespace ros4c;
  extern __shared__ double sm[];
  __shared__ long long s_next;
  RosShared s = ros_carve(sm, m.K, m.R, G);
  const int N = m.K + 1, lda = ros_lda(N), tid = threadIdx.x;
  long long c_att = 0, c_acc = 0, c_rej = 0, c_rhs = 0, c_jac = 0, c_fail = 0;
  long long r = blockIdx.x;
  for (;;) {
    if (a.use_queue) {
      __syncthreads();
      if (tid == 0) s_next = (long long)atomicAdd(&a.stats->queue, 1ULL);
      __syncthreads();
      r = s_next;
    }
    const bool resume = a.list != nullptr;   // tail of the batched rounds: reactors of an active list continue
    if (r >= (resume ? (long long)*a.list_n : a.n)) break;
    if (resume) r = a.list[r];
    const double p = a.p[r];
    __syncthreads();
    for (int i = tid; i < N; i += G) s.y[i] = a.y[(size_t)i * a.ld + r];
    __syncthreads();
    double tcur = 0.0, h, fac_max = 5.0, h_used = 0.0;
    int nacc = 0, nrej = 0, status = CK_ST_OK;
    if (resume) { tcur = a.rt[r]; h = a.rh[r]; fac_max = a.rfac[r]; nacc = a.racc[r]; nrej = a.rrej[r]; }
    else if (a.h0 > 0.0) h = a.h0;
    else { h = estimate_h0_coop<G>(m, s, p, a.dt, a.rtol, a.atol); c_rhs += 2; }
    const int nacc0 = nacc, nrej0 = nrej;
    while (tcur < a.dt) {
      if (nacc + nrej >= a.max_steps) { status = CK_ST_MAX_STEPS; break; }
      if (!isfinite(h)) { status = CK_ST_NONFINITE; break; }
      if (h < 1e-12 * a.dt) { status = CK_ST_H_UNDERFLOW; break; }
      bool last = false;
      if (h >= a.dt - tcur) { h = a.dt - tcur; last = true; }
      // ---- one attempt ----
      c_rhs += jacobian_coop<G>(m, s, p, a.jac_mode, h, a.rtol, a.atol);
      c_jac++;
      const double ihg = 1.0 / (h * gam), ih = 1.0 / h;
      constexpr bool REG_FULL = NS > 0;   // compile-time N, rows in registers, fully unrolled
      for (int idx = tid; idx < N * lda; idx += G) s.A[idx] = -s.A[idx];
      __syncthreads();
      for (int i = tid; i < N; i += G) s.A[(size_t)i * lda + i] += ihg;
      __syncthreads();
      bool ok;
      int pstep = -2;
      if constexpr (REG_FULL) {  // compile-time N: rows in registers, implicit pivoting (ck_linalg.cuh)
        double arow[NS];
        if (tid < NS) {
#pragma unroll
          for (int j = 0; j < NS; ++j) arow[j] = s.A[(size_t)tid * lda + j];
        } else {
#pragma unroll
          for (int j = 0; j < NS; ++j) arow[j] = 0.0;
        }
        ok = lu_factor_rows<NS, G>(arow, pstep, s.tmp, s.c.red);
        if (tid < NS) {
#pragma unroll
          for (int j = 0; j < NS; ++j) s.A[(size_t)tid * lda + j] = arow[j];
        }
        __syncthreads();
      } else if constexpr (NS < 0) {  // any N <= G: rows in shared memory, implicit pivoting, 8-wide updates
        ok = lu_factor_rows_smem<G>(s.A, lda, N, pstep, s.e, s.c.red);
      } else {
        ok = lu_factor_block<G>(s.A, lda, N, s.piv, s.c.red);
      }
      if (!ok) { status = CK_ST_ZERO_PIVOT; break; }
      // compact copies of the 4 x 4 diagonal blocks for the blocked stage solves; the derivative chunk arrays are
      // dead until the next Jacobian (the stage evaluations below run rhs_coop<G, false>)
      double* const Lb = s.c.dqs;
      double* const Ub = s.c.dqs + 3 * N;
      if constexpr (NS < 0) lu_compact4<G>(s.A, lda, N, pstep, Lb, Ub);
      if constexpr (REG_FULL) solve_rows_smem<NS, G>(s.A, lda, pstep, s.f0, s.u1, s.c.red + 36);
      else if constexpr (NS < 0) {
        double bb = (tid < N) ? s.f0[tid] : 0.0;
        lu_solve_rows_blk<G>(s.A, lda, N, pstep, s.e, Lb, Ub, bb, s.c.red + 32);
        if (pstep >= 0) s.u1[pstep] = bb;
        __syncthreads();
      } else { if (tid < 32) lu_solve_warp<NR>(s.A, lda, N, s.piv, s.f0, s.u1); __syncthreads(); }
      for (int i = tid; i < N; i += G) s.yt[i] = fma(a21, s.u1[i], s.y[i]);
      __syncthreads();
      rhs_stage<G>(&m, (int)(s.yt - s.A), p, (int)(s.ft - s.A));
      for (int i = tid; i < N; i += G) s.rhs[i] = fma(c21 * ih, s.u1[i], s.ft[i]);
      __syncthreads();
      if constexpr (REG_FULL) solve_rows_smem<NS, G>(s.A, lda, pstep, s.rhs, s.u2, s.c.red + 36);
      else if constexpr (NS < 0) {
        double bb = (tid < N) ? s.rhs[tid] : 0.0;
        lu_solve_rows_blk<G>(s.A, lda, N, pstep, s.e, Lb, Ub, bb, s.c.red + 32);
        if (pstep >= 0) s.u2[pstep] = bb;
        __syncthreads();
      } else { if (tid < 32) lu_solve_warp<NR>(s.A, lda, N, s.piv, s.rhs, s.u2); __syncthreads(); }
      for (int i = tid; i < N; i += G) s.yt[i] = s.y[i] + a31 * s.u1[i] + a32 * s.u2[i];
      __syncthreads();
      rhs_stage<G>(&m, (int)(s.yt - s.A), p, (int)(s.ft - s.A));
      c_rhs += 2;
      for (int i = tid; i < N; i += G) s.rhs[i] = s.ft[i] + (c31 * s.u1[i] + c32 * s.u2[i]) * ih;
      __syncthreads();
      if constexpr (REG_FULL) solve_rows_smem<NS, G>(s.A, lda, pstep, s.rhs, s.u3, s.c.red + 36);
      else if constexpr (NS < 0) {
        double bb = (tid < N) ? s.rhs[tid] : 0.0;
        lu_solve_rows_blk<G>(s.A, lda, N, pstep, s.e, Lb, Ub, bb, s.c.red + 32);
        if (pstep >= 0) s.u3[pstep] = bb;
        __syncthreads();
      } else { if (tid < 32) lu_solve_warp<NR>(s.A, lda, N, s.piv, s.rhs, s.u3); __syncthreads(); }
      for (int i = tid; i < N; i += G) s.rhs[i] = s.ft[i] + (c41 * s.u1[i] + c42 * s.u2[i] + c43 * s.u3[i]) * ih;
      __syncthreads();
      if constexpr (REG_FULL) solve_rows_smem<NS, G>(s.A, lda, pstep, s.rhs, s.u4, s.c.red + 36);
      else if constexpr (NS < 0) {
        double bb = (tid < N) ? s.rhs[tid] : 0.0;
        lu_solve_rows_blk<G>(s.A, lda, N, pstep, s.e, Lb, Ub, bb, s.c.red + 32);
        if (pstep >= 0) s.u4[pstep] = bb;
        __syncthreads();
      } else { if (tid < 32) lu_solve_warp<NR>(s.A, lda, N, s.piv, s.rhs, s.u4); __syncthreads(); }
      double es = 0.0;
      for (int i = tid; i < N; i += G) {
        const double yn = s.y[i] + m1 * s.u1[i] + m2 * s.u2[i] + m3 * s.u3[i] + m4 * s.u4[i];
        const double e = e1 * s.u1[i] + e2 * s.u2[i] + e3 * s.u3[i] + e4 * s.u4[i];
        s.yn[i] = yn;
        const double w = e / fma(a.rtol, fmax(fabs(s.y[i]), fabs(yn)), a.atol);
        es = fma(w, w, es);
      }
      const double err = sqrt(block_sum<G>(es, s.c.red) / N);
      h_used = h;
      // ---- accept / reject, new h (same for both solvers except the exponent) ----
      if (isfinite(err) && err < 1.0) {
        __syncthreads();
        for (int i = tid; i < N; i += G) s.y[i] = s.yn[i];
        __syncthreads();
        tcur = last ? a.dt : tcur + h;
        nacc++;
        h *= fmin(fac_max, fmax(0.2, 0.9 * pow(fmax(err, 1e-10), -0.25)));
        fac_max = 5.0;
      } else {
        nrej++;
        h *= isfinite(err) ? fmin(1.0, fmax(0.2, 0.9 * pow(fmax(err, 1e-10), -0.25))) : 0.2;
        fac_max = 1.0;
      }
    }
    __syncthreads();
    for (int i = tid; i < N; i += G) a.y[(size_t)i * a.ld + r] = s.y[i];
    if (tid == 0) {
      if (a.n_accept) a.n_accept[r] = nacc;
      if (a.n_reject) a.n_reject[r] = nrej;
      if (a.status) a.status[r] = status;
      if (a.h_last) a.h_last[r] = h_used;
      a.att[r] = nacc + nrej;
    }
    c_att += (nacc - nacc0) + (nrej - nrej0); c_acc += nacc - nacc0; c_rej += nrej - nrej0; c_fail += (status != CK_ST_OK);
    if (!a.use_queue) { r += gridDim.x; }
  }
  if (tid == 0) {
    atomicAdd(&a.stats->attempts, (unsigned long long)c_att);
    atomicAdd(&a.stats->accepted, (unsigned long long)c_acc);
    atomicAdd(&a.stats->rejected, (unsigned long long)c_rej);
    atomicAdd(&a.stats->rhs_evals, (unsigned long long)c_rhs);
    atomicAdd(&a.stats->jac_evals, (unsigned long long)c_jac);
    atomicAdd(&a.stats->failed, (unsigned long long)c_fail);
  }
}

}  // namespace ck

using namespace ck;

namespace {
inline int group_size(int N) { return N <= 32 ? 32 : (N <= 64 ? 64 : 128); }
constexpr size_t SMEM_CAP = 227 * 1024;

template <int G>
int32_t launch_jac(const ck_mech* m, long long n, const double* y, long long ld, const double* p, int mode, double h,
                   double rtol, double atol, double* J, long long ldJ, cudaStream_t st) {
  const size_t smem = ros_smem_doubles(m->K, m->R, G) * sizeof(double);
  CK_CUDA(cudaFuncSetAttribute(jac_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0, sms = 0;
  CK_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, jac_kernel<G>, G, smem));
  CK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, m->device));
  const long long grid = std::min<long long>(n, (long long)std::max(per_sm, 1) * sms);
  jac_kernel<G><<<(unsigned)grid, G, smem, st>>>(m->dev, n, y, ld, p, mode, h, rtol, atol, J, ldJ);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}

template <int G, int NR, int NS>
int32_t launch_ros(const ck_mech* m, const RosArgs& a, long long n_hint, cudaStream_t st) {
  const size_t smem = ros_smem_doubles(m->K, m->R, G) * sizeof(double);
  CK_CUDA(cudaFuncSetAttribute(ros4_kernel<G, NR, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0, sms = 0;
  CK_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ros4_kernel<G, NR, NS>, G, smem));
  CK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, m->device));
  const long long grid = std::max<long long>(1, std::min<long long>(n_hint, (long long)std::max(per_sm, 1) * sms));
  ros4_kernel<G, NR, NS><<<(unsigned)grid, G, smem, st>>>(m->dev, a);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}
}  // namespace

extern "C" int32_t ck_jac(const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, int32_t mode, double h,
                          double rtol, double atol, double* J, int64_t ldJ, void* stream) {
  if (!m) { set_error("ck_jac: null mechanism"); return CK_EINVAL; }
  if (n < 0 || ld < n || ldJ < n) { set_error("ck_jac: bad n/ld"); return CK_EINVAL; }
  if (mode != CK_JAC_ANALYTIC && mode != CK_JAC_FD) { set_error("ck_jac: bad mode %d", mode); return CK_EINVAL; }
  if (n == 0) return CK_OK;
  if (!y || !p || !J) { set_error("ck_jac: null batch pointer"); return CK_EINVAL; }
  const int N = m->K + 1;
  if (ros_smem_doubles(m->K, m->R, group_size(N)) * sizeof(double) > SMEM_CAP) { set_error("ck_jac: %d x %d matrix does not fit shared memory", N, N); return CK_EUNSUPPORTED; }
  CK_CUDA(cudaSetDevice(m->device));
  cudaStream_t st = (cudaStream_t)stream;
  switch (group_size(N)) {
    case 32: return launch_jac<32>(m, n, y, ld, p, mode, h, rtol, atol, J, ldJ, st);
    case 64: return launch_jac<64>(m, n, y, ld, p, mode, h, rtol, atol, J, ldJ, st);
    default: return launch_jac<128>(m, n, y, ld, p, mode, h, rtol, atol, J, ldJ, st);
  }
}

namespace ck {
// shared by both integrators: validate, zero the stats header, and (after the kernels) assemble the report
int32_t integrate_prologue(const char* who, const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double dt,
                           const ck_opts* o, void* ws, size_t ws_bytes, size_t need, cudaStream_t st) {
  if (!m) { set_error("%s: null mechanism", who); return CK_EINVAL; }
  if (!o || o->struct_size != (int32_t)sizeof(ck_opts)) { set_error("%s: bad ck_opts", who); return CK_EINVAL; }
  if (n < 0 || ld < n) { set_error("%s: bad n/ld", who); return CK_EINVAL; }
  if (!(dt > 0) || !(o->rtol >= 0) || !(o->atol >= 0) || !(o->rtol + o->atol > 0) || !(o->h0 >= 0)) { set_error("%s: bad dt/tolerances", who); return CK_EINVAL; }
  if (n == 0) return CK_OK;
  if (!y || !p) { set_error("%s: null batch pointer", who); return CK_EINVAL; }
  if (!ws || ws_bytes < need) { set_error("%s: workspace of %zu bytes needed, %zu given", who, need, ws_bytes); return CK_EWORKSPACE; }
  CK_CUDA(cudaSetDevice(m->device));
  CK_CUDA(cudaMemsetAsync(ws, 0, sizeof(DevStats), st));
  return CK_OK;
}

int32_t integrate_report(const ck_mech* m, int64_t n, const int32_t* att_dev, const DevStats* stats_dev, int rounds,
                         long long lu_per_jac, ck_report* rep, cudaStream_t st) {
  if (!rep) return CK_OK;
  DevStats hs;
  std::vector<int> att((size_t)n);
  CK_CUDA(cudaMemcpyAsync(&hs, stats_dev, sizeof hs, cudaMemcpyDeviceToHost, st));
  CK_CUDA(cudaMemcpyAsync(att.data(), att_dev, (size_t)n * sizeof(int), cudaMemcpyDeviceToHost, st));
  CK_CUDA(cudaStreamSynchronize(st));
  rep->attempts = (int64_t)hs.attempts; rep->accepted = (int64_t)hs.accepted; rep->rejected = (int64_t)hs.rejected;
  rep->rhs_evals = (int64_t)hs.rhs_evals; rep->jac_evals = (int64_t)hs.jac_evals;
  rep->lu_factor = (int64_t)hs.attempts * lu_per_jac;   // one factorisation per attempt (the Jacobian may be older: ck_ros_rounds.cu)
  rep->simt_efficiency = hs.lane_total ? (double)hs.lane_active / (double)hs.lane_total : 1.0;
  rep->waste_p32 = waste_static(att, 32);
  rep->rounds = rounds;
  rep->n_failed = (int32_t)hs.failed;
  (void)m;
  return CK_OK;
}
}  // namespace ck

// workspace of the fused kernel: [DevStats][int attempts[n]]
namespace ck {
size_t ros_fused_workspace(int64_t n) { return sizeof(DevStats) + (((size_t)n * sizeof(int) + 255) & ~size_t(255)); }

int32_t ros_fused_launch(const ck_mech* m, const RosArgs& a, long long n_hint, int* G_used, cudaStream_t st) {
  const int N = m->K + 1;
  if (ros_smem_doubles(m->K, m->R, group_size(N)) * sizeof(double) > SMEM_CAP || N > 256) {
    set_error("ck_integrate_ros: %d x %d matrix does not fit shared memory", N, N);
    return CK_EUNSUPPORTED;
  }
  if (G_used) *G_used = group_size(N);
  const int NRv = (N + 31) / 32;
  // compile-time-N instantiations (register-resident LU) for the two small model sizes of the paper's Table 1 shapes
  // (K = 9 is config 1, K = 14 the H2/CO-sized model); any other size runs the generic shared-memory path
  if (N == 10) return launch_ros<32, 1, 10>(m, a, n_hint, st);
  if (N == 15) return launch_ros<32, 1, 15>(m, a, n_hint, st);
  if (N <= 32) return launch_ros<32, 1, -1>(m, a, n_hint, st);
  if (N <= 64) return launch_ros<64, 2, -1>(m, a, n_hint, st);
  if (N <= 128) return launch_ros<128, 4, -1>(m, a, n_hint, st);
  if (NRv <= 4) return launch_ros<128, 4, 0>(m, a, n_hint, st);
  return launch_ros<128, 8, 0>(m, a, n_hint, st);
}
}  // namespace ck

size_t ck_ros_workspace(const ck_mech* m, int64_t n) {
  return std::max(ros_fused_workspace(n), ros_rounds_supported(m) ? ros_rounds_workspace(m, n) : (size_t)0);
}

// ck_opts.flags (ROS4): bit 0 static mapping in the fused kernel; bit 2 force the fused CTA-per-reactor kernel;
// bit 3 force the batched rounds (tests run both drivers on the same small batches)
extern "C" int32_t ck_integrate_ros(const ck_mech* m, int64_t n, double* y, int64_t ld, const double* p, double dt,
                                    const ck_opts* o, int32_t* n_accept, int32_t* n_reject, int32_t* status, double* h_last,
                                    void* ws, size_t ws_bytes, ck_report* report, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  if (!m) { set_error("ck_integrate_ros: null mechanism"); return CK_EINVAL; }
  int32_t rc = integrate_prologue("ck_integrate_ros", m, n, y, ld, p, dt, o, ws, ws_bytes, ck_ros_workspace(m, n), st);
  if (rc) return rc;
  if (n == 0) { if (report) *report = ck_report{}; return CK_OK; }
  if (o->jac_mode != CK_JAC_ANALYTIC && o->jac_mode != CK_JAC_FD) { set_error("ck_integrate_ros: bad jac_mode"); return CK_EINVAL; }
  const int N = m->K + 1;
  const bool can_rounds = ros_rounds_supported(m) && o->jac_mode == CK_JAC_ANALYTIC && !(o->flags & 1);
  const bool want_rounds = (o->flags & 8) || (!(o->flags & 4) && N >= 33 && n >= 16384);
  int32_t* att = (int32_t*)((char*)ws + sizeof(DevStats));
  DevStats* stats = (DevStats*)ws;
  int rounds = 1;
  double lane_util;
  if (can_rounds && want_rounds) {
    rc = ros_rounds_run(m, n, y, ld, p, dt, o, n_accept, n_reject, status, h_last, ws, ws_bytes, &rounds, &lane_util, st);
    if (rc) return rc;
  } else {
    RosArgs a{};
    a.n = n; a.ld = ld; a.y = y; a.p = p; a.dt = dt; a.rtol = o->rtol; a.atol = o->atol; a.h0 = o->h0;
    a.jac_mode = o->jac_mode; a.max_steps = o->max_steps > 0 ? o->max_steps : 100000; a.use_queue = !(o->flags & 1);
    a.n_accept = n_accept; a.n_reject = n_reject; a.status = status; a.h_last = h_last;
    a.stats = stats; a.att = att;
    int G = 0;
    rc = ros_fused_launch(m, a, n, &G, st);
    if (rc) return rc;
    // CTA per reactor + work queue: no step-count divergence by construction.  What is reported is the ANALYTIC lane
    // utilisation of the cooperative loops (R reactions resp. N rows dealt over G lanes), not a device counter; ncu's
    // warp execution efficiency of the kernel is quoted beside it in DESIGN.md.
    const double ur = (double)m->R / (G * ((m->R + G - 1) / G)), un = (double)N / (G * ((N + G - 1) / G));
    lane_util = 0.5 * (ur + un);
  }
  if (report) {
    rc = integrate_report(m, n, att, stats, rounds, 1, report, st);
    if (!(can_rounds && want_rounds)) report->simt_efficiency = lane_util;
  }
  return rc;
}
