// ck_integrate_rkf45: embedded Runge-Kutta-Fehlberg 4(5) (Eq. 2-3; Table B.2
// with the repaired cells a42 = -7200/2197, a54 = -845/4104, a64 = 1859/4104 -- DESIGN.md reading G3),
// thread-per-reactor, with the DIVERGENCE-CONTROL LAYER the paper's results call for (PAPER.md:218, 255,
// 363, 419): a persistent kernel in which every lane is a slot that runs the adaptive driver of
// Algorithm 1/2 as a small state machine, one RHS evaluation per loop trip, and
// REFILLS itself from a device-side work queue as soon as its reactor reaches t_f (warp-aggregated
// atomic fetch), so a reactor that needs 900 attempts never keeps the other 31 lanes of its warp waiting.
// flags bit 0 switches the refill off (a warp takes 32 consecutive reactors and waits for the slowest, the
// paper's static mapping) so that both can be measured.  SIMT efficiency = active / issued lane-slots.
//
// Per-slot vectors (y_n, k1..k6, stage argument) live in the caller's workspace, component-major over
// SLOTS (coalesced for every access of the stage loops); the reactor's own column in y_inout is touched
// twice, at fetch and at completion.
#include <algorithm>
#include <vector>

#include <cstdlib>

#include "ck_rhs_tmem.cuh"
#include "ck_coop.cuh"
#include "ck_stats.h"

namespace ck {

// a[s][j]: argument of evaluation s+1 is y + h sum_j a[s][j] k_j ; row 5: 4th-order weights b ; row 6: bhat - b
__constant__ double RKF_T[7][6] = {
    {1.0 / 4, 0, 0, 0, 0, 0},
    {3.0 / 32, 9.0 / 32, 0, 0, 0, 0},
    {1932.0 / 2197, -7200.0 / 2197, 7296.0 / 2197, 0, 0, 0},
    {439.0 / 216, -8.0, 3680.0 / 513, -845.0 / 4104, 0, 0},
    {-8.0 / 27, 2.0, -3544.0 / 2565, 1859.0 / 4104, -11.0 / 40, 0},
    {25.0 / 216, 0, 1408.0 / 2565, 2197.0 / 4104, -1.0 / 5, 0},
    {16.0 / 135 - 25.0 / 216, 0, 6656.0 / 12825 - 1408.0 / 2565, 28561.0 / 56430 - 2197.0 / 4104, -9.0 / 50 + 1.0 / 5,
     2.0 / 55}};

struct RkfArgs {
  long long n, ld, nslots;
  double* y;
  const double* p;
  double dt, rtol, atol, h0;
  int max_steps, refill;
  int *n_accept, *n_reject, *status;
  double* h_last;
  int* att;
  // hand-over records of reactors evicted at an attempt boundary (finished by rkf45_coop_kernel)
  int* elist;           // [n] after the classification phase: reactors to resume (from the front), stragglers (from the back)
  int* elist2;          // [n] reactors evicted at the end-game (narrow finisher, from the front); middle class (from the back)
  int* tmp;             // [n] scratch of rkf_bucket_kernel
  double* rec_t;        // [n] time reached
  double* rec_h;        // [n] next step size
  double* rec_fac;      // [n] fac_max (1 right after a reject)
  int* rec_acc;         // [n]
  int* rec_rej;         // [n]
  int evict;            // 1: end-game eviction enabled
  int cap;              // > 0: classification phase -- every reactor is handed on after `cap` attempts
  double big_steps;     // predicted remaining attempts above which a reactor counts as a straggler (wide finisher)
  double mid_steps;     // ... above which it goes to the narrow finisher at once instead of being resumed thread-per-reactor
  // work list: null = reactors 0..n-1 from stats->queue; else resume reactors rlist[0 .. *rcount) (queue head *rqueue)
  const int* rlist;
  const unsigned long long* rcount;
  unsigned long long* rqueue;
  double* V;  // [8][N][nslots]: 0 = y_n, 1..6 = f evaluations, 7 = stage argument
  DevStats* stats;
};

// Finisher work lists: cls 0 = end-game evictions (front of elist2), 1 = stragglers (back of elist), 2 = middle class
// (back of elist2).  Lists 1 and 2 may be re-ordered longest-first by rkf_order_kernel before they are consumed.
__device__ __forceinline__ long long fin_count(const RkfArgs& a, int cls) {
  return (long long)(cls == 1 ? a.stats->n_evicted_b : (cls == 2 ? a.stats->n_evicted_m : a.stats->n_evicted_n));
}
__device__ __forceinline__ unsigned long long* fin_queue(const RkfArgs& a, int cls) {
  return cls == 1 ? &a.stats->queue_b : (cls == 2 ? &a.stats->queue_m : &a.stats->queue2);
}
__device__ __forceinline__ int* fin_entry(const RkfArgs& a, int cls, long long i) {
  return cls == 1 ? &a.elist[a.n - 1 - i] : (cls == 2 ? &a.elist2[a.n - 1 - i] : &a.elist2[i]);
}

// Longest first: the finisher lists 1 / 2 sorted by predicted remaining attempts, descending (one CTA; rank sort in
// shared memory, n <= RKF_ORDER_MAX).  A straggler that starts late ends late; the order costs nothing else.
constexpr int RKF_ORDER_MAX = 6144;
__global__ void __launch_bounds__(1024) rkf_order_kernel(const RkfArgs a, const int cls) {
  extern __shared__ double sm[];
  const int n = (int)fin_count(a, cls);
  if (n < 2 || n > RKF_ORDER_MAX) return;
  double* key = sm;
  int* id = reinterpret_cast<int*>(sm + RKF_ORDER_MAX);
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const int r = *fin_entry(a, cls, i);
    id[i] = r;
    key[i] = (a.dt - a.rec_t[r]) / a.rec_h[r];
  }
  __syncthreads();
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const double k = key[i];
    int rank = 0;
    for (int j = 0; j < n; ++j) rank += (key[j] > k || (key[j] == k && j < i)) ? 1 : 0;
    *fin_entry(a, cls, rank) = id[i];
  }
}

}  // namespace ck
#include "ck_rkf_wide.cuh"
namespace ck {

// Lists too long for the rank sort are ordered coarsely: four buckets by predicted remaining attempts, descending (order
// inside a bucket is arbitrary).  which = -1: the list of the resumed thread-per-reactor phase (front of elist; a reactor
// that needs 1000 more attempts and is fetched last would add a second to the run), buckets at top / 2, / 4, / 8 with
// top = mid_steps; which = 2: the middle class, top = big_steps.  One CTA; `tmp` (n ints) is the buffer.
__global__ void __launch_bounds__(1024) rkf_bucket_kernel(const RkfArgs a, const int which, int* __restrict__ tmp) {
  __shared__ int cnt[4], cur[4];
  const int n = (int)(which < 0 ? a.stats->n_evicted : fin_count(a, which));
  const double top = which < 0 ? a.mid_steps : a.big_steps;
  if (threadIdx.x < 4) cnt[threadIdx.x] = 0;
  __syncthreads();
  auto entry = [&](int i) -> int* { return which < 0 ? &a.elist[i] : fin_entry(a, which, i); };
  auto bucket = [&](int r) {
    const double pred = (a.dt - a.rec_t[r]) / a.rec_h[r];
    return pred > 0.5 * top ? 0 : (pred > 0.25 * top ? 1 : (pred > 0.125 * top ? 2 : 3));
  };
  for (int i = threadIdx.x; i < n; i += blockDim.x) atomicAdd(&cnt[bucket(*entry(i))], 1);
  __syncthreads();
  if (threadIdx.x == 0) { cur[0] = 0; cur[1] = cnt[0]; cur[2] = cnt[0] + cnt[1]; cur[3] = cnt[0] + cnt[1] + cnt[2]; }
  __syncthreads();
  for (int i = threadIdx.x; i < n; i += blockDim.x) { const int r = *entry(i); tmp[atomicAdd(&cur[bucket(r)], 1)] = r; }
  __syncthreads();
  for (int i = threadIdx.x; i < n; i += blockDim.x) *entry(i) = tmp[i];
}

enum { ST_H0A = -2, ST_H0B = -1 };  // EstimateH0 evaluations; 0..5 = RK stages

// TM = true: production-rate accumulators in tensor memory (ck_rhs_tmem.cuh), BLOCK = 512
template <int BLOCK, bool TM>
__global__ void __launch_bounds__(BLOCK, 1) rkf45_kernel(const MechDev m, const RkfArgs a) {
  extern __shared__ double sm[];
  const int tid = threadIdx.x, lane = tid & 31;
  const int N = m.K + 1;
  double* Cs = sm + tid;
  double* wsm = sm + (size_t)(m.K + 1) * BLOCK + tid;
  double* stage_buf = sm + (size_t)(TM ? 1 : 2) * (m.K + 1) * BLOCK;
  __shared__ uint32_t s_tmem;
  uint32_t wt = 0;
  if (TM) {
    if (tid < 32) {
      const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&s_tmem);
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(dst));
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);  // warp-uniform for the compiler (ck_rhs_tmem.cuh)
    wt = s_tmem + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 2 * (m.K + 1));
  }
  const long long slot = (long long)blockIdx.x * BLOCK + tid;
  const size_t vs = (size_t)N * a.nslots;  // stride between vectors
  double* Vy = a.V + slot;                 // component c of vector v: Vy[v*vs + c*nslots]
  const long long ns = a.nslots;

  long long r = -1;
  int st = 0, nacc = 0, nrej = 0, status = CK_ST_OK;
  double t = 0, h = 0, fac_max = 5.0, p = P_0, ha = 0, d1 = 0, h_used = 0;
  bool last = false, endgame = false;
  __shared__ int s_qempty;
  if (tid == 0) s_qempty = 0;
  __syncthreads();
  unsigned long long lane_act = 0, lane_tot = 0, c_rhs = 0, c_att = 0, c_acc = 0, c_rej = 0, c_fail = 0;
  const long long q_limit = a.rlist ? (long long)*a.rcount : a.n;

  // start an attempt from y_n: step-size guards of Algorithm 1, clip to t_f, stage argument = y_n
  auto begin_attempt = [&]() -> bool {
    if (nacc + nrej >= a.max_steps) { status = CK_ST_MAX_STEPS; return false; }
    if (!isfinite(h)) { status = CK_ST_NONFINITE; return false; }
    if (h < 1e-12 * a.dt) { status = CK_ST_H_UNDERFLOW; return false; }
    const bool capped = a.cap > 0 && nacc + nrej >= a.cap;
    if (endgame || capped) {  // re-batch: hand this reactor on (its state is at an attempt boundary)
      for (int c = 0; c < N; ++c) a.y[(size_t)c * a.ld + r] = Vy[c * ns];
      a.rec_t[r] = t; a.rec_h[r] = h; a.rec_fac[r] = fac_max; a.rec_acc[r] = nacc; a.rec_rej[r] = nrej;
      if (capped) {
        // classification: reactors whose predicted number of remaining attempts (t_f - t) / h is large are the critical
        // chains of the batch -- they go to the wide, latency-optimised finisher AT ONCE (it runs beside the resumed
        // thread-per-reactor phase of everybody else)
        const double pred = fmin((a.dt - t) / h, 1e9);
        const int kind = (pred > a.big_steps) ? 2 : ((pred > a.mid_steps) ? 1 : 0);
        if (kind == 2) a.elist[a.n - 1 - (long long)atomicAdd(&a.stats->n_evicted_b, 1ULL)] = (int)r;
        else if (kind == 1) a.elist2[a.n - 1 - (long long)atomicAdd(&a.stats->n_evicted_m, 1ULL)] = (int)r;
        else a.elist[atomicAdd(&a.stats->n_evicted, 1ULL)] = (int)r;
        atomicAdd(&a.stats->sum_pred[kind], (unsigned long long)pred);
      } else {
        a.elist2[atomicAdd(&a.stats->n_evicted_n, 1ULL)] = (int)r;   // end-game: the throughput-oriented finisher
      }
      r = -1;
      return true;
    }
    last = false;
    if (h >= a.dt - t) { h = a.dt - t; last = true; }
    for (int c = 0; c < N; ++c) Vy[7 * vs + c * ns] = Vy[c * ns];
    st = 0;
    return true;
  };
  auto finish = [&]() {
    for (int c = 0; c < N; ++c) a.y[(size_t)c * a.ld + r] = Vy[c * ns];
    if (a.n_accept) a.n_accept[r] = nacc;
    if (a.n_reject) a.n_reject[r] = nrej;
    if (a.status) a.status[r] = status;
    if (a.h_last) a.h_last[r] = h_used;
    a.att[r] = nacc + nrej;
    c_att += nacc + nrej; c_acc += nacc; c_rej += nrej; c_fail += (status != CK_ST_OK);
    r = -1;
  };
  auto wrms2 = [&](int v, int v2) -> double {  // || V[v] (- V[v2]) || weighted by y_n
    double s = 0.0;
    for (int c = 0; c < N; ++c) {
      double x = Vy[(size_t)v * vs + c * ns];
      if (v2 >= 0) x -= Vy[(size_t)v2 * vs + c * ns];
      const double w = x / fma(a.rtol, fabs(Vy[c * ns]), a.atol);
      s = fma(w, w, s);
    }
    return sqrt(s / N);
  };

  for (;;) {
    // ---- divergence control: refill idle lanes from the work queue --------------------------------
    const unsigned idle = __ballot_sync(0xffffffffu, r < 0);
    if (idle && (a.refill || idle == 0xffffffffu)) {
      const int cnt = a.refill ? __popc(idle) : 32;
      unsigned long long base = 0;
      if (lane == 0) base = atomicAdd(a.rqueue, (unsigned long long)cnt);
      base = __shfl_sync(0xffffffffu, base, 0);
      if (r < 0) {
        const long long cand = (long long)base + (a.refill ? __popc(idle & ((1u << lane) - 1)) : lane);
        if (cand < q_limit) {
          r = a.rlist ? (long long)a.rlist[cand] : cand;
          p = a.p[r];
          for (int c = 0; c < N; ++c) {
            const double v = a.y[(size_t)c * a.ld + r];
            Vy[c * ns] = v;
            Vy[7 * vs + c * ns] = v;
          }
          status = CK_ST_OK; h_used = 0; last = false;
          if (a.rlist) {  // resume from the hand-over record
            t = a.rec_t[r]; h = a.rec_h[r]; fac_max = a.rec_fac[r]; nacc = a.rec_acc[r]; nrej = a.rec_rej[r];
            if (!begin_attempt()) finish();
          } else {
            t = 0; nacc = 0; nrej = 0; fac_max = 5.0;
            if (a.h0 > 0.0) { h = a.h0; if (!begin_attempt()) finish(); }
            else st = ST_H0A;
          }
        } else {
          s_qempty = 1;  // the queue ran dry (benign race: every writer stores 1)
        }
      }
    }
    const int n_active = __syncthreads_count(r >= 0);
    if (n_active == 0) break;
    endgame = a.evict && s_qempty && (n_active * 4 < BLOCK);
    const bool act = r >= 0;
    lane_act += act; lane_tot += 1;
    // ---- one RHS evaluation for every lane: f(stage argument) -> evaluation vector of this stage -----
    const int dstv = (st < 0) ? (st + 3) : (st + 1);  // H0A -> 1, H0B -> 2, stage s -> s+1
    if constexpr (TM) rhs_thread_tmem<BLOCK>(m, Vy + 7 * vs, ns, p, Vy + (size_t)dstv * vs, ns, Cs, wt, stage_buf, act);
    else rhs_thread<BLOCK>(m, Vy + 7 * vs, ns, p, Vy + (size_t)dstv * vs, ns, Cs, wsm, stage_buf, act);
    if (!act) continue;
    c_rhs++;
    // ---- per-lane state machine ---------------------------------------------------------------------
    if (st == ST_H0A) {           // EstimateH0, first evaluation: f0 = f(y) (reading G8)
      const double d0 = wrms2(0, -1);
      d1 = wrms2(1, -1);
      ha = (d0 < 1e-5 || d1 < 1e-5) ? 1e-6 * a.dt : 0.01 * d0 / d1;
      for (int c = 0; c < N; ++c) Vy[7 * vs + c * ns] = fma(ha, Vy[vs + c * ns], Vy[c * ns]);
      st = ST_H0B;
    } else if (st == ST_H0B) {    // second evaluation: f(y + ha f0)
      const double d2 = wrms2(2, 1) / ha;
      const double dm = fmax(d1, d2);
      const double hb = (dm <= 1e-15) ? fmax(1e-6 * a.dt, 1e-3 * ha) : pow(0.01 / dm, 0.2);
      h = fmin(fmin(100.0 * ha, hb), a.dt);
      if (!begin_attempt()) finish();
    } else if (st < 5) {          // argument of the next evaluation
      for (int c = 0; c < N; ++c) {
        double acc = 0.0;
#pragma unroll
        for (int j = 0; j < 5; ++j)
          if (j <= st) acc = fma(RKF_T[st][j], Vy[(size_t)(j + 1) * vs + c * ns], acc);
        Vy[7 * vs + c * ns] = fma(h, acc, Vy[c * ns]);
      }
      st++;
    } else {                      // all six evaluations done: 4th-order solution, error, accept / reject
      double es = 0.0;
      for (int c = 0; c < N; ++c) {
        double yb = 0.0, eb = 0.0;
#pragma unroll
        for (int j = 0; j < 6; ++j) {
          const double k = Vy[(size_t)(j + 1) * vs + c * ns];
          yb = fma(RKF_T[5][j], k, yb);
          eb = fma(RKF_T[6][j], k, eb);
        }
        const double y0 = Vy[c * ns];
        const double yn = fma(h, yb, y0);
        Vy[7 * vs + c * ns] = yn;  // candidate kept in the stage-argument vector
        const double w = (h * eb) / fma(a.rtol, fmax(fabs(y0), fabs(yn)), a.atol);
        es = fma(w, w, es);
      }
      const double err = sqrt(es / N);
      h_used = h;
      if (isfinite(err) && err < 1.0) {
        for (int c = 0; c < N; ++c) Vy[c * ns] = Vy[7 * vs + c * ns];
        t = last ? a.dt : t + h;
        nacc++;
        h *= fmin(fac_max, fmax(0.2, 0.9 * pow(fmax(err, 1e-10), -0.2)));
        fac_max = 5.0;
      } else {
        nrej++;
        h *= isfinite(err) ? fmin(1.0, fmax(0.2, 0.9 * pow(fmax(err, 1e-10), -0.2))) : 0.2;
        fac_max = 1.0;
      }
      if (!(t < a.dt) || !begin_attempt()) finish();
    }
  }
  // ---- statistics: one atomic set per warp -------------------------------------------------------------
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lane_act += __shfl_xor_sync(0xffffffffu, lane_act, o); lane_tot += __shfl_xor_sync(0xffffffffu, lane_tot, o);
    c_rhs += __shfl_xor_sync(0xffffffffu, c_rhs, o); c_att += __shfl_xor_sync(0xffffffffu, c_att, o);
    c_acc += __shfl_xor_sync(0xffffffffu, c_acc, o); c_rej += __shfl_xor_sync(0xffffffffu, c_rej, o);
    c_fail += __shfl_xor_sync(0xffffffffu, c_fail, o);
  }
  if (lane == 0) {
    atomicAdd(&a.stats->lane_active, lane_act); atomicAdd(&a.stats->lane_total, lane_tot);
    atomicAdd(&a.stats->rhs_evals, c_rhs); atomicAdd(&a.stats->attempts, c_att);
    atomicAdd(&a.stats->accepted, c_acc); atomicAdd(&a.stats->rejected, c_rej);
    atomicAdd(&a.stats->failed, c_fail);
  }
  if (TM) {
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(s_tmem));
  }
}

// Finisher of the divergence-control layer: reactors evicted from the thread-per-reactor phase (the
// stragglers of the step-count distribution) are completed CTA-per-reactor, so that one
// reactor's long serial chain of attempts runs at the latency of a cooperative RHS (G lanes share one
// evaluation) instead of holding a mostly idle CTA of the throughput kernel.
__host__ __device__ inline size_t rkf_coop_smem_doubles(int K, int R, int n_tent) {
  return (size_t)8 * (K + 1) + coop_chem_doubles(K, R, false) + (size_t)((n_tent + K + 2 + 1) >> 1);
}

template <int G>
__global__ void __launch_bounds__(G) rkf45_coop_kernel(const MechDev m, const RkfArgs a, const int cls) {
  extern __shared__ double sm[];
  __shared__ long long s_next;
  const int N = m.K + 1, tid = threadIdx.x;
  double* Y = sm;            // y_n
  double* F = sm + N;        // six evaluation vectors F[j*N + c]
  double* YT = sm + 7 * N;   // stage argument / candidate
  CoopChem c = coop_carve(sm + 8 * N, m.K, m.R, false);
  const long long n_ev = fin_count(a, cls);
  unsigned long long c_rhs = 0, c_att = 0, c_acc = 0, c_rej = 0, c_fail = 0;
  for (;;) {
    __syncthreads();
    if (tid == 0) s_next = (long long)atomicAdd(fin_queue(a, cls), 1ULL);
    __syncthreads();
    if (s_next >= n_ev) break;
    const long long r = *fin_entry(a, cls, s_next);
    const double p = a.p[r];
    for (int i = tid; i < N; i += G) Y[i] = a.y[(size_t)i * a.ld + r];
    double t = a.rec_t[r], h = a.rec_h[r], fac_max = a.rec_fac[r], h_used = 0.0;
    int nacc = a.rec_acc[r], nrej = a.rec_rej[r], status = CK_ST_OK;
    __syncthreads();
    while (t < a.dt) {
      if (nacc + nrej >= a.max_steps) { status = CK_ST_MAX_STEPS; break; }
      if (!isfinite(h)) { status = CK_ST_NONFINITE; break; }
      if (h < 1e-12 * a.dt) { status = CK_ST_H_UNDERFLOW; break; }
      bool last = false;
      if (h >= a.dt - t) { h = a.dt - t; last = true; }
      TState ts;
      rhs_coop<G, false>(m, Y, p, F, c, ts);
      for (int s = 0; s < 5; ++s) {
        for (int i = tid; i < N; i += G) {
          double acc = 0.0;
          for (int j = 0; j <= s; ++j) acc = fma(RKF_T[s][j], F[j * N + i], acc);
          YT[i] = fma(h, acc, Y[i]);
        }
        __syncthreads();
        rhs_coop<G, false>(m, YT, p, F + (s + 1) * N, c, ts);
      }
      c_rhs += 6;
      double es = 0.0;
      for (int i = tid; i < N; i += G) {
        double yb = 0.0, eb = 0.0;
#pragma unroll
        for (int j = 0; j < 6; ++j) { const double k = F[j * N + i]; yb = fma(RKF_T[5][j], k, yb); eb = fma(RKF_T[6][j], k, eb); }
        const double yn = fma(h, yb, Y[i]);
        YT[i] = yn;
        const double w = (h * eb) / fma(a.rtol, fmax(fabs(Y[i]), fabs(yn)), a.atol);
        es = fma(w, w, es);
      }
      const double err = sqrt(block_sum<G>(es, c.red) / N);
      h_used = h;
      if (isfinite(err) && err < 1.0) {
        __syncthreads();
        for (int i = tid; i < N; i += G) Y[i] = YT[i];
        t = last ? a.dt : t + h;
        nacc++;
        h *= fmin(fac_max, fmax(0.2, 0.9 * pow(fmax(err, 1e-10), -0.2)));
        fac_max = 5.0;
      } else {
        nrej++;
        h *= isfinite(err) ? fmin(1.0, fmax(0.2, 0.9 * pow(fmax(err, 1e-10), -0.2))) : 0.2;
        fac_max = 1.0;
      }
      __syncthreads();
    }
    __syncthreads();
    for (int i = tid; i < N; i += G) a.y[(size_t)i * a.ld + r] = Y[i];
    if (tid == 0) {
      if (a.n_accept) a.n_accept[r] = nacc;
      if (a.n_reject) a.n_reject[r] = nrej;
      if (a.status) a.status[r] = status;
      if (a.h_last) a.h_last[r] = h_used;
      a.att[r] = nacc + nrej;
    }
    c_att += nacc + nrej; c_acc += nacc; c_rej += nrej; c_fail += (status != CK_ST_OK);
  }
  if (tid == 0) {
    atomicAdd(&a.stats->rhs_evals, c_rhs); atomicAdd(&a.stats->attempts, c_att);
    atomicAdd(&a.stats->accepted, c_acc); atomicAdd(&a.stats->rejected, c_rej);
    atomicAdd(&a.stats->failed, c_fail);
  }
}

}  // namespace ck

using namespace ck;

namespace ck {
int32_t integrate_prologue(const char* who, const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double dt,
                           const ck_opts* o, void* ws, size_t ws_bytes, size_t need, cudaStream_t st);
int32_t integrate_report(const ck_mech* m, int64_t n, const int32_t* att_dev, const DevStats* stats_dev, int rounds,
                         long long lu_per_jac, ck_report* rep, cudaStream_t st);
}

namespace {
struct RkfPlan { int block = 0; long long grid = 0; size_t smem = 0; bool tmem = false; };

template <int BLOCK, bool TM>
cudaError_t plan_for(const ck_mech* m, long long n, RkfPlan* pl) {
  pl->block = BLOCK;
  pl->tmem = TM;
  pl->smem = TM ? rhs_tmem_smem_bytes(m->K, m->dev.rstride, BLOCK) : rhs_smem_bytes(m->K, m->dev.rstride, BLOCK);
  cudaError_t e = cudaFuncSetAttribute(rkf45_kernel<BLOCK, TM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem);
  if (e != cudaSuccess) return e;
  int per_sm = 0, sms = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, rkf45_kernel<BLOCK, TM>, BLOCK, pl->smem);
  if (TM) per_sm = std::min(per_sm, 1);  // one CTA owns all 512 tensor-memory columns
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, m->device);
  if (e != cudaSuccess) return e;
  pl->grid = std::min<long long>((n + BLOCK - 1) / BLOCK, (long long)std::max(per_sm, 1) * sms);
  return cudaSuccess;
}

int32_t rkf_plan(const ck_mech* m, long long n, RkfPlan* pl) {
  CK_CUDA(cudaSetDevice(m->device));
  if (m->K + 1 <= 64 && rhs_tmem_smem_bytes(m->K, m->dev.rstride, 512) <= 227 * 1024 && n >= (long long)m->sms * 256) {
    CK_CUDA((plan_for<512, true>(m, n, pl)));
    return CK_OK;
  }
  const int block = rhs_pick_block(m->K, m->dev.rstride, n, m->sms);
  switch (block) {
    case 256: CK_CUDA((plan_for<256, false>(m, n, pl))); break;
    case 128: CK_CUDA((plan_for<128, false>(m, n, pl))); break;
    case 64: CK_CUDA((plan_for<64, false>(m, n, pl))); break;
    case 32: CK_CUDA((plan_for<32, false>(m, n, pl))); break;
    default: set_error("ck_integrate_rkf45: %d species do not fit the shared-memory columns", m->K); return CK_EUNSUPPORTED;
  }
  return CK_OK;
}
inline size_t al256(size_t x) { return (x + 255) & ~size_t(255); }
}  // namespace

namespace {
// slots of the per-slot stage vectors: the plan for n reactors, with room for the plan of any smaller resumed batch
inline size_t rkf_vslots(const RkfPlan& pl, int64_t n) { return std::max<size_t>((size_t)pl.grid * pl.block, (size_t)n + 512); }

int32_t launch_main(const ck_mech* m, const RkfPlan& pl, const RkfArgs& a, long long grid, cudaStream_t st) {
  switch (pl.block) {
    case 512: rkf45_kernel<512, true><<<(unsigned)grid, 512, pl.smem, st>>>(m->dev, a); break;
    case 256: rkf45_kernel<256, false><<<(unsigned)grid, 256, pl.smem, st>>>(m->dev, a); break;
    case 128: rkf45_kernel<128, false><<<(unsigned)grid, 128, pl.smem, st>>>(m->dev, a); break;
    case 64: rkf45_kernel<64, false><<<(unsigned)grid, 64, pl.smem, st>>>(m->dev, a); break;
    default: rkf45_kernel<32, false><<<(unsigned)grid, 32, pl.smem, st>>>(m->dev, a); break;
  }
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}
}  // namespace

// workspace: [DevStats][int attempts[n]][hand-over: 5 int + 3 double per reactor][double V[8][N][slots]]
size_t ck_rkf_workspace(const ck_mech* m, int64_t n) {
  if (n == 0) return sizeof(DevStats);
  RkfPlan pl;
  if (rkf_plan(m, n, &pl) != CK_OK) return sizeof(DevStats);  // the integrate call reports the error
  return sizeof(DevStats) + 6 * al256((size_t)n * sizeof(int)) + 3 * al256((size_t)n * sizeof(double)) +
         (size_t)8 * (m->K + 1) * rkf_vslots(pl, n) * sizeof(double);
}

// Flow (flags = 0, models with N > 32):
//   1  classification: the thread-per-reactor kernel over all reactors, every reactor handed on after RKF_CAP attempts
//      (most of config 4's reactors need more) into one of three lists by its predicted remaining attempts (t_f - t) / h:
//      stragglers (> RKF_BIG), middle class (> RKF_MID), the rest
//   2a the wide finisher over the stragglers, longest first, one 384-thread CTA and one SM per straggler: their serial
//      chains are the critical path of the batch (ck_rkf_wide.cuh: 18 us per attempt against 0.8-1 ms thread-per-reactor)
//   2b the thread-per-reactor kernel resumes the rest, long ones first (lane refill; end-game eviction -> list N): the
//      cheapest mode per attempt (2.1 us of an SM), usable only where ~1 ms per attempt does not make the reactor late
//   2c the narrow finisher over the middle class, longest first (64 / 128-thread CTAs, eight per SM: 7.4 us of an SM per
//      attempt, 40-60 us per attempt for one reactor)
//      2a, 2b and 2c run side by side on three streams over disjoint SMs (shares from the predicted work, see below)
//   3  the narrow finisher over list N
// N <= 32: phases 1 (uncapped, with end-game eviction) and 3 only.  flags bit 0 / 1: one kernel, no eviction.
extern "C" int32_t ck_integrate_rkf45(const ck_mech* m, int64_t n, double* y, int64_t ld, const double* p, double dt,
                                      const ck_opts* o, int32_t* n_accept, int32_t* n_reject, int32_t* status,
                                      double* h_last, void* ws, size_t ws_bytes, ck_report* report, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  if (!m) { set_error("ck_integrate_rkf45: null mechanism"); return CK_EINVAL; }
  RkfPlan pl;
  if (n > 0) { int32_t rc0 = rkf_plan(m, n, &pl); if (rc0) return rc0; }
  const size_t nslots = n > 0 ? rkf_vslots(pl, n) : 0;
  const size_t bi = al256((size_t)n * sizeof(int)), bd = al256((size_t)n * sizeof(double));
  const size_t need = n > 0 ? sizeof(DevStats) + 6 * bi + 3 * bd + (size_t)8 * (m->K + 1) * nslots * sizeof(double) : sizeof(DevStats);
  int32_t rc = integrate_prologue("ck_integrate_rkf45", m, n, y, ld, p, dt, o, ws, ws_bytes, need, st);
  if (rc) return rc;
  if (n == 0) { if (report) *report = ck_report{}; return CK_OK; }
  const int N = m->K + 1;
  RkfArgs a{};
  a.n = n; a.ld = ld; a.nslots = (long long)nslots; a.y = y; a.p = p; a.dt = dt; a.rtol = o->rtol; a.atol = o->atol; a.h0 = o->h0;
  a.max_steps = o->max_steps > 0 ? o->max_steps : 100000; a.refill = !(o->flags & 1);
  a.n_accept = n_accept; a.n_reject = n_reject; a.status = status; a.h_last = h_last;
  a.stats = (DevStats*)ws;
  char* wp = (char*)ws + sizeof(DevStats);
  a.att = (int*)wp; wp += bi;
  a.elist = (int*)wp; wp += bi;
  a.elist2 = (int*)wp; wp += bi;
  a.tmp = (int*)wp; wp += bi;
  a.rec_acc = (int*)wp; wp += bi;
  a.rec_rej = (int*)wp; wp += bi;
  a.rec_t = (double*)wp; wp += bd;
  a.rec_h = (double*)wp; wp += bd;
  a.rec_fac = (double*)wp; wp += bd;
  a.V = (double*)wp;
  const bool finishers = !(o->flags & 3);          // bit 0: static mapping, bit 1: refill only (no finisher)
  const bool classify = finishers && N > 32;
  constexpr int RKF_CAP = 24;                       // attempts before a reactor is classified
  constexpr double RKF_BIG = 8000.0;                // predicted remaining attempts that make a straggler (wide finisher)
  constexpr double RKF_MID = 400.0;                 // ... that send a reactor to the narrow finisher at once
  a.rlist = nullptr; a.rcount = nullptr; a.rqueue = &a.stats->queue;
  a.cap = classify ? std::min(RKF_CAP, a.max_steps) : 0;
  a.big_steps = (o->flags & 16) ? -1.0 : RKF_BIG;   // bit 4 (measurement): every classified reactor counts as a straggler
  // small batches cannot fill the lanes of the thread-per-reactor kernel, whose ~1 ms per attempt then is all they would
  // get from it: everything goes to the finishers after the classification pass (n = 4096: 0.4 s instead of 1.9 s)
  a.mid_steps = (n < 16384) ? -1.0 : RKF_MID;
  a.evict = (finishers && !classify) ? 1 : 0;
  // everything the finishers need is validated BEFORE the first launch: a failure must not leave y half-integrated
  const size_t smem2 = rkf_coop_smem_doubles(m->K, m->R, m->dev.n_tent) * sizeof(double);
  if (finishers && smem2 > 227 * 1024) { set_error("ck_integrate_rkf45: mechanism too large for the cooperative finisher"); return CK_EUNSUPPORTED; }
  int sms = 0;
  CK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, m->device));
  if (finishers) {
    // Touch every kernel of the flow BEFORE the first launch: CUDA loads kernels lazily, and a first-use load issued while
    // another kernel runs waits for it -- the side-by-side phases of the first call of a process would run one after
    // the other (measured: 3.4 s instead of 1.45 s for config 4).
    // The shared-memory opt-ins are made here as well, so that nothing that can fail is left for the time when y is
    // half-integrated.
    cudaFuncAttributes fa;
    const size_t smem_w0 = rkf_wide_smem_doubles(m->K, m->R, m->dev.r_tb, m->dev.n_tent) * sizeof(double);
    if (m->K <= 128 && smem_w0 <= 227 * 1024)
      CK_CUDA(cudaFuncSetAttribute(rkf45_wide_kernel<WIDE_G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_w0));
    CK_CUDA(cudaFuncSetAttribute(rkf45_coop_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2));
    CK_CUDA(cudaFuncSetAttribute(rkf45_coop_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2));
    CK_CUDA(cudaFuncSetAttribute(rkf45_coop_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2));
    CK_CUDA(cudaFuncSetAttribute(rkf_order_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, RKF_ORDER_MAX * 12));
    CK_CUDA(cudaFuncGetAttributes(&fa, rkf_bucket_kernel));
    CK_CUDA(cudaFuncGetAttributes(&fa, rkf45_kernel<512, true>));
  }
  rc = launch_main(m, pl, a, pl.grid, st);
  if (rc) return rc;
  int rounds = 1;
  if (finishers) {
    int per_sm = 0;
    auto launch_fin = [&](auto kern, int G, int cls, long long want, cudaStream_t s, size_t smem = 0) -> int32_t {
      if (smem == 0) smem = smem2;
      CK_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      CK_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, G, smem));
      const long long grid = std::max<long long>(1, std::min<long long>(want, (long long)std::max(per_sm, 1) * sms));
      kern<<<(unsigned)grid, G, smem, s>>>(m->dev, a, cls);
      CK_CUDA(cudaGetLastError());
      return CK_OK;
    };
    cudaStream_t s2 = nullptr, s3 = nullptr;
    cudaEvent_t ev_fin = nullptr, ev_fin3 = nullptr;
    if (classify) {
      DevStats hs;   // the list lengths size the next launches (one small read-back; this call synchronises anyway)
      CK_CUDA(cudaMemcpyAsync(&hs, a.stats, sizeof hs, cudaMemcpyDeviceToHost, st));
      CK_CUDA(cudaStreamSynchronize(st));
      const long long nW = (long long)hs.n_evicted_b, nM = (long long)hs.n_evicted_m, nC = (long long)hs.n_evicted;
      const size_t smem_w = rkf_wide_smem_doubles(m->K, m->R, m->dev.r_tb, m->dev.n_tent) * sizeof(double);
      const bool wide_ok = m->K <= 128 && smem_w <= 227 * 1024 && !(o->flags & 32);
      // SM shares.  The three phases that follow run side by side, and the resumed thread-per-reactor kernel and the wide
      // finisher each need a whole SM per CTA, so the split is made here: the stragglers get one SM each (at most 30 % of
      // the machine: measured on config 4, 20 % makes their queue the long pole, 40 % starves the other two), the rest is divided between the resumed kernel and the narrow finisher in proportion to their
      // predicted work (measured cost per attempt: 2.1 us of an SM thread-per-reactor, 7.4 us on narrow CTAs); the narrow
      // finisher is launched with more CTAs than fit, so it also takes over every SM the other two give back.
      const long long gW = std::min<long long>(nW, (nC + nM > 0) ? (3 * sms) / 10 : sms);
      const double eb = 2.1 * (double)hs.sum_pred[0], em = 7.4 * (double)hs.sum_pred[1];
      const long long rem = sms - (wide_ok ? gW : 0);
      long long gC = rem;
      if (nM > 0 || (nW > 0 && !wide_ok)) gC = std::max<long long>(8, std::min<long long>(rem - 8, (long long)((double)rem * eb / std::max(eb + em, 1.0) + 0.5)));
      cudaEvent_t ev_main = nullptr;
      if (nW > 0 || nM > 0) {
        CK_CUDA(cudaEventCreateWithFlags(&ev_main, cudaEventDisableTiming));
        CK_CUDA(cudaEventRecord(ev_main, st));
      }
      if (nC > 0) {   // 2b: resume the rest thread-per-reactor (first: its CTAs take their SMs before the others are placed)
        RkfPlan pl2;
        rc = rkf_plan(m, nC, &pl2);
        if (rc) return rc;
        rkf_bucket_kernel<<<1, 1024, 0, st>>>(a, -1, a.tmp);
        RkfArgs ac = a;
        ac.cap = 0; ac.evict = 1;
        ac.rlist = a.elist; ac.rcount = &a.stats->n_evicted; ac.rqueue = &a.stats->queue_c;
        rc = launch_main(m, pl2, ac, std::min<long long>(pl2.grid, gC), st);
        if (rc) return rc;
        rounds++;
      }
      const int order_smem = RKF_ORDER_MAX * 12;
      if (nW > 0) {   // 2a: the stragglers, longest first
        CK_CUDA(cudaStreamCreateWithFlags(&s2, cudaStreamNonBlocking));
        CK_CUDA(cudaEventCreateWithFlags(&ev_fin, cudaEventDisableTiming));
        CK_CUDA(cudaStreamWaitEvent(s2, ev_main, 0));
        CK_CUDA(cudaFuncSetAttribute(rkf_order_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, order_smem));
        rkf_order_kernel<<<1, 1024, order_smem, s2>>>(a, 1);
        if (wide_ok) rc = launch_fin(rkf45_wide_kernel<WIDE_G>, WIDE_G, 1, gW, s2, smem_w);
        else rc = (N <= 64) ? launch_fin(rkf45_coop_kernel<64>, 64, 1, nW, s2) : launch_fin(rkf45_coop_kernel<128>, 128, 1, nW, s2);
        if (rc) return rc;
        CK_CUDA(cudaEventRecord(ev_fin, s2));
        rounds++;
      }
      if (nM > 0) {   // 2c: the middle class on narrow CTAs, longest first, oversubscribed
        CK_CUDA(cudaStreamCreateWithFlags(&s3, cudaStreamNonBlocking));
        CK_CUDA(cudaEventCreateWithFlags(&ev_fin3, cudaEventDisableTiming));
        CK_CUDA(cudaStreamWaitEvent(s3, ev_main, 0));
        CK_CUDA(cudaFuncSetAttribute(rkf_order_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, order_smem));
        if (nM <= RKF_ORDER_MAX) rkf_order_kernel<<<1, 1024, order_smem, s3>>>(a, 2);
        else rkf_bucket_kernel<<<1, 1024, 0, s3>>>(a, 2, a.tmp + nC);   // the two bucket passes may overlap: disjoint halves
        if (wide_ok && nC == 0 && nW + nM <= sms)   // SMs to spare: everybody gets the low-latency kernel
          rc = launch_fin(rkf45_wide_kernel<WIDE_G>, WIDE_G, 2, nM, s3, smem_w);
        else
          rc = (N <= 64) ? launch_fin(rkf45_coop_kernel<64>, 64, 2, nM, s3) : launch_fin(rkf45_coop_kernel<128>, 128, 2, nM, s3);
        if (rc) return rc;
        CK_CUDA(cudaEventRecord(ev_fin3, s3));
        rounds++;
      }
      if (ev_main) cudaEventDestroy(ev_main);
      a.cap = 0; a.evict = 1;
    }
    // 3: whatever the end-game evicted (its count is read on the device)
    if (N <= 32) rc = launch_fin(rkf45_coop_kernel<32>, 32, 0, n, st);
    else if (N <= 64) rc = launch_fin(rkf45_coop_kernel<64>, 64, 0, n, st);
    else rc = launch_fin(rkf45_coop_kernel<128>, 128, 0, n, st);
    if (rc) return rc;
    rounds++;
    if (s2) {   // join the side streams; the objects are released once their work has drained
      CK_CUDA(cudaStreamWaitEvent(st, ev_fin, 0));
      cudaEventDestroy(ev_fin);
      cudaStreamDestroy(s2);
    }
    if (s3) {
      CK_CUDA(cudaStreamWaitEvent(st, ev_fin3, 0));
      cudaEventDestroy(ev_fin3);
      cudaStreamDestroy(s3);
    }
  }
  return integrate_report(m, n, a.att, a.stats, rounds, 0, report, st);
}
