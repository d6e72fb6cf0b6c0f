// ck_rhs: f(y; p) of Eq. 12-19 for a batch of reactor states, thread-per-reactor.
//
// Mapping: one thread owns one reactor; consecutive threads own consecutive
// reactors so every HBM access to the component-major state is a fully coalesced 256 B row segment.
// The only per-thread arrays with data-dependent indices -- concentrations C_k and the production-rate
// accumulators omega_k -- live in shared memory as conflict-free columns (C[k*BLOCK + tid]); reaction
// constants are warp-uniform loads.  All arithmetic is FP64.
#include "ck_chem.cuh"

namespace ck {

// One RHS evaluation for the reactor of this thread.  yin / fout are pre-offset to the reactor's column.
// Cs, ws: shared-memory columns of this thread (pre-offset by tid), stride BLOCK.
template <int BLOCK>
__device__ __forceinline__ void rhs_thread(const MechDev& m, const double* __restrict__ yin, long long ldin, double p,
                                           double* __restrict__ fout, long long ldout, double* __restrict__ Cs,
                                           double* __restrict__ ws, bool store) {
  const int K = m.K, R = m.R;
  const TState t = make_tstate(m, yin[0]);
  // (2) ideal gas: S = sum Y_k/W_k, rho = p/(R_u T S), C_k = rho Y_k/W_k; cp sum on the way
  double S = 0.0, cps = 0.0;
  for (int k = 0; k < K; ++k) {
    const double Yk = yin[(size_t)(k + 1) * ldin];
    const double yw = Yk * __ldg(m.invW + k);
    double cpR, hRT;
    thermo_cp_h(m, k, t, cpR, hRT);
    S += yw;
    cps = fma(yw, cpR, cps);
    Cs[(size_t)k * BLOCK] = yw;
    ws[(size_t)k * BLOCK] = 0.0;
  }
  const double Ctot = p / (R_U * t.T);  // = rho * S
  const double rho = Ctot / S;
  for (int k = 0; k < K; ++k) Cs[(size_t)k * BLOCK] *= rho;
  // (3) reactions
  for (int r = 0; r < R; ++r) {
    const double q = reaction_q<BLOCK, false>(m, r, t, Cs, Ctot, nullptr);
#pragma unroll
    for (int s = 0; s < 6; ++s) {
      const int e = __ldg(m.part + (size_t)s * R + r);
      if (e) {
        const double nu = (double)(e & 255);
        double* w = ws + (size_t)(e >> 8) * BLOCK;
        *w = fma(s < 3 ? -nu : nu, q, *w);
      }
    }
  }
  // (4) Eq. 12-13 (13 in reading G2)
  const double irho = 1.0 / rho;
  double hw = 0.0;
  for (int k = 0; k < K; ++k) {
    double cpR, hRT;
    thermo_cp_h(m, k, t, cpR, hRT);
    const double w = ws[(size_t)k * BLOCK];
    hw = fma(hRT, w, hw);
    if (store) fout[(size_t)(k + 1) * ldout] = w * __ldg(m.W + k) * irho;
  }
  if (store) fout[0] = -(t.T * hw) / (rho * cps);  // R_u cancels: -R_u T hw / (rho R_u cps)
}

template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) rhs_kernel(const MechDev m, long long n, const double* __restrict__ y,
                                                    long long ld, const double* __restrict__ p,
                                                    double* __restrict__ f, long long ldf) {
  extern __shared__ double sm[];
  const int tid = threadIdx.x;
  const long long r = (long long)blockIdx.x * BLOCK + tid;
  const bool act = r < n;
  const long long rr = act ? r : n - 1;  // idle lanes of the ragged tail recompute the last reactor, store nothing
  double* Cs = sm + tid;
  double* ws = sm + (size_t)m.K * BLOCK + tid;
  rhs_thread<BLOCK>(m, y + rr, ld, p[rr], f + rr, ldf, Cs, ws, act);
}

template <int BLOCK>
static int32_t launch_rhs(const ck_mech* m, long long n, const double* y, long long ld, const double* p, double* f,
                          long long ldf, cudaStream_t st) {
  const size_t smem = (size_t)2 * m->K * BLOCK * sizeof(double);
  CK_CUDA(cudaFuncSetAttribute(rhs_kernel<BLOCK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const long long grid = (n + BLOCK - 1) / BLOCK;
  rhs_kernel<BLOCK><<<(unsigned)grid, BLOCK, smem, st>>>(m->dev, n, y, ld, p, f, ldf);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}

}  // namespace ck

using namespace ck;

extern "C" int32_t ck_rhs(const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double* dydt,
                          int64_t ld_out, void* stream) {
  if (!m) { set_error("ck_rhs: null mechanism"); return CK_EINVAL; }
  if (n < 0 || ld < n || ld_out < n) { set_error("ck_rhs: bad n/ld (n=%lld ld=%lld ld_out=%lld)", (long long)n, (long long)ld, (long long)ld_out); return CK_EINVAL; }
  if (n == 0) return CK_OK;
  if (!y || !p || !dydt) { set_error("ck_rhs: null batch pointer"); return CK_EINVAL; }
  if ((n + 31) / 32 > 0x7fffffffLL) { set_error("ck_rhs: n too large"); return CK_EINVAL; }
  CK_CUDA(cudaSetDevice(m->device));
  cudaStream_t st = (cudaStream_t)stream;
  const size_t per_thread = (size_t)2 * m->K * sizeof(double);
  const size_t cap = 227 * 1024;
  if (per_thread * 128 * 2 <= cap) return launch_rhs<128>(m, n, y, ld, p, dydt, ld_out, st);
  if (per_thread * 64 <= cap / 2) return launch_rhs<64>(m, n, y, ld, p, dydt, ld_out, st);
  if (per_thread * 32 <= cap) return launch_rhs<32>(m, n, y, ld, p, dydt, ld_out, st);
  set_error("ck_rhs: %d species need %zu B of shared memory per thread (unsupported)", m->K, per_thread);
  return CK_EUNSUPPORTED;
}
