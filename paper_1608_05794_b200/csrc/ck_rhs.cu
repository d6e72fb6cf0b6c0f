// ck_rhs: f(y; p) of Eq. 12-19 for a batch of reactor states, thread-per-reactor.
//
// Mapping: one thread owns one reactor; consecutive threads own consecutive
// reactors so every HBM access to the component-major state is a fully coalesced 256 B row segment.
// The only per-thread arrays with data-dependent indices -- concentrations C_k and the production-rate
// accumulators omega_k -- live in shared memory as conflict-free columns (C[k*BLOCK + tid]); reaction
// constants are warp-uniform loads.  All arithmetic is FP64.
#include <algorithm>
#include <cstdlib>

#include "ck_rhs_tmem.cuh"

namespace ck {

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
  double* ws = sm + (size_t)(m.K + 1) * BLOCK + tid;
  double* stage = sm + (size_t)2 * (m.K + 1) * BLOCK;
  rhs_thread<BLOCK>(m, y + rr, ld, p[rr], f + rr, ldf, Cs, ws, stage, act);
}

template <int BLOCK>
static int32_t launch_rhs(const ck_mech* m, long long n, const double* y, long long ld, const double* p, double* f,
                          long long ldf, cudaStream_t st) {
  const size_t smem = rhs_smem_bytes(m->K, m->dev.rstride, BLOCK);
  CK_CUDA(cudaFuncSetAttribute(rhs_kernel<BLOCK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const long long grid = (n + BLOCK - 1) / BLOCK;
  rhs_kernel<BLOCK><<<(unsigned)grid, BLOCK, smem, st>>>(m->dev, n, y, ld, p, f, ldf);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}

// accumulators in tensor memory: BLOCK threads per CTA, persistent over batches of BLOCK reactors.  512 threads (one
// CTA per SM) for large batches of models with K + 1 <= 64; 128 threads (up to three CTAs per SM) when the batch
// would leave most SMs without a 512-thread CTA; 224 threads (seven warps, two column sets) for 64 < K + 1 <= 124.
template <int BLOCK, int CVM>
static int32_t launch_rhs_tmem_kind(const ck_mech* m, long long n, const double* y, long long ld, const double* p, double* f,
                                    long long ldf, cudaStream_t st) {
  const size_t smem = rhs_tmem_smem_bytes(m->K, m->dev.rstride, BLOCK);
  CK_CUDA(cudaFuncSetAttribute(rhs_kernel_tmem<BLOCK, CVM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int sms = 0;
  CK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, m->device));
  const int cols = rhs_tmem_cols(m->K, BLOCK);
  const long long per_sm = std::max<long long>(1, std::min<long long>(512 / cols, (long long)((227 * 1024) / (smem + 1024))));
  const long long batches = (n + BLOCK - 1) / BLOCK;
  const long long grid = std::min<long long>(batches, per_sm * sms);
  rhs_kernel_tmem<BLOCK, CVM><<<(unsigned)grid, BLOCK, smem, st>>>(m->dev, n, y, ld, p, f, ldf);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}
template <int BLOCK>
static int32_t launch_rhs_tmem(const ck_mech* m, long long n, const double* y, long long ld, const double* p, double* f,
                               long long ldf, cudaStream_t st) {
  return m->dev.cv ? launch_rhs_tmem_kind<BLOCK, 1>(m, n, y, ld, p, f, ldf, st) : launch_rhs_tmem_kind<BLOCK, 0>(m, n, y, ld, p, f, ldf, st);
}

// CTA width of the tensor-memory kernel for this batch; 0: use the shared-memory kernel
int rhs_tmem_block(const ck_mech* m, long long n) {
  const int K = m->K, rs = m->dev.rstride;
  if (K + 1 <= 64) {
    if (n >= (long long)m->sms * 256 && rhs_tmem_smem_bytes(K, rs, 512) <= 227 * 1024) return 512;
    if (n >= 2048 && rhs_tmem_cols(K, 128) != 0) return 128;
    return 0;
  }
  if (n >= 4096 && rhs_tmem_cols(K, 224) != 0 && rhs_tmem_smem_bytes(K, rs, 224) <= 227 * 1024) return 224;
  return 0;
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
  if (m->dev.rstride > 64) { set_error("ck_rhs: too many temperature intervals"); return CK_EUNSUPPORTED; }
  switch (ck::rhs_tmem_block(m, n)) {
    case 512: return launch_rhs_tmem<512>(m, n, y, ld, p, dydt, ld_out, st);
    case 224: return launch_rhs_tmem<224>(m, n, y, ld, p, dydt, ld_out, st);
    case 128: return launch_rhs_tmem<128>(m, n, y, ld, p, dydt, ld_out, st);
    default: break;
  }
  switch (rhs_pick_block(m->K, m->dev.rstride, n, m->sms)) {
    case 256: return launch_rhs<256>(m, n, y, ld, p, dydt, ld_out, st);
    case 128: return launch_rhs<128>(m, n, y, ld, p, dydt, ld_out, st);
    case 64: return launch_rhs<64>(m, n, y, ld, p, dydt, ld_out, st);
    case 32: return launch_rhs<32>(m, n, y, ld, p, dydt, ld_out, st);
    default: break;
  }
  set_error("ck_rhs: %d species do not fit the shared-memory columns (unsupported)", m->K);
  return CK_EUNSUPPORTED;
}

// which kernel ck_rhs launches for a batch of n states: CTA width, and whether the production-rate accumulators live
// in tensor memory (for the roofline record of bench.py: the kernel name comes from the dispatch, not from a constant)
extern "C" int32_t ck_rhs_variant(const ck_mech* m, int64_t n, int32_t* block, int32_t* tmem) {
  if (!m || !block || !tmem) { set_error("ck_rhs_variant: null argument"); return CK_EINVAL; }
  const int b = ck::rhs_tmem_block(m, n);
  *tmem = b != 0;
  *block = b ? b : rhs_pick_block(m->K, m->dev.rstride, n, m->sms);
  return CK_OK;
}
