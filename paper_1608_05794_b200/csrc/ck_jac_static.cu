// ck_jac_batched_static: the thread-per-reactor analytic Jacobian of ck_jac_batched (ck_jac_tpr.cuh) for callers that
// cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The scratch
// the kernel needs (f(y), the row-0 vectors HC, the per-reaction derivative pieces G2) lives in a file-scope device array
// of fixed size instead of a caller-supplied workspace.  The entry point calls no cudaMalloc / cudaFree and no allocating
// library routine; it only launches kernels on the caller's stream.
//
// The array's name is a host-side stand-in in host code, NOT a device address: its address is taken with
// cudaGetSymbolAddress once per device, with that device current, and that pointer is what the kernels get.
// Every GPU that loads the library holds the array (CK_JAC_STATIC_BYTES) until the process exits.  Every call on a device
// shares it: the array keeps the last call's contents (the kernels write every entry they later read, so nothing has
// to be cleared), and two calls that overlap on the GPU (different streams, or graphs replayed concurrently) RACE.
#include <algorithm>
#include <mutex>

#include "ck_jac_tpr.cuh"

namespace ck {
constexpr size_t JAC_STATIC_DOUBLES = CK_JAC_STATIC_BYTES / sizeof(double);
static __device__ __align__(256) double g_jac_scratch[JAC_STATIC_DOUBLES];
}  // namespace ck

using namespace ck;

namespace {
constexpr int MAX_DEV = 64;
std::mutex g_mu;
double* g_ptr[MAX_DEV] = {};   // device address of g_jac_scratch on each device (set up once per device)

inline size_t al32(size_t doubles) { return (doubles + 31) & ~size_t(31); }   // 256-byte pieces
inline size_t need_doubles(const ck_mech* m, int64_t n) {
  const size_t N = m->K + 1;
  return al32(N * (size_t)n) + al32((size_t)jac_hc_rows(m->K) * n) + al32((size_t)jac_g2_rows(m->R, m->dev.r_tb) * n);
}

int32_t scratch_address(int device, double** out) {
  if (device < 0 || device >= MAX_DEV) { set_error("ck_jac_batched_static: device %d out of range", device); return CK_EINVAL; }
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_ptr[device]) {
    CK_CUDA(cudaSetDevice(device));   // the symbol's address belongs to the CURRENT device's copy of the module
    double* p = nullptr;
    CK_CUDA(cudaGetSymbolAddress((void**)&p, g_jac_scratch));
    g_ptr[device] = p;
  }
  *out = g_ptr[device];
  return CK_OK;
}

template <int BLOCK>
int32_t launch_rows(const ck_mech* m, long long n, const double* y, long long ld, const double* p, const JacOut& o, cudaStream_t st) {
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

extern "C" int32_t ck_jac_static_max_reactors(const ck_mech* m, int64_t* n_max) {
  if (!m || !n_max) { set_error("ck_jac_static_max_reactors: null argument"); return CK_EINVAL; }
  int64_t lo = 0, hi = (int64_t)JAC_STATIC_DOUBLES;   // largest n whose scratch fits (need_doubles is monotone in n)
  while (lo < hi) {
    const int64_t mid = lo + (hi - lo + 1) / 2;
    if (need_doubles(m, mid) <= JAC_STATIC_DOUBLES) lo = mid; else hi = mid - 1;
  }
  *n_max = lo;
  return CK_OK;
}

extern "C" int32_t ck_jac_batched_static(const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double* J,
                                         int64_t ldJ, void* stream) {
  if (!m) { set_error("ck_jac_batched_static: null mechanism"); return CK_EINVAL; }
  if (n < 0 || ld < n || ldJ < n) { set_error("ck_jac_batched_static: bad n/ld"); return CK_EINVAL; }
  if (n == 0) return CK_OK;
  if (!y || !p || !J) { set_error("ck_jac_batched_static: null batch pointer"); return CK_EINVAL; }
  const int block = jac_tpr_block(m->dev);
  if (block == 0 || m->dev.rstride > 64) { set_error("ck_jac_batched_static: %d species do not fit the thread-per-reactor kernel (use ck_jac)", m->K); return CK_EUNSUPPORTED; }
  const size_t need = need_doubles(m, n);
  if (need > JAC_STATIC_DOUBLES) {
    int64_t nmax = 0;
    ck_jac_static_max_reactors(m, &nmax);
    set_error("ck_jac_batched_static: %lld reactors need %zu bytes of scratch, the static array holds %zu (at most %lld reactors of this model per call; use ck_jac_batched with a workspace beyond that)",
              (long long)n, need * sizeof(double), (size_t)CK_JAC_STATIC_BYTES, (long long)nmax);
    return CK_EWORKSPACE;
  }
  double* base = nullptr;
  int32_t rc = scratch_address(m->device, &base);
  if (rc) return rc;
  CK_CUDA(cudaSetDevice(m->device));
  cudaStream_t st = (cudaStream_t)stream;
  const size_t N = m->K + 1;
  JacOut o{};
  o.f = base; o.ldf = n;
  o.hc = o.f + al32(N * (size_t)n); o.ldh = n;
  o.g2 = o.hc + al32((size_t)jac_hc_rows(m->K) * n); o.ldg = n;
  o.J = J; o.ldJ = ldJ; o.ldr = 0; o.sstride = 0;
  rc = (block == 512) ? launch_rows<512>(m, n, y, ld, p, o, st) : launch_rows<224>(m, n, y, ld, p, o, st);
  if (rc) return rc;
  jac_trow_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(m->K, n, o.f, o.ldf, o.hc, o.ldh, J, ldJ);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}
