// ck_waste: Eq. 20, the waste of each SIMD work unit of width P under the static linear
// reactor -> lane mapping: W_j = 1 - sum_i N_i / (P max_i N_i), N_i = attempts of reactor i.
// One warp per work unit; lanes stride over the unit's reactors, sum and maximum by REDUX.
#include <algorithm>

#include "ck_internal.h"

using namespace ck;

namespace {

// m tasks per lane (m = 1: Eq. 20 as printed): unit j holds the P m consecutive reactors from b = j P m, lane l takes
// reactors b + l, b + l + P, ... (interleaved, so that a warp still reads consecutive reactors), its cost is the SUM of
// their attempts, and W_j = 1 - sum_i N_i / (lanes x max_l cost_l) with `lanes` = lanes that own at least one reactor.
__global__ void __launch_bounds__(256) waste_kernel(long long n, const int* __restrict__ na, const int* __restrict__ nr, int P, int m,
                                                    double* __restrict__ W) {
  const long long per = (long long)P * m;
  const long long units = (n + per - 1) / per;
  const int lane = threadIdx.x & 31;
  const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
  for (long long j = warp0; j < units; j += nwarps) {
    const long long b = j * per, e = (b + per < n) ? b + per : n;
    unsigned long long mx = 0, tot = 0;
    for (long long l = lane; l < P; l += 32) {
      unsigned long long cost = 0;
      for (long long i = b + l; i < e; i += P) cost += (unsigned)(na[i] + (nr ? nr[i] : 0));
      tot += cost;
      mx = cost > mx ? cost : mx;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      tot += __shfl_xor_sync(0xffffffffu, tot, o);
      const unsigned long long x = __shfl_xor_sync(0xffffffffu, mx, o);
      mx = x > mx ? x : mx;
    }
    const long long lanes = (e - b < P) ? e - b : P;
    if (lane == 0) W[j] = mx ? 1.0 - (double)tot / ((double)lanes * (double)mx) : 0.0;
  }
}

int32_t waste_launch(int64_t n, const int32_t* n_accept, const int32_t* n_reject, int32_t P, int32_t m, double* W, void* stream,
                     const char* who) {
  if (n < 0 || P < 1 || P > 1024 || m < 1 || m > 4096) { set_error("%s: bad n / P / tasks (%lld, %d, %d)", who, (long long)n, P, m); return CK_EINVAL; }
  if (n == 0) return CK_OK;
  if (!n_accept || !W) { set_error("%s: null pointer", who); return CK_EINVAL; }
  const long long units = (n + (long long)P * m - 1) / ((long long)P * m);
  int dev = 0, sms = 148;   // no mechanism handle here: ask the current device
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const long long blocks = std::max<long long>(1, std::min<long long>((units + 7) / 8, (long long)sms * 8));
  waste_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(n, n_accept, n_reject, P, m, W);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}

}  // namespace

extern "C" int32_t ck_waste(int64_t n, const int32_t* n_accept, const int32_t* n_reject, int32_t P, double* W, void* stream) {
  return waste_launch(n, n_accept, n_reject, P, 1, W, stream, "ck_waste");
}
extern "C" int32_t ck_waste_tasks(int64_t n, const int32_t* n_accept, const int32_t* n_reject, int32_t P, int32_t tasks,
                                  double* W, void* stream) {
  return waste_launch(n, n_accept, n_reject, P, tasks, W, stream, "ck_waste_tasks");
}
