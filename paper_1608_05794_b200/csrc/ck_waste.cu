// ck_waste: Eq. 20, the waste of each SIMD work unit of width P under the static linear
// reactor -> lane mapping: W_j = 1 - sum_i N_i / (P max_i N_i), N_i = attempts of reactor i.
// One warp per work unit; lanes stride over the unit's reactors, sum and maximum by REDUX.
#include <algorithm>

#include "ck_internal.h"

using namespace ck;

namespace {

__global__ void __launch_bounds__(256) waste_kernel(long long n, const int* __restrict__ na, const int* __restrict__ nr, int P,
                                                    double* __restrict__ W) {
  const long long units = (n + P - 1) / P;
  const int lane = threadIdx.x & 31;
  const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
  for (long long j = warp0; j < units; j += nwarps) {
    const long long b = j * P, e = (b + P < n) ? b + P : n;
    unsigned mx = 0;
    unsigned long long tot = 0;
    for (long long i = b + lane; i < e; i += 32) {
      const unsigned a = (unsigned)(na[i] + (nr ? nr[i] : 0));
      tot += a;
      mx = a > mx ? a : mx;
    }
    mx = __reduce_max_sync(0xffffffffu, mx);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    if (lane == 0) W[j] = mx ? 1.0 - (double)tot / ((double)(e - b) * (double)mx) : 0.0;
  }
}

}  // namespace

extern "C" int32_t ck_waste(int64_t n, const int32_t* n_accept, const int32_t* n_reject, int32_t P, double* W, void* stream) {
  if (n < 0 || P < 1 || P > 1024) { set_error("ck_waste: bad n / P (%lld, %d)", (long long)n, P); return CK_EINVAL; }
  if (n == 0) return CK_OK;
  if (!n_accept || !W) { set_error("ck_waste: null pointer"); return CK_EINVAL; }
  const long long units = (n + P - 1) / P;
  const long long blocks = std::min<long long>((units + 7) / 8, 148 * 8);
  waste_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(n, n_accept, n_reject, P, W);
  CK_CUDA(cudaGetLastError());
  return CK_OK;
}
