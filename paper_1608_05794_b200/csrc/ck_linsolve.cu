// ck_lu_solve_batched: the per-reactor dense linear algebra of the Rosenbrock stage equations (Eq. 6, PAPER.md:72-76;
// cost ~ N^3) exposed on its own: factor each A_r with partial pivoting and solve A_r x_r = b_r.
// One warp per system (ck_lu_warp.cuh).
#include <algorithm>

#include "ck_lu_warp.cuh"

namespace ck {

template <int NR>
__global__ void __launch_bounds__(32) lu_solve_batched_kernel(int N, long long n, const double* __restrict__ A,
                                                              const double* __restrict__ b, double* __restrict__ x,
                                                              int* __restrict__ status) {
  extern __shared__ double sm[];
  const int lane = threadIdx.x, lda = luw_lda(N), NP = luw_np(N);
  double* As = sm;
  double* dinv = As + (size_t)NP * lda;
  int* perm = reinterpret_cast<int*>(dinv + NP);
  for (long long s = blockIdx.x; s < n; s += gridDim.x) {
    __syncwarp();
    for (int idx = lane; idx < NP * lda; idx += 32) As[idx] = 0.0;
    __syncwarp();
    const double* src = A + (size_t)s * N * N;
    for (int idx = lane; idx < N * N; idx += 32) { const int i = idx / N, j = idx - i * N; As[(size_t)i * lda + j] = src[idx]; }
    __syncwarp();
    const bool ok = lu_factor_warp_dmma<NR>(As, lda, N, perm, dinv);
    double bb[NR];
#pragma unroll
    for (int r = 0; r < NR; ++r) { const int i = lane + 32 * r; bb[r] = (i < N) ? b[(size_t)s * N + perm[i]] : 0.0; }
    lu_solve_warp_regs<NR>(As, lda, N, dinv, bb);
#pragma unroll
    for (int r = 0; r < NR; ++r) { const int i = lane + 32 * r; if (i < N) x[(size_t)s * N + i] = bb[r]; }
    if (lane == 0 && status) status[s] = ok ? CK_ST_OK : CK_ST_ZERO_PIVOT;
  }
}

}  // namespace ck

using namespace ck;

extern "C" int32_t ck_lu_solve_batched(int32_t N, int64_t n, const double* A, const double* b, double* x, int32_t* status,
                                       void* stream) {
  if (N < 1 || N > 128 || n < 0) { set_error("ck_lu_solve_batched: bad sizes (1 <= N <= 128)"); return CK_EINVAL; }
  if (n == 0) return CK_OK;
  if (!A || !b || !x) { set_error("ck_lu_solve_batched: null pointer"); return CK_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream;
  const size_t smem = ((size_t)luw_block_doubles(N) + luw_np(N)) * sizeof(double) + (size_t)luw_np(N) * sizeof(int);
  int dev = 0, sms = 0, per_sm = 0;
  CK_CUDA(cudaGetDevice(&dev));
  CK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  auto run = [&](auto kern) -> int32_t {
    CK_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CK_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 32, smem));
    const long long grid = std::max<long long>(1, std::min<long long>(n, (long long)std::max(per_sm, 1) * sms));
    kern<<<(unsigned)grid, 32, smem, st>>>(N, n, A, b, x, status);
    CK_CUDA(cudaGetLastError());
    return CK_OK;
  };
  switch ((N + 31) / 32) {
    case 1: return run(lu_solve_batched_kernel<1>);
    case 2: return run(lu_solve_batched_kernel<2>);
    case 3: return run(lu_solve_batched_kernel<3>);
    default: return run(lu_solve_batched_kernel<4>);
  }
}
