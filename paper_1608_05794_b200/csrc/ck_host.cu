// Host-buffer entry points (end-to-end path: transfers inside the call) and the FP64 peak probe.
#include <algorithm>

#include "ck_internal.h"

using namespace ck;

namespace {

// grow-only device staging buffer cached in the handle
int32_t stage_reserve(ck_mech* m, size_t bytes) {
  if (m->stage_bytes >= bytes) return CK_OK;
  if (m->stage) { cudaFree(m->stage); m->stage = nullptr; m->stage_bytes = 0; }
  CK_CUDA(cudaMalloc(&m->stage, bytes));
  m->stage_bytes = bytes;
  return CK_OK;
}
inline size_t al(size_t x) { return (x + 255) & ~size_t(255); }

// register-resident DFMA chains: 8 independent accumulators per thread, ITER x 8 DFMA per thread
__global__ void __launch_bounds__(256) dfma_probe(double* out, double a, double b, int iters) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

// the same for the FP64 tensor-core path: 8 independent m8n8k4 accumulator tiles per warp (256 FMA per instruction)
__global__ void __launch_bounds__(256) dmma_probe(double* out, double a, double b, int iters) {
  double c[8][2];
#pragma unroll
  for (int i = 0; i < 8; ++i) { c[i][0] = threadIdx.x + i; c[i][1] = i; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

extern "C" int32_t ck_fp64_mma_peak(int32_t device, double* fma_per_s, void* stream) {
  if (!fma_per_s) { set_error("ck_fp64_mma_peak: null output"); return CK_EINVAL; }
  CK_CUDA(cudaSetDevice(device));
  cudaStream_t st = (cudaStream_t)stream;
  int sms = 0;
  CK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
  const int blocks = sms * 4, threads = 256, iters = 8192;
  double* out = nullptr;
  CK_CUDA(cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)));
  cudaEvent_t e0, e1;
  CK_CUDA(cudaEventCreate(&e0));
  CK_CUDA(cudaEventCreate(&e1));
  double best = 0;
  for (int rep = 0; rep < 6; ++rep) {
    CK_CUDA(cudaEventRecord(e0, st));
    dmma_probe<<<blocks, threads, 0, st>>>(out, 1.0000001, 0.9999999, iters);
    CK_CUDA(cudaEventRecord(e1, st));
    CK_CUDA(cudaEventSynchronize(e1));
    float ms = 0;
    CK_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    const double rate = (double)blocks * (threads / 32) * iters * 8.0 * 256.0 / (ms * 1e-3);
    if (rep >= 1) best = std::max(best, rate);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
  *fma_per_s = best;
  return CK_OK;
}

extern "C" int32_t ck_fp64_peak(int32_t device, double* dfma_per_s, void* stream) {
  if (!dfma_per_s) { set_error("ck_fp64_peak: null output"); return CK_EINVAL; }
  CK_CUDA(cudaSetDevice(device));
  cudaStream_t st = (cudaStream_t)stream;
  int sms = 0;
  CK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
  const int blocks = sms * 8, threads = 256, iters = 4096;
  double* out = nullptr;
  CK_CUDA(cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)));
  cudaEvent_t e0, e1;
  CK_CUDA(cudaEventCreate(&e0));
  CK_CUDA(cudaEventCreate(&e1));
  double best = 0;
  for (int rep = 0; rep < 6; ++rep) {
    CK_CUDA(cudaEventRecord(e0, st));
    dfma_probe<<<blocks, threads, 0, st>>>(out, 0.999999, 1e-9, iters);
    CK_CUDA(cudaEventRecord(e1, st));
    CK_CUDA(cudaEventSynchronize(e1));
    float ms = 0;
    CK_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    const double rate = (double)blocks * threads * iters * 64.0 / (ms * 1e-3);
    if (rep >= 1) best = std::max(best, rate);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
  *dfma_per_s = best;
  return CK_OK;
}

// Chunked pipeline: the batch is column-separable, PCIe is full duplex, so the states are cut into column blocks
// that travel H2D / through the kernel / D2H on three streams -- while block c is evaluated, block c + 1 is on its way
// in and block c - 1 on its way out.  Host buffers should be pinned (pageable memory makes the copies synchronous).
extern "C" int32_t ck_rhs_host(ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double* dydt,
                               int64_t ld_out) {
  if (!m) { set_error("ck_rhs_host: null mechanism"); return CK_EINVAL; }
  if (n < 0 || ld < n || ld_out < n) { set_error("ck_rhs_host: bad n/ld"); return CK_EINVAL; }
  if (n == 0) return CK_OK;
  if (!y || !p || !dydt) { set_error("ck_rhs_host: null batch pointer"); return CK_EINVAL; }
  CK_CUDA(cudaSetDevice(m->device));
  constexpr int NS = 3;
  for (int i = 0; i < NS; ++i)
    if (!m->pstream[i]) CK_CUDA(cudaStreamCreateWithFlags(&m->pstream[i], cudaStreamNonBlocking));
  const int N = m->K + 1;
  // block width: at least the batch the tensor-memory kernel wants, at most an eighth of the batch
  const int64_t blk = std::min<int64_t>(n, std::max<int64_t>(65536, (n + 7) / 8));
  const size_t by = al((size_t)N * blk * sizeof(double)), bp = al((size_t)blk * sizeof(double));
  int32_t rc = stage_reserve(m, NS * (2 * by + bp));
  if (rc) return rc;
  int c = 0;
  for (int64_t b = 0; b < n; b += blk, ++c) {
    const int64_t nb = std::min<int64_t>(blk, n - b);
    const int sidx = c % NS;
    cudaStream_t st = m->pstream[sidx];
    char* base = (char*)m->stage + (size_t)sidx * (2 * by + bp);
    double* dy = (double*)base;
    double* df = (double*)(base + by);
    double* dp = (double*)(base + 2 * by);
    CK_CUDA(cudaMemcpy2DAsync(dy, nb * sizeof(double), y + b, ld * sizeof(double), nb * sizeof(double), N, cudaMemcpyHostToDevice, st));
    CK_CUDA(cudaMemcpyAsync(dp, p + b, nb * sizeof(double), cudaMemcpyHostToDevice, st));
    rc = ck_rhs(m, nb, dy, nb, dp, df, nb, st);
    if (rc) return rc;
    CK_CUDA(cudaMemcpy2DAsync(dydt + b, ld_out * sizeof(double), df, nb * sizeof(double), nb * sizeof(double), N, cudaMemcpyDeviceToHost, st));
  }
  for (int i = 0; i < NS; ++i) CK_CUDA(cudaStreamSynchronize(m->pstream[i]));
  return CK_OK;
}

extern "C" int32_t ck_integrate_host(ck_mech* m, int32_t op, int64_t n, double* y, int64_t ld, const double* p, double dt,
                                     const ck_opts* opts, int32_t* n_accept, int32_t* n_reject, int32_t* status,
                                     double* h_last, ck_report* report) {
  if (!m) { set_error("ck_integrate_host: null mechanism"); return CK_EINVAL; }
  if (op != CK_OP_ROS && op != CK_OP_RKF45) { set_error("ck_integrate_host: bad op %d", op); return CK_EINVAL; }
  if (n < 0 || ld < n) { set_error("ck_integrate_host: bad n/ld"); return CK_EINVAL; }
  if (n == 0) { if (report) *report = ck_report{}; return CK_OK; }
  if (!y || !p) { set_error("ck_integrate_host: null batch pointer"); return CK_EINVAL; }
  CK_CUDA(cudaSetDevice(m->device));
  if (!m->hstream) CK_CUDA(cudaStreamCreateWithFlags(&m->hstream, cudaStreamNonBlocking));
  const int N = m->K + 1;
  size_t wsb = 0;
  int32_t rc = ck_workspace_bytes(m, op, n, &wsb);
  if (rc) return rc;
  const size_t by = al((size_t)N * n * sizeof(double)), bp = al((size_t)n * sizeof(double)), bi = al((size_t)n * sizeof(int32_t));
  rc = stage_reserve(m, by + 2 * bp + 3 * bi + al(wsb));
  if (rc) return rc;
  char* b = (char*)m->stage;
  double* dy = (double*)b; b += by;
  double* dp = (double*)b; b += bp;
  double* dh = (double*)b; b += bp;
  int32_t* da = (int32_t*)b; b += bi;
  int32_t* dr = (int32_t*)b; b += bi;
  int32_t* ds = (int32_t*)b; b += bi;
  void* ws = b;
  cudaStream_t st = m->hstream;
  CK_CUDA(cudaMemcpy2DAsync(dy, n * sizeof(double), y, ld * sizeof(double), n * sizeof(double), N, cudaMemcpyHostToDevice, st));
  CK_CUDA(cudaMemcpyAsync(dp, p, n * sizeof(double), cudaMemcpyHostToDevice, st));
  ck_report local;
  ck_report* rep = report ? report : &local;
  if (op == CK_OP_ROS) rc = ck_integrate_ros(m, n, dy, n, dp, dt, opts, da, dr, ds, dh, ws, wsb, rep, st);
  else rc = ck_integrate_rkf45(m, n, dy, n, dp, dt, opts, da, dr, ds, dh, ws, wsb, rep, st);
  if (rc) return rc;
  CK_CUDA(cudaMemcpy2DAsync(y, ld * sizeof(double), dy, n * sizeof(double), n * sizeof(double), N, cudaMemcpyDeviceToHost, st));
  if (n_accept) CK_CUDA(cudaMemcpyAsync(n_accept, da, n * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (n_reject) CK_CUDA(cudaMemcpyAsync(n_reject, dr, n * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (status) CK_CUDA(cudaMemcpyAsync(status, ds, n * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (h_last) CK_CUDA(cudaMemcpyAsync(h_last, dh, n * sizeof(double), cudaMemcpyDeviceToHost, st));
  CK_CUDA(cudaStreamSynchronize(st));
  return CK_OK;
}
