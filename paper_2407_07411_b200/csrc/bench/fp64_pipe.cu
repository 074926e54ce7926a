// libhpsi_bench.so (include/hpsi_bench.h): register-resident DMMA.8x8x4 / DFMA issue-rate probes that bench.py loads to
// state what the FP64 pipes of this B200 can do next to the cuBLAS DGEMM calibration.  Stand-alone: shares nothing with
// the product library.
#include <cuda_runtime.h>

#include <string>

#include "../../../include/hpsi_bench.h"

namespace {

thread_local std::string g_err;
int fail(cudaError_t e, const char* what) {
  g_err = std::string("CUDA error: ") + cudaGetErrorString(e) + " in " + what;
  cudaGetLastError();
  return -3;
}
#define BENCH_CUDA(call)                                   \
  do {                                                     \
    cudaError_t e_ = (call);                               \
    if (e_ != cudaSuccess) return fail(e_, #call);         \
  } while (0)

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// KIND 0: 16 independent DMMA chains per warp; 1: 32 independent DFMA chains per thread; 2: both interleaved.
template <int KIND>
__global__ void __launch_bounds__(256) pipe_kernel(int iters, double* sink, double a0, double b0) {
  double c[16][2], f[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) { c[i][0] = c[i][1] = 0.0; f[i] = threadIdx.x * 1e-9 + i; }
  double a = a0 + threadIdx.x * 1e-12, b = b0;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      if (KIND == 0 || KIND == 2) dmma(c[i][0], c[i][1], a, b);
      if (KIND == 1 || KIND == 2) {
        asm volatile("fma.rn.f64 %0, %1, %2, %0;\n" : "+d"(f[i]) : "d"(a), "d"(b));
        if (KIND == 1) asm volatile("fma.rn.f64 %0, %1, %2, %0;\n" : "+d"(f[i]) : "d"(b), "d"(a));
      }
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1] + f[i];
  if (s == 12345.678) sink[0] = s;
}

}  // namespace

extern "C" int hpsi_bench_fp64_pipe(int kind, int iters, double* ms_out, double* flops_out) {
  int wps = 0;                                   // kind = 100 + w: DMMA probe with w warps per SM (one CTA per SM)
  if (kind >= 101 && kind <= 132) { wps = kind - 100; kind = 0; }
  if (kind < 0 || kind > 2 || iters < 1 || !ms_out || !flops_out) { g_err = "bad argument"; return -1; }
  int dev = 0, n_sm = 0;
  BENCH_CUDA(cudaGetDevice(&dev));
  BENCH_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  double* sink = nullptr;
  BENCH_CUDA(cudaMalloc(&sink, 8));
  cudaEvent_t e0, e1;
  BENCH_CUDA(cudaEventCreate(&e0));
  BENCH_CUDA(cudaEventCreate(&e1));
  const int grid = wps ? n_sm * wps : n_sm * 4, threads = wps ? 32 : 256;   // w one-warp CTAs per SM
  auto run = [&](int n) {
    if (kind == 0) pipe_kernel<0><<<grid, threads>>>(n, sink, 1.0, 1e-9);
    else if (kind == 1) pipe_kernel<1><<<grid, threads>>>(n, sink, 1.0, 1e-9);
    else pipe_kernel<2><<<grid, threads>>>(n, sink, 1.0, 1e-9);
  };
  run(iters / 10 + 1);
  BENCH_CUDA(cudaDeviceSynchronize());
  BENCH_CUDA(cudaEventRecord(e0));
  run(iters);
  BENCH_CUDA(cudaEventRecord(e1));
  BENCH_CUDA(cudaEventSynchronize(e1));
  float ms = 0.f;
  BENCH_CUDA(cudaEventElapsedTime(&ms, e0, e1));
  const double warps = (double)grid * threads / 32.0;
  double flops = 0.0;
  if (kind == 0 || kind == 2) flops += warps * iters * 16.0 * 512.0;                 // 8x8x4 MMA = 512 flops
  if (kind == 1) flops += warps * 32.0 * iters * 32.0 * 2.0;                         // 32 DFMA per thread per iter
  if (kind == 2) flops += warps * 32.0 * iters * 16.0 * 2.0;
  *ms_out = ms;
  *flops_out = flops;
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  return 0;
}

extern "C" const char* hpsi_bench_last_error(void) { return g_err.c_str(); }
