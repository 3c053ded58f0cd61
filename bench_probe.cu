// bench_probe.cu -- bench.py's helper, NOT part of libsfd.so: measured FP64 FMA throughput of the device, the roofline
// denominator of the direct sum (A4), which MEASURED_PEAKS.json does not carry.  8 independent DFMA chains per thread,
// 256 threads x 8 CTAs per SM.  Built by __graft_entry__.build() / bench.py into libbench_probe.so (repo root).
#include <cuda_runtime.h>

namespace {

constexpr int kChains = 8;
constexpr int kInner = 64;

__global__ void __launch_bounds__(256) fp64_fma_kernel(int iters, double a, double b, double* __restrict__ sink) {
  double v[kChains];
#pragma unroll
  for (int c = 0; c < kChains; ++c) v[c] = (double)(threadIdx.x + c) * 1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < kInner; ++u) {
#pragma unroll
      for (int c = 0; c < kChains; ++c) v[c] = __fma_rn(v[c], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int c = 0; c < kChains; ++c) s += v[c];
  if (s == 123.456) sink[0] = s;  // never true: keeps the chains alive
}

}  // namespace

// Returns 0 and the achieved TFLOP/s (FMA = 2 flops) / kernel time of a dependency-free DFMA loop covering every SM of the
// current device; a CUDA error code otherwise.  `stream` is a cudaStream_t.  Synchronises it.
extern "C" int bench_probe_fp64(int iters, void* stream, double* h_tflops, double* h_ms) {
  if (!h_tflops || !h_ms || iters < 1 || iters > (1 << 20)) return -1;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  double* sink = nullptr;
  if (e == cudaSuccess) e = cudaMalloc(&sink, 256);
  if (e != cudaSuccess) return (int)e;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int blocks = sms * 8;
  fp64_fma_kernel<<<blocks, 256, 0, st>>>(16, 0.999999, 1e-9, sink);  // warm-up
  cudaEventRecord(e0, st);
  fp64_fma_kernel<<<blocks, 256, 0, st>>>(iters, 0.999999, 1e-9, sink);
  cudaEventRecord(e1, st);
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (e != cudaSuccess) return (int)e;
  const double flops = 2.0 * (double)blocks * 256.0 * kChains * kInner * (double)iters;
  *h_ms = ms;
  *h_tflops = flops / (ms * 1e-3) * 1e-12;
  return 0;
}
