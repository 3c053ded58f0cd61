// probe.cu -- measured FP64 FMA throughput of the device: the roofline denominator of the direct sum (A4), which
// MEASURED_PEAKS.json does not carry.  8 independent DFMA chains per thread, 256 threads x 8 CTAs per SM.
#include "internal.cuh"

namespace sfd {
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

int probe_fp64(int iters, cudaStream_t st, double* h_tflops, double* h_ms) {
  SFD_REQUIRE(h_tflops && h_ms, SFD_ERR_NULL, "sfd_probe_fp64: NULL output");
  SFD_REQUIRE(iters >= 1 && iters <= (1 << 20), SFD_ERR_INVALID_ARG, "sfd_probe_fp64: iters out of range");
  double* sink = nullptr;
  SFD_CUDA_TRY(cudaMalloc(&sink, 256));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int blocks = num_sms() * 8;
  fp64_fma_kernel<<<blocks, 256, 0, st>>>(16, 0.999999, 1e-9, sink);  // warm-up
  cudaEventRecord(e0, st);
  fp64_fma_kernel<<<blocks, 256, 0, st>>>(iters, 0.999999, 1e-9, sink);
  cudaEventRecord(e1, st);
  int rc = launch_check("fp64_fma_kernel");
  cudaError_t e = cudaStreamSynchronize(st);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (rc != SFD_OK) return rc;
  SFD_CUDA_TRY(e);
  const double flops = 2.0 * (double)blocks * 256.0 * kChains * kInner * (double)iters;
  *h_ms = ms;
  *h_tflops = flops / (ms * 1e-3) * 1e-12;
  return SFD_OK;
}

}  // namespace sfd
