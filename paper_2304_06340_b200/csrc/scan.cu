// scan.cu -- exclusive prefix sum over int32 counts: the integer backbone of A1 (midpoint ranks) and of
// the A5 bin sorts ("sort ... so that consecutive indices contribute to close memory addresses").
// Three-phase hierarchical scan (chunk scan -> scan of chunk totals -> add), deterministic, integer-exact.
#include "internal.cuh"

namespace sfd {
namespace {

constexpr int kScanThreads = 512;
constexpr int kItems = 4;
constexpr int kChunk = kScanThreads * kItems;  // 2048 counts per CTA

__device__ __forceinline__ int warp_inclusive_scan(int v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += t;
  }
  return v;
}

// out[i] = exclusive prefix inside the chunk; sums[blockIdx.x] = chunk total.
__global__ void __launch_bounds__(kScanThreads) chunk_scan_kernel(const int32_t* __restrict__ in, int32_t* __restrict__ out,
                                                                 int64_t n, int32_t* __restrict__ sums) {
  __shared__ int warp_tot[kScanThreads / 32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int64_t base = (int64_t)blockIdx.x * kChunk + (int64_t)tid * kItems;
  int v[kItems];
  int tsum = 0;
#pragma unroll
  for (int i = 0; i < kItems; ++i) {
    v[i] = base + i < n ? in[base + i] : 0;
    tsum += v[i];
  }
  const int incl = warp_inclusive_scan(tsum, lane);
  if (lane == 31) warp_tot[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    const int t = lane < kScanThreads / 32 ? warp_tot[lane] : 0;
    const int s = warp_inclusive_scan(t, lane);
    if (lane < kScanThreads / 32) warp_tot[lane] = s - t;  // exclusive offset of each warp
    if (lane == kScanThreads / 32 - 1 && sums) sums[blockIdx.x] = s;
  }
  __syncthreads();
  int run = warp_tot[wid] + incl - tsum;
#pragma unroll
  for (int i = 0; i < kItems; ++i) {
    if (base + i < n) out[base + i] = run;
    run += v[i];
  }
}

__global__ void __launch_bounds__(kScanThreads) chunk_add_kernel(int32_t* __restrict__ out, int64_t n,
                                                                const int32_t* __restrict__ sums) {
  const int add = sums[blockIdx.x];
  const int64_t base = (int64_t)blockIdx.x * kChunk + (int64_t)threadIdx.x * kItems;
#pragma unroll
  for (int i = 0; i < kItems; ++i)
    if (base + i < n) out[base + i] += add;
}

__global__ void total_kernel(const int32_t* __restrict__ last_in_copy, const int32_t* __restrict__ out, int64_t n,
                             int32_t* __restrict__ total) {
  *total = out[n - 1] + *last_in_copy;
}

__global__ void save_last_kernel(const int32_t* __restrict__ in, int64_t n, int32_t* __restrict__ slot) { *slot = in[n - 1]; }

int64_t chunks(int64_t n) { return (n + kChunk - 1) / kChunk; }

}  // namespace

size_t scan_workspace(int64_t n) {
  size_t bytes = 256;  // slot for the last input value
  for (int64_t m = chunks(n); m > 1; m = chunks(m)) bytes += align_up((size_t)m * sizeof(int32_t));
  bytes += 256;
  return bytes;
}

static int scan_rec(const int32_t* in, int32_t* out, int64_t n, char* work, cudaStream_t st) {
  const int64_t nb = chunks(n);
  if (nb <= 1) {
    chunk_scan_kernel<<<1, kScanThreads, 0, st>>>(in, out, n, nullptr);
    return launch_check("chunk_scan_kernel");
  }
  int32_t* sums = reinterpret_cast<int32_t*>(work);
  chunk_scan_kernel<<<(unsigned)nb, kScanThreads, 0, st>>>(in, out, n, sums);
  SFD_TRY(launch_check("chunk_scan_kernel"));
  SFD_TRY(scan_rec(sums, sums, nb, work + align_up((size_t)nb * sizeof(int32_t)), st));
  chunk_add_kernel<<<(unsigned)nb, kScanThreads, 0, st>>>(out, n, sums);
  return launch_check("chunk_add_kernel");
}

int exclusive_scan_i32(const int32_t* d_in, int32_t* d_out, int64_t n, int32_t* d_total, void* d_work,
                       size_t work_bytes, cudaStream_t st) {
  if (n <= 0) {
    if (d_total) SFD_CUDA_TRY(cudaMemsetAsync(d_total, 0, sizeof(int32_t), st));
    return SFD_OK;
  }
  SFD_REQUIRE(n / kChunk < 0x7fffffffLL, SFD_ERR_INVALID_ARG, "scan too long");
  SFD_REQUIRE(d_work && work_bytes >= scan_workspace(n), SFD_ERR_WORKSPACE_TOO_SMALL,
              "scan needs %zu workspace bytes, got %zu", scan_workspace(n), work_bytes);
  char* work = static_cast<char*>(d_work);
  int32_t* last = reinterpret_cast<int32_t*>(work);
  if (d_total) {
    save_last_kernel<<<1, 1, 0, st>>>(d_in, n, last);  // in-place scans overwrite in[n-1]
    SFD_TRY(launch_check("save_last_kernel"));
  }
  SFD_TRY(scan_rec(d_in, d_out, n, work + 256, st));
  if (d_total) {
    total_kernel<<<1, 1, 0, st>>>(last, d_out, n, d_total);
    SFD_TRY(launch_check("total_kernel"));
  }
  return SFD_OK;
}

}  // namespace sfd
