// noalloc.cu -- sfd_surface_ft_direct_static (include/sfd.h): the fp64 direct sum of A4 for callers that
// cannot allocate -- code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  The one piece of
// scratch the direct sum needs (the partial sums of its source splits, direct.cu: nsplit x K complex128 values, combined
// in a fixed order) lives in a file-scope device array of SFD_STATIC_SCRATCH_BYTES instead of a caller's workspace.
// Every GPU that loads the library holds that array until the process exits.
//
// The array is shared by every call on the device and keeps the last call's contents.  Nothing in it has to start at
// zero: each (split, target) entry is written by exactly one thread of direct_sum_kernel before combine_splits_kernel
// reads it, so there is nothing to clear.  Two calls that overlap on the GPU (different streams, or graphs replayed
// concurrently) race on it; calls on one stream are ordered and safe.
//
// In host code the array's name is a host-side stand-in, not a device address: the address the kernels get is looked up
// with cudaGetSymbolAddress here, in the file that defines the array, once per device with that device current.
#include <mutex>

#include "direct.cuh"

namespace sfd {
namespace {

static __device__ __align__(256) unsigned char g_static_scratch[SFD_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;

// Device address of g_static_scratch on the current device.
int static_scratch(void** out) {
  static std::mutex mu;
  static void* ptr[kMaxDevices] = {};
  int dev = 0;
  SFD_CUDA_TRY(cudaGetDevice(&dev));
  SFD_REQUIRE(dev >= 0 && dev < kMaxDevices, SFD_ERR_UNSUPPORTED, "device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lk(mu);
  if (!ptr[dev]) {
    void* p = nullptr;
    SFD_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scratch));
    SFD_REQUIRE(p && (reinterpret_cast<uintptr_t>(p) & 255) == 0, SFD_ERR_CUDA,
                "static scratch array has no usable device address on device %d", dev);
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return SFD_OK;
}

}  // namespace
}  // namespace sfd

using namespace sfd;

extern "C" {

int sfd_surface_ft_direct_static_scratch(int64_t J, int64_t K, size_t* bytes) {
  SFD_REQUIRE(bytes, SFD_ERR_NULL, "sfd_surface_ft_direct_static_scratch: bytes is NULL");
  SFD_REQUIRE(J >= 0 && K >= 0, SFD_ERR_INVALID_ARG, "J and K must be >= 0");
  *bytes = (J == 0 || K == 0) ? 0 : direct_plan(J, K).work_bytes;
  return SFD_OK;
}

int sfd_surface_ft_direct_static(const double* d_x, const double* d_w, int64_t J, const double* d_xi, int64_t K,
                                 double* d_nuhat, sfd_stream stream) {
  SFD_REQUIRE(J >= 0 && K >= 0, SFD_ERR_INVALID_ARG, "J and K must be >= 0");
  if (K == 0) return SFD_OK;
  SFD_REQUIRE(d_xi && d_nuhat, SFD_ERR_NULL, "sfd_surface_ft_direct_static: NULL target buffer");
  SFD_REQUIRE(J == 0 || (d_x && d_w), SFD_ERR_NULL, "sfd_surface_ft_direct_static: NULL source buffer");
  const size_t need = J == 0 ? 0 : direct_plan(J, K).work_bytes;
  SFD_REQUIRE(need <= (size_t)SFD_STATIC_SCRATCH_BYTES, SFD_ERR_UNSUPPORTED,
              "sfd_surface_ft_direct_static: J = %lld sources x K = %lld targets need %zu bytes of scratch for the partial "
              "sums of the source splits, the static array holds %zu (SFD_STATIC_SCRATCH_BYTES); use sfd_surface_ft with a "
              "workspace",
              (long long)J, (long long)K, need, (size_t)SFD_STATIC_SCRATCH_BYTES);
  void* scratch = nullptr;
  SFD_TRY(static_scratch(&scratch));
  // the kernels of direct.cu, with the static array where the caller's workspace would be
  return direct_sum(d_x, d_w, J, d_xi, K, d_nuhat, scratch, (size_t)SFD_STATIC_SCRATCH_BYTES, static_cast<cudaStream_t>(stream));
}

}  // extern "C"
