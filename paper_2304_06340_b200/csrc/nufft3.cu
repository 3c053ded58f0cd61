// placeholder, replaced by the type-3 NUFFT
#include "internal.cuh"
namespace sfd {
int nufft3_sizes(int64_t, int64_t, const double*, const double*, double, Nufft3Sizes*) {
  set_error("type-3 NUFFT not built yet");
  return SFD_ERR_UNSUPPORTED;
}
int nufft3(const double*, const double*, int64_t, const double*, int64_t, double, double*, void*, size_t, cudaStream_t) {
  set_error("type-3 NUFFT not built yet");
  return SFD_ERR_UNSUPPORTED;
}
int nufft3_release_cache() { return SFD_OK; }
}  // namespace sfd
