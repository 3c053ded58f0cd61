// common.cuh -- shared plumbing of the CUDA path: status/error handling, launch helpers,
// device sincos.  Not shared with oracle/ (which includes nothing from this tree).
#pragma once

#include <cuda_runtime.h>

#include <atomic>
#include <cstdarg>
#include <cstdint>
#include <cstdio>

#include "../../include/sfd.h"

namespace sfd {

void set_error(const char* fmt, ...);

#define SFD_CUDA_TRY(expr)                                                                 \
  do {                                                                                     \
    cudaError_t _e = (expr);                                                               \
    if (_e != cudaSuccess) {                                                               \
      ::sfd::set_error("%s:%d: %s failed: %s", __FILE__, __LINE__, #expr, cudaGetErrorString(_e)); \
      return SFD_ERR_CUDA;                                                                 \
    }                                                                                      \
  } while (0)

#define SFD_TRY(expr)          \
  do {                         \
    int _s = (expr);           \
    if (_s != SFD_OK) return _s; \
  } while (0)

#define SFD_REQUIRE(cond, code, ...) \
  do {                               \
    if (!(cond)) {                   \
      ::sfd::set_error(__VA_ARGS__); \
      return (code);                 \
    }                                \
  } while (0)

// number of kernels of this library launched so far in the process (sfd_launch_count)
extern std::atomic<long long> g_launches;

// Device-side error word, one per device, owned by the library (api.cu).  A kernel that meets invalid input it can
// only see on the device -- a face index outside [0, nV) -- sets kFlagBadIndex with atomicOr; the final kernel of
// every reduction collects and clears the word, and the synchronising call that reads the result back returns
// SFD_ERR_INVALID_ARG ("checked on device, reported at the next synchronising call").
constexpr int kFlagBadIndex = 1;
int32_t* device_flags();   // device address of the word on the current device (nullptr if the lookup fails)

inline int launch_check(const char* what) {
  ++g_launches;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    set_error("launch of %s failed: %s", what, cudaGetErrorString(e));
    return SFD_ERR_CUDA;
  }
  return SFD_OK;
}

inline size_t align_up(size_t n, size_t a = 256) { return (n + a - 1) / a * a; }

// Bump allocator over the caller's workspace.
struct Arena {
  char* base;
  size_t cap, off;
  Arena(void* p, size_t bytes) : base(static_cast<char*>(p)), cap(bytes), off(0) {}
  template <class T>
  T* take(size_t count) {
    size_t o = align_up(off);
    off = o + count * sizeof(T);
    return reinterpret_cast<T*>(base + o);  // validity is checked once via fits()
  }
  bool fits() const { return off <= cap; }
};

int num_sms();

// Kernel attributes (the opt-in to > 48 KB of dynamic shared memory) are per device: true when the calling thread has
// not yet seen the current device with this slot (`last` is a static thread_local int initialised to -1).
inline bool first_use_on_device(int& last) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return true;
  if (last == dev) return false;
  last = dev;
  return true;
}

// stage timing (sfd_set_profiling)
void prof_begin(cudaStream_t st);
void prof_mark(const char* name, cudaStream_t st);
void prof_end(cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// fp64 sincos for arbitrary finite arguments up to |t| ~ 2^30 (every phase xi.x of this library):
// n = round(t * 2/pi); two-term Cody-Waite reduction with FMA (t - n*PIO2_HI is exact, see
// DESIGN.md "direct sum"); degree-13/14 polynomials on [-pi/4, pi/4]; quadrant fix-up on the
// integer pipe.  Max error ~1 ulp of the result + the fp64 rounding of t itself.
// Coefficients: Chebyshev-node interpolants of (sin(sqrt z)/sqrt z - 1)/z and (cos(sqrt z) - 1 + z/2)/z^2 on
// [0, (1.02 pi/4)^2], computed at 60 digits; the literals are checked against mpmath by tests/test_kernel_constants_cpu.py.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void sincos_fp64(double t, double& s, double& c) {
  const double kTwoOverPi = 6.36619772367581382433e-01;
  const double kMagic = 6755399441055744.0;         // 1.5 * 2^52: adds round-to-nearest-integer
  const double kPio2Hi = 1.57079632679489655800e+00;  // fp64(pi/2)
  const double kPio2Lo = 6.12323399573676603587e-17;  // pi/2 - fp64(pi/2)
  const double nm = __fma_rn(t, kTwoOverPi, kMagic);
  const int q = __double2loint(nm);
  const double n = nm - kMagic;
  double r = __fma_rn(-n, kPio2Hi, t);
  r = __fma_rn(-n, kPio2Lo, r);
  const double z = r * r;
  // sin(r) = r + r z P(z), cos(r) = 1 - z/2 + z^2 Q(z); P, Q: see above
  double ps = 1.59124614998394676947e-10;
  ps = __fma_rn(ps, z, -2.50510515868469095197e-8);
  ps = __fma_rn(ps, z, 2.75573157096352918481e-6);
  ps = __fma_rn(ps, z, -1.98412698359855841056e-4);
  ps = __fma_rn(ps, z, 8.33333333333042701245e-3);
  ps = __fma_rn(ps, z, -1.66666666666666640762e-1);
  const double sr = __fma_rn(r * z, ps, r);
  double pc = -1.13790866347294788724e-11;
  pc = __fma_rn(pc, z, 2.08760960589953694532e-9);
  pc = __fma_rn(pc, z, -2.75573170259234590869e-7);
  pc = __fma_rn(pc, z, 2.4801587298282115935e-5);
  pc = __fma_rn(pc, z, -1.38888888888870710153e-3);
  pc = __fma_rn(pc, z, 4.16666666666666650464e-2);
  pc = __fma_rn(pc, z, -0.5);
  const double cr = __fma_rn(pc, z, 1.0);
  // quadrant: q&1 swaps, sign of sin flips for q&2, sign of cos flips for (q+1)&2
  double so = (q & 1) ? cr : sr;
  double co = (q & 1) ? sr : cr;
  const int shi = __double2hiint(so) ^ ((q & 2) << 30);
  const int chi = __double2hiint(co) ^ (((q + 1) & 2) << 30);
  s = __hiloint2double(shi, __double2loint(so));
  c = __hiloint2double(chi, __double2loint(co));
}

}  // namespace sfd
