// reduce.cu -- A6: fused target-side kernel.  For every frequency node: r = |xi_k|, sigmahat = 4 pi sin r / r (the
// unit sphere's transform, eq. 2.14 in the e^{-i xi.x} convention), Sobolev weight (1+r^2)^{-s} (eq. 2.7),
// quadrature weight W_k, then I = (2 pi)^-3 sum_k W_k |nuhat_k - sigmahat|^2 (1+r^2)^{-s} (Plancherel, eq. 2.5).
// The paper leaves this step out of its timings ("can be ideally accelerated by GPUs").
//
// HBM-bound, 48 B per target, one pass.  The sum is carried as a (sum, compensation) fp64 pair (TwoSum) from the
// per-thread accumulators through warp shuffles, the block tree and a fixed-order final pass over the per-CTA
// partials: deterministic for a given K.
#include <algorithm>
#include <cmath>

#include "internal.cuh"

namespace sfd {
namespace {

constexpr int kThreads = 256;
constexpr int kMaxBlocks = 2048;   // upper bound of the per-CTA partials (the grid is 8 CTAs per SM of the device)

struct Comp {
  double s, c;
};

__device__ __forceinline__ void two_sum_add(Comp& a, double v) {
  const double t = __dadd_rn(a.s, v);
  const double bp = __dsub_rn(t, a.s);
  const double e = __dadd_rn(__dsub_rn(a.s, __dsub_rn(t, bp)), __dsub_rn(v, bp));
  a.s = t;
  a.c = __dadd_rn(a.c, e);
}
__device__ __forceinline__ void comp_merge(Comp& a, const Comp& b) {
  two_sum_add(a, b.s);
  a.c = __dadd_rn(a.c, b.c);
}
__device__ __forceinline__ Comp comp_shfl_down(const Comp& a, int d) {
  Comp b;
  b.s = __shfl_down_sync(0xffffffffu, a.s, d);
  b.c = __shfl_down_sync(0xffffffffu, a.c, d);
  return b;
}

__device__ __forceinline__ Comp block_reduce(Comp v) {
  __shared__ Comp part[kThreads / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    const Comp o = comp_shfl_down(v, d);
    comp_merge(v, o);
  }
  if (lane == 0) part[wid] = v;
  __syncthreads();
  if (wid == 0) {
    v = lane < kThreads / 32 ? part[lane] : Comp{0.0, 0.0};
#pragma unroll
    for (int d = 4; d > 0; d >>= 1) {
      const Comp o = comp_shfl_down(v, d);
      comp_merge(v, o);
    }
  }
  return v;  // valid in thread 0
}

__device__ __forceinline__ double sigma_hat(double r) {
  const double four_pi = 12.566370614359172;
  if (r < 1e-4) {
    const double r2 = r * r;
    return four_pi * (1.0 - r2 / 6.0 + r2 * r2 / 120.0);
  }
  return four_pi * sin(r) / r;
}

// (1+r^2)^-s: s = 1, 2 directly; other integer s <= 64 by binary powering (the paper's s = 5, 10; the generic pow costs
// more FP64 instructions than the rest of the node put together and made the pass ALU-bound); pow otherwise.
__device__ __forceinline__ double sobolev_weight(double q, double s, int s_kind) {
  if (s_kind == 1) return 1.0 / q;
  if (s_kind == 2) return 1.0 / (q * q);
  if (s_kind > 2) {
    double r = 1.0, b = q;
    for (int e = s_kind; e > 0; e >>= 1) {   // uniform across the grid
      if (e & 1) r *= b;
      b *= b;
    }
    return 1.0 / r;
  }
  return pow(q, -s);
}

// nuhat2 == nullptr: difference against the unit sphere's closed form; else against a second transform (mesh vs mesh).
// LATTICE: the nodes are the paper's lattice in the order of nodes.cu lattice_kernel and are recomputed
// from the index with the same roundings (xi = 2 pi (m h), W = h^3 / 2^{faces}) instead of being read: 16 B per node.
template <bool LATTICE>
__global__ void __launch_bounds__(kThreads) reduce_terms_kernel(const double2* __restrict__ nuhat,
                                                               const double2* __restrict__ nuhat2, const double* __restrict__ xi,
                                                               const double* __restrict__ W, int64_t K, double s, int s_kind,
                                                               double scale2, int M, double h, Comp* __restrict__ partial) {
  Comp acc{0.0, 0.0};
  const int64_t stride = (int64_t)gridDim.x * kThreads;
  for (int64_t k = (int64_t)blockIdx.x * kThreads + threadIdx.x; k < K; k += stride) {
    double a, b, c, wk;
    if (LATTICE) {
      const unsigned n = (unsigned)M + 1u, ku = (unsigned)k;
      const unsigned ab = ku / n;
      const int ic = (int)(ku - ab * n) - M / 2, ib = (int)(ab % n) - M / 2, ia = (int)(ab / n) - M / 2;
      const double two_pi = 6.283185307179586476925286766559;
      a = __dmul_rn(two_pi, __dmul_rn((double)ia, h));
      b = __dmul_rn(two_pi, __dmul_rn((double)ib, h));
      c = __dmul_rn(two_pi, __dmul_rn((double)ic, h));
      wk = __dmul_rn(__dmul_rn(h, h), h);
      if (ia == -M / 2 || ia == M / 2) wk = __dmul_rn(wk, 0.5);
      if (ib == -M / 2 || ib == M / 2) wk = __dmul_rn(wk, 0.5);
      if (ic == -M / 2 || ic == M / 2) wk = __dmul_rn(wk, 0.5);
    } else {
      a = xi[3 * k], b = xi[3 * k + 1], c = xi[3 * k + 2];
      wk = W[k];
    }
    const double2 nu = nuhat[k];
    const double r2 = a * a + b * b + c * c;
    const double r = sqrt(r2);
    double dre, dim;
    if (nuhat2) {
      const double2 nb = nuhat2[k];
      dre = nu.x - nb.x;
      dim = nu.y - nb.y;
    } else {
      dre = nu.x - sigma_hat(r);
      dim = nu.y;
    }
    const double term = wk * (dre * dre + dim * dim) * sobolev_weight(__fma_rn(scale2, r2, 1.0), s, s_kind);
    two_sum_add(acc, term);
  }
  const Comp tot = block_reduce(acc);
  if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

// The paper's lattice straight from the type-1 transform's FFT output (internal.cuh Nufft1Band): mode (m0, m1, m2 >= 0)
// -> nuhat = v dec0[|m0|] dec1[|m1|] dec2[m2] e^{-i xi.C}, xi = 2 pi (m h); its mirror mode has the conjugate transform
// and the same radius and weight, hence the same term: modes with m2 > 0 count twice.
__global__ void __launch_bounds__(kThreads) lattice_band_terms_kernel(const double2* __restrict__ v, const double* __restrict__ dec,
                                                                     double c0, double c1, double c2, int M, double h,
                                                                     double s, int s_kind, double scale2, int f32,
                                                                     Comp* __restrict__ partial) {
  const int n = M + 1, nh = M / 2 + 1;
  const int64_t Kh = (int64_t)n * n * nh;
  const bool phase = c0 != 0.0 || c1 != 0.0 || c2 != 0.0;
  Comp acc{0.0, 0.0};
  const int64_t stride = (int64_t)gridDim.x * kThreads;
  for (int64_t k = (int64_t)blockIdx.x * kThreads + threadIdx.x; k < Kh; k += stride) {
    const unsigned ku = (unsigned)k, ab = ku / (unsigned)nh;
    const int m2 = (int)(ku - ab * (unsigned)nh), m1 = (int)(ab % (unsigned)n) - M / 2, m0 = (int)(ab / (unsigned)n) - M / 2;
    const double two_pi = 6.283185307179586476925286766559;
    const double a = __dmul_rn(two_pi, __dmul_rn((double)m0, h)), b = __dmul_rn(two_pi, __dmul_rn((double)m1, h)),
                 c = __dmul_rn(two_pi, __dmul_rn((double)m2, h));
    double wk = __dmul_rn(__dmul_rn(h, h), h);
    if (m0 == -M / 2 || m0 == M / 2) wk = __dmul_rn(wk, 0.5);
    if (m1 == -M / 2 || m1 == M / 2) wk = __dmul_rn(wk, 0.5);
    if (m2 == M / 2) wk = __dmul_rn(wk, 0.5);
    if (m2 > 0) wk = __dmul_rn(wk, 2.0);
    double2 g;
    if (f32) {   // single-precision band (N3Params::f32)
      const float2 gf = reinterpret_cast<const float2*>(v)[k];
      g = make_double2((double)gf.x, (double)gf.y);
    } else {
      g = v[k];
    }
    const double f = dec[abs(m0)] * dec[nh + abs(m1)] * dec[2 * nh + m2];
    g.x *= f;
    g.y *= f;
    if (phase) {
      double sn, cs;
      sincos_fp64(__fma_rn(a, c0, __fma_rn(b, c1, c * c2)), sn, cs);
      g = make_double2(g.x * cs + g.y * sn, g.y * cs - g.x * sn);
    }
    const double r2 = a * a + b * b + c * c;
    const double dre = g.x - sigma_hat(sqrt(r2));
    const double term = wk * (dre * dre + g.y * g.y) * sobolev_weight(__fma_rn(scale2, r2, 1.0), s, s_kind);
    two_sum_add(acc, term);
  }
  const Comp tot = block_reduce(acc);
  if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

// result[0] = I; result[1] = the device error word (collected and cleared: common.cuh device_flags); result[2..3] =
// the (sum, compensation) pair scaled by pref, for consumers that keep adding (the shards of a multi-GPU run).
__global__ void __launch_bounds__(kThreads) reduce_final_kernel(const Comp* __restrict__ partial, int n, double pref,
                                                               double* __restrict__ result, int32_t* __restrict__ flags) {
  Comp acc{0.0, 0.0};
  for (int i = threadIdx.x; i < n; i += kThreads) comp_merge(acc, partial[i]);
  const Comp tot = block_reduce(acc);
  if (threadIdx.x == 0) {
    result[0] = (tot.s + tot.c) * pref;
    result[1] = flags ? (double)atomicExch(flags, 0) : 0.0;
    result[2] = tot.s * pref;
    result[3] = tot.c * pref;
  }
}

int reduce_blocks(int64_t K) {
  const int64_t want = (K + kThreads - 1) / kThreads;
  const int64_t cap = std::min<int64_t>(kMaxBlocks, (int64_t)num_sms() * 8);
  return (int)(want < 1 ? 1 : (want > cap ? cap : want));
}

}  // namespace

size_t reduce_workspace(int64_t K) {
  (void)K;
  return 256 + align_up(sizeof(Comp) * kMaxBlocks);
}

namespace {
int reduce_any(const double* d_nuhat, const double* d_xi, const double* d_W, int64_t K, double s, void* d_work,
               size_t work_bytes, cudaStream_t st, double** d_result, double scale, double pref, const double* d_nuhat2,
               int M, double h) {
  if (pref < 0.0) pref = 1.0 / (6.283185307179586 * 6.283185307179586 * 6.283185307179586);   // (2 pi)^-3
  SFD_REQUIRE(K >= 0, SFD_ERR_INVALID_ARG, "K must be >= 0");
  SFD_REQUIRE(s > 0.5 && s < 1e6, SFD_ERR_INVALID_ARG, "Sobolev order s must exceed 1/2 (P:113), got %g", s);
  SFD_REQUIRE(d_work && work_bytes >= reduce_workspace(K), SFD_ERR_WORKSPACE_TOO_SMALL,
              "reduction needs %zu workspace bytes, got %zu", reduce_workspace(K), work_bytes);
  SFD_REQUIRE(K == 0 || (d_nuhat && (M > 0 || (d_xi && d_W))), SFD_ERR_NULL, "sfd_reduce: NULL input buffer");
  double* result = static_cast<double*>(d_work);
  Comp* partial = reinterpret_cast<Comp*>(static_cast<char*>(d_work) + 256);
  *d_result = result;
  if (K == 0) {
    SFD_CUDA_TRY(cudaMemsetAsync(result, 0, 4 * sizeof(double), st));
    return SFD_OK;
  }
  const int blocks = reduce_blocks(K);
  const int s_kind = (s == std::floor(s) && s >= 1.0 && s <= 64.0) ? (int)s : 0;   // integer exponent, else 0
  const double2* nu = reinterpret_cast<const double2*>(d_nuhat);
  const double2* nu2 = reinterpret_cast<const double2*>(d_nuhat2);
  if (M > 0)
    reduce_terms_kernel<true><<<blocks, kThreads, 0, st>>>(nu, nu2, nullptr, nullptr, K, s, s_kind, scale * scale, M, h, partial);
  else
    reduce_terms_kernel<false><<<blocks, kThreads, 0, st>>>(nu, nu2, d_xi, d_W, K, s, s_kind, scale * scale, 0, 0.0, partial);
  SFD_TRY(launch_check("reduce_terms_kernel"));
  reduce_final_kernel<<<1, kThreads, 0, st>>>(partial, blocks, pref, result, device_flags());
  return launch_check("reduce_final_kernel");
}
}  // namespace

int reduce_enqueue(const double* d_nuhat, const double* d_xi, const double* d_W, int64_t K, double s, void* d_work,
                   size_t work_bytes, cudaStream_t st, double** d_result, double scale, double pref,
                   const double* d_nuhat2) {
  return reduce_any(d_nuhat, d_xi, d_W, K, s, d_work, work_bytes, st, d_result, scale, pref, d_nuhat2, 0, 0.0);
}

int reduce_lattice_enqueue(const double* d_nuhat, int M, double xi_max, double s, void* d_work, size_t work_bytes,
                           cudaStream_t st, double** d_result, double scale, double pref) {
  SFD_REQUIRE(M >= 2 && (M & 1) == 0 && M <= 1624, SFD_ERR_INVALID_ARG, "lattice size M must be even, 2..1624 (got %d)", M);
  const int64_t K = (int64_t)(M + 1) * (M + 1) * (M + 1);
  return reduce_any(d_nuhat, nullptr, nullptr, K, s, d_work, work_bytes, st, d_result, scale, pref, nullptr, M,
                    2.0 * xi_max / M);
}

int reduce_lattice_band_enqueue(const Nufft1Band& band, int M, double xi_max, double s, void* d_work, size_t work_bytes,
                                cudaStream_t st, double** d_result, double scale, double pref) {
  SFD_REQUIRE(M >= 2 && (M & 1) == 0 && M <= 1624, SFD_ERR_INVALID_ARG, "lattice size M must be even, 2..1624 (got %d)", M);
  SFD_REQUIRE(s > 0.5 && s < 1e6, SFD_ERR_INVALID_ARG, "Sobolev order s must exceed 1/2 (P:113), got %g", s);
  SFD_REQUIRE(band.v && band.dec, SFD_ERR_NULL, "reduce_lattice_band: NULL band");
  const int64_t Kh = (int64_t)(M + 1) * (M + 1) * (M / 2 + 1);
  SFD_REQUIRE(d_work && work_bytes >= reduce_workspace(Kh), SFD_ERR_WORKSPACE_TOO_SMALL,
              "reduction needs %zu workspace bytes, got %zu", reduce_workspace(Kh), work_bytes);
  double* result = static_cast<double*>(d_work);
  Comp* partial = reinterpret_cast<Comp*>(static_cast<char*>(d_work) + 256);
  *d_result = result;
  const int blocks = reduce_blocks(Kh);
  const int s_kind = (s == std::floor(s) && s >= 1.0 && s <= 64.0) ? (int)s : 0;
  lattice_band_terms_kernel<<<blocks, kThreads, 0, st>>>(reinterpret_cast<const double2*>(band.v), band.dec, band.C[0],
                                                         band.C[1], band.C[2], M, 2.0 * xi_max / M, s, s_kind,
                                                         scale * scale, band.f32, partial);
  SFD_TRY(launch_check("lattice_band_terms_kernel"));
  reduce_final_kernel<<<1, kThreads, 0, st>>>(partial, blocks, pref, result, device_flags());
  return launch_check("reduce_final_kernel");
}

}  // namespace sfd
