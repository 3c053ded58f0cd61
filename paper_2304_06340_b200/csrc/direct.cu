// direct.cu -- A4: fp64 direct summation nuhat_k = sum_j w_j exp(-i xi_k . x_j)  (eq. 2.8
// applied to the atoms of P:152).  FP64-pipe bound: per pair 3 FMA (phase) + 20 (sincos) + 2 (accumulate).
//
// Layout: one CTA = 128 threads x T targets held in registers (xi and the two accumulators); the sources
// stream through shared memory in tiles of kTile atoms, double-buffered with 1-D bulk TMA copies
// (cp.async.bulk + mbarrier) issued by one elected thread; every thread reads the same source at the same
// time (shared-memory broadcast, no bank conflicts).  For small K the source range is split over
// gridDim.y and the partial sums are combined in a fixed order by a second kernel (deterministic).
#include <algorithm>

#include "common.cuh"
#include "direct.cuh"

namespace sfd {
namespace {

constexpr int kThreads = 128;
constexpr int kTile = 512;  // atoms per stage: 512*32 B = 16 KB; two stages

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

struct __align__(16) Stage {
  double x[kTile * 3];
  double w[kTile];
};

template <int T>
__global__ void __launch_bounds__(kThreads) direct_sum_kernel(const double* __restrict__ x, const double* __restrict__ w,
                                                             int64_t J, const double* __restrict__ xi, int64_t K,
                                                             double* __restrict__ out, int64_t j_per_split, int use_tma) {
  __shared__ Stage stage[2];
  __shared__ __align__(8) uint64_t bar[2];
  const int tid = threadIdx.x;
  const int64_t k0 = (int64_t)blockIdx.x * (kThreads * T);
  const int64_t jb = (int64_t)blockIdx.y * j_per_split;
  const int64_t je = min(J, jb + j_per_split);
  const int ntiles = (int)((je - jb + kTile - 1) / kTile);

  double a0[T], a1[T], a2[T], re[T], im[T];
#pragma unroll
  for (int t = 0; t < T; ++t) {
    const int64_t k = min(k0 + t * kThreads + tid, K - 1);
    a0[t] = xi[3 * k];
    a1[t] = xi[3 * k + 1];
    a2[t] = xi[3 * k + 2];
    re[t] = 0.0;
    im[t] = 0.0;
  }

  if (tid == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // a tile goes by TMA when it is full (sizes and addresses are then multiples of 16 B)
  auto issue = [&](int t) {
    const int64_t j0 = jb + (int64_t)t * kTile;
    Stage& s = stage[t & 1];
    mbar_expect_tx(&bar[t & 1], kTile * 32);
    bulk_g2s(s.x, x + 3 * j0, kTile * 24, &bar[t & 1]);
    bulk_g2s(s.w, w + j0, kTile * 8, &bar[t & 1]);
  };
  auto tile_n = [&](int t) { return (int)min((int64_t)kTile, je - (jb + (int64_t)t * kTile)); };

  if (tid == 0 && ntiles > 0 && use_tma && tile_n(0) == kTile) issue(0);

  for (int t = 0; t < ntiles; ++t) {
    const int n = tile_n(t);
    Stage& s = stage[t & 1];
    const bool tma = use_tma && n == kTile;
    if (tid == 0 && t + 1 < ntiles && use_tma && tile_n(t + 1) == kTile) issue(t + 1);
    if (tma) {
      mbar_wait(&bar[t & 1], (t >> 1) & 1);
    } else {
      const int64_t j0 = jb + (int64_t)t * kTile;
      for (int i = tid; i < 3 * n; i += kThreads) s.x[i] = x[3 * j0 + i];
      for (int i = tid; i < n; i += kThreads) s.w[i] = w[j0 + i];
      __syncthreads();
    }
#pragma unroll 2
    for (int j = 0; j < n; ++j) {
      const double x0 = s.x[3 * j], x1 = s.x[3 * j + 1], x2 = s.x[3 * j + 2], wj = s.w[j];
#pragma unroll
      for (int u = 0; u < T; ++u) {
        const double th = __fma_rn(a0[u], x0, __fma_rn(a1[u], x1, a2[u] * x2));
        double sn, cs;
        sincos_fp64(th, sn, cs);
        re[u] = __fma_rn(wj, cs, re[u]);
        im[u] = __fma_rn(wj, sn, im[u]);
      }
    }
    __syncthreads();  // everyone is done with this stage before it is refilled
  }

  double* o = out + (size_t)blockIdx.y * (size_t)K * 2;
#pragma unroll
  for (int t = 0; t < T; ++t) {
    const int64_t k = k0 + t * kThreads + tid;
    if (k < K) reinterpret_cast<double2*>(o)[k] = make_double2(re[t], -im[t]);
  }
}

__global__ void combine_splits_kernel(const double* __restrict__ part, int nsplit, int64_t n2, double* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n2) return;
  double acc = 0.0;
  for (int s = 0; s < nsplit; ++s) acc += part[(size_t)s * n2 + i];
  out[i] = acc;
}

}  // namespace

DirectPlan direct_plan(int64_t J, int64_t K) {
  DirectPlan p;
  const int64_t sms = num_sms();
  p.T = K >= sms * kThreads * 4 * 6 ? 4 : (K >= sms * kThreads * 2 * 4 ? 2 : 1);
  p.blocks_k = (K + (int64_t)kThreads * p.T - 1) / ((int64_t)kThreads * p.T);
  // few target tiles (small K): split the sources over gridDim.y so that every SM has work
  const int64_t tiles = std::max<int64_t>(1, (J + kTile - 1) / kTile);
  const int64_t want = (4 * sms + p.blocks_k - 1) / std::max<int64_t>(1, p.blocks_k);
  const int64_t nsplit = std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(want, tiles), 64));
  const int64_t tiles_per = (tiles + nsplit - 1) / nsplit;
  p.j_per_split = tiles_per * kTile;
  p.nsplit = (int)std::max<int64_t>(1, (J + p.j_per_split - 1) / p.j_per_split);
  p.work_bytes = p.nsplit > 1 ? align_up((size_t)p.nsplit * (size_t)K * 16) : 0;
  return p;
}

int direct_sum(const double* d_x, const double* d_w, int64_t J, const double* d_xi, int64_t K, double* d_nuhat,
               void* d_work, size_t work_bytes, cudaStream_t st) {
  if (K == 0) return SFD_OK;
  if (J == 0) {
    SFD_CUDA_TRY(cudaMemsetAsync(d_nuhat, 0, (size_t)K * 16, st));
    return SFD_OK;
  }
  const DirectPlan p = direct_plan(J, K);
  SFD_REQUIRE(work_bytes >= p.work_bytes && (p.work_bytes == 0 || d_work), SFD_ERR_WORKSPACE_TOO_SMALL,
              "direct sum needs %zu workspace bytes, got %zu", p.work_bytes, work_bytes);
  SFD_REQUIRE(p.blocks_k <= 0x7fffffffLL, SFD_ERR_INVALID_ARG, "K too large");
  const int use_tma = ((reinterpret_cast<uintptr_t>(d_x) | reinterpret_cast<uintptr_t>(d_w)) & 15) == 0;
  double* out = p.nsplit > 1 ? static_cast<double*>(d_work) : d_nuhat;
  dim3 grid((unsigned)p.blocks_k, (unsigned)p.nsplit);
  switch (p.T) {
    case 4: direct_sum_kernel<4><<<grid, kThreads, 0, st>>>(d_x, d_w, J, d_xi, K, out, p.j_per_split, use_tma); break;
    case 2: direct_sum_kernel<2><<<grid, kThreads, 0, st>>>(d_x, d_w, J, d_xi, K, out, p.j_per_split, use_tma); break;
    default: direct_sum_kernel<1><<<grid, kThreads, 0, st>>>(d_x, d_w, J, d_xi, K, out, p.j_per_split, use_tma); break;
  }
  SFD_TRY(launch_check("direct_sum_kernel"));
  if (p.nsplit > 1) {
    const int64_t n2 = 2 * K;
    combine_splits_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>(out, p.nsplit, n2, d_nuhat);
    SFD_TRY(launch_check("combine_splits_kernel"));
  }
  return SFD_OK;
}

}  // namespace sfd
