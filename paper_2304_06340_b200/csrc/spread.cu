// spread.cu -- A5-4: spreading of the type-3 NUFFT.  g[l] += c'_j psi(l1 h - x'_j1) psi(l2 h - x'_j2) psi(l3 h - x'_j3)
// over the w^3 cells around every source, psi(y) = phi(2y/(w h)), phi(z) = exp(beta (sqrt(1-z^2) - 1)) (the
// "exponential of semicircle" kernel, P:185 refs [2,3]; convolution step of P:180-185).
//
// The paper's GPU library spreads bin-sorted subproblems in shared memory with atomics and had to fall back to
// single precision because fp64 subgrids did not fit.  Here: one persistent CTA per SM pulls work items
// (an occupied bin, or a slice of a heavy bin) from a device-side queue; the bin's padded subgrid (bs+w)^3 lives
// in up to ~200 KB of shared memory in fp64; there are w warps and x-plane ix of the subgrid is owned by warp
// ix mod w, so a source's w planes go to w different warps and no two warps ever touch the same cell: the
// accumulation needs no atomics at all (fp64 shared-memory atomics would be CAS loops).  Inside a warp the 32
// lanes cover the w x w cells of the plane.  Only the final write-back of the subgrid uses fp64 global reductions
// (RED.ADD.F64), because neighbouring bins' paddings overlap.
#include "nufft3.cuh"

namespace sfd {
namespace {

constexpr int kChunk = 32;          // sources whose 3w kernel values are tabulated at a time (one per lane)
constexpr int kMaxCellsPerLane = (kMaxW * kMaxW + 31) / 32;

struct ChunkTables {
  double k[3][kChunk][kMaxW];   // kernel values per dimension
  double c[kChunk][2];          // strengths
  int i0[kChunk][3];            // first cell of the footprint, relative to the subgrid origin
};

constexpr int kRealMaxP = 29;   // 29^3 * 8 B  = 195 KB
constexpr int kCplxMaxP = 23;   // 23^3 * 16 B = 195 KB

template <bool REAL>
__global__ void __launch_bounds__(32 * kMaxW, 1)
spread_kernel(N3Params p, const double* __restrict__ ptab, const SrcRec* __restrict__ src,
              const int32_t* __restrict__ item_bin,
              const int32_t* __restrict__ item_start, const int32_t* __restrict__ item_count,
              const int32_t* __restrict__ n_items, int32_t* __restrict__ counter, double* __restrict__ grid) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  ChunkTables& tab = *reinterpret_cast<ChunkTables*>(smem_raw);
  double* sub = reinterpret_cast<double*>(smem_raw + sizeof(ChunkTables));
  __shared__ int s_item;
  __shared__ double s_poly[(kMaxDeg + 1) * kPolyStride];   // piecewise-polynomial kernel table (footprint())
  for (int i = threadIdx.x; i < (kMaxDeg + 1) * kPolyStride; i += blockDim.x) s_poly[i] = ptab[i];

  const int w = p.w, P = p.bs + w, fw = w / 2;
  const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5, nthreads = blockDim.x;
  const int ncell = P * P * P;
  constexpr int CW = REAL ? 1 : 2;

  // the lane's cells of a w x w plane: c = lane + 32 i -> (iy, iz)
  int cy[kMaxCellsPerLane], cz[kMaxCellsPerLane];
  const int ncl = (w * w + 31) / 32;
#pragma unroll
  for (int i = 0; i < kMaxCellsPerLane; ++i) {
    const int c = lane + 32 * i;
    cy[i] = c < w * w ? c / w : -1;
    cz[i] = c < w * w ? c % w : 0;
  }

  const int total = *n_items;
  for (;;) {
    if (tid == 0) s_item = atomicAdd(counter, 1);
    __syncthreads();
    const int item = s_item;
    if (item >= total) break;
    const int bin = item_bin[item];
    const int start = item_start[item], count = item_count[item];
    const int bz = bin % p.nbs[2], by = (bin / p.nbs[2]) % p.nbs[1], bx = bin / (p.nbs[2] * p.nbs[1]);
    const int o[3] = {bx * p.bs - fw, by * p.bs - fw, bz * p.bs - fw};

    for (int i = tid; i < ncell * CW; i += nthreads) sub[i] = 0.0;

    for (int c0 = 0; c0 < count; c0 += kChunk) {
      const int nch = min(kChunk, count - c0);
      __syncthreads();  // zero-fill / previous sweep finished
      if (lane < nch) {
        const SrcRec r = src[start + c0 + lane];
        // warp wq evaluates interval wq of the three 1-D kernels for 32 sources at once (coefficients: broadcast)
        int i0[3];
        double sv[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) footprint(r.u[d], w, i0[d], sv[d]);
        double k0 = s_poly[p.deg * kPolyStride + wq], k1 = k0, k2 = k0;
        for (int q = p.deg - 1; q >= 0; --q) {
          const double c = s_poly[q * kPolyStride + wq];
          k0 = __fma_rn(k0, sv[0], c);
          k1 = __fma_rn(k1, sv[1], c);
          k2 = __fma_rn(k2, sv[2], c);
        }
        tab.k[0][lane][wq] = k0;
        tab.k[1][lane][wq] = k1;
        tab.k[2][lane][wq] = k2;
        if (wq == 0) {
          tab.i0[lane][0] = i0[0] - o[0];
          tab.i0[lane][1] = i0[1] - o[1];
          tab.i0[lane][2] = i0[2] - o[2];
        }
        if (wq == 0) {
          tab.c[lane][0] = r.re;
          tab.c[lane][1] = r.im;
        }
      }
      __syncthreads();
      for (int s = 0; s < nch; ++s) {
        const int ix0 = tab.i0[s][0];
        int a = (wq - ix0) % w;   // the plane of this footprint that warp wq owns: (ix0 + a) mod w == wq
        if (a < 0) a += w;
        const double kx = tab.k[0][s][a];
        const double cre = tab.c[s][0] * kx;
        const double cim = REAL ? 0.0 : tab.c[s][1] * kx;
        const int base = ((ix0 + a) * P + tab.i0[s][1]) * P + tab.i0[s][2];
#pragma unroll
        for (int i = 0; i < kMaxCellsPerLane; ++i) {
          if (i < ncl && cy[i] >= 0) {
            const double kyz = tab.k[1][s][cy[i]] * tab.k[2][s][cz[i]];
            const int idx = base + cy[i] * P + cz[i];
            if (REAL) {
              sub[idx] = __fma_rn(cre, kyz, sub[idx]);
            } else {
              double2 v = reinterpret_cast<double2*>(sub)[idx];
              v.x = __fma_rn(cre, kyz, v.x);
              v.y = __fma_rn(cim, kyz, v.y);
              reinterpret_cast<double2*>(sub)[idx] = v;
            }
          }
        }
        __syncwarp();
      }
    }
    __syncthreads();
    // write-back: neighbouring bins overlap in their paddings -> fp64 reductions into the global fine grid
    for (int i = tid; i < ncell; i += nthreads) {
      const int iz = i % P, iy = (i / P) % P, ix = i / (P * P);
      const int gx = o[0] + ix, gy = o[1] + iy, gz = o[2] + iz;
      if (gx < 0 || gy < 0 || gz < 0 || gx >= p.nf[0] || gy >= p.nf[1] || gz >= p.nf[2]) continue;
      const size_t g = ((size_t)gx * p.nf[1] + gy) * p.nf[2] + gz;
      if (REAL) {
        const double v = sub[i];
        if (v != 0.0) atomicAdd(&grid[g], v);
      } else {
        const double2 v = reinterpret_cast<double2*>(sub)[i];
        if (v.x != 0.0) atomicAdd(&grid[2 * g], v.x);
        if (v.y != 0.0) atomicAdd(&grid[2 * g + 1], v.y);
      }
    }
    __syncthreads();  // s_item and the subgrid are reused
  }
}

}  // namespace

int spread_max_bin(int w, bool real_c) { return (real_c ? kRealMaxP : kCplxMaxP) - w; }

size_t spread_smem_bytes(const N3Params& p) {
  const size_t P = p.bs + p.w;
  return sizeof(ChunkTables) + P * P * P * (p.real_c ? 8 : 16);
}

int spread(const N3Params& p, const double* d_ptab, const SrcRec* d_src, const int32_t* d_item_bin, const int32_t* d_item_start,
           const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter, double* d_grid, cudaStream_t st) {
  const size_t smem = spread_smem_bytes(p);
  SFD_REQUIRE(smem <= 227 * 1024 - 4096, SFD_ERR_INVALID_ARG, "spread subgrid does not fit shared memory (%zu B)", smem);
  SFD_CUDA_TRY(cudaMemsetAsync(d_counter, 0, sizeof(int32_t), st));
  const int threads = 32 * p.w;
  const int blocks = num_sms();
  if (p.real_c) {
    static bool attr = false;
    if (!attr) {
      SFD_CUDA_TRY(cudaFuncSetAttribute(spread_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 4096));
      attr = true;
    }
    spread_kernel<true><<<blocks, threads, smem, st>>>(p, d_ptab, d_src, d_item_bin, d_item_start, d_item_count,
                                                      d_n_items, d_counter, d_grid);
  } else {
    static bool attr = false;
    if (!attr) {
      SFD_CUDA_TRY(cudaFuncSetAttribute(spread_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 4096));
      attr = true;
    }
    spread_kernel<false><<<blocks, threads, smem, st>>>(p, d_ptab, d_src, d_item_bin, d_item_start, d_item_count,
                                                       d_n_items, d_counter, d_grid);
  }
  return launch_check("spread_kernel");
}

}  // namespace sfd
