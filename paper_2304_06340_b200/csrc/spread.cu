// spread.cu -- A5-4: spreading of the type-3 NUFFT.  g[l] += c'_j psi(l1 h - x'_j1) psi(l2 h - x'_j2) psi(l3 h - x'_j3)
// over the w^3 cells around every source, psi(y) = phi(2y/(w h)), phi(z) = exp(beta (sqrt(1-z^2) - 1)) (the
// "exponential of semicircle" kernel, P:185 refs [2,3]; convolution step of P:180-185).
//
// The paper's GPU library spreads bin-sorted subproblems in shared memory with atomics and had to fall back to
// single precision because fp64 subgrids did not fit.  Here:
//   * one persistent CTA per SM pulls work items (an occupied bin, or a slice of <= kSrcCap sources of a heavy bin)
//     from a device-side queue; the bin's padded subgrid lives in up to ~200 KB of shared memory in fp64 (real when
//     the strengths are real, i.e. ball-centred targets; complex otherwise);
//   * no atomics in shared memory: cell (ix, iy, .) of the subgrid is owned by warp (ix mod W, iy mod NSPLIT) -- an
//     absolute assignment, the same for every source -- so the W planes of a source go to W different warp groups,
//     each plane's rows to NSPLIT warps, and no two warps ever touch the same cell;
//   * the z extent of a bin is 16 (real) or 8/16 (complex) cells, which makes the row pitch congruent to W modulo
//     the number of bank groups: the lanes' cells c = y W + z of a plane fall into distinct banks for every W;
//   * kernel values are piecewise polynomials (nufft3.cuh footprint()): for a chunk of 32 sources (one per lane) warp
//     group a evaluates interval a with the coefficients in registers; the next chunk's records are prefetched
//     while the current one is accumulated;
//   * only the final write-back of the subgrid uses fp64 global reductions (RED.ADD.F64), because neighbouring
//     bins' paddings overlap; all-zero cells are skipped (the sources lie on a 2-D shell).
#include <algorithm>

#include "nufft3.cuh"

namespace sfd {
namespace {

constexpr int kChunk = 32;               // sources whose 3W kernel values are tabulated at a time (one per lane)
constexpr int kSmemBytes = 200 * 1024;   // subgrid budget

constexpr int nsplit_for(int W) {
  int n = (20 + W / 2) / W;
  if (n < 1) n = 1;
  if (n > W) n = W;
  return n;
}

struct ChunkTables {
  double k[3][kChunk][16];   // kernel values per dimension
  double c[kChunk][2];       // strengths
  int i0[kChunk][3];         // first cell of the footprint, relative to the subgrid origin
};

template <int W, bool REAL>
__global__ void __launch_bounds__(32 * W * nsplit_for(W), 1)
spread_kernel(N3Params p, const double* __restrict__ ptab, const SrcRec* __restrict__ src,
              const int32_t* __restrict__ item_bin, const int32_t* __restrict__ item_start,
              const int32_t* __restrict__ item_count, const int32_t* __restrict__ n_items,
              int32_t* __restrict__ counter, double* __restrict__ grid) {
  constexpr int NSPLIT = nsplit_for(W);
  constexpr int NWARPS = W * NSPLIT;
  constexpr int RS = (W + NSPLIT - 1) / NSPLIT;     // rows of a footprint plane that one warp can own (at most)
  constexpr int NCL = (RS * W + 31) / 32;
  constexpr int DEG = W + 3;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  ChunkTables& tab = *reinterpret_cast<ChunkTables*>(smem_raw);
  double* sub = reinterpret_cast<double*>(smem_raw + sizeof(ChunkTables));
  __shared__ int s_item;

  const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
  const int a_own = wq % W, slab = wq / W;
  const int Px = p.bs[0] + W, Py = p.bs[1] + W, Pz = p.bs[2] + W;

  double pc[DEG + 1];
#pragma unroll
  for (int q = 0; q <= DEG; ++q) pc[q] = ptab[q * kPolyStride + a_own];

  // the lane's cells: c = lane + 32 i -> (m, cz); the warp's m-th row of a footprint is cy = r0 + NSPLIT m, where
  // r0 = (slab - i0y) mod NSPLIT depends on the source
  int cm[NCL], cz[NCL], off[NCL];
#pragma unroll
  for (int i = 0; i < NCL; ++i) {
    const int c = min(lane + 32 * i, RS * W - 1);
    cm[i] = NSPLIT * (c / W);
    cz[i] = c % W;
    off[i] = cm[i] * Pz + cz[i];
  }

  const int total = *n_items;
  for (;;) {
    __syncthreads();  // s_item and the subgrid are reused
    if (tid == 0) s_item = atomicAdd(counter, 1);
    __syncthreads();
    const int item = s_item;
    if (item >= total) break;
    const int bin = item_bin[item];
    const int start = item_start[item], count = item_count[item];
    const int bz = bin % p.nbs[2], by = (bin / p.nbs[2]) % p.nbs[1], bx = bin / (p.nbs[2] * p.nbs[1]);
    const int ox = bx * p.bs[0] - W / 2, oy = by * p.bs[1] - W / 2, oz = bz * p.bs[2] - W / 2;

    const int ncell = Px * Py * Pz;
    for (int i = tid; i < ncell * (REAL ? 1 : 2); i += 32 * NWARPS) sub[i] = 0.0;

    SrcRec rn = src[start + min(lane, count - 1)];
    for (int c0 = 0; c0 < count; c0 += kChunk) {
      const int nch = min(kChunk, count - c0);
      const SrcRec r = rn;
      if (c0 + kChunk < count) rn = src[start + min(c0 + kChunk + lane, count - 1)];   // prefetch the next chunk
      __syncthreads();  // zero-fill / previous sweep finished: the tables may be overwritten
      // warp group a_own evaluates interval a_own for 32 sources at once; slab s takes the dimensions d = s mod NSPLIT
      if (lane < nch && slab < 3) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
          if (d % NSPLIT == slab) {
            int i0;
            double s;
            footprint(r.u[d], W, i0, s);
            double kv = pc[DEG];
#pragma unroll
            for (int q = DEG - 1; q >= 0; --q) kv = __fma_rn(kv, s, pc[q]);
            tab.k[d][lane][a_own] = kv;
            if (a_own == 0) tab.i0[lane][d] = i0 - (d == 0 ? ox : (d == 1 ? oy : oz));
          }
        }
        if (wq == 0) {
          tab.c[lane][0] = r.re;
          tab.c[lane][1] = r.im;
        }
      }
      __syncthreads();
      {
        for (int s = 0; s < nch; ++s) {
          const int ix0 = tab.i0[s][0], iy0 = tab.i0[s][1];
          int a = (a_own - ix0) % W;   // the plane of this footprint that this warp group owns
          if (a < 0) a += W;
          int r0 = (slab - iy0) % NSPLIT;   // its first row of that plane
          if (r0 < 0) r0 += NSPLIT;
          const double kx = tab.k[0][s][a];
          const double cre = tab.c[s][0] * kx;
          const double cim = REAL ? 0.0 : tab.c[s][1] * kx;
          const int base = ((ix0 + a) * Py + iy0 + r0) * Pz + tab.i0[s][2];
#pragma unroll
          for (int i = 0; i < NCL; ++i) {
            if (lane + 32 * i < RS * W && r0 + cm[i] < W) {
              const double kyz = tab.k[1][s][r0 + cm[i]] * tab.k[2][s][cz[i]];
              const int idx = base + off[i];
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
    }
    __syncthreads();
    // write-back: neighbouring bins overlap in their paddings -> fp64 reductions into the global fine grid.
    // One (x,y) row of Pz <= 32 cells per warp pass, coalesced along z.
    for (int row = wq; row < Px * Py; row += NWARPS) {
      const int ix = row / Py, iy = row - ix * Py;
      const int gx = ox + ix, gy = oy + iy, gz = oz + lane;
      if (lane < Pz && gx >= 0 && gy >= 0 && gz >= 0 && gx < p.nf[0] && gy < p.nf[1] && gz < p.nf[2]) {
        const size_t g = ((size_t)gx * p.nf[1] + gy) * p.nf[2] + gz;
        if (REAL) {
          const double v = sub[row * Pz + lane];
          if (v != 0.0) atomicAdd(&grid[g], v);
        } else {
          const double2 v = reinterpret_cast<double2*>(sub)[row * Pz + lane];
          if (v.x != 0.0) atomicAdd(&grid[2 * g], v.x);
          if (v.y != 0.0) atomicAdd(&grid[2 * g + 1], v.y);
        }
      }
    }
  }
}

template <int W, bool REAL>
int launch(const N3Params& p, const double* d_ptab, const SrcRec* d_src, const int32_t* d_item_bin,
           const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
           double* d_grid, size_t smem, cudaStream_t st) {
  static bool attr = false;
  if (!attr) {
    SFD_CUDA_TRY(cudaFuncSetAttribute(spread_kernel<W, REAL>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 2048));
    attr = true;
  }
  spread_kernel<W, REAL><<<num_sms(), 32 * W * nsplit_for(W), smem, st>>>(p, d_ptab, d_src, d_item_bin, d_item_start,
                                                                         d_item_count, d_n_items, d_counter, d_grid);
  return launch_check("spread_kernel");
}

}  // namespace

// Source-bin shape: z extent 16 (real grid: 16 eight-byte bank groups) or 8/16 (complex), x and y as large as the
// shared-memory budget allows (at most 24: the sources lie on a shell, and smaller bins balance better).
void spread_bins(int w, bool real_c, int bs[3]) {
  const int cell = real_c ? 8 : 16;
  const int cap = (kSmemBytes - (int)sizeof(ChunkTables)) / cell;
  double best = -1.0;
  for (int bz = real_c ? 16 : 8; bz <= 16; bz += 8) {
    const int pz = bz + w;
    int m = 1;
    while ((m + 1) * (m + 1) * pz <= cap) ++m;
    const int b = std::min(m - w, 24);
    if (b < 1) continue;
    const double ratio = (double)b * b * bz / ((double)(b + w) * (b + w) * pz);
    if (ratio > best) {
      best = ratio;
      bs[0] = bs[1] = b;
      bs[2] = bz;
    }
  }
}

size_t spread_smem_bytes(const N3Params& p) {
  return sizeof(ChunkTables) + (size_t)(p.bs[0] + p.w) * (p.bs[1] + p.w) * (p.bs[2] + p.w) * (p.real_c ? 8 : 16);
}

int spread(const N3Params& p, const double* d_ptab, const SrcRec* d_src, const int32_t* d_item_bin,
           const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
           double* d_grid, cudaStream_t st) {
  const size_t smem = spread_smem_bytes(p);
  SFD_REQUIRE(smem <= 227 * 1024 - 2048 && p.bs[2] + p.w <= 32, SFD_ERR_INVALID_ARG,
              "spread subgrid does not fit shared memory (%zu B)", smem);
  SFD_CUDA_TRY(cudaMemsetAsync(d_counter, 0, sizeof(int32_t), st));
#define SFD_SPREAD_CASE(W_)                                                                                          \
  case W_:                                                                                                           \
    return p.real_c ? launch<W_, true>(p, d_ptab, d_src, d_item_bin, d_item_start, d_item_count, d_n_items,          \
                                       d_counter, d_grid, smem, st)                                                  \
                    : launch<W_, false>(p, d_ptab, d_src, d_item_bin, d_item_start, d_item_count, d_n_items,         \
                                        d_counter, d_grid, smem, st);
  switch (p.w) {
    SFD_SPREAD_CASE(2) SFD_SPREAD_CASE(3) SFD_SPREAD_CASE(4) SFD_SPREAD_CASE(5) SFD_SPREAD_CASE(6)
    SFD_SPREAD_CASE(7) SFD_SPREAD_CASE(8) SFD_SPREAD_CASE(9) SFD_SPREAD_CASE(10) SFD_SPREAD_CASE(11)
    SFD_SPREAD_CASE(12) SFD_SPREAD_CASE(13) SFD_SPREAD_CASE(14) SFD_SPREAD_CASE(15) SFD_SPREAD_CASE(16)
  }
#undef SFD_SPREAD_CASE
  set_error("spread: unsupported kernel width %d", p.w);
  return SFD_ERR_UNSUPPORTED;
}

}  // namespace sfd
