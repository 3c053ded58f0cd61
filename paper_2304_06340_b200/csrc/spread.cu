// spread.cu -- A5-4: spreading of the type-3 NUFFT.  g[l] += c'_j psi(l1 h - x'_j1) psi(l2 h - x'_j2) psi(l3 h - x'_j3)
// over the w^3 cells around every source, psi(y) = phi(2y/(w h)), phi(z) = exp(beta (sqrt(1-z^2) - 1)) (the
// "exponential of semicircle" kernel, P:185 refs [2,3]; convolution step of P:180-185).
//
// The paper's GPU library spreads bin-sorted subproblems in shared memory with atomics and had to fall back to
// single precision because fp64 subgrids did not fit.  Here:
//   * persistent CTAs (two per SM up to w = 11, one beyond) pull work items (an occupied bin, or a slice of <= kSrcCap
//     sources of a heavy bin) from a device-side queue; the bin's padded subgrid lives in up to ~100 / ~200 KB of shared
//     memory in fp64 (real when the strengths are real, i.e. ball-centred targets; complex otherwise);
//   * no atomics in shared memory: x-plane ix of the subgrid is owned by warp ix mod W -- an absolute assignment, the
//     same for every source -- so the W planes of a footprint go to the W warps of the CTA and no two warps ever
//     touch the same cell; inside a warp the 32 lanes cover the W x W cells of the plane;
//   * per chunk of 32 sources the per-source set-up (owned plane, its address, strength x x-kernel) is computed with
//     one source per lane and broadcast by shuffles in the sweep, which keeps the sweep at ~10 instructions per
//     source and 32 cells;
//   * the z extent of a bin is 16 (real) or 8/16 (complex) cells, which makes the row pitch congruent to W modulo
//     the number of bank groups: the lanes' cells c = y W + z of a plane fall into distinct banks for every W;
//   * kernel values are piecewise polynomials (nufft3.cuh footprint()): for a chunk of 32 sources (one per lane) warp
//     group a evaluates interval a with the coefficients in registers; the next chunk's records are prefetched
//     while the current one is accumulated;
//   * consecutive sources whose footprints cover the same cells of the warp's plane are summed in registers and
//     added to the subgrid once: with many sources per cell (the paper's lattice variant maps 2e7 atoms onto a
//     54^3 grid) and the sort by footprint (N3Params::fine) this removes almost all shared-memory traffic;
//   * only the final write-back of the subgrid uses fp64 global reductions (RED.ADD.F64), because neighbouring
//     bins' paddings overlap; all-zero cells are skipped (the sources lie on a 2-D shell).
#include <algorithm>

#include "nufft3.cuh"

namespace sfd {
namespace {

constexpr int kChunk = 32;               // sources whose 3W kernel values are tabulated at a time (one per lane)
constexpr int kSmemBytes = 200 * 1024;   // subgrid budget of a CTA that has the SM to itself
// Kernels up to w = 11 run two CTAs per SM on half the budget each: the sweep is latency-bound and every warp walks
// every source of its CTA's item, so a second, independent CTA doubles the sources in flight.  Measured: spread
// 0.93 -> 0.76 ms at w = 7 (config 3), 3.45 -> 3.06 ms at w = 10 (config 4), 17.1 -> 16.5 ms at w = 11 (config 5);
// at w = 13 the 78-register budget spills and the gain is within the noise, so wider kernels keep one CTA.
// Three CTAs (80 registers, bins of a third of the shared memory) at w <= 8: 0.416 -> 0.343 ms at w = 5, 0.505 -> 0.466 at
// w = 6, 0.626 -> 0.596 at w = 7, 0.670 -> 0.641 at w = 8 (config 3's sources); four at w <= 6 lose again (0.373 / 0.483:
// the bins shrink to 5 cells a side).  As in the FFT passes, CTAs in different phases fill the pipes, not warps.
constexpr int kTwoCtaMaxW = 11;
constexpr int kThreeCtaMaxW = 8;
constexpr int ctas_per_sm(int w) { return w <= kThreeCtaMaxW ? 3 : (w <= kTwoCtaMaxW ? 2 : 1); }

// Sources of a chunk whose W x W products ky[cy] kz[cz] are tabulated at a time: every one of the W warps that visit a
// source needs the same W^2 products -- computed once and read as ceil(W^2/32) contiguous LDS.64, instead of twice as
// many gathers from the ky and kz columns plus a DMUL per cell and visit.  The whole chunk of 32 where the shared memory
// allows it (one CTA per SM above w = 11: 49 KB at w = 13; ~17 KB at w <= 8), half a chunk at w = 9 ... 11 (two CTAs per
// SM: a whole chunk would shrink the bins too far).  Measured at config 3's sources, sub-chunks of 8 / 16 / 32 sources:
// w = 12 2.00 / 1.87 / 1.80 ms, w = 13 2.56 / 2.41 / 2.31 ms, w = 14 3.01 / 2.87 / 2.77 ms (every sub-chunk costs two
// barriers); w = 10 (config 4) 2.88 / 2.80 / 2.86 ms, w = 11 (config 5) 15.0 / 14.7 / 15.3 ms; w = 7 16 / 32: 0.613 / 0.594 ms.
constexpr int kyz_sub(int W) { return (W <= 8 || W > 11) ? 32 : 16; }
constexpr int kyz_pitch(int W) { return ((W * W + 31) / 32) * 32 + 1; }   // odd: lanes = consecutive sources write a column
constexpr int kyz_bytes(int W) { return kyz_sub(W) * kyz_pitch(W) * 8; }

struct ChunkTables {
  double k[3][kChunk][17];   // kernel values per dimension (pitch 17: the lanes of a warp, one source each, write and
                             // read column a of 32 rows -- with a pitch of 16 doubles all 32 land in one bank pair)
  double c[kChunk][2];       // strengths
  int i0[kChunk][3];         // first cell of the footprint, relative to the subgrid origin
};

template <int W, bool REAL, bool RUNS>
__global__ void __launch_bounds__(32 * W, ctas_per_sm(W))
spread_kernel(N3Params p, const double* __restrict__ ptab, const SrcRec* __restrict__ src,
              const int32_t* __restrict__ item_bin, const int32_t* __restrict__ item_start,
              const int32_t* __restrict__ item_count, const int32_t* __restrict__ n_items,
              int32_t* __restrict__ counter, double* __restrict__ grid) {
  constexpr int NCL = (W * W + 31) / 32;
  constexpr int DEG = W + 3;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  ChunkTables& tab = *reinterpret_cast<ChunkTables*>(smem_raw);
  constexpr int KS = kyz_sub(W), KP = kyz_pitch(W);
  double* kyzt = reinterpret_cast<double*>(smem_raw + sizeof(ChunkTables));          // [KS][KP]
  double* sub = reinterpret_cast<double*>(smem_raw + sizeof(ChunkTables) + ((kyz_bytes(W) + 15) & ~15));
  __shared__ int s_item;

  const int tid = threadIdx.x, lane = tid & 31, a_own = tid >> 5;   // warp a_own owns the x-planes ix = a_own mod W
  const int Px = p.bs[0] + W, Py = p.bs[1] + W, Pz = p.bs[2] + W;

  double pc[DEG + 1];
#pragma unroll
  for (int q = 0; q <= DEG; ++q) pc[q] = ptab[q * kPolyStride + a_own];

  // the lane's cells of a W x W plane: c = lane + 32 i -> (cy, cz)
  int cy[NCL], cz[NCL], off[NCL];
  bool on[NCL];
#pragma unroll
  for (int i = 0; i < NCL; ++i) {
    on[i] = lane + 32 * i < W * W;
    const int c = min(lane + 32 * i, W * W - 1);
    cy[i] = c / W;
    cz[i] = c % W;
    off[i] = cy[i] * Pz + cz[i];
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
    for (int i = tid; i < ncell * (REAL ? 1 : 2); i += 32 * W) sub[i] = 0.0;

    // RUNS (N3Params::fine == 1, the sort is by footprint): consecutive sources with the same footprint cells in this
    // warp's plane form a run, which is accumulated in registers and added to the subgrid once.
    int run_base = -1;
    double acc_re[NCL], acc_im[NCL];
#pragma unroll
    for (int i = 0; i < NCL; ++i) acc_re[i] = acc_im[i] = 0.0;
    auto flush = [&]() {
      if (run_base >= 0) {
#pragma unroll
        for (int i = 0; i < NCL; ++i) {
          if (on[i]) {
            const int idx = run_base + off[i];
            if (REAL) {
              sub[idx] += acc_re[i];
            } else {
              double2 v = reinterpret_cast<double2*>(sub)[idx];
              v.x += acc_re[i];
              v.y += acc_im[i];
              reinterpret_cast<double2*>(sub)[idx] = v;
            }
          }
          acc_re[i] = acc_im[i] = 0.0;
        }
        __syncwarp();   // the next run's cells may be ones other lanes have just written
      }
    };

    SrcRec rn = src[start + min(lane, count - 1)];
    for (int c0 = 0; c0 < count; c0 += kChunk) {
      const int nch = min(kChunk, count - c0);
      const SrcRec r = rn;
      if (c0 + kChunk < count) rn = src[start + min(c0 + kChunk + lane, count - 1)];   // prefetch the next chunk
      __syncthreads();  // zero-fill / previous sweep finished: the tables may be overwritten
      // lane = source of the chunk; warp a_own evaluates interval a_own of the three 1-D kernels for 32 sources at once
      int i0[3];
      {
        double sv[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) footprint(r.u[d], W, i0[d], sv[d]);
        double k0 = pc[DEG], k1 = pc[DEG], k2 = pc[DEG];
#pragma unroll
        for (int q = DEG - 1; q >= 0; --q) {
          k0 = __fma_rn(k0, sv[0], pc[q]);
          k1 = __fma_rn(k1, sv[1], pc[q]);
          k2 = __fma_rn(k2, sv[2], pc[q]);
        }
        i0[0] -= ox;
        i0[1] -= oy;
        i0[2] -= oz;
        if (lane < nch) {
          tab.k[0][lane][a_own] = k0;
          tab.k[1][lane][a_own] = k1;
          tab.k[2][lane][a_own] = k2;
        }
      }
      __syncthreads();
      // per-source quantities of this warp, one source per lane: the plane of the footprint that the warp owns, the
      // address of that plane's first cell and the strength times the x-kernel; broadcast by shuffles in the sweep
      int a = (a_own - i0[0]) % W;
      if (a < 0) a += W;
      const int base_l = ((i0[0] + a) * Py + i0[1]) * Pz + i0[2];
      const double kx = lane < nch ? tab.k[0][lane][a] : 0.0;
      const double cre_l = r.re * kx;
      const double cim_l = REAL ? 0.0 : r.im * kx;
      // sweep over the chunk's sources in sub-chunks of KS: first every thread of the CTA fills its share of the
      // sub-chunk's ky kz products (index p = source + KS * cell: consecutive lanes are consecutive sources, so the
      // pitch-17 columns and the odd-pitch product rows are read and written without bank conflicts), then every warp
      // sweeps the KS sources, software-pipelined: the broadcasts and the products of source s+1 are fetched while
      // source s is accumulated
      for (int sc0 = 0; sc0 < nch; sc0 += KS) {
      const int nsc = min(KS, nch - sc0);
      if (sc0 > 0) __syncthreads();   // the previous sub-chunk's products are no longer read
      for (int pidx = tid; pidx < KS * W * W; pidx += 32 * W) {
        const int sl = pidx % KS, c = pidx / KS;
        const int ccy = c / W, ccz = c - ccy * W;
        if (sl < nsc) kyzt[sl * KP + c] = tab.k[1][sc0 + sl][ccy] * tab.k[2][sc0 + sl][ccz];
      }
      __syncthreads();
      int base_n = __shfl_sync(0xffffffffu, base_l, sc0);
      double cre_n = __shfl_sync(0xffffffffu, cre_l, sc0);
      double cim_n = REAL ? 0.0 : __shfl_sync(0xffffffffu, cim_l, sc0);
      double kyz_n[NCL];
#pragma unroll
      for (int i = 0; i < NCL; ++i) kyz_n[i] = on[i] ? kyzt[lane + 32 * i] : 0.0;
      for (int s = 0; s < nsc; ++s) {
        const int base = base_n;
        const double cre = cre_n, cim = cim_n;
        double kyz[NCL];
#pragma unroll
        for (int i = 0; i < NCL; ++i) kyz[i] = kyz_n[i];
        const int sn = min(s + 1, nsc - 1);
        base_n = __shfl_sync(0xffffffffu, base_l, sc0 + sn);
        cre_n = __shfl_sync(0xffffffffu, cre_l, sc0 + sn);
        if (!REAL) cim_n = __shfl_sync(0xffffffffu, cim_l, sc0 + sn);
#pragma unroll
        for (int i = 0; i < NCL; ++i) kyz_n[i] = on[i] ? kyzt[sn * KP + lane + 32 * i] : 0.0;
        if (RUNS) {
          if (base != run_base) {   // warp-uniform
            flush();
            run_base = base;
          }
#pragma unroll
          for (int i = 0; i < NCL; ++i) {
            acc_re[i] = __fma_rn(cre, kyz[i], acc_re[i]);
            if (!REAL) acc_im[i] = __fma_rn(cim, kyz[i], acc_im[i]);
          }
        } else {
#pragma unroll
          for (int i = 0; i < NCL; ++i) {
            if (on[i]) {
              const int idx = base + off[i];
              if (REAL) {
                sub[idx] = __fma_rn(cre, kyz[i], sub[idx]);
              } else {
                double2 v = reinterpret_cast<double2*>(sub)[idx];
                v.x = __fma_rn(cre, kyz[i], v.x);
                v.y = __fma_rn(cim, kyz[i], v.y);
                reinterpret_cast<double2*>(sub)[idx] = v;
              }
            }
          }
          __syncwarp();
        }
      }
      }   // sub-chunks
    }
    if (RUNS) flush();
    __syncthreads();
    // write-back: neighbouring bins overlap in their paddings -> fp64 reductions into the global fine grid.
    // One (x,y) row of Pz <= 32 cells per warp pass, coalesced along z.
    for (int row = a_own; row < Px * Py; row += W) {
      const int ix = row / Py, iy = row - ix * Py;
      const int gx = ox + ix, gy = oy + iy, gz = oz + lane;
      if (lane < Pz && gx >= 0 && gy >= 0 && gz >= 0 && gx < p.nf[0] && gy < p.nf[1] && gz < p.nf[2]) {
        const size_t g = ((size_t)gx * p.nf[1] + gy) * p.nf[2] + gz;
        // (p.f32: the global grid is single precision -- the subgrid sum, accumulated in fp64, is rounded once per bin)
        float* gridf = reinterpret_cast<float*>(grid);
        if (REAL) {
          const double v = sub[row * Pz + lane];
          if (v != 0.0) {
            if (p.f32) atomicAdd(&gridf[g], (float)v);
            else atomicAdd(&grid[g], v);
          }
        } else {
          const double2 v = reinterpret_cast<double2*>(sub)[row * Pz + lane];
          if (p.f32) {
            if (v.x != 0.0) atomicAdd(&gridf[2 * g], (float)v.x);
            if (v.y != 0.0) atomicAdd(&gridf[2 * g + 1], (float)v.y);
          } else {
            if (v.x != 0.0) atomicAdd(&grid[2 * g], v.x);
            if (v.y != 0.0) atomicAdd(&grid[2 * g + 1], v.y);
          }
        }
      }
    }
  }
}

template <int W, bool REAL, bool RUNS>
int launch(const N3Params& p, const double* d_ptab, const SrcRec* d_src, const int32_t* d_item_bin,
           const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
           double* d_grid, size_t smem, cudaStream_t st) {
  static thread_local int attr_dev = -1;
  if (first_use_on_device(attr_dev)) {
    SFD_CUDA_TRY(cudaFuncSetAttribute(spread_kernel<W, REAL, RUNS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (227 * 1024 - 2048) / ctas_per_sm(W) - 1024));
  }
  spread_kernel<W, REAL, RUNS><<<num_sms() * ctas_per_sm(W), 32 * W, smem, st>>>(p, d_ptab, d_src, d_item_bin, d_item_start, d_item_count,
                                                                d_n_items, d_counter, d_grid);
  return launch_check("spread_kernel");
}


// ---- many sources per cell ("highly clustered"): one warp per run of equal footprints --------------------
// With the sources ordered by footprint (N3Params::fine == 2) a work item is a slice of <= kRunCap consecutive
// sources that all start at the same cell i0.  One warp takes the whole item: the lanes evaluate the 3 W kernel
// values of 32 sources at once (one source per lane, Horner), the sweep then adds c kx[a] * (ky kz)[cell] into
// W x NCL register accumulators per lane -- 16 DFMA per source at W = 8, no shared-memory read-modify-write and no
// redundancy between warps -- and the W^3 sums go to the global grid by fp64 reductions once per item.  Warps are
// independent (dynamic queue), so many of them hide each other's latencies.  Real strengths, W <= 10.
constexpr int kRunWarps = 16;
constexpr int kRunCap = 512;

template <int W>
__global__ void __launch_bounds__(32 * kRunWarps, 1)
spread_runs_kernel(N3Params p, const double* __restrict__ ptab, const SrcRec* __restrict__ src,
                   const int32_t* __restrict__ item_key, const int32_t* __restrict__ item_start,
                   const int32_t* __restrict__ item_count, const int32_t* __restrict__ n_items,
                   int32_t* __restrict__ counter, double* __restrict__ grid) {
  constexpr int NCL = (W * W + 31) / 32;
  constexpr int DEG = W + 3;
  constexpr int PITCH = 33;                      // kv[d][a][lane]: conflict-free for reads across a at a fixed lane
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* s_pc = reinterpret_cast<double*>(smem_raw);   // polynomial coefficients, [q][a]
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  for (int i = tid; i < (DEG + 1) * W; i += 32 * kRunWarps) s_pc[i] = ptab[(i / W) * kPolyStride + (i % W)];
  __syncthreads();
  double* kv = s_pc + (DEG + 1) * W + wrp * (3 * W * PITCH);

  int cy[NCL], cz[NCL];
  bool on[NCL];
#pragma unroll
  for (int i = 0; i < NCL; ++i) {
    on[i] = lane + 32 * i < W * W;
    const int c = min(lane + 32 * i, W * W - 1);
    cy[i] = c / W;
    cz[i] = c % W;
  }
  const int sub1 = p.bs[1] + 1, sub2 = p.bs[2] + 1, sub0 = p.bs[0] + 1;
  const int total = *n_items;
  for (;;) {
    int item = 0;
    if (lane == 0) item = atomicAdd(counter, 1);
    item = __shfl_sync(0xffffffffu, item, 0);
    if (item >= total) break;
    const int key = item_key[item], start = item_start[item], count = item_count[item];
    // key = ((bin * sub0 + c0) * sub1 + c1) * sub2 + c2 (nufft3_glue.cu source_keys_kernel)
    const int c2 = key % sub2, c1 = (key / sub2) % sub1, c0 = (key / (sub2 * sub1)) % sub0, bin = key / (sub2 * sub1 * sub0);
    const int bz = bin % p.nbs[2], by = (bin / p.nbs[2]) % p.nbs[1], bx = bin / (p.nbs[2] * p.nbs[1]);
    const int i0x = bx * p.bs[0] - W / 2 + c0, i0y = by * p.bs[1] - W / 2 + c1, i0z = bz * p.bs[2] - W / 2 + c2;

    double acc[W][NCL];
#pragma unroll
    for (int a = 0; a < W; ++a)
#pragma unroll
      for (int i = 0; i < NCL; ++i) acc[a][i] = 0.0;

    for (int c0s = 0; c0s < count; c0s += 32) {
      const int nch = min(32, count - c0s);
      const SrcRec r = src[start + min(c0s + lane, count - 1)];
      double sv[3];
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        int i0;
        footprint(r.u[d], W, i0, sv[d]);
      }
      __syncwarp();   // the previous chunk's sweep has finished reading kv
      // phi is even, so interval W-1-a is interval a mirrored: P_{W-1-a}(s) = P_a(-s).  With P_a(s) = E(s^2) + s O(s^2)
      // one pair of intervals costs two half-degree Horner chains per dimension instead of two full ones.
      {
        constexpr int QE = DEG & ~1, QO = (DEG - 1) | 1;   // highest even / odd power
        const double z0 = sv[0] * sv[0], z1 = sv[1] * sv[1], z2 = sv[2] * sv[2];
        const double cw = lane < nch ? r.re : 0.0;
#pragma unroll
        for (int a = 0; a < (W + 1) / 2; ++a) {
          double e0 = s_pc[QE * W + a], e1 = e0, e2 = e0;
#pragma unroll
          for (int q = QE - 2; q >= 0; q -= 2) {
            const double cq = s_pc[q * W + a];
            e0 = __fma_rn(e0, z0, cq);
            e1 = __fma_rn(e1, z1, cq);
            e2 = __fma_rn(e2, z2, cq);
          }
          double o0 = s_pc[QO * W + a], o1 = o0, o2 = o0;
#pragma unroll
          for (int q = QO - 2; q >= 1; q -= 2) {
            const double cq = s_pc[q * W + a];
            o0 = __fma_rn(o0, z0, cq);
            o1 = __fma_rn(o1, z1, cq);
            o2 = __fma_rn(o2, z2, cq);
          }
          kv[(0 * W + a) * PITCH + lane] = __fma_rn(sv[0], o0, e0) * cw;
          kv[(1 * W + a) * PITCH + lane] = __fma_rn(sv[1], o1, e1);
          kv[(2 * W + a) * PITCH + lane] = __fma_rn(sv[2], o2, e2);
          if (a != W - 1 - a) {
            kv[(0 * W + (W - 1 - a)) * PITCH + lane] = __fma_rn(-sv[0], o0, e0) * cw;
            kv[(1 * W + (W - 1 - a)) * PITCH + lane] = __fma_rn(-sv[1], o1, e1);
            kv[(2 * W + (W - 1 - a)) * PITCH + lane] = __fma_rn(-sv[2], o2, e2);
          }
        }
      }
      __syncwarp();
#pragma unroll 2
      for (int s2 = 0; s2 < nch; ++s2) {
        double kyz[NCL];
#pragma unroll
        for (int i = 0; i < NCL; ++i) kyz[i] = kv[(W + cy[i]) * PITCH + s2] * kv[(2 * W + cz[i]) * PITCH + s2];
#pragma unroll
        for (int a = 0; a < W; ++a) {
          const double ck = kv[a * PITCH + s2];
#pragma unroll
          for (int i = 0; i < NCL; ++i) acc[a][i] = __fma_rn(ck, kyz[i], acc[a][i]);
        }
      }
    }
    // W^3 sums of the item -> global grid (footprints of different items overlap: fp64 reductions)
#pragma unroll
    for (int a = 0; a < W; ++a) {
#pragma unroll
      for (int i = 0; i < NCL; ++i) {
        if (on[i] && acc[a][i] != 0.0) {
          const size_t g = ((size_t)(i0x + a) * p.nf[1] + (i0y + cy[i])) * p.nf[2] + (i0z + cz[i]);
          if (p.f32) atomicAdd(reinterpret_cast<float*>(grid) + g, (float)acc[a][i]);
          else atomicAdd(&grid[g], acc[a][i]);
        }
      }
    }
  }
}

template <int W>
int launch_runs(const N3Params& p, const double* d_ptab, const SrcRec* d_src, const int32_t* d_item_key,
                const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
                double* d_grid, cudaStream_t st) {
  constexpr size_t smem = ((size_t)(W + 4) * W + (size_t)kRunWarps * 3 * W * 33) * sizeof(double);
  static thread_local int attr_dev = -1;
  if (first_use_on_device(attr_dev)) {
    SFD_CUDA_TRY(cudaFuncSetAttribute(spread_runs_kernel<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  }
  spread_runs_kernel<W><<<num_sms(), 32 * kRunWarps, smem, st>>>(p, d_ptab, d_src, d_item_key, d_item_start, d_item_count,
                                                              d_n_items, d_counter, d_grid);
  return launch_check("spread_runs_kernel");
}

}  // namespace

int spread_runs_cap() { return kRunCap; }
bool spread_runs_ok(int w, bool real_c) { return real_c && w >= 2 && w <= 10; }

int spread_runs(const N3Params& p, const double* d_ptab, const SrcRec* d_src, const int32_t* d_item_key,
                const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
                double* d_grid, cudaStream_t st) {
  SFD_REQUIRE(spread_runs_ok(p.w, p.real_c != 0), SFD_ERR_INVALID_ARG, "spread_runs: unsupported width %d", p.w);
  SFD_CUDA_TRY(cudaMemsetAsync(d_counter, 0, sizeof(int32_t), st));
#define SFD_RUNS_CASE(W_) \
  case W_: return launch_runs<W_>(p, d_ptab, d_src, d_item_key, d_item_start, d_item_count, d_n_items, d_counter, d_grid, st);
  switch (p.w) {
    SFD_RUNS_CASE(2) SFD_RUNS_CASE(3) SFD_RUNS_CASE(4) SFD_RUNS_CASE(5) SFD_RUNS_CASE(6)
    SFD_RUNS_CASE(7) SFD_RUNS_CASE(8) SFD_RUNS_CASE(9) SFD_RUNS_CASE(10)
  }
#undef SFD_RUNS_CASE
  return SFD_ERR_UNSUPPORTED;
}

// Source-bin shape: z extent 16 (real grid: 16 eight-byte bank groups) or 8/16 (complex), x and y as large as the
// shared-memory budget allows (at most 24: the sources lie on a shell, and smaller bins balance better).
void spread_bins(int w, bool real_c, int bs[3]) {
  const int cell = real_c ? 8 : 16;
  const int cap = (kSmemBytes / ctas_per_sm(w) - (int)sizeof(ChunkTables) - ((kyz_bytes(w) + 15) & ~15)) / cell;
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
  return sizeof(ChunkTables) + ((kyz_bytes(p.w) + 15) & ~15) +
         (size_t)(p.bs[0] + p.w) * (p.bs[1] + p.w) * (p.bs[2] + p.w) * (p.real_c ? 8 : 16);
}

int spread(const N3Params& p, const double* d_ptab, const SrcRec* d_src, const int32_t* d_item_bin,
           const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
           double* d_grid, cudaStream_t st) {
  const size_t smem = spread_smem_bytes(p);
  SFD_REQUIRE(smem <= (size_t)((227 * 1024 - 2048) / ctas_per_sm(p.w) - 1024) && p.bs[2] + p.w <= 32, SFD_ERR_INVALID_ARG,
              "spread subgrid does not fit shared memory (%zu B)", smem);
  SFD_CUDA_TRY(cudaMemsetAsync(d_counter, 0, sizeof(int32_t), st));
#define SFD_SPREAD_ARGS p, d_ptab, d_src, d_item_bin, d_item_start, d_item_count, d_n_items, d_counter, d_grid, smem, st
#define SFD_SPREAD_CASE(W_)                                                                        \
  case W_:                                                                                         \
    if (p.fine == 1) return p.real_c ? launch<W_, true, true>(SFD_SPREAD_ARGS) : launch<W_, false, true>(SFD_SPREAD_ARGS); \
    return p.real_c ? launch<W_, true, false>(SFD_SPREAD_ARGS) : launch<W_, false, false>(SFD_SPREAD_ARGS);
  switch (p.w) {
    SFD_SPREAD_CASE(2) SFD_SPREAD_CASE(3) SFD_SPREAD_CASE(4) SFD_SPREAD_CASE(5) SFD_SPREAD_CASE(6)
    SFD_SPREAD_CASE(7) SFD_SPREAD_CASE(8) SFD_SPREAD_CASE(9) SFD_SPREAD_CASE(10) SFD_SPREAD_CASE(11)
    SFD_SPREAD_CASE(12) SFD_SPREAD_CASE(13) SFD_SPREAD_CASE(14) SFD_SPREAD_CASE(15) SFD_SPREAD_CASE(16)
  }
#undef SFD_SPREAD_CASE
#undef SFD_SPREAD_ARGS
  set_error("spread: unsupported kernel width %d", p.w);
  return SFD_ERR_UNSUPPORTED;
}

}  // namespace sfd
