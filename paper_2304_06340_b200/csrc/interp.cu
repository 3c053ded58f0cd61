// interp.cu -- A5-8: interpolation step of the inner type-2 transform of the type-3 NUFFT ("Type-2 ...
// its adjoint").  G_k = sum over the w^3 cells m around t_k of v[m] psi2(m h2 - t_k), the gather twin of the
// spreading step: same kernel, no write conflicts.
//
// Roofline: every target reads w^3 complex128 cells = 16 w^3 bytes of shared memory and does 2 w^3 DFMAs; at
// 128 B/clk/SM of shared-memory bandwidth against 64 DFMA/clk/SM the gather is shared-memory-bandwidth bound by 4x
// (w = 10: 125 clk per target and SM), far above its HBM traffic (the band of the inner grid, read once per bin).
// The kernel is built to sit on that bound:
//   * one persistent CTA per SM pulls work items (a target bin, or a slice of one: 512 to 4096 targets, nufft3.cu) from a
//     device-side queue and stages the bin's padded subgrid (bt+w cells per axis) in shared memory as complex128 -- one 3-D
//     TMA box copy (cp.async.bulk.tensor, zero fill outside the band) issued by one thread, so that the staging costs the
//     LSU pipe (the kernel's bottleneck) nothing; the bins at the centre plane of the Hermitian half band, whose lower
//     cells are reflections, and the single-precision grids are staged with 16-byte LDGSTS copies instead;
//   * the z extent of a bin is 8 or 16 cells, so the row pitch Pz = bt_z + w is congruent to w modulo 8 and the
//     flattened (y,z) cell index c = y w + z lands in bank group c mod 8: any 8 consecutive lanes of an LDS.128 hit 8
//     distinct 16-byte bank groups -- no bank conflicts for any w;
//   * each of the 16 warps gathers one target at a time: the 32 lanes cover the w x w cells of an x-plane
//     (ceil(w^2/32) cells per lane, fixed for the whole kernel), walk the w planes accumulating v * kx in registers,
//     weight by ky kz at the end and finish with a warp-shuffle sum;
//   * the 3w kernel values of a target are piecewise polynomials (nufft3.cuh footprint()) whose coefficients live
//     in registers: lane i (mod 16) owns interval i, lanes 0-15 evaluate x then z, lanes 16-31 evaluate y;
//   * w is a template parameter: plane loop, cell map and polynomial degree are compile-time.
#include <cuda.h>   // CUtensorMap (the encoder is looked up through the runtime: no link against libcuda)

#include <cstdlib>
#include <cstring>
#include <type_traits>

#include "nufft3.cuh"

namespace sfd {
namespace {

constexpr int kWarps = 16;
constexpr int kMaxTpw = 2;           // targets a warp works on at a time (2 where the accumulators fit the registers)
constexpr int tpw_for(int W) { return W <= 10 ? 2 : 1; }   // (w = 11..13 measured slower with 2: spills)
constexpr int kTabBytes = sizeof(double) * kWarps * kMaxTpw * 3 * 16;   // per-warp kernel values: 12 KB
constexpr int kSmemCells = 13600;   // complex128 cells of the subgrid: 217,600 B

// Target-bin shape for kernel width w, as compile-time functions (host and device use the same numbers): z extent 8
// or 16 (conflict-free pitch), x and y as large as the shared-memory budget allows; the shape with the best
// owned-cells / staged-cells ratio wins.  With the shape fixed per W every subgrid stride is an immediate.
constexpr int bin_xy(int w, int bz) {
  int m = 1;
  while ((m + 1) * (m + 1) * (bz + w) <= kSmemCells) ++m;
  return m - w;
}
constexpr int bin_z(int w) {
  const int b8 = bin_xy(w, 8), b16 = bin_xy(w, 16);
  if (b8 < 1) return 16;
  if (b16 < 1) return 8;
  // ratio b^2 bz / ((b+w)^2 (bz+w)), compared by cross-multiplication in 64-bit
  const long long l8 = (long long)b8 * b8 * 8 * (b16 + w) * (b16 + w) * (16 + w);
  const long long l16 = (long long)b16 * b16 * 16 * (b8 + w) * (b8 + w) * (8 + w);
  return l16 > l8 ? 16 : 8;
}

// Single-precision subgrid (N3Params::f32): 8-byte cells, so the same shared memory holds a bin of twice the cells;
// z extent 16, i.e. the row pitch is congruent to w modulo 16 and the 16 lanes of an LDS.64 phase hit 16 distinct 8-byte
// bank groups.  The plane loop accumulates in fp32 (w terms per accumulator), everything after it is fp64.
constexpr int kSmemCells32 = 2 * kSmemCells;
constexpr int bin_xy32(int w) {
  int m = 1;
  while ((m + 1) * (m + 1) * (16 + w) <= kSmemCells32) ++m;
  return m - w;
}
constexpr int kMaxW32 = 8;   // eps >= 1e-6 (w <= 7, one more for a handful of sources)

template <int W, bool F32>
__global__ void __launch_bounds__(32 * kWarps, 1)
interp_kernel(N3Params p, const __grid_constant__ CUtensorMap tmap, int use_tma, const double* __restrict__ ptab,
              const void* __restrict__ v_raw, const TgtRec* __restrict__ tgt,
              const int32_t* __restrict__ item_bin, const int32_t* __restrict__ item_start,
              const int32_t* __restrict__ item_count, const int32_t* __restrict__ n_items,
              int32_t* __restrict__ counter, double2* __restrict__ G) {
  constexpr int DEG = W + 3;
  constexpr int NCL = (W * W + 31) / 32;
  constexpr int TPW = tpw_for(W);
  extern __shared__ __align__(128) unsigned char smem_raw[];   // (the TMA destination wants 128-byte alignment)
  using CT = std::conditional_t<F32, float2, double2>;   // a cell of the subgrid (and of the band in global memory)
  using AT = std::conditional_t<F32, float, double>;     // the plane loop's accumulators
  const CT* __restrict__ v = static_cast<const CT*>(v_raw);
  double (*ktab)[kMaxTpw][3][16] = reinterpret_cast<double (*)[kMaxTpw][3][16]>(smem_raw);
  CT* sub = reinterpret_cast<CT*>(smem_raw + kTabBytes);
  __shared__ int s_item;
  __shared__ __align__(8) uint64_t s_bar;   // completion of the TMA box copy
  uint32_t bar_phase = 0;

  const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5, li = lane & 15;
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((uint32_t)__cvta_generic_to_shared(&s_bar)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  constexpr int BZ = F32 ? 16 : bin_z(W), BXY = F32 ? bin_xy32(W) : bin_xy(W, BZ);
  constexpr int Px = BXY + W, Py = BXY + W, Pz = BZ + W;
  constexpr int plane = Py * Pz;

  // the polynomial of interval li, in registers
  double pc[DEG + 1];
#pragma unroll
  for (int q = 0; q <= DEG; ++q) pc[q] = li < W ? ptab[q * kPolyStride + li] : 0.0;

  // the lane's cells of a W x W plane: c = lane + 32 i -> (cy, cz); offset inside the plane cy Pz + cz
  // (lanes beyond the last cell of the last round load nothing in the plane loop and get weight 0)
  int off[NCL], cy[NCL], cz[NCL];
  bool on[NCL];
#pragma unroll
  for (int i = 0; i < NCL; ++i) {
    on[i] = lane + 32 * i < W * W;
    const int c = on[i] ? lane + 32 * i : 0;
    cy[i] = c / W;
    cz[i] = c - cy[i] * W;
    off[i] = cy[i] * Pz + cz[i];
  }

  const int total = *n_items;
  for (;;) {
    // (the subgrid is read, and on the LDGSTS path written, through the generic proxy; the next box copy writes it
    // through the async proxy)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();  // everyone is done with s_item and the previous subgrid
    if (tid == 0) s_item = atomicAdd(counter, 1);
    __syncthreads();
    const int tick = s_item;
    if (tick >= total) break;
    // Items are in bin order, x slowest: the crowded bins around the origin (the rule's nodes cluster as 1/r^2) sit in
    // the middle of the list.  Hand them out from the middle outwards, so that the long items start first and the
    // short ones fill the tail.
    const int mid = total / 2;
    int item = (tick & 1) ? mid - 1 - (tick >> 1) : mid + (tick >> 1);
    if (item < 0) item = tick;                 // the lower side is exhausted (odd totals): the rest of the upper side
    else if (item >= total) item = total - 1 - tick;   // the upper side is exhausted: the rest of the lower side
    const int bin = item_bin[item];
    const int start = item_start[item], count = item_count[item];
    const int bz = bin % p.nbt[2], by = (bin / p.nbt[2]) % p.nbt[1], bx = bin / (p.nbt[2] * p.nbt[1]);
    const int ox = p.t0[0] + bx * p.bt[0] - W / 2, oy = p.t0[1] + by * p.bt[1] - W / 2, oz = p.t0[2] + bz * p.bt[2] - W / 2;

    const int cx2 = p.n2[0], cy2 = p.n2[1], czc = p.n2[2] / 2;   // reflection m -> n2 - m about the centre n2/2
    // The subgrid as one TMA box [Px][Py][2 Pz] of doubles at (ox, oy, oz) - lo, zero-filled outside the band: possible
    // unless the box reaches below the centre plane of a half band (those cells are reflections of stored ones).
    const bool box = !F32 && use_tma && !(p.zh && oz < czc);
    if (box) {
      if (tid == 0) {
        constexpr uint32_t bytes = (uint32_t)Px * Py * Pz * sizeof(double2);
        const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&s_bar), dst = (uint32_t)__cvta_generic_to_shared(sub);
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
        asm volatile(
            "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst),
            "l"(reinterpret_cast<uint64_t>(&tmap)), "r"(2 * (oz - p.lo[2])), "r"(oy - p.lo[1]), "r"(ox - p.lo[0]), "r"(bar)
            : "memory");
      }
    } else {
    // stage the subgrid with 16-byte asynchronous copies (LDGSTS; zero-filled outside the band): every warp issues
    // all of its rows back to back and waits once, so the staging runs at L2 bandwidth instead of one round trip per
    // row.  One (x,y) row of Pz <= 32 cells per warp pass, coalesced along z.
    for (int row = wq; row < Px * Py; row += kWarps) {
      const int ix = row / Py, iy = row - ix * Py;
      if (lane < Pz) {
        int mx = ox + ix, my = oy + iy, mz = oz + lane;          // absolute inner-grid indices of the cell
        if (p.zh && mz < czc) {                                   // lower half: the conjugate of the mirror cell (sign applied in the gather)
          mx = cx2 - mx;
          my = cy2 - my;
          mz = 2 * czc - mz;
        }
        const int gx = mx - p.lo[0], gy = my - p.lo[1], gz = mz - p.lo[2];
        const bool inside = gx >= 0 && gy >= 0 && gz >= 0 && gx < p.nout[0] && gy < p.nout[1] && gz < p.nout[2];
        const CT* srcp = inside ? v + (((size_t)gx * p.nout[1] + gy) * p.nout[2] + gz) : v;
        const unsigned dst = (unsigned)__cvta_generic_to_shared(sub + row * Pz + lane);
        const int nbytes = inside ? (int)sizeof(CT) : 0;   // src-size 0: the destination bytes are zero-filled
        if (F32)
          asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(srcp), "r"(nbytes) : "memory");
        else
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(srcp), "r"(nbytes) : "memory");
      }
    }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    TgtRec r[TPW];
#pragma unroll
    for (int u = 0; u < TPW; ++u) r[u] = tgt[start + min(wq + u * kWarps, count - 1)];
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (box) {
      const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&s_bar);
      asm volatile(
          "{\n"
          ".reg .pred p;\n"
          "WAIT_%=:\n"
          "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
          "@p bra DONE_%=;\n"
          "bra WAIT_%=;\n"
          "DONE_%=:\n"
          "}\n" ::"r"(bar),
          "r"(bar_phase)
          : "memory");
      bar_phase ^= 1;
    }
    __syncthreads();

    for (int t = wq; t < count; t += kWarps * TPW) {
      // TPW targets per warp and iteration: their dependency chains (polynomials, gathers, shuffles) are independent
      // and interleave, which hides the latencies that 16 warps per SM cannot
      TgtRec cur[TPW];
      bool live[TPW];
#pragma unroll
      for (int u = 0; u < TPW; ++u) {
        cur[u] = r[u];
        live[u] = t + u * kWarps < count;
        const int nx = t + (TPW + u) * kWarps;
        if (nx < count) r[u] = tgt[start + nx];   // prefetch the warp's next targets
      }
      // kernel values: lanes 0-15 do x then z, lanes 16-31 do y
      int i0x[TPW], i0y[TPW], i0z[TPW];
      double k1[TPW], k2[TPW], s1[TPW], sz[TPW];
#pragma unroll
      for (int u = 0; u < TPW; ++u) {
        double sx, sy;
        footprint(cur[u].u[0], W, i0x[u], sx);
        footprint(cur[u].u[1], W, i0y[u], sy);
        footprint(cur[u].u[2], W, i0z[u], sz[u]);
        s1[u] = lane < 16 ? sx : sy;
        k1[u] = k2[u] = pc[DEG];
      }
#pragma unroll
      for (int q = DEG - 1; q >= 0; --q) {
#pragma unroll
        for (int u = 0; u < TPW; ++u) {
          k1[u] = __fma_rn(k1[u], s1[u], pc[q]);
          k2[u] = __fma_rn(k2[u], sz[u], pc[q]);
        }
      }
      __syncwarp();   // the previous targets' reads of ktab are done
      if (li < W) {
#pragma unroll
        for (int u = 0; u < TPW; ++u) {
          ktab[wq][u][lane < 16 ? 0 : 1][li] = k1[u];
          if (lane < 16) ktab[wq][u][2][li] = k2[u];
        }
      }
      __syncwarp();

      AT are[TPW][NCL], aim[TPW][NCL];
      const CT* cell[TPW][NCL];   // the lane's cells in plane 0 of the footprint; plane a is an immediate offset
#pragma unroll
      for (int u = 0; u < TPW; ++u) {
        const CT* base = sub + ((i0x[u] - ox) * Py + (i0y[u] - oy)) * Pz + (i0z[u] - oz);
#pragma unroll
        for (int i = 0; i < NCL; ++i) {
          are[u][i] = aim[u][i] = (AT)0;
          cell[u][i] = base + off[i];
        }
      }
#pragma unroll
      for (int a = 0; a < W; ++a) {
#pragma unroll
        for (int u = 0; u < TPW; ++u) {
          const AT kx = (AT)ktab[wq][u][0][a];
#pragma unroll
          for (int i = 0; i < NCL; ++i) {
            // the last round of a plane covers only W*W - 32 (NCL-1) cells: lanes beyond them issue no load (a load
            // of a dummy cell would still cost its shared-memory wavefronts: 2 of 9 per plane at W = 7)
            CT c{};
            if (i + 1 < NCL || on[i]) c = cell[u][i][a * plane];
            are[u][i] = fma(c.x, kx, are[u][i]);
            aim[u][i] = fma(c.y, kx, aim[u][i]);
          }
        }
      }
      double re[TPW], im[TPW];
#pragma unroll
      for (int u = 0; u < TPW; ++u) {
        re[u] = im[u] = 0.0;
#pragma unroll
        for (int i = 0; i < NCL; ++i) {
          const double kyz = on[i] ? ktab[wq][u][1][cy[i]] * ktab[wq][u][2][cz[i]] : 0.0;
          re[u] = __fma_rn((double)are[u][i], kyz, re[u]);
          // cells below the centre plane hold the mirror cell un-conjugated: flip the sign of their imaginary part
          im[u] = __fma_rn((double)aim[u][i], (p.zh && i0z[u] + cz[i] < czc) ? -kyz : kyz, im[u]);
        }
      }
      if (TPW == 2) {
        // two targets: the first exchange hands target 0 to lanes 0-15 and target 1 to lanes 16-31, the remaining
        // four rounds reduce both at once -- 10 fp64 shuffles for two targets instead of 20
        const bool up = (lane & 16) != 0;
        const double sre = up ? re[0] : re[TPW - 1], sim = up ? im[0] : im[TPW - 1];
        double rr = (up ? re[TPW - 1] : re[0]) + __shfl_xor_sync(0xffffffffu, sre, 16);
        double ri = (up ? im[TPW - 1] : im[0]) + __shfl_xor_sync(0xffffffffu, sim, 16);
#pragma unroll
        for (int d = 8; d > 0; d >>= 1) {
          rr += __shfl_xor_sync(0xffffffffu, rr, d);
          ri += __shfl_xor_sync(0xffffffffu, ri, d);
        }
        if (lane == 0 && live[0]) G[cur[0].k] = make_double2(rr, ri);
        if (lane == 16 && live[TPW - 1]) G[cur[TPW - 1].k] = make_double2(rr, ri);
      } else {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
          re[0] += __shfl_xor_sync(0xffffffffu, re[0], d);
          im[0] += __shfl_xor_sync(0xffffffffu, im[0], d);
        }
        if (lane == 0 && live[0]) G[cur[0].k] = make_double2(re[0], im[0]);
      }
    }
  }
}

// Tensor map of the band [nout0][nout1][nout2] of complex128 cells, seen as doubles [nout0][nout1][2 nout2], with the box
// of one staged subgrid.  *ok = false when the driver offers no encoder or rejects the shape: LDGSTS staging then.
void band_tensor_map(const N3Params& p, const double* d_v, CUtensorMap* tm, bool* ok) {
  using Encode = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                              const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                              CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static Encode encode = [] {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess ||
        qr != cudaDriverEntryPointSuccess)
      fn = nullptr;
    cudaGetLastError();
    return reinterpret_cast<Encode>(fn);
  }();
  *ok = false;
  std::memset(tm, 0, sizeof(*tm));
  if (!encode || p.f32) return;
  const cuuint64_t dim[3] = {2ull * p.nout[2], (cuuint64_t)p.nout[1], (cuuint64_t)p.nout[0]};
  const cuuint64_t stride[2] = {16ull * p.nout[2], 16ull * p.nout[2] * p.nout[1]};   // bytes, dimensions 1 and 2
  const cuuint32_t boxd[3] = {2u * (p.bt[2] + p.w), (cuuint32_t)(p.bt[1] + p.w), (cuuint32_t)(p.bt[0] + p.w)};
  const cuuint32_t estr[3] = {1, 1, 1};
  if (boxd[0] > 256 || boxd[1] > 256 || boxd[2] > 256 || (reinterpret_cast<uintptr_t>(d_v) & 15) != 0) return;
  *ok = encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(d_v), dim, stride, boxd, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int W, bool F32>
int launch(const N3Params& p, const double* d_ptab, const double* d_v, const TgtRec* d_tgt, const int32_t* d_item_bin,
           const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
           double* d_G, size_t smem, cudaStream_t st) {
  static thread_local int attr_dev = -1;
  if (first_use_on_device(attr_dev)) {
    SFD_CUDA_TRY(cudaFuncSetAttribute(interp_kernel<W, F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024));
  }
  CUtensorMap tm;
  bool tma = false;
  band_tensor_map(p, d_v, &tm, &tma);
  const char* no_tma = std::getenv("SFD_INTERP_NO_TMA");   // A-B measurements
  if (no_tma && no_tma[0] == '1') tma = false;
  interp_kernel<W, F32><<<num_sms(), 32 * kWarps, smem, st>>>(p, tm, tma ? 1 : 0, d_ptab, d_v, d_tgt,
                                                        d_item_bin, d_item_start, d_item_count, d_n_items, d_counter,
                                                        reinterpret_cast<double2*>(d_G));
  return launch_check("interp_kernel");
}

}  // namespace

void interp_bins(int w, bool f32, int bt[3]) {
  if (f32 && w <= kMaxW32) {
    bt[2] = 16;
    bt[0] = bt[1] = bin_xy32(w);
    return;
  }
  bt[2] = bin_z(w);
  bt[0] = bt[1] = bin_xy(w, bt[2]);
}

size_t interp_smem_bytes(const N3Params& p) {
  return kTabBytes + (size_t)(p.bt[0] + p.w) * (p.bt[1] + p.w) * (p.bt[2] + p.w) * (p.f32 ? 8 : 16);
}

int interp(const N3Params& p, const double* d_ptab, const double* d_v, const TgtRec* d_tgt, const int32_t* d_item_bin,
           const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
           double* d_G, cudaStream_t st) {
  const size_t smem = interp_smem_bytes(p);
  SFD_REQUIRE(smem <= 227 * 1024 - 1024 && p.bt[2] + p.w <= 32, SFD_ERR_INVALID_ARG,
              "interp subgrid does not fit shared memory (%zu B)", smem);
  SFD_CUDA_TRY(cudaMemsetAsync(d_counter, 0, sizeof(int32_t), st));
  if (p.f32) {
#define SFD_INTERP_CASE32(W_) \
  case W_: return launch<W_, true>(p, d_ptab, d_v, d_tgt, d_item_bin, d_item_start, d_item_count, d_n_items, d_counter, d_G, smem, st);
    switch (p.w) {
      SFD_INTERP_CASE32(2) SFD_INTERP_CASE32(3) SFD_INTERP_CASE32(4) SFD_INTERP_CASE32(5) SFD_INTERP_CASE32(6)
      SFD_INTERP_CASE32(7) SFD_INTERP_CASE32(8)
    }
#undef SFD_INTERP_CASE32
    set_error("interp: single-precision grids support kernel widths up to %d (eps >= 1e-6), got %d", kMaxW32, p.w);
    return SFD_ERR_UNSUPPORTED;
  }
#define SFD_INTERP_CASE(W_) \
  case W_: return launch<W_, false>(p, d_ptab, d_v, d_tgt, d_item_bin, d_item_start, d_item_count, d_n_items, d_counter, d_G, smem, st);
  switch (p.w) {
    SFD_INTERP_CASE(2) SFD_INTERP_CASE(3) SFD_INTERP_CASE(4) SFD_INTERP_CASE(5) SFD_INTERP_CASE(6)
    SFD_INTERP_CASE(7) SFD_INTERP_CASE(8) SFD_INTERP_CASE(9) SFD_INTERP_CASE(10) SFD_INTERP_CASE(11)
    SFD_INTERP_CASE(12) SFD_INTERP_CASE(13) SFD_INTERP_CASE(14) SFD_INTERP_CASE(15) SFD_INTERP_CASE(16)
  }
#undef SFD_INTERP_CASE
  set_error("interp: unsupported kernel width %d", p.w);
  return SFD_ERR_UNSUPPORTED;
}

}  // namespace sfd
