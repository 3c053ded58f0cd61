// interp.cu -- A5-8: interpolation step of the inner type-2 transform of the type-3 NUFFT ("Type-2 ...
// its adjoint").  G_k = sum over the w^3 cells m around t_k of v[m] psi2(m h2 - t_k), the gather twin of the
// spreading step: same kernel, no write conflicts.
//
// One persistent CTA per SM pulls work items (an occupied target bin or a slice of one) from a device-side queue,
// stages the bin's padded subgrid (bt+w)^3 of the inner grid in shared memory as complex128 (16 B LDG/STS) and
// lets each of its 16 warps gather one target at a time: the 32 lanes cover the w x w cells of an x-plane, walk
// the w planes accumulating v * kx in registers, weight by ky kz at the end and finish with a warp-shuffle sum.
#include "nufft3.cuh"

namespace sfd {
namespace {

constexpr int kWarps = 16;
constexpr int kMaxCellsPerLane = (kMaxW * kMaxW + 31) / 32;
constexpr int kMaxP = 23;  // 23^3 * 16 B = 195 KB

__global__ void __launch_bounds__(32 * kWarps, 1)
interp_kernel(N3Params p, const double2* __restrict__ v, const TgtRec* __restrict__ tgt,
              const int32_t* __restrict__ item_bin, const int32_t* __restrict__ item_start,
              const int32_t* __restrict__ item_count, const int32_t* __restrict__ n_items,
              int32_t* __restrict__ counter, double2* __restrict__ G) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double (*ktab)[3][kMaxW] = reinterpret_cast<double (*)[3][kMaxW]>(smem_raw);
  double2* sub = reinterpret_cast<double2*>(smem_raw + sizeof(double) * kWarps * 3 * kMaxW);
  __shared__ int s_item;

  const int w = p.w, P = p.bt + w, fw = w / 2;
  const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
  const int ncell = P * P * P;

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
    __syncthreads();  // everyone is done with s_item and the previous subgrid
    if (tid == 0) s_item = atomicAdd(counter, 1);
    __syncthreads();
    const int item = s_item;
    if (item >= total) break;
    const int bin = item_bin[item];
    const int start = item_start[item], count = item_count[item];
    const int bz = bin % p.nbt[2], by = (bin / p.nbt[2]) % p.nbt[1], bx = bin / (p.nbt[2] * p.nbt[1]);
    const int o[3] = {p.t0[0] + bx * p.bt - fw, p.t0[1] + by * p.bt - fw, p.t0[2] + bz * p.bt - fw};

    for (int i = tid; i < ncell; i += 32 * kWarps) {
      const int iz = i % P, iy = (i / P) % P, ix = i / (P * P);
      const int gx = o[0] + ix, gy = o[1] + iy, gz = o[2] + iz;
      double2 val = make_double2(0.0, 0.0);
      if (gx >= 0 && gy >= 0 && gz >= 0 && gx < p.n2[0] && gy < p.n2[1] && gz < p.n2[2])
        val = v[((size_t)gx * p.n2[1] + gy) * p.n2[2] + gz];
      sub[i] = val;
    }
    __syncthreads();

    for (int t = wq; t < count; t += kWarps) {
      const TgtRec r = tgt[start + t];
      int i0[3];
#pragma unroll
      for (int d = 0; d < 3; ++d) i0[d] = (int)ceil(r.u[d] - 0.5 * w);
      __syncwarp();
      for (int e = lane; e < 3 * w; e += 32) {
        const int d = e / w, i = e - d * w;
        const double ud = d == 0 ? r.u[0] : (d == 1 ? r.u[1] : r.u[2]);
        const int id = d == 0 ? i0[0] : (d == 1 ? i0[1] : i0[2]);
        ktab[wq][d][i] = es_kernel(((double)(id + i) - ud) * (2.0 / w), p.beta);
      }
      __syncwarp();
      double are[kMaxCellsPerLane], aim[kMaxCellsPerLane];
#pragma unroll
      for (int i = 0; i < kMaxCellsPerLane; ++i) are[i] = aim[i] = 0.0;
      const int base = ((i0[0] - o[0]) * P + (i0[1] - o[1])) * P + (i0[2] - o[2]);
      for (int a = 0; a < w; ++a) {
        const double kx = ktab[wq][0][a];
#pragma unroll
        for (int i = 0; i < kMaxCellsPerLane; ++i) {
          if (i < ncl && cy[i] >= 0) {
            const double2 c = sub[base + (a * P + cy[i]) * P + cz[i]];
            are[i] = __fma_rn(c.x, kx, are[i]);
            aim[i] = __fma_rn(c.y, kx, aim[i]);
          }
        }
      }
      double re = 0.0, im = 0.0;
#pragma unroll
      for (int i = 0; i < kMaxCellsPerLane; ++i) {
        if (i < ncl && cy[i] >= 0) {
          const double kyz = ktab[wq][1][cy[i]] * ktab[wq][2][cz[i]];
          re = __fma_rn(are[i], kyz, re);
          im = __fma_rn(aim[i], kyz, im);
        }
      }
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) {
        re += __shfl_xor_sync(0xffffffffu, re, d);
        im += __shfl_xor_sync(0xffffffffu, im, d);
      }
      if (lane == 0) G[r.k] = make_double2(re, im);
    }
  }
}

}  // namespace

int interp_max_bin(int w) { return kMaxP - w; }

size_t interp_smem_bytes(const N3Params& p) {
  const size_t P = p.bt + p.w;
  return sizeof(double) * kWarps * 3 * kMaxW + P * P * P * 16;
}

int interp(const N3Params& p, const double* d_v, const TgtRec* d_tgt, const int32_t* d_item_bin,
           const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
           double* d_G, cudaStream_t st) {
  const size_t smem = interp_smem_bytes(p);
  SFD_REQUIRE(smem <= 227 * 1024 - 1024, SFD_ERR_INVALID_ARG, "interp subgrid does not fit shared memory (%zu B)", smem);
  SFD_CUDA_TRY(cudaMemsetAsync(d_counter, 0, sizeof(int32_t), st));
  static bool attr = false;
  if (!attr) {
    SFD_CUDA_TRY(cudaFuncSetAttribute(interp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024));
    attr = true;
  }
  interp_kernel<<<num_sms(), 32 * kWarps, smem, st>>>(p, reinterpret_cast<const double2*>(d_v), d_tgt, d_item_bin,
                                                     d_item_start, d_item_count, d_n_items, d_counter,
                                                     reinterpret_cast<double2*>(d_G));
  return launch_check("interp_kernel");
}

}  // namespace sfd
