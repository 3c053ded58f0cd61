// exact.cu -- S:8(f) NEXT-3: direct summation of the exact triangle transform, the O(N_S N_F) method of the prior-art
// codes the paper compares with ("several previous studies including [8, 38] employ the exact formula (2.19) and
// implement the direct summation in the frequency space"; timings P:244).  In the e^{-i xi.x} convention
//
//   T^(xi_k) = sum_f Q_f^(xi_k),   Q^(xi) = int_Q e^{-i xi.x} dS = 2A e^{-i alpha_0} g(u, v),
//   alpha_0 = xi.p_0, u = xi.(p_1 - p_0), v = xi.(p_2 - p_0),   g(u, v) = exp[0, -iu, -iv]
//
// with exp[.,.,.] the second divided difference of exp; for distinct nodes this is P:128 eq. 2.19 (gamma = 2A).
// Eq. 2.19 itself "suffers from large cancellation errors when a simplex is almost degenerate or when the vector xi is
// almost orthogonal to one of the edges" and the prior art regularises the denominators or switches to a degenerate
// formula, "both of which limit accuracy".  Here the divided difference is evaluated without cancellation in
// fp64, every pair to ~1e-15 absolute whatever the configuration:
//   * max(|u|, |v|, |v-u|) <= 1 (always the case once |xi| h <= 1, i.e. for fine meshes): the power series
//     g = sum_n (-i)^n H_n(u,v)/(n+2)!, H_n = u H_{n-1} + v^n, 8 to 18 terms by the warp's largest argument
//     (3 FP64 instructions per term), then one sincos for e^{-i alpha_0};
//   * otherwise the recursion exp[a,b,c] = (exp[b,c] - exp[a,b]) / (z_c - z_a) over the pair (a,c) farthest apart
//     (|z_c - z_a| > 1, so the division amplifies nothing), with first differences in the cancellation-free form
//     exp[-ix, -iy] = e^{-i(x+y)/2} sinc((y-x)/2).
// Faces are preprocessed once into 80-byte records (p_0, e_1, e_2, 2A) and staged through shared memory; one thread
// per frequency, all lanes of a warp read the same record (broadcast).  FP64-ALU-bound like the atoms' direct sum:
// ~65-110 FP64 instructions per (face, frequency) pair in the series branch.
#include <algorithm>

#include "internal.cuh"

namespace sfd {
namespace {

struct __align__(16) FaceRec {
  double p0[3], e1[3], e2[3], a2;
};
static_assert(sizeof(FaceRec) == 80, "FaceRec layout");

constexpr int kThreads = 256;
constexpr int kTile = 128;   // faces per shared-memory tile (10 KB)

// c[n] = (-i)^n / (n+2)! split into the real coefficients of the even and odd terms: Re g = sum_{n even} c[n] H_n,
// Im g = sum_{n odd} c[n] H_n.
__constant__ double c_series[18] = {
    1.0 / 2.0,                 -1.0 / 6.0,                 -1.0 / 24.0,                1.0 / 120.0,
    1.0 / 720.0,               -1.0 / 5040.0,              -1.0 / 40320.0,             1.0 / 362880.0,
    1.0 / 3628800.0,           -1.0 / 39916800.0,          -1.0 / 479001600.0,         1.0 / 6227020800.0,
    1.0 / 87178291200.0,       -1.0 / 1307674368000.0,     -1.0 / 20922789888000.0,    1.0 / 355687428096000.0,
    1.0 / 6402373705728000.0,  -1.0 / 121645100408832000.0};

__global__ void __launch_bounds__(256) face_prep_kernel(const double* __restrict__ V, int64_t nV, const int32_t* __restrict__ F,
                                                       int64_t nF, FaceRec* __restrict__ out, int32_t* __restrict__ flags) {
  const int64_t f = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (f >= nF) return;
  const int32_t i0 = F[3 * f], i1 = F[3 * f + 1], i2 = F[3 * f + 2];
  FaceRec r;
  if (i0 < 0 || i1 < 0 || i2 < 0 || i0 >= nV || i1 >= nV || i2 >= nV) {
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
#pragma unroll
    for (int c = 0; c < 3; ++c) r.p0[c] = r.e1[c] = r.e2[c] = nan;
    r.a2 = nan;
    if (flags) atomicOr(flags, kFlagBadIndex);
  } else {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      r.p0[c] = V[3 * (int64_t)i0 + c];
      r.e1[c] = V[3 * (int64_t)i1 + c] - r.p0[c];
      r.e2[c] = V[3 * (int64_t)i2 + c] - r.p0[c];
    }
    const double cx = r.e1[1] * r.e2[2] - r.e1[2] * r.e2[1];
    const double cy = r.e1[2] * r.e2[0] - r.e1[0] * r.e2[2];
    const double cz = r.e1[0] * r.e2[1] - r.e1[1] * r.e2[0];
    r.a2 = sqrt(cx * cx + cy * cy + cz * cz);   // 2A = gamma of eq. 2.19
  }
  out[f] = r;
}

// g(u, v) = sum_{n < NT} (-i)^n H_n(u, v) / (n+2)!,  H_n = u H_{n-1} + v^n
template <int NT>
__device__ __forceinline__ void series(double u, double v, double& sr, double& si) {
  double H = 1.0, P = 1.0;
  sr = c_series[0];
  si = 0.0;
#pragma unroll
  for (int n = 1; n < NT; ++n) {
    P *= v;
    H = __fma_rn(u, H, P);
    if (n & 1) si = __fma_rn(c_series[n], H, si);
    else sr = __fma_rn(c_series[n], H, sr);
  }
}

// sin(h)/h
__device__ __forceinline__ double sinc_fp64(double h) {
  double s, c;
  sincos_fp64(h, s, c);
  return h == 0.0 ? 1.0 : s / h;
}

__global__ void __launch_bounds__(kThreads) exact_sum_kernel(const FaceRec* __restrict__ faces, int64_t nF,
                                                            const double* __restrict__ xi, int64_t K, int64_t faces_per_split,
                                                            double2* __restrict__ out) {
  __shared__ FaceRec tile[kTile];
  const int64_t k = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  const bool live = k < K;
  const double x0 = live ? xi[3 * k] : 0.0, x1 = live ? xi[3 * k + 1] : 0.0, x2 = live ? xi[3 * k + 2] : 0.0;
  const int64_t f_begin = (int64_t)blockIdx.y * faces_per_split;
  const int64_t f_end = min(nF, f_begin + faces_per_split);
  double re = 0.0, im = 0.0;
  for (int64_t f0 = f_begin; f0 < f_end; f0 += kTile) {
    const int nt = (int)min((int64_t)kTile, f_end - f0);
    __syncthreads();
    {
      const double* src = reinterpret_cast<const double*>(faces + f0);
      double* dst = reinterpret_cast<double*>(tile);
      for (int i = threadIdx.x; i < nt * 10; i += kThreads) dst[i] = src[i];
    }
    __syncthreads();
    for (int j = 0; j < nt; ++j) {
      const FaceRec& r = tile[j];
      const double a0 = __fma_rn(x0, r.p0[0], __fma_rn(x1, r.p0[1], x2 * r.p0[2]));
      const double u = __fma_rn(x0, r.e1[0], __fma_rn(x1, r.e1[1], x2 * r.e1[2]));
      const double v = __fma_rn(x0, r.e2[0], __fma_rn(x1, r.e2[1], x2 * r.e2[2]));
      const double t = v - u;
      const double au = fabs(u), av = fabs(v), at = fabs(t);
      const double dmax = fmax(au, fmax(av, at));
      double gre, gim;   // e^{-i alpha_0} g(u, v)
      if (dmax <= 1.0) {
        // terms 0..nterm-1; remainder (n+1) d^n / (n+2)! below 1e-17
        int nterm = dmax <= 0.03 ? 8 : (dmax <= 0.1 ? 10 : (dmax <= 0.25 ? 12 : (dmax <= 0.5 ? 15 : 18)));
        nterm = __reduce_max_sync(__activemask(), nterm);
        double sr, si;
        switch (nterm) {   // uniform in the warp: one fully unrolled series per length, no per-term test
          case 8: series<8>(u, v, sr, si); break;
          case 10: series<10>(u, v, sr, si); break;
          case 12: series<12>(u, v, sr, si); break;
          case 15: series<15>(u, v, sr, si); break;
          default: series<18>(u, v, sr, si); break;
        }
        double s, c;
        sincos_fp64(a0, s, c);
        gre = __fma_rn(c, sr, s * si);
        gim = __fma_rn(c, si, -s * sr);
      } else {
        double oa, ob, oc;   // offsets from alpha_0 of the farthest pair (a, c) and the node between
        if (av >= au && av >= at) {
          oa = 0.0; ob = u; oc = v;
        } else if (au >= at) {
          oa = 0.0; ob = v; oc = u;
        } else {
          oa = u; ob = 0.0; oc = v;
        }
        const double k1 = sinc_fp64(0.5 * (oc - ob)), k2 = sinc_fp64(0.5 * (ob - oa));
        double s1, c1, s2, c2;
        sincos_fp64(a0 + 0.5 * (ob + oc), s1, c1);
        sincos_fp64(a0 + 0.5 * (oa + ob), s2, c2);
        const double nx = c1 * k1 - c2 * k2, ny = -(s1 * k1 - s2 * k2);   // exp[b,c] - exp[a,b]
        const double inv = 1.0 / (oc - oa);
        gre = -ny * inv;   // divide by z_c - z_a = -i (oc - oa): i (nx + i ny) / D
        gim = nx * inv;
      }
      re = __fma_rn(r.a2, gre, re);
      im = __fma_rn(r.a2, gim, im);
    }
  }
  if (!live) return;
  if (gridDim.y == 1) {
    out[k] = make_double2(re, im);
  } else {
    atomicAdd(&out[k].x, re);
    atomicAdd(&out[k].y, im);
  }
}

}  // namespace

size_t exact_ft_workspace(int64_t nF) { return align_up((size_t)std::max<int64_t>(nF, 1) * sizeof(FaceRec)); }

int exact_ft(const double* d_V, int64_t nV, const int32_t* d_F, int64_t nF, const double* d_xi, int64_t K, double* d_out,
             void* d_work, size_t work_bytes, cudaStream_t st) {
  if (K == 0) return SFD_OK;
  if (nF == 0) {
    SFD_CUDA_TRY(cudaMemsetAsync(d_out, 0, (size_t)K * 16, st));
    return SFD_OK;
  }
  SFD_REQUIRE(d_work && work_bytes >= exact_ft_workspace(nF), SFD_ERR_WORKSPACE_TOO_SMALL,
              "sfd_exact_ft needs %zu workspace bytes, got %zu", exact_ft_workspace(nF), work_bytes);
  FaceRec* faces = static_cast<FaceRec*>(d_work);
  face_prep_kernel<<<(unsigned)((nF + 255) / 256), 256, 0, st>>>(d_V, nV, d_F, nF, faces, device_flags());
  SFD_TRY(launch_check("face_prep_kernel"));
  const int64_t blocks = (K + kThreads - 1) / kThreads;
  // few frequencies: split the faces over blockIdx.y so that every SM has work (partial sums meet in fp64 reductions)
  int64_t nsplit = std::max<int64_t>(1, ((int64_t)num_sms() * 4 + blocks - 1) / blocks);
  nsplit = std::min<int64_t>(nsplit, (nF + kTile - 1) / kTile);
  nsplit = std::min<int64_t>(nsplit, 65535);
  const int64_t per = ((nF + nsplit - 1) / nsplit + kTile - 1) / kTile * kTile;
  nsplit = (nF + per - 1) / per;
  if (nsplit > 1) SFD_CUDA_TRY(cudaMemsetAsync(d_out, 0, (size_t)K * 16, st));
  SFD_REQUIRE(blocks <= 0x7fffffffLL, SFD_ERR_UNSUPPORTED, "sfd_exact_ft: too many frequencies");
  exact_sum_kernel<<<dim3((unsigned)blocks, (unsigned)nsplit), kThreads, 0, st>>>(faces, nF, d_xi, K, per,
                                                                                reinterpret_cast<double2*>(d_out));
  return launch_check("exact_sum_kernel");
}

}  // namespace sfd
