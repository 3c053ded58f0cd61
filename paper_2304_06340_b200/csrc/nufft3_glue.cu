// nufft3_glue.cu -- the one-pass, HBM-bound kernels of the type-3 NUFFT around spread / FFT / interp:
// bounds (A5-1), source rescaling + pre-phase + bin sort (A5-2, A5-3; "sort"), deconvolution + zero padding
// (A5-5), target rescaling + bin sort (A5-7), post-deconvolution + post-phase (A5-9).  Formulas: DESIGN.md
// "type-3 NUFFT"; layouts: nufft3.cuh.
#include <algorithm>

#include "internal.cuh"
#include "atoms.cuh"
#include "nufft3.cuh"

namespace sfd {
namespace {

constexpr int kT = 256;

__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, d));
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, d));
  return v;
}

// ---- A5-1 bounds ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kT) bounds_partial_kernel(const double* __restrict__ pts, int64_t n, double* __restrict__ part) {
  __shared__ double sm[kT / 32][6];
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  double lo[3] = {inf, inf, inf}, hi[3] = {-inf, -inf, -inf};
  for (int64_t i = (int64_t)blockIdx.x * kT + threadIdx.x; i < n; i += (int64_t)gridDim.x * kT) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double v = pts[3 * i + c];
      lo[c] = fmin(lo[c], v);
      hi[c] = fmax(hi[c], v);
    }
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    lo[c] = warp_min(lo[c]);
    hi[c] = warp_max(hi[c]);
  }
  if (lane == 0)
    for (int c = 0; c < 3; ++c) {
      sm[wid][c] = lo[c];
      sm[wid][3 + c] = hi[c];
    }
  __syncthreads();
  if (threadIdx.x < 6) {
    double v = sm[0][threadIdx.x];
    for (int i = 1; i < kT / 32; ++i) v = threadIdx.x < 3 ? fmin(v, sm[i][threadIdx.x]) : fmax(v, sm[i][threadIdx.x]);
    part[blockIdx.x * 6 + threadIdx.x] = v;
  }
}
// one warp per component: the lanes stride over the per-block partials, then a shuffle reduction
__global__ void __launch_bounds__(192) bounds_final_kernel(const double* __restrict__ part, int nblocks, double* __restrict__ out6) {
  const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  double v = c < 3 ? inf : -inf;
  for (int i = lane; i < nblocks; i += 32) v = c < 3 ? fmin(v, part[i * 6 + c]) : fmax(v, part[i * 6 + c]);
  v = c < 3 ? warp_min(v) : warp_max(v);
  if (lane == 0) out6[c] = v;
}

// Warp-aggregated counter update: lanes of a warp that hold the same key share one atomicAdd (consecutive points
// fall into the same bin -- 256 points of a phi-ring near the origin, the 6 atoms of a face -- so per-lane atomics
// serialise on a handful of counters).  Returns the lane's slot: value of counter[key] before the add + its rank.
__device__ __forceinline__ int warp_agg_inc(int32_t* counter, int key, bool active) {
  const unsigned live = __ballot_sync(0xffffffffu, active);
  if (!active) return 0;
  const unsigned peers = __match_any_sync(live, key);
  const int lane = threadIdx.x & 31;
  const int leader = __ffs(peers) - 1;
  const int rank = __popc(peers & ((1u << lane) - 1u));
  int base = 0;
  if (lane == leader) base = atomicAdd(&counter[key], __popc(peers));
  base = __shfl_sync(peers, base, leader);
  return base + rank;
}

// ---- bin keys ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

// Fine-grid coordinate of a source (A5-2).  Analytically u lies in [(w+1)/2, nf-(w+1)/2]; the clamp only guards
// the rounding of the caller's extents, so that the w-cell footprint can never leave the grid.
__device__ __forceinline__ double src_coord(const N3Params& p, double x, int d) {
  const double u = __fma_rn(x - p.C[d], p.sx[d], 0.5 * p.nf[d]);
  const double lo = 0.5 * p.w + 1e-9;
  return fmin(fmax(u, lo), p.nf[d] - lo);
}
// Inner-grid coordinate of a target (A5-7): analytically in [n2/4, 3 n2/4].
__device__ __forceinline__ double tgt_coord(const N3Params& p, double xi, int d) {
  const double u = __fma_rn(xi - p.D[d], p.st[d], 0.5 * p.n2[d]);
  return fmin(fmax(u, (double)p.t0[d]), (double)(p.t0[d] + p.n2[d] / 2));
}

// Where the sources come from: the arrays x[J][3], w[J], or (V != nullptr) the atoms of a mesh generated on the fly
// (atoms.cuh) -- the lattice variant's 2e7 atoms are then never written to or read from memory as (x, w).
struct SrcView {
  const double* x;
  const double* w;
  const double* V;
  const int32_t* F;
  int64_t nV;
  const double* rule;   // 4 x Q columns (device)
  int Q;
  int32_t* flags;       // device error word (common.cuh): a bad face index is reported, not only poisoned
};
__device__ __forceinline__ void stage_rule(const SrcView& v, double* s_rule) {
  if (v.V) {
    for (int t = threadIdx.x; t < 4 * v.Q; t += kT) s_rule[t] = v.rule[t];
    __syncthreads();
  }
}
__device__ __forceinline__ void load_source(const SrcView& v, const double* s_rule, int64_t j, double& x0, double& x1,
                                            double& x2, double& w) {
  if (v.V) {
    atom_eval(v.V, v.nV, v.F, j, v.Q, s_rule, x0, x1, x2, w, v.flags);
  } else {
    x0 = v.x[3 * j];
    x1 = v.x[3 * j + 1];
    x2 = v.x[3 * j + 2];
    w = v.w[j];
  }
}

__global__ void __launch_bounds__(kT) source_keys_kernel(N3Params p, SrcView v, int64_t J, int32_t* __restrict__ key,
                                                        int32_t* __restrict__ hist) {
  __shared__ double s_rule[4 * 64];
  stage_rule(v, s_rule);
  const int64_t j = (int64_t)blockIdx.x * kT + threadIdx.x;
  const bool active = j < J;
  int k = 0;
  if (active) {
    double xs[3], wj;
    load_source(v, s_rule, j, xs[0], xs[1], xs[2], wj);
    int b[3], c[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double u = src_coord(p, xs[d], d);
      b[d] = clampi((int)floor(u / p.bs[d]), 0, p.nbs[d] - 1);
      // first cell of the footprint relative to the bin's padded subgrid: in [0, bs] (the footprint fits the subgrid)
      int i0;
      double s;
      footprint(u, p.w, i0, s);
      c[d] = clampi(i0 - (b[d] * p.bs[d] - p.w / 2), 0, p.bs[d]);
    }
    k = (b[0] * p.nbs[1] + b[1]) * p.nbs[2] + b[2];
    if (p.fine) k = (k * (p.bs[0] + 1) + c[0]) * (p.bs[1] + 1) * (p.bs[2] + 1) + c[1] * (p.bs[2] + 1) + c[2];
    key[j] = k;
  }
  warp_agg_inc(hist, k, active);
}

__global__ void __launch_bounds__(kT) bin_ranges_kernel(const int32_t* __restrict__ off, int64_t nbins, int64_t cpb, int64_t J,
                                                       int32_t* __restrict__ bhist, int32_t* __restrict__ boff) {
  const int64_t b = (int64_t)blockIdx.x * kT + threadIdx.x;
  if (b > nbins) return;
  const int32_t lo = b < nbins ? off[b * cpb] : (int32_t)J;
  boff[b] = lo;
  if (b < nbins) bhist[b] = (b + 1 < nbins ? off[(b + 1) * cpb] : (int32_t)J) - lo;
}

__global__ void __launch_bounds__(kT) source_scatter_kernel(N3Params p, SrcView v, int64_t J, const int32_t* __restrict__ key,
                                                           const int32_t* __restrict__ off, int32_t* __restrict__ cursor,
                                                           SrcRec* __restrict__ out) {
  __shared__ double s_rule[4 * 64];
  stage_rule(v, s_rule);
  const int64_t j = (int64_t)blockIdx.x * kT + threadIdx.x;
  const bool active = j < J;
  const int k = active ? key[j] : 0;
  const int slot = warp_agg_inc(cursor, k, active);
  if (!active) return;
  const int pos = off[k] + slot;
  SrcRec r;
  double x0, x1, x2, wj;
  load_source(v, s_rule, j, x0, x1, x2, wj);
  r.u[0] = src_coord(p, x0, 0);
  r.u[1] = src_coord(p, x1, 1);
  r.u[2] = src_coord(p, x2, 2);
  if (p.real_c) {
    r.re = wj;
    r.im = 0.0;
  } else {
    double s, c;
    sincos_fp64(__fma_rn(p.D[0], x0, __fma_rn(p.D[1], x1, p.D[2] * x2)), s, c);
    r.re = wj * c;
    r.im = -wj * s;
  }
  out[pos] = r;
}

__global__ void __launch_bounds__(kT) target_keys_kernel(N3Params p, const double* __restrict__ xi, int64_t K,
                                                        int32_t* __restrict__ key, int32_t* __restrict__ hist) {
  const int64_t k = (int64_t)blockIdx.x * kT + threadIdx.x;
  const bool active = k < K;
  int kk = 0;
  if (active) {
    int b[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double u = tgt_coord(p, xi[3 * k + d], d);
      b[d] = clampi((int)floor((u - p.t0[d]) / p.bt[d]), 0, p.nbt[d] - 1);
    }
    kk = (b[0] * p.nbt[1] + b[1]) * p.nbt[2] + b[2];
    key[k] = kk;
  }
  warp_agg_inc(hist, kk, active);
}

__global__ void __launch_bounds__(kT) target_scatter_kernel(N3Params p, const double* __restrict__ xi, int64_t K,
                                                           const int32_t* __restrict__ key, const int32_t* __restrict__ off,
                                                           int32_t* __restrict__ cursor, TgtRec* __restrict__ out) {
  const int64_t k = (int64_t)blockIdx.x * kT + threadIdx.x;
  const bool active = k < K;
  const int kk = active ? key[k] : 0;
  const int slot = warp_agg_inc(cursor, kk, active);
  if (!active) return;
  const int pos = off[kk] + slot;
  TgtRec r;
#pragma unroll
  for (int d = 0; d < 3; ++d) r.u[d] = tgt_coord(p, xi[3 * k + d], d);
  r.k = k;
  out[pos] = r;
}

// ---- work items ----------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kT) item_counts_kernel(const int32_t* __restrict__ hist, int64_t nbins, int cap,
                                                        int32_t* __restrict__ nit) {
  const int64_t b = (int64_t)blockIdx.x * kT + threadIdx.x;
  if (b < nbins) nit[b] = (hist[b] + cap - 1) / cap;
}
__global__ void __launch_bounds__(kT) item_fill_kernel(const int32_t* __restrict__ hist, const int32_t* __restrict__ off,
                                                      const int32_t* __restrict__ pos, int64_t nbins, int cap,
                                                      int64_t max_items, int32_t* __restrict__ items) {
  const int64_t b = (int64_t)blockIdx.x * kT + threadIdx.x;
  if (b >= nbins) return;
  const int n = hist[b];
  int at = pos[b];
  for (int s = 0; s < n; s += cap, ++at) {
    items[at] = (int32_t)b;
    items[max_items + at] = off[b] + s;
    items[2 * max_items + at] = min(cap, n - s);
  }
}

// ---- A5-5 deconvolution + zero padding -----------------------------------------------------------------------
__global__ void __launch_bounds__(kT) deconv_tables_kernel(N3Params p, ChebTable q, double* __restrict__ dec) {
  const int i = blockIdx.x * kT + threadIdx.x;
  const int n0 = p.nf[0], n1 = p.nf[1], n2 = p.nf[2];
  if (i >= n0 + n1 + n2) return;
  const int d = i < n0 ? 0 : (i < n0 + n1 ? 1 : 2);
  const int ii = i - (d == 0 ? 0 : (d == 1 ? n0 : n0 + n1));
  const int l = ii - p.nf[d] / 2;
  const double kappa = (double)l * p.w * 3.14159265358979323846 / (double)p.n2[d];
  const double v = 1.0 / half_w_phihat(q, kappa);
  dec[i] = (l & 1) ? -v : v;   // (-1)^l: shifts the inner grid by half a period, t_m = m h2 - pi
}

// ---- A5-9 post-deconvolution + post-phase --------------------------------------------------------------------
__global__ void __launch_bounds__(kT) post_deconv_kernel(N3Params p, ChebTable q, const double* __restrict__ xi, int64_t K,
                                                        double2* __restrict__ nuhat) {
  const int64_t k = (int64_t)blockIdx.x * kT + threadIdx.x;
  if (k >= K) return;
  const double a0 = xi[3 * k] - p.D[0], a1 = xi[3 * k + 1] - p.D[1], a2 = xi[3 * k + 2] - p.D[2];
  const double den = half_w_phihat(q, a0 * p.kap[0]) * half_w_phihat(q, a1 * p.kap[1]) * half_w_phihat(q, a2 * p.kap[2]);
  double s, c;
  sincos_fp64(__fma_rn(a0, p.C[0], __fma_rn(a1, p.C[1], a2 * p.C[2])), s, c);
  const double2 g = nuhat[k];
  const double inv = 1.0 / den;
  // G * (c - i s) / den
  nuhat[k] = make_double2((g.x * c + g.y * s) * inv, (g.y * c - g.x * s) * inv);
}

// ---- type-1 tail (eq. 3.6): lattice modes out of the FFT band ---------------------------------------------
// dec[d * (M/2+1) + m] = 1 / ((w/2) phihat(m w pi / N_d)), m = |mode| (phihat is even)
__global__ void __launch_bounds__(kT) lattice_tables_kernel(N3Params p, ChebTable q, int M, double* __restrict__ dec) {
  const int i = blockIdx.x * kT + threadIdx.x;
  const int nh = M / 2 + 1;
  if (i >= 3 * nh) return;
  const int d = i / nh, m = i - d * nh;
  dec[i] = 1.0 / half_w_phihat(q, (double)m * p.w * 3.14159265358979323846 / (double)p.n2[d]);
}

// v = complex[M+1][M+1][M/2+1], modes (m0, m1, m2 >= 0); the other half by v(-m) = conj v(m) (real strengths).
// nuhat[k], k = ((a (M+1)) + b)(M+1) + c as in lattice_kernel (nodes.cu), m = (a, b, c) - M/2:
//   nuhat = v(m) e^{-i xi.C} prod_d dec_d[|m_d|],  xi_d = 2 pi (m_d h)
__global__ void __launch_bounds__(kT) lattice_post_kernel(N3Params p, int M, double h, const double* __restrict__ dec,
                                                         const double2* __restrict__ v, double2* __restrict__ nuhat) {
  const int n = M + 1, nh = M / 2 + 1;
  const int64_t K = (int64_t)n * n * n;
  const int64_t k = (int64_t)blockIdx.x * kT + threadIdx.x;
  if (k >= K) return;
  const int c = (int)(k % n);
  const int64_t ab = k / n;
  const int b = (int)(ab % n), a = (int)(ab / n);
  const int m0 = a - M / 2, m1 = b - M / 2, m2 = c - M / 2;
  const bool refl = m2 < 0;
  const int ia = refl ? M - a : a, ib = refl ? M - b : b, ic = refl ? -m2 : m2;
  const int64_t cell = ((int64_t)ia * n + ib) * nh + ic;
  double2 g;
  if (p.f32) {   // single-precision band
    const float2 gf = reinterpret_cast<const float2*>(v)[cell];
    g = make_double2((double)gf.x, (double)gf.y);
  } else {
    g = v[cell];
  }
  if (refl) g.y = -g.y;
  const double f = dec[abs(m0)] * dec[nh + abs(m1)] * dec[2 * nh + ic];
  g.x *= f;
  g.y *= f;
  if (p.C[0] != 0.0 || p.C[1] != 0.0 || p.C[2] != 0.0) {
    const double two_pi = 6.283185307179586476925286766559;
    const double x0 = __dmul_rn(two_pi, __dmul_rn((double)m0, h)), x1 = __dmul_rn(two_pi, __dmul_rn((double)m1, h)),
                 x2 = __dmul_rn(two_pi, __dmul_rn((double)m2, h));
    double sn, cs;
    sincos_fp64(__fma_rn(x0, p.C[0], __fma_rn(x1, p.C[1], x2 * p.C[2])), sn, cs);
    g = make_double2(g.x * cs + g.y * sn, g.y * cs - g.x * sn);
  }
  nuhat[k] = g;
}

}  // namespace

static inline unsigned blocks_for(int64_t n) { return (unsigned)((n + kT - 1) / kT); }

int bounds_minmax(const double* d_pts, int64_t n, double* d_out6, double* d_scratch, cudaStream_t st) {
  const int nb = (int)std::min<int64_t>(kBoundsBlocks, std::max<int64_t>(1, (n + kT - 1) / kT));
  bounds_partial_kernel<<<nb, kT, 0, st>>>(d_pts, n, d_scratch);
  SFD_TRY(launch_check("bounds_partial_kernel"));
  bounds_final_kernel<<<1, 192, 0, st>>>(d_scratch, nb, d_out6);
  return launch_check("bounds_final_kernel");
}

static SrcView src_view(const double* d_x, const double* d_w, const MeshAtoms* mesh, const double* d_rule) {
  SrcView v{};
  v.x = d_x;
  v.w = d_w;
  if (mesh) {
    v.V = mesh->d_V;
    v.F = mesh->d_F;
    v.nV = mesh->nV;
    v.rule = d_rule;
    v.Q = mesh->rule;
    v.flags = device_flags();
  }
  return v;
}

int source_keys(const N3Params& p, const double* d_x, int64_t J, int32_t* d_key, int32_t* d_hist, cudaStream_t st,
                const MeshAtoms* mesh, const double* d_rule) {
  source_keys_kernel<<<blocks_for(J), kT, 0, st>>>(p, src_view(d_x, nullptr, mesh, d_rule), J, d_key, d_hist);
  return launch_check("source_keys_kernel");
}
int source_bin_ranges(const N3Params& p, const int32_t* d_off, int64_t nbins, int64_t J, int32_t* d_bhist,
                      int32_t* d_boff, cudaStream_t st) {
  bin_ranges_kernel<<<blocks_for(nbins + 1), kT, 0, st>>>(d_off, nbins, source_subkeys(p), J, d_bhist, d_boff);
  return launch_check("bin_ranges_kernel");
}
int source_scatter(const N3Params& p, const double* d_x, const double* d_w, int64_t J, const int32_t* d_key,
                   const int32_t* d_off, int32_t* d_cursor, SrcRec* d_out, cudaStream_t st, const MeshAtoms* mesh,
                   const double* d_rule) {
  source_scatter_kernel<<<blocks_for(J), kT, 0, st>>>(p, src_view(d_x, d_w, mesh, d_rule), J, d_key, d_off, d_cursor, d_out);
  return launch_check("source_scatter_kernel");
}
int target_keys(const N3Params& p, const double* d_xi, int64_t K, int32_t* d_key, int32_t* d_hist, cudaStream_t st) {
  target_keys_kernel<<<blocks_for(K), kT, 0, st>>>(p, d_xi, K, d_key, d_hist);
  return launch_check("target_keys_kernel");
}
int target_scatter(const N3Params& p, const double* d_xi, int64_t K, const int32_t* d_key, const int32_t* d_off,
                   int32_t* d_cursor, TgtRec* d_out, cudaStream_t st) {
  target_scatter_kernel<<<blocks_for(K), kT, 0, st>>>(p, d_xi, K, d_key, d_off, d_cursor, d_out);
  return launch_check("target_scatter_kernel");
}

int make_items(const int32_t* d_hist, const int32_t* d_off, int64_t nbins, int cap, int32_t* d_tmp, int32_t* d_items,
               int64_t max_items, int32_t* d_n_items, void* d_scan, size_t scan_bytes, cudaStream_t st) {
  item_counts_kernel<<<blocks_for(nbins), kT, 0, st>>>(d_hist, nbins, cap, d_tmp);
  SFD_TRY(launch_check("item_counts_kernel"));
  SFD_TRY(exclusive_scan_i32(d_tmp, d_tmp, nbins, d_n_items, d_scan, scan_bytes, st));
  item_fill_kernel<<<blocks_for(nbins), kT, 0, st>>>(d_hist, d_off, d_tmp, nbins, cap, max_items, d_items);
  return launch_check("item_fill_kernel");
}


int deconv_tables(const N3Params& p, const ChebTable& q, double* d_dec, cudaStream_t st) {
  deconv_tables_kernel<<<blocks_for(p.nf[0] + p.nf[1] + p.nf[2]), kT, 0, st>>>(p, q, d_dec);
  return launch_check("deconv_tables_kernel");
}

int post_deconv(const N3Params& p, const ChebTable& q, const double* d_xi, int64_t K, double* d_nuhat, cudaStream_t st) {
  post_deconv_kernel<<<blocks_for(K), kT, 0, st>>>(p, q, d_xi, K, reinterpret_cast<double2*>(d_nuhat));
  return launch_check("post_deconv_kernel");
}

int lattice_tables(const N3Params& p, const ChebTable& q, int M, double* d_dec, cudaStream_t st) {
  lattice_tables_kernel<<<blocks_for(3 * (M / 2 + 1)), kT, 0, st>>>(p, q, M, d_dec);
  return launch_check("lattice_tables_kernel");
}

int lattice_post(const N3Params& p, int M, double h, const double* d_dec, const double* d_v, double* d_nuhat,
                 cudaStream_t st) {
  const int64_t K = (int64_t)(M + 1) * (M + 1) * (M + 1);
  lattice_post_kernel<<<blocks_for(K), kT, 0, st>>>(p, M, h, d_dec, reinterpret_cast<const double2*>(d_v),
                                                    reinterpret_cast<double2*>(d_nuhat));
  return launch_check("lattice_post_kernel");
}

}  // namespace sfd
