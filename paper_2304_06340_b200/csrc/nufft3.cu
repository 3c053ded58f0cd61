// nufft3.cu -- A5: 3-D type-3 nonuniform FFT, nuhat_k = sum_j w_j exp(-i xi_k . x_j) to tolerance eps, for
// nonuniform sources AND nonuniform targets ("in general it is required to compute contributions from
// nonuniform sources to nonuniform targets, which can be accelerated by the Type-3 NUFFT [18]").  The paper
// itself runs the type-1 special case on a lattice (eq. 3.6, eq. 3.7) through a library; this is a
// from-scratch implementation of the general case in fp64.  DESIGN.md "type-3 NUFFT" derives the formulas.
//
//   xi.x = (xi-D).(x-C) + D.x + (xi-D).C            C, D = centres of sources / targets
//   1. c'_j = w_j e^{-i D.x_j};  u_j = (x_j-C) sigma S/pi + nf/2   (rescaling: analogue of P:188 eq. 3.7)
//   2. bin-sort sources ("sort"), spread onto the fine grid nf^3 (spread.cu)
//   3. deconvolve by the kernel's transform on the integer modes (folded into the first FFT pass)
//   4. uniform FFT of size n2^3, n2 = 2 nf, pruned to the nf^3 non-zero inputs and to the band of outputs the
//      targets touch: three passes of in-shared-memory 1-D transforms (fft.cu).  The paper's library calls cuFFT on
//      the full lattice; a full n2^3 transform would move 8-16x more data and not fit at config 5.
//   5. bin-sort targets, interpolate at u2_k = (xi_k-D) n2/(2 sigma S) + n2/2 (interp.cu)
//   6. divide by the kernel's transform at the non-integer frequencies, multiply by e^{-i (xi_k-D).C}
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>
#include <functional>
#include <mutex>
#include <tuple>
#include <vector>

#include "atoms.cuh"
#include "fft.cuh"
#include "internal.cuh"
#include "nufft3.cuh"

namespace sfd {
namespace {

constexpr double kPi = 3.14159265358979323846;
constexpr int kSrcCap = 1024;   // sources per spread work item
constexpr int kTgtCap = 512;    // targets per interp work item (lower bound; nufft3() raises it with K)
// fixed head of the workspace: [0,96) bounds of x and xi; [128,144) n_items_s, n_items_t, queue counters;
// [1024, ...) scratch of the bounds reduction; [kRuleOff, +2048) the triangle rule when the sources are a mesh's atoms
constexpr size_t kMiscBytes = 32768;
constexpr size_t kRuleOff = 24576;

// Grid size: the smallest even n' >= n of the form 2^a 3^b 5^c (the radices 4, 2, 3, 5 of fft.cu), or of the form
// 2^a 3^b 5^c 7^d when that is at least 3 % smaller (a radix-7 stage costs more per point, and an extra stage when it
// does not pair up: 1344 is not worth it against 1350, 336 against 360 and 672 against 720 are).
int64_t next_smooth_even_of(int64_t n, bool with7) {
  if (n < 2) n = 2;
  if (n & 1) ++n;
  for (;; n += 2) {
    int64_t m = n;
    while (m % 2 == 0) m /= 2;
    while (m % 3 == 0) m /= 3;
    while (m % 5 == 0) m /= 5;
    if (with7)
      while (m % 7 == 0) m /= 7;
    if (m == 1) return n;
  }
}
int64_t next_smooth_even(int64_t n) {
  const int64_t n5 = next_smooth_even_of(n, false), n7 = next_smooth_even_of(n, true);
  return (double)n7 <= 0.97 * (double)n5 ? n7 : n5;
}

// Kernel width and shape for tolerance eps at upsampling 2 (parameter choice of the ES-kernel papers, refs [2,3]
// of P:185; reading R10): w = ceil(log10(1/eps)) + 1, beta = 2.30 w.  `careful`: one more cell of width --
// for a handful of sources (nothing averages the kernel's pointwise error, which reaches ~25 eps) and for a
// space-bandwidth product below one (a grid of a few cells); both cost nothing.
void kernel_params(double eps, bool careful, int* w, double* beta) {
  int ww = (int)std::ceil(std::log10(1.0 / eps) - 1e-9) + 1 + (careful ? 1 : 0);
  if (ww < 2) ww = 2;
  if (ww > kMaxW) ww = kMaxW;
  *w = ww;
  *beta = 2.30 * ww;
}

struct Layout {
  size_t src, skey, shist, soff, scur, sbhist, sboff, sitems, tgt, tkey, thist, toff, tcur, titems, fine, bufx, bufy, ffttab, dec,
      scan, scan_t, misc, ptab, total;
  int64_t ns_bins, ns_keys, nt_bins, ns_items, nt_items;
  size_t fine_bytes;
};

// Geometry from half-widths X (sources) and S (targets); centres are filled in by the caller.
constexpr int64_t kFewSources = 64;

int make_params(const double X_in[3], const double S_in[3], double eps, bool real_c, int64_t J, N3Params* p,
                bool f32 = false) {
  bool careful = J < kFewSources;
  for (int d = 0; d < 3; ++d)
    if (X_in[d] * (S_in[d] < 1e-150 ? 1.0 : S_in[d]) < 1.0) careful = true;
  kernel_params(eps, careful, &p->w, &p->beta);
  p->real_c = real_c ? 1 : 0;
  p->f32 = f32 ? 1 : 0;
  for (int d = 0; d < 3; ++d) {
    double X = X_in[d], S = S_in[d];
    SFD_REQUIRE(std::isfinite(X) && std::isfinite(S) && X >= 0 && S >= 0, SFD_ERR_INVALID_ARG,
                "type-3 NUFFT: extents must be finite and >= 0");
    if (S < 1e-150) S = 1.0;
    if (X * S < 1.0) X = 1.0 / S;
    const double need = 2.0 * kSigma * X * S / kPi + p->w + 1;
    SFD_REQUIRE(need < 8192.0, SFD_ERR_UNSUPPORTED, "type-3 NUFFT: fine grid of %.0f points per axis is too large", need);
    const int64_t nf = next_smooth_even((int64_t)std::ceil(need));
    p->nf[d] = (int)nf;
    p->n2[d] = (int)(2 * nf);
    p->sx[d] = kSigma * S / kPi;
    p->st[d] = (double)p->n2[d] / (2.0 * kSigma * S);
    p->kap[d] = p->w * kPi / (2.0 * kSigma * S);
  }
  p->deg = p->w + 3;
  spread_bins(p->w, real_c, p->bs);
  interp_bins(p->w, f32, p->bt);
  for (int d = 0; d < 3; ++d) {
    p->nbs[d] = (p->nf[d] + p->bs[d] - 1) / p->bs[d];
    p->t0[d] = p->n2[d] / 4;                      // targets occupy u2 in [n2/4, 3 n2/4]
    p->nbt[d] = (p->n2[d] / 2) / p->bt[d] + 1;
    // cells any footprint can touch: ceil(n2/4 - w/2) ... ceil(3 n2/4 - w/2) + w - 1, plus one cell of slack
    // (+1 for odd w: the band is then symmetric about n2/2, which the Hermitian reflection needs)
    p->lo[d] = std::max(0, p->n2[d] / 4 - (p->w + 1) / 2 - 1);
    p->nout[d] = std::min(p->n2[d] - p->lo[d], p->n2[d] / 2 + p->w + 3 + (p->w & 1));
  }
  // real strengths: keep only the upper half of the band along z (the last FFT-pass axis to be produced first)
  p->zh = 0;
  if (real_c && p->lo[2] > 0 && p->lo[0] > 0 && p->lo[1] > 0) {
    const int c2 = p->n2[2] / 2, hi2 = p->lo[2] + p->nout[2] - 1;
    p->zh = 1;
    p->lo[2] = c2;
    p->nout[2] = hi2 - c2 + 1;
  }
  return SFD_OK;
}

// Order the sources of a bin by footprint (N3Params::fine) when there are enough of them per cell for runs of equal
// footprints to form -- the clustered case of the paper's lattice variant -- and the key table stays small.
// sizing = true (workspace queries): whenever the table is small enough, so that the query bounds either choice.
void choose_sort(N3Params* p, int64_t J, bool sizing = false) {
  const int64_t nkeys = (int64_t)p->nbs[0] * p->nbs[1] * p->nbs[2] * source_subkeys(*p);
  p->fine = (nkeys <= (int64_t(1) << 22) && (sizing || J * 16 >= nkeys)) ? 1 : 0;
  // tens of sources per occupied cell (the sources lie on a surface: a few per cent of the cells): one warp per run
  if (p->fine && (sizing || J >= nkeys) && spread_runs_ok(p->w, p->real_c != 0)) p->fine = 2;
}

int make_layout(const N3Params& p, int64_t J, int64_t K, Layout* L) {
  L->ns_bins = (int64_t)p.nbs[0] * p.nbs[1] * p.nbs[2];
  L->nt_bins = (int64_t)p.nbt[0] * p.nbt[1] * p.nbt[2];
  L->ns_items = L->ns_bins + J / kSrcCap + 1;   // upper bound for any cap >= kSrcCap
  if (p.fine == 2) L->ns_items = std::max(L->ns_items, L->ns_bins * source_subkeys(p) + J / spread_runs_cap() + 1);
  L->nt_items = L->nt_bins + K / kTgtCap + 1;
  SFD_REQUIRE(L->ns_bins < 0x7fffffffLL && L->nt_bins < 0x7fffffffLL && J < 0x7fffffffLL && K < 0x7fffffffLL,
              SFD_ERR_UNSUPPORTED, "type-3 NUFFT: problem too large for 32-bit bin bookkeeping");
  size_t o = 0;
  auto put = [&](size_t bytes) {
    const size_t at = o;
    o += align_up(bytes);
    return at;
  };
  L->misc = put(kMiscBytes);
  L->ptab = put((size_t)(kMaxDeg + 1) * kPolyStride * 8);
  L->ns_keys = p.fine ? L->ns_bins * source_subkeys(p) : L->ns_bins;
  L->src = put((size_t)J * sizeof(SrcRec));
  L->skey = put((size_t)J * 4);
  L->shist = put((size_t)(L->ns_keys + 1) * 4);
  L->soff = put((size_t)(L->ns_keys + 1) * 4);
  L->scur = put((size_t)(L->ns_keys + 1) * 4);
  L->sbhist = put(p.fine ? (size_t)(L->ns_bins + 1) * 4 : 0);
  L->sboff = put(p.fine ? (size_t)(L->ns_bins + 1) * 4 : 0);
  L->sitems = put((size_t)L->ns_items * 4 * 3);
  L->tgt = put((size_t)K * sizeof(TgtRec));
  L->tkey = put((size_t)K * 4);
  L->thist = put((size_t)(L->nt_bins + 1) * 4);
  L->toff = put((size_t)(L->nt_bins + 1) * 4);
  L->tcur = put((size_t)(L->nt_bins + 1) * 4);
  L->titems = put((size_t)L->nt_items * 4 * 3);
  L->dec = put((size_t)(p.nf[0] + p.nf[1] + p.nf[2] + p.nout[0] + p.nout[1] + p.nout[2]) * 8);
  L->scan = put(scan_workspace(std::max(L->ns_keys, L->nt_bins) + 1));
  L->scan_t = put(scan_workspace(L->nt_bins + 1));   // the target sort runs beside the source side, on a stream of its own
  L->ffttab = put(fft_tables_bytes(p.n2));
  const size_t cb = p.f32 ? 8 : 16;   // bytes of a complex cell of the grids
  L->fine_bytes = (size_t)p.nf[0] * p.nf[1] * p.nf[2] * (p.real_c ? cb / 2 : cb);
  L->fine = put(L->fine_bytes);
  // FFT passes: fine -> X [nf0][nf1][nout2] -> Y [nf0][nout1][nout2] -> X [nout0][nout1][nout2]
  const size_t xa = (size_t)p.nf[0] * p.nf[1] * p.nout[2], xc = (size_t)p.nout[0] * p.nout[1] * p.nout[2];
  L->bufx = put(std::max(xa, xc) * cb);
  L->bufy = put((size_t)p.nf[0] * p.nout[1] * p.nout[2] * cb);
  L->total = o;
  return SFD_OK;
}

}  // namespace
}  // namespace sfd

// ================================================================================================================
namespace sfd {
namespace {

// (w/2) phihat(kappa) = (w/2) * 2 int_0^1 phi(z) cos(kappa z) dz; with z = sin(theta) the integrand
// exp(beta (cos(theta) - 1)) cos(kappa sin(theta)) cos(theta) is analytic on [0, pi/2] and 64 Gauss-Legendre nodes
// in long double give it to ~1e-18.  Sampled at the Chebyshev nodes of y = 2 (kappa/kmax)^2 - 1 and turned into the
// Chebyshev coefficients that the device evaluates (nufft3.cuh ChebTable).
long double half_w_phihat_host(const N3Params& p, const std::vector<long double>& gt, const std::vector<long double>& gw,
                               long double kappa) {
  const long double pi = 3.14159265358979323846264338327950288L;
  long double acc = 0.0L;
  for (size_t i = 0; i < gt.size(); ++i) {
    const long double th = (gt[i] + 1.0L) * pi / 4.0L;
    const long double om = gw[i] * pi / 4.0L;
    acc += (long double)p.w * om * cosl(th) * expl((long double)p.beta * (cosl(th) - 1.0L)) * cosl(kappa * sinl(th));
  }
  return acc;
}

void make_cheb(const N3Params& p, ChebTable* t) {
  const int nq = 64;
  std::vector<long double> gt, gw;
  gauss_legendre_host(nq, gt, gw);
  const long double pi = 3.14159265358979323846264338327950288L;
  const long double kmax = (long double)p.w * pi / 4.0L * (1.0L + 1e-9L);
  const int n = kChebN;
  std::vector<long double> fv(n);
  for (int k = 0; k < n; ++k) {
    const long double y = cosl(pi * (2 * k + 1) / (2.0L * n));
    fv[k] = half_w_phihat_host(p, gt, gw, kmax * sqrtl((y + 1.0L) / 2.0L));
  }
  for (int j = 0; j < n; ++j) {
    long double acc = 0.0L;
    for (int k = 0; k < n; ++k) acc += fv[k] * cosl(j * pi * (2 * k + 1) / (2.0L * n));
    t->c[j] = (double)(acc * (j == 0 ? 1.0L : 2.0L) / n);
  }
  t->inv_kmax2_x2 = (double)(2.0L / (kmax * kmax));
}

// Piecewise-polynomial kernel table (nufft3.cuh footprint()): on interval i the function s -> phi((t + i - w/2) 2/w),
// t = (s+1)/2, is interpolated at the deg+1 Chebyshev nodes of [-1,1] (discrete Chebyshev transform in long double)
// and converted to monomial coefficients by the T_j recurrence (|coefficients| <= 1: Horner in fp64 is accurate to
// ~1e-15).  tab[q * kPolyStride + i] = coefficient of s^q.
void make_poly(const N3Params& p, double* tab) {
  const int n = p.deg + 1;
  const long double pi = 3.14159265358979323846264338327950288L;
  std::vector<long double> x(n), fx(n), co(n);
  std::vector<std::vector<long double>> T(n, std::vector<long double>(n, 0.0L));
  T[0][0] = 1.0L;
  if (n > 1) T[1][1] = 1.0L;
  for (int j = 2; j < n; ++j) {
    for (int q = 1; q < n; ++q) T[j][q] = 2.0L * T[j - 1][q - 1];
    for (int q = 0; q < n; ++q) T[j][q] -= T[j - 2][q];
  }
  for (int k = 0; k < n; ++k) x[k] = cosl(pi * (2 * k + 1) / (2.0L * n));
  for (int i = 0; i < (kMaxDeg + 1) * kPolyStride; ++i) tab[i] = 0.0;
  for (int i = 0; i < p.w; ++i) {
    for (int k = 0; k < n; ++k) {
      const long double z = ((x[k] + 1.0L) / 2.0L + i - p.w / 2.0L) * 2.0L / p.w;
      const long double a = 1.0L - z * z;
      fx[k] = expl((long double)p.beta * (sqrtl(a > 0 ? a : 0.0L) - 1.0L));
    }
    for (int j = 0; j < n; ++j) {
      long double acc = 0.0L;
      for (int k = 0; k < n; ++k) acc += fx[k] * cosl(j * pi * (2 * k + 1) / (2.0L * n));
      co[j] = acc * (j == 0 ? 1.0L : 2.0L) / n;
    }
    for (int q = 0; q < n; ++q) {
      long double m = 0.0L;
      for (int j = q; j < n; ++j) m += co[j] * T[j][q];
      tab[q * kPolyStride + i] = (double)m;
    }
  }
}

// host-side tables are pure functions of (w, beta): computed once per width (long-double work, ~ms), then reused
void width_tables(const N3Params& p, ChebTable* quad, double* h_ptab) {
  struct WidthTables {
    bool ready = false;
    double beta = 0.0;
    ChebTable cheb;
    double poly[(kMaxDeg + 1) * kPolyStride];
  };
  static WidthTables wt_cache[kMaxW + 1];
  static std::mutex wt_mu;
  std::lock_guard<std::mutex> lk(wt_mu);
  WidthTables& wt = wt_cache[p.w];
  if (!wt.ready || wt.beta != p.beta) {
    make_cheb(p, &wt.cheb);
    make_poly(p, wt.poly);
    wt.beta = p.beta;
    wt.ready = true;
  }
  *quad = wt.cheb;
  std::memcpy(h_ptab, wt.poly, sizeof(wt.poly));
}

// Work items of the spreader and the spread itself (shared by the type-3 and the type-1 transform).
int items_and_spread(const N3Params& p, int64_t J, int64_t ns_bins, int64_t ns_keys, int64_t ns_items, int32_t* hist,
                     int32_t* off, int32_t* tmp, int32_t* sitems, int32_t* d_ctl, void* scan_w, size_t scan_b,
                     const double* ptab, const SrcRec* src, double* fine, size_t fine_bytes, cudaStream_t st,
                     const std::function<int()>& before_spread = nullptr) {
  if (p.fine == 2) {
    // one item per run of equal footprints (hist / off are the per-footprint tables), cut at spread_runs_cap()
    SFD_TRY(make_items(hist, off, ns_keys, spread_runs_cap(), tmp, sitems, ns_items, d_ctl + 0, scan_w, scan_b, st));
    prof_mark("src_sort", st);
    SFD_CUDA_TRY(cudaMemsetAsync(fine, 0, fine_bytes, st));
    if (before_spread) SFD_TRY(before_spread());
    SFD_TRY(spread_runs(p, ptab, src, sitems, sitems + ns_items, sitems + 2 * ns_items, d_ctl + 0, d_ctl + 2, fine, st));
    prof_mark("spread", st);
    return SFD_OK;
  }
  // items of <= cap sources: 1024 normally; when the sources crowd into few bins (the paper's lattice variant maps
  // 2e7 atoms onto ~60^3 cells, "highly clustered") larger slices keep the number of subgrid write-backs --
  // global fp64 reductions onto the same few cells -- proportional to the SM count instead of to J
  const int src_cap = (int)std::max<int64_t>(kSrcCap, J / ((int64_t)num_sms() * 8));
  SFD_TRY(make_items(hist, off, ns_bins, src_cap, tmp, sitems, ns_items, d_ctl + 0, scan_w, scan_b, st));
  prof_mark("src_sort", st);
  SFD_CUDA_TRY(cudaMemsetAsync(fine, 0, fine_bytes, st));
  if (before_spread) SFD_TRY(before_spread());
  SFD_TRY(spread(p, ptab, src, sitems, sitems + ns_items, sitems + 2 * ns_items, d_ctl + 0, d_ctl + 2, fine, st));
  prof_mark("spread", st);
  return SFD_OK;
}

}  // namespace

int nufft3_release_cache() { return SFD_OK; }   // nothing is cached on the device any more

int nufft3_sizes(int64_t J, int64_t K, const double X[3], const double S[3], double eps, Nufft3Sizes* out, bool real_only) {
  SFD_REQUIRE(X && S && out, SFD_ERR_NULL, "nufft3_sizes: NULL argument");
  // the call recomputes the extents from the data; the query leaves room for their rounding
  double Xi[3], Si[3];
  for (int d = 0; d < 3; ++d) {
    Xi[d] = X[d] * (1.0 + 1e-6);
    Si[d] = S[d] * (1.0 + 1e-6);
  }
  size_t total = 0;
  N3Params p{};
  // whether the strengths stay real is only known from the data, unless the caller knows the targets to be centred at
  // the origin (the distance calls: real_only)
  for (int real_c = real_only ? 1 : 0; real_c < 2; ++real_c) {
    // (the call decides on the wider kernel from the data's own extents: near the threshold size for both)
    bool near = false;
    for (int d = 0; d < 3; ++d) near = near || (X[d] * S[d] < 1.01 && X[d] * S[d] > 0.98);
    for (int pass = 0; pass < (near ? 2 : 1); ++pass) {
      SFD_TRY(make_params(Xi, Si, eps, real_c != 0, pass == 0 ? J : 0, &p));
      choose_sort(&p, J, true);
      Layout L;
      SFD_TRY(make_layout(p, J, K, &L));
      total = std::max(total, L.total);
    }
    SFD_TRY(make_params(Xi, Si, eps, real_c != 0, J, &p));
  }
  out->w = p.w;
  out->beta = p.beta;
  for (int d = 0; d < 3; ++d) {
    out->nf[d] = p.nf[d];
    out->n2[d] = p.n2[d];
    out->nout[d] = p.nout[d];
  }
  out->work_bytes = total;
  return SFD_OK;
}

}  // namespace sfd

// ================================================================================================================
namespace sfd {

namespace {
// The target sort (A5-7) depends on the geometry only, not on the source side, and is bandwidth-light work that fits beside
// the spreader (LSU-bound) and the FFT passes: it runs on a second stream, forked from the caller's stream once the geometry
// is known and joined before the interpolation.  One stream and two events per host thread and device, created on first use.
struct SideStream {
  cudaStream_t s = nullptr;
  cudaEvent_t fork = nullptr, join = nullptr;
  int dev = -1;
};
int side_stream(SideStream** out) {
  static thread_local SideStream side;
  int dev = 0;
  SFD_CUDA_TRY(cudaGetDevice(&dev));
  if (side.dev != dev) {
    // (a stream of another device is left alone: the thread may come back to it)
    side = SideStream{};
    SFD_CUDA_TRY(cudaStreamCreateWithFlags(&side.s, cudaStreamNonBlocking));
    SFD_CUDA_TRY(cudaEventCreateWithFlags(&side.fork, cudaEventDisableTiming));
    SFD_CUDA_TRY(cudaEventCreateWithFlags(&side.join, cudaEventDisableTiming));
    side.dev = dev;
  }
  *out = &side;
  return SFD_OK;
}
// Leaves no work of the second stream unordered with the caller's stream, whichever way the function returns (an error
// between fork and join included: the caller may free the workspace as soon as its own stream has drained).
struct SideJoin {
  SideStream* side = nullptr;
  cudaStream_t st = nullptr;
  bool forked = false;
  ~SideJoin() {
    if (!forked) return;
    if (cudaEventRecord(side->join, side->s) == cudaSuccess) cudaStreamWaitEvent(st, side->join, 0);
  }
};
}  // namespace

int nufft3(const double* d_x, const double* d_w, int64_t J, const double* d_xi, int64_t K, double eps, double* d_nuhat,
           void* d_work, size_t work_bytes, cudaStream_t st, bool origin_centred, const ExtentHint* hint) {
  if (K == 0) return SFD_OK;
  SFD_REQUIRE(J > 0, SFD_ERR_INVALID_ARG, "nufft3: J must be > 0 (the caller handles J == 0)");
  SFD_REQUIRE(d_work && work_bytes >= kMiscBytes, SFD_ERR_WORKSPACE_TOO_SMALL,
              "type-3 NUFFT needs a workspace (sfd_surface_ft_workspace), got %zu bytes", work_bytes);
  char* base = static_cast<char*>(d_work);
  double* d_bounds = reinterpret_cast<double*>(base);
  int32_t* d_ctl = reinterpret_cast<int32_t*>(base + 128);
  double* d_scratch = reinterpret_cast<double*>(base + 1024);

  // A5-1: extents of sources and targets (the one host synchronisation of the transform); a caller that knows a
  // hull of the sources or the reach of the targets saves the pass over all of them
  const bool hull = hint && hint->d_hull && hint->n_hull > 0;
  const bool reach_known = hint && hint->target_reach > 0.0;
  SFD_TRY(bounds_minmax(hull ? hint->d_hull : d_x, hull ? hint->n_hull : J, d_bounds, d_scratch, st));
  if (!reach_known) SFD_TRY(bounds_minmax(d_xi, K, d_bounds + 6, d_scratch, st));
  double hb[12];
  SFD_CUDA_TRY(cudaMemcpyAsync(hb, d_bounds, (reach_known ? 6 : 12) * sizeof(double), cudaMemcpyDeviceToHost, st));
  SFD_CUDA_TRY(cudaStreamSynchronize(st));
  if (reach_known)
    for (int d = 0; d < 3; ++d) {
      hb[6 + d] = -hint->target_reach;
      hb[9 + d] = hint->target_reach;
    }
  prof_mark("bounds", st);

  N3Params p{};
  double X[3], S[3];
  bool real_c = true;
  for (int d = 0; d < 3; ++d) {
    SFD_REQUIRE(std::isfinite(hb[d]) && std::isfinite(hb[3 + d]) && std::isfinite(hb[6 + d]) && std::isfinite(hb[9 + d]),
                SFD_ERR_INVALID_ARG, "type-3 NUFFT: non-finite source or target coordinate");
    p.C[d] = 0.5 * (hb[d] + hb[3 + d]);
    X[d] = (0.5 * (hb[3 + d] - hb[d])) * (1.0 + 1e-12) + 1e-300;
    p.D[d] = 0.5 * (hb[6 + d] + hb[9 + d]);
    S[d] = (0.5 * (hb[9 + d] - hb[6 + d])) * (1.0 + 1e-12) + 1e-300;
    // targets centred at the origin up to rounding (the ball quadrature): snap D to 0 so that c'_j = w_j is real
    const double reach = std::fmax(std::fabs(hb[6 + d]), std::fabs(hb[9 + d]));
    if (origin_centred || std::fabs(p.D[d]) <= 1e-9 * reach) {
      p.D[d] = 0.0;
      S[d] = reach * (1.0 + 1e-12) + 1e-300;
    } else {
      real_c = false;
    }
  }
  const bool f32 = grid_f32();
  SFD_REQUIRE(!f32 || eps >= 1e-6, SFD_ERR_INVALID_ARG,
              "single-precision grids (sfd_set_grid_precision(32)) carry tolerances eps >= 1e-6 only, got %g", eps);
  SFD_TRY(make_params(X, S, eps, real_c, J, &p, f32));
  choose_sort(&p, J);
  Layout L;
  SFD_TRY(make_layout(p, J, K, &L));
  SFD_REQUIRE(work_bytes >= L.total, SFD_ERR_WORKSPACE_TOO_SMALL,
              "type-3 NUFFT (w=%d, fine grid %dx%dx%d) needs %zu workspace bytes, got %zu", p.w, p.nf[0], p.nf[1], p.nf[2],
              L.total, work_bytes);
  ChebTable quad;
  double h_ptab[(kMaxDeg + 1) * kPolyStride];
  width_tables(p, &quad, h_ptab);
  double* ptab = reinterpret_cast<double*>(base + L.ptab);
  SFD_CUDA_TRY(cudaMemcpyAsync(ptab, h_ptab, sizeof(h_ptab), cudaMemcpyHostToDevice, st));
  SrcRec* src = reinterpret_cast<SrcRec*>(base + L.src);
  TgtRec* tgt = reinterpret_cast<TgtRec*>(base + L.tgt);
  int32_t* skey = reinterpret_cast<int32_t*>(base + L.skey);
  int32_t* shist = reinterpret_cast<int32_t*>(base + L.shist);
  int32_t* soff = reinterpret_cast<int32_t*>(base + L.soff);
  int32_t* scur = reinterpret_cast<int32_t*>(base + L.scur);
  int32_t* sitems = reinterpret_cast<int32_t*>(base + L.sitems);
  int32_t* tkey = reinterpret_cast<int32_t*>(base + L.tkey);
  int32_t* thist = reinterpret_cast<int32_t*>(base + L.thist);
  int32_t* toff = reinterpret_cast<int32_t*>(base + L.toff);
  int32_t* tcur = reinterpret_cast<int32_t*>(base + L.tcur);
  int32_t* titems = reinterpret_cast<int32_t*>(base + L.titems);
  double* dec = reinterpret_cast<double*>(base + L.dec);
  double* fine = reinterpret_cast<double*>(base + L.fine);
  double* bufx = reinterpret_cast<double*>(base + L.bufx);
  double* bufy = reinterpret_cast<double*>(base + L.bufy);
  void* scan_w = base + L.scan;
  const size_t scan_b = L.scan_t - L.scan;
  const size_t fine_bytes = L.fine_bytes;

  // A5-7: rescale and bin-sort the targets
  auto target_sort = [&](cudaStream_t ts, void* sw, size_t sb) -> int {
    SFD_CUDA_TRY(cudaMemsetAsync(thist, 0, (size_t)(L.nt_bins + 1) * 4, ts));
    SFD_CUDA_TRY(cudaMemsetAsync(tcur, 0, (size_t)(L.nt_bins + 1) * 4, ts));
    SFD_TRY(target_keys(p, d_xi, K, tkey, thist, ts));
    SFD_TRY(exclusive_scan_i32(thist, toff, L.nt_bins, nullptr, sw, sb, ts));
    SFD_TRY(target_scatter(p, d_xi, K, tkey, toff, tcur, tgt, ts));
    // slices of a crowded bin each stage the bin's subgrid again: larger slices when there are enough targets to keep
    // every SM busy (measured: interp -15 % at config 3 with 4096, +25 % at config 2 where 4096 leaves SMs idle)
    const int tgt_cap = (int)std::min<int64_t>(4096, std::max<int64_t>(kTgtCap, K / ((int64_t)num_sms() * 4)));
    return make_items(thist, toff, L.nt_bins, tgt_cap, tcur, titems, L.nt_items, d_ctl + 1, sw, sb, ts);
  };
  const char* no_overlap = std::getenv("SFD_NO_OVERLAP");   // A-B measurements: everything on the caller's stream
  const bool overlap = !(no_overlap && no_overlap[0] == '1');
  SideStream* side = nullptr;
  SideJoin side_join;

  // A5-2/A5-3: rescale, pre-phase and bin-sort the sources
  SFD_CUDA_TRY(cudaMemsetAsync(shist, 0, (size_t)(L.ns_keys + 1) * 4, st));
  SFD_CUDA_TRY(cudaMemsetAsync(scur, 0, (size_t)(L.ns_keys + 1) * 4, st));
  SFD_TRY(source_keys(p, d_x, J, skey, shist, st));
  SFD_TRY(exclusive_scan_i32(shist, soff, L.ns_keys, nullptr, scan_w, scan_b, st));
  SFD_TRY(source_scatter(p, d_x, d_w, J, skey, soff, scur, src, st));
  if (p.fine == 1) {   // per-bin ranges out of the per-footprint ones
    int32_t* bh = reinterpret_cast<int32_t*>(base + L.sbhist);
    int32_t* bo = reinterpret_cast<int32_t*>(base + L.sboff);
    SFD_TRY(source_bin_ranges(p, soff, L.ns_bins, J, bh, bo, st));
    shist = bh;
    soff = bo;
  }
  // A5-4: work items and spread.  The fork sits between the zero-fill and the spreader's launch: the target sort's kernels
  // fill the machine on their own, so made eligible any earlier they only run ahead of the source side; from here on they
  // share the SMs with the spreader's persistent CTAs (no shared memory, few registers) and with the FFT passes.
  auto fork = [&]() -> int {
    if (!overlap) return SFD_OK;
    SFD_TRY(side_stream(&side));
    SFD_CUDA_TRY(cudaEventRecord(side->fork, st));
    SFD_CUDA_TRY(cudaStreamWaitEvent(side->s, side->fork, 0));
    side_join.side = side;
    side_join.st = st;
    side_join.forked = true;
    return SFD_OK;
  };
  SFD_TRY(items_and_spread(p, J, L.ns_bins, L.ns_keys, L.ns_items, shist, soff, scur, sitems, d_ctl, scan_w, scan_b, ptab,
                           src, fine, fine_bytes, st, fork));
  if (overlap) {   // (submitted behind the spreader)
    SFD_TRY(target_sort(side->s, base + L.scan_t, L.ffttab - L.scan_t));
    SFD_CUDA_TRY(cudaEventRecord(side->join, side->s));
  }

  // A5-5 + A5-6: deconvolution folded into the first of three pruned 1-D FFT passes (timed on its own)
  SFD_TRY(deconv_tables(p, quad, dec, st));
  FftTables ft;
  SFD_TRY(fft_upload_tables(p.n2, base + L.ffttab, &ft, st));
  {
    const int64_t nf0 = p.nf[0], nf1 = p.nf[1], nf2 = p.nf[2], no0 = p.nout[0], no1 = p.nout[1], no2 = p.nout[2];
    (void)no0;
    FftPass A{};   // axis 2 (contiguous): rows (i0, i1) of the fine grid -> X[i0][i1][m2]
    A.N = p.n2[2]; A.n_in = p.nf[2]; A.lo = p.lo[2]; A.nout = p.nout[2];
    A.n_hi = nf0; A.n_lo = nf1;
    A.in_hi = nf1 * nf2; A.in_lo = nf2; A.in_el = 1;
    A.out_hi = nf1 * no2; A.out_lo = no2; A.out_el = 1;
    A.contig = 1; A.real_in = p.real_c; A.f32 = p.f32;
    A.dec_axis = dec + p.nf[0] + p.nf[1]; A.dec_hi = dec; A.dec_lo = dec + p.nf[0];
    SFD_TRY(fft_pass(A, ft, 2, fine, bufx, st));
    FftPass B{};   // axis 1: columns (i0, m2) of X -> Y[i0][m1][m2]
    B.N = p.n2[1]; B.n_in = p.nf[1]; B.lo = p.lo[1]; B.nout = p.nout[1];
    B.n_hi = nf0; B.n_lo = no2;
    B.in_hi = nf1 * no2; B.in_lo = 1; B.in_el = no2;
    B.out_hi = no1 * no2; B.out_lo = 1; B.out_el = no2; B.f32 = p.f32;
    // Targets inside the ball |xi| <= R (the ball rule): in inner-grid cells they fill the ellipsoid E with semi-axes
    // a_d = n2_d / 4 about the centre (the axes differ when the mesh's bounding box is not a cube).  What the
    // interpolation reads is E (+) the footprint cube of half-width w/2 + 1 cells, inside E (+) Ball(r), r = sqrt 3 times
    // that plus a cell of slack, and since E contains Ball(a_min): E (+) Ball(r) is inside (1 + r / a_min) E.  Only that
    // scaled ellipsoid of the band is computed and stored (for a cubic box this is the ball of radius a + r).  Pass B
    // stops storing the m1 outside the ellipsoid's section at its m2; pass C skips the (m1, m2) columns outside its
    // projection and stores only the m0 inside it.
    const bool ball = hint && hint->target_ball && hint->target_reach > 0.0;
    const double reach = (0.5 * p.w + 1.0) * 1.7321 + 1.0;
    const double a_min = 0.25 * std::min(p.n2[0], std::min(p.n2[1], p.n2[2]));
    const double grow = 1.0 + reach / a_min;
    if (ball) {
      B.ball = 2;
      B.ball_nb = 0;
      B.ball_ca = 0.0; B.ball_ira = 0.0;
      B.ball_cb = 0.5 * p.n2[2] - p.lo[2];
      B.ball_irb = 1.0 / (0.25 * p.n2[2] * grow);
      B.ball_ct = 0.5 * p.n2[1] - p.lo[1];
      B.ball_rt = 0.25 * p.n2[1] * grow;
    }
    // SFD_DEBUG_POISON_BAND=1 (tests): fill each pass's output buffer with NaN first, so that any cell the pruned passes
    // leave unstored and a later stage reads anyway shows up as a NaN distance (tests/test_gpu_fullsize.py)
    const char* poison_env = std::getenv("SFD_DEBUG_POISON_BAND");
    const bool poison = poison_env && poison_env[0] == '1';
    if (poison) SFD_CUDA_TRY(cudaMemsetAsync(bufy, 0xff, (size_t)p.nf[0] * p.nout[1] * p.nout[2] * (p.f32 ? 8 : 16), st));
    SFD_TRY(fft_pass(B, ft, 1, bufx, bufy, st));
    if (poison) SFD_CUDA_TRY(cudaMemsetAsync(bufx, 0xff, L.bufy - L.bufx, st));
    FftPass C{};   // axis 0: columns (m1, m2) of Y -> X[m0][m1][m2]
    C.N = p.n2[0]; C.n_in = p.nf[0]; C.lo = p.lo[0]; C.nout = p.nout[0];
    C.n_hi = 1; C.n_lo = no1 * no2;
    C.in_hi = 0; C.in_lo = 1; C.in_el = no1 * no2;
    C.out_hi = 0; C.out_lo = 1; C.out_el = no1 * no2; C.f32 = p.f32;
    if (ball) {
      C.ball = 1;
      C.ball_nb = (int)no2;
      C.ball_ca = 0.5 * p.n2[1] - p.lo[1];
      C.ball_cb = 0.5 * p.n2[2] - p.lo[2];
      C.ball_ira = 1.0 / (0.25 * p.n2[1] * grow);
      C.ball_irb = 1.0 / (0.25 * p.n2[2] * grow);
      C.ball_ct = 0.5 * p.n2[0] - p.lo[0];
      C.ball_rt = 0.25 * p.n2[0] * grow;
    }
    SFD_TRY(fft_pass(C, ft, 0, bufy, bufx, st));
  }
  prof_mark("fft", st);

  // A5-7 (enqueued above on the second stream): the interpolation waits for it
  if (overlap) {
    SFD_CUDA_TRY(cudaStreamWaitEvent(st, side->join, 0));
    side_join.forked = false;
  } else {
    SFD_TRY(target_sort(st, scan_w, scan_b));
  }
  prof_mark("tgt_sort", st);

  // A5-8: interpolate;  A5-9: post-deconvolve + post-phase
  SFD_TRY(interp(p, ptab, bufx, tgt, titems, titems + L.nt_items, titems + 2 * L.nt_items, d_ctl + 1, d_ctl + 3, d_nuhat, st));
  prof_mark("interp", st);
  SFD_TRY(post_deconv(p, quad, d_xi, K, d_nuhat, st));
  prof_mark("post", st);
  return SFD_OK;
}

}  // namespace sfd

// ================================================================================================================
// Type-1 NUFFT on the paper's lattice (eq. 3.6, eq. 3.7): nuhat(xi_m) = sum_j w_j e^{-i xi_m . x_j} at
// xi_m = 2 pi h m, m in [-M/2, M/2]^3 (nodes.cu lattice_kernel).  With x' = 2 pi h (x - C) in [-pi, pi) -- the
// rescaling x -> h x of eq. 3.7 -- the sum is a Fourier series on integer modes: spread onto a grid of N >= 2(M+1)
// points per period, FFT, keep the band |m| <= M/2, divide by the kernel's transform.  Everything is shared with the
// type-3 transform: the same sort, spread.cu and fft.cu with other geometry (the spread grid is only the n_in^3
// cells around the origin that the rescaled sources reach, the "highly clustered" case of P:236; the FFT is pruned
// to those inputs and to the band; real strengths keep the half m_2 >= 0).  No interpolation step.
namespace sfd {
namespace {

// *ok = false: the lattice is too coarse for the extent of the sources (2 pi h X >= pi up to the kernel's
// footprint: the periodic images would overlap) or the transform is too long for fft.cu -- use the type-3 path.
int make_params_lattice(const double X_in[3], const double C[3], int M, double h, double eps, int64_t J, N3Params* p,
                        bool* ok, bool f32 = false) {
  kernel_params(eps, J < kFewSources, &p->w, &p->beta);
  p->real_c = 1;
  p->f32 = f32 ? 1 : 0;
  p->zh = 1;
  p->deg = p->w + 3;
  *ok = false;
  const double hx = 2.0 * kPi * h;   // lattice step in the e^{-i xi.x} convention
  const int64_t N = next_smooth_even((int64_t)std::ceil(kSigma * (M + 1)));
  int tbp = 0;
  if (!fft_length_ok((int)N) || fft_tile((int)N, 0, &tbp) == 0 || fft_tile((int)N, 1, &tbp) == 0) return SFD_OK;
  for (int d = 0; d < 3; ++d) {
    SFD_REQUIRE(std::isfinite(X_in[d]) && X_in[d] >= 0, SFD_ERR_INVALID_ARG, "type-1 NUFFT: extents must be finite and >= 0");
    p->n2[d] = (int)N;
    p->sx[d] = hx * (double)N / (2.0 * kPi);
    const int64_t nin = 2 * (int64_t)std::ceil(X_in[d] * p->sx[d] + 0.5 * (p->w + 1)) + 2;
    if (nin > N) return SFD_OK;
    p->nf[d] = (int)nin;
    p->C[d] = C[d];
    p->D[d] = 0.0;
    p->st[d] = 0.0;
    p->kap[d] = p->w * kPi / ((double)N * hx);
    p->lo[d] = -(M / 2);
    p->nout[d] = M + 1;
    p->bt[d] = 1;
    p->nbt[d] = 1;
    p->t0[d] = 0;
  }
  p->lo[2] = 0;
  p->nout[2] = M / 2 + 1;
  spread_bins(p->w, true, p->bs);
  for (int d = 0; d < 3; ++d) p->nbs[d] = (p->nf[d] + p->bs[d] - 1) / p->bs[d];
  *ok = true;
  return SFD_OK;
}

}  // namespace

int nufft1_lattice_sizes(int64_t J, int M, double h, const double X[3], double eps, bool* applicable, size_t* bytes) {
  SFD_REQUIRE(X && applicable && bytes, SFD_ERR_NULL, "nufft1_lattice_sizes: NULL argument");
  double Xi[3];
  const double C0[3] = {0.0, 0.0, 0.0};
  for (int d = 0; d < 3; ++d) Xi[d] = X[d] * (1.0 + 1e-6);
  N3Params p{};
  SFD_TRY(make_params_lattice(Xi, C0, M, h, eps, J, &p, applicable));
  *bytes = 0;
  if (!*applicable) return SFD_OK;
  choose_sort(&p, J, true);
  Layout L;
  SFD_TRY(make_layout(p, J, 0, &L));
  *bytes = L.total;
  return SFD_OK;
}

int nufft1_lattice(const double* d_x, const double* d_w, int64_t J, int M, double h, double eps, double* d_nuhat,
                   void* d_work, size_t work_bytes, cudaStream_t st, bool* applicable, const ExtentHint* hint,
                   const MeshAtoms* mesh, Nufft1Band* band) {
  SFD_REQUIRE(J > 0 && applicable, SFD_ERR_INVALID_ARG, "nufft1_lattice: J must be > 0");
  SFD_REQUIRE(d_work && work_bytes >= kMiscBytes, SFD_ERR_WORKSPACE_TOO_SMALL,
              "type-1 NUFFT needs a workspace (sfd_surface_ft_lattice_workspace), got %zu bytes", work_bytes);
  char* base = static_cast<char*>(d_work);
  double* d_bounds = reinterpret_cast<double*>(base);
  int32_t* d_ctl = reinterpret_cast<int32_t*>(base + 128);
  double* d_scratch = reinterpret_cast<double*>(base + 1024);

  // extents: a hull the caller knows, else the mesh's vertices (the atoms are convex combinations), else the sources
  const bool hull = hint && hint->d_hull && hint->n_hull > 0;
  const double* bsrc = hull ? hint->d_hull : (mesh ? mesh->d_V : d_x);
  const int64_t nb = hull ? hint->n_hull : (mesh ? mesh->nV : J);
  SFD_TRY(bounds_minmax(bsrc, nb, d_bounds, d_scratch, st));
  double hb[6];
  SFD_CUDA_TRY(cudaMemcpyAsync(hb, d_bounds, sizeof(hb), cudaMemcpyDeviceToHost, st));
  SFD_CUDA_TRY(cudaStreamSynchronize(st));
  prof_mark("bounds", st);
  double X[3], C[3];
  for (int d = 0; d < 3; ++d) {
    SFD_REQUIRE(std::isfinite(hb[d]) && std::isfinite(hb[3 + d]), SFD_ERR_INVALID_ARG,
                "type-1 NUFFT: non-finite source coordinate");
    C[d] = 0.5 * (hb[d] + hb[3 + d]);
    X[d] = (0.5 * (hb[3 + d] - hb[d])) * (1.0 + 1e-12) + 1e-300;
    // sources centred at the origin up to rounding (a closed surface around it): snap C to 0, no post-phase
    const double reach = std::fmax(std::fabs(hb[d]), std::fabs(hb[3 + d]));
    if (std::fabs(C[d]) <= 1e-9 * reach) {
      C[d] = 0.0;
      X[d] = reach * (1.0 + 1e-12) + 1e-300;
    }
  }
  N3Params p{};
  const bool f32 = grid_f32();
  SFD_REQUIRE(!f32 || eps >= 1e-7, SFD_ERR_INVALID_ARG,
              "single-precision grids (sfd_set_grid_precision(32)) carry tolerances eps >= 1e-7 on the lattice (the paper's "
              "setting, P:238) and >= 1e-6 otherwise, got %g", eps);
  SFD_TRY(make_params_lattice(X, C, M, h, eps, J, &p, applicable, f32));
  if (!*applicable) return SFD_OK;
  choose_sort(&p, J);
  Layout L;
  SFD_TRY(make_layout(p, J, 0, &L));
  SFD_REQUIRE(work_bytes >= L.total, SFD_ERR_WORKSPACE_TOO_SMALL,
              "type-1 NUFFT (w=%d, spread grid %dx%dx%d, FFT length %d) needs %zu workspace bytes, got %zu", p.w, p.nf[0],
              p.nf[1], p.nf[2], p.n2[0], L.total, work_bytes);
  ChebTable quad;
  double h_ptab[(kMaxDeg + 1) * kPolyStride];
  width_tables(p, &quad, h_ptab);
  double* ptab = reinterpret_cast<double*>(base + L.ptab);
  SFD_CUDA_TRY(cudaMemcpyAsync(ptab, h_ptab, sizeof(h_ptab), cudaMemcpyHostToDevice, st));
  SrcRec* src = reinterpret_cast<SrcRec*>(base + L.src);
  int32_t* skey = reinterpret_cast<int32_t*>(base + L.skey);
  int32_t* shist = reinterpret_cast<int32_t*>(base + L.shist);
  int32_t* soff = reinterpret_cast<int32_t*>(base + L.soff);
  int32_t* scur = reinterpret_cast<int32_t*>(base + L.scur);
  int32_t* sitems = reinterpret_cast<int32_t*>(base + L.sitems);
  double* dec = reinterpret_cast<double*>(base + L.dec);
  double* fine = reinterpret_cast<double*>(base + L.fine);
  double* bufx = reinterpret_cast<double*>(base + L.bufx);
  double* bufy = reinterpret_cast<double*>(base + L.bufy);
  void* scan_w = base + L.scan;
  const size_t scan_b = L.scan_t - L.scan;

  // rescale (eq. 3.7) and bin-sort the sources, as in the type-3 transform
  SFD_CUDA_TRY(cudaMemsetAsync(shist, 0, (size_t)(L.ns_keys + 1) * 4, st));
  SFD_CUDA_TRY(cudaMemsetAsync(scur, 0, (size_t)(L.ns_keys + 1) * 4, st));
  double* d_rule = reinterpret_cast<double*>(base + kRuleOff);
  if (mesh) {
    SFD_REQUIRE(mesh->nF * mesh->rule == J, SFD_ERR_INVALID_ARG, "nufft1_lattice: J does not match the mesh");
    SFD_TRY(rule_table_device(mesh->rule, d_rule, st));
  }
  SFD_TRY(source_keys(p, d_x, J, skey, shist, st, mesh, d_rule));
  SFD_TRY(exclusive_scan_i32(shist, soff, L.ns_keys, nullptr, scan_w, scan_b, st));
  SFD_TRY(source_scatter(p, d_x, d_w, J, skey, soff, scur, src, st, mesh, d_rule));
  if (p.fine == 1) {   // per-bin ranges out of the per-footprint ones
    int32_t* bh = reinterpret_cast<int32_t*>(base + L.sbhist);
    int32_t* bo = reinterpret_cast<int32_t*>(base + L.sboff);
    SFD_TRY(source_bin_ranges(p, soff, L.ns_bins, J, bh, bo, st));
    shist = bh;
    soff = bo;
  }
  SFD_TRY(items_and_spread(p, J, L.ns_bins, L.ns_keys, L.ns_items, shist, soff, scur, sitems, d_ctl, scan_w, scan_b, ptab,
                           src, fine, L.fine_bytes, st));

  // three pruned FFT passes: position l = i - n_in/2 <-> x' = 2 pi l / N, output = the lattice modes
  SFD_TRY(lattice_tables(p, quad, M, dec, st));
  FftTables ft;
  SFD_TRY(fft_upload_tables(p.n2, base + L.ffttab, &ft, st));
  {
    const int64_t nf0 = p.nf[0], nf1 = p.nf[1], nf2 = p.nf[2], no1 = p.nout[1], no2 = p.nout[2];
    FftPass A{};
    A.N = p.n2[2]; A.n_in = p.nf[2]; A.lo = p.lo[2]; A.nout = p.nout[2];
    A.n_hi = nf0; A.n_lo = nf1;
    A.in_hi = nf1 * nf2; A.in_lo = nf2; A.in_el = 1;
    A.out_hi = nf1 * no2; A.out_lo = no2; A.out_el = 1;
    A.contig = 1; A.real_in = 1; A.f32 = p.f32;
    SFD_TRY(fft_pass(A, ft, 2, fine, bufx, st));
    FftPass B{};
    B.N = p.n2[1]; B.n_in = p.nf[1]; B.lo = p.lo[1]; B.nout = p.nout[1];
    B.n_hi = nf0; B.n_lo = no2;
    B.in_hi = nf1 * no2; B.in_lo = 1; B.in_el = no2;
    B.out_hi = no1 * no2; B.out_lo = 1; B.out_el = no2; B.f32 = p.f32;
    // SFD_DEBUG_POISON_BAND=1 (tests): fill each pass's output buffer with NaN first, so that any cell the pruned passes
    // leave unstored and a later stage reads anyway shows up as a NaN distance (tests/test_gpu_fullsize.py)
    const char* poison_env = std::getenv("SFD_DEBUG_POISON_BAND");
    const bool poison = poison_env && poison_env[0] == '1';
    if (poison) SFD_CUDA_TRY(cudaMemsetAsync(bufy, 0xff, (size_t)p.nf[0] * p.nout[1] * p.nout[2] * (p.f32 ? 8 : 16), st));
    SFD_TRY(fft_pass(B, ft, 1, bufx, bufy, st));
    if (poison) SFD_CUDA_TRY(cudaMemsetAsync(bufx, 0xff, L.bufy - L.bufx, st));
    FftPass C3{};
    C3.N = p.n2[0]; C3.n_in = p.nf[0]; C3.lo = p.lo[0]; C3.nout = p.nout[0];
    C3.n_hi = 1; C3.n_lo = no1 * no2;
    C3.in_hi = 0; C3.in_lo = 1; C3.in_el = no1 * no2;
    C3.out_hi = 0; C3.out_lo = 1; C3.out_el = no1 * no2; C3.f32 = p.f32;
    SFD_TRY(fft_pass(C3, ft, 0, bufy, bufx, st));
  }
  prof_mark("fft", st);

  if (!d_nuhat && band) {   // the consumer deconvolves while it reduces
    band->v = bufx;
    band->f32 = p.f32;
    band->dec = dec;
    for (int d = 0; d < 3; ++d) band->C[d] = p.C[d];
    return SFD_OK;
  }
  SFD_REQUIRE(d_nuhat, SFD_ERR_NULL, "nufft1_lattice: NULL output");
  SFD_TRY(lattice_post(p, M, h, dec, bufx, d_nuhat, st));
  prof_mark("post", st);
  return SFD_OK;
}

}  // namespace sfd
