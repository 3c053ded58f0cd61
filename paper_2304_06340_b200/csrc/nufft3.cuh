// nufft3.cuh -- internal interfaces of the 3-D type-3 nonuniform FFT (A5; "contributions from nonuniform
// sources to nonuniform targets, which can be accelerated by the Type-3 NUFFT [18]").
// derives every formula used here.  Shared by nufft3.cu (plan, glue kernels), spread.cu and interp.cu.
#pragma once
#include "common.cuh"

namespace sfd {

constexpr int kMaxW = 16;        // widest kernel (eps = 1e-14 -> w = 15)
constexpr double kSigma = 2.0;   // upsampling factor of both the spreading and the inner type-2 step

// Everything the kernels need to know about one transform (passed by value).
struct N3Params {
  int w;              // kernel width in cells
  double beta;        // ES kernel: phi(z) = exp(beta (sqrt(1-z^2) - 1)), |z| <= 1   (P:185 refs [2,3])
  int nf[3];          // fine (spreading) grid, index i = l + nf/2 for mode l in [-nf/2, nf/2)
  int n2[3];          // inner type-2 grid (2 nf), index m <-> t = m h2 - pi
  double C[3], D[3];  // centres of the sources / of the targets
  double sx[3];       // source  -> fine-grid coordinate: u  = (x - C) sx + nf/2,   sx = sigma S / pi
  double st[3];       // target  -> inner-grid coordinate: u2 = (xi - D) st + n2/2, st = n2 / (2 sigma S)
  double kap[3];      // target  -> argument of phihat:    kappa = (xi - D) kap,    kap = w pi / (2 sigma S)
  int real_c;         // 1 when D == 0: the strengths c'_j = w_j stay real and so does the fine grid
  int bs[3], nbs[3];  // source bins: bs[0] x bs[1] x bs[2] cells (bs[2] = 8 or 16), nbs[d] = ceil(nf[d] / bs[d])
  int bt[3], nbt[3], t0[3];  // target bins (bt[0] x bt[1] x bt[2] cells) over the band [t0, t0 + nbt*bt) of the
                             // inner grid that holds every target; bt[2] is 8 or 16 (bank-conflict-free pitch)
  int deg;                   // degree of the piecewise-polynomial kernel evaluation (w + 3)
  int fine;                  // 1: inside a bin the sources are also ordered by the first cell of their footprint
                             // ((bs+1)^3 sub-keys per bin), so that sources with the same footprint are consecutive
                             // and the spreader accumulates them in registers (many sources per cell: P:236)
                             // 2: so many per cell that one warp spreads a whole run (spread.cu spread_runs_kernel)
  int lo[3], nout[3];        // band of the inner grid that is computed and stored: v[m - lo], m in [lo, lo + nout)
  int f32;                   // 1: the grids in global memory (fine grid, FFT intermediates, band) and the interpolation's
                             // subgrid are single precision (S:8(f) NEXT-4); everything else stays fp64
  int zh;                    // 1: real strengths => v is Hermitian about the centre m = n2/2 (v[c+k] = conj v[c-k]) and
                             // only the half m_2 >= n2_2/2 of the band is computed and stored (lo[2] = n2_2/2); the
                             // interpolation reads the other half by reflection (all three indices) and conjugation
};

constexpr int kMaxDeg = kMaxW + 3;
constexpr int kPolyStride = 16;   // ptab[q * kPolyStride + i]: coefficient of s^q on interval i (i < w)

struct __align__(8) SrcRec { double u[3]; double re, im; };   // sorted source: grid coordinate + strength (40 B)
struct __align__(8) TgtRec { double u[3]; int64_t k; };       // sorted target: grid coordinate + original index

// (w/2) phihat(kappa) = (w/2) 2 int_0^1 phi(z) cos(kappa z) dz, the kernel's Fourier transform that both
// deconvolutions divide by, as a Chebyshev series in y = 2 (kappa/kmax)^2 - 1 on |kappa| <= kmax = w pi / 4 (the whole
// range either deconvolution reaches at sigma = 2).  phihat is even and entire and only falls to ~0.1-0.6 of its peak
// there, so 17 coefficients reproduce it to ~1e-14 relative; coefficients come from a long-double Gauss-Legendre
// quadrature on the host (nufft3.cu make_cheb).  Evaluated by Clenshaw's recurrence: 17 FMAs instead of 2w+6 cosines.
constexpr int kChebN = 17;
struct ChebTable {
  double inv_kmax2_x2;   // 2 / kmax^2
  double c[kChebN];
};
__device__ __forceinline__ double half_w_phihat(const ChebTable& t, double kappa) {
  const double y = __fma_rn(kappa * kappa, t.inv_kmax2_x2, -1.0);
  const double y2 = y + y;
  double b1 = 0.0, b2 = 0.0;
#pragma unroll
  for (int k = kChebN - 1; k >= 1; --k) {
    const double b0 = __fma_rn(y2, b1, t.c[k] - b2);
    b2 = b1;
    b1 = b0;
  }
  return __fma_rn(y, b1, t.c[0] - b2);
}

__device__ __forceinline__ double es_kernel(double z, double beta) {
  const double t = fmax(0.0, __fma_rn(-z, z, 1.0));
  return exp(beta * (sqrt(t) - 1.0));
}

// Piecewise-polynomial evaluation of the kernel (the "Horner" evaluation of the ES-kernel papers [2,3]): for a point
// at grid coordinate u the footprint starts at i0 = ceil(u - w/2); with t = i0 - (u - w/2) in [0,1) and s = 2t - 1 the
// value on cell i0 + i is phi((t + i - w/2) 2/w) = P_i(s), a polynomial of degree p.deg per interval i whose
// coefficients (Chebyshev-node interpolants, host long double; nufft3.cu make_poly) sit in ptab.  Interior intervals
// are accurate to ~1e-15; the two edge intervals, where phi has a square-root singularity and is ~e^-beta, to
// ~0.05 eps.
__device__ __forceinline__ void footprint(double u, int w, int& i0, double& s) {
  const double lo = u - 0.5 * w;
  const double c = ceil(lo);
  i0 = (int)c;
  s = __fma_rn(2.0, c - lo, -1.0);
}

// ---- spread.cu (A5-4) ------------------------------------------------------------------------------------
// Work item i: sources [item_start[i], item_start[i]+item_count[i]) of bin item_bin[i].  *n_items on the device.
// grid is real double[nf0][nf1][nf2] (real_c) or complex double[nf0][nf1][nf2][2] -- float instead of double when
// p.f32 --; must be zero on entry.
void spread_bins(int w, bool real_c, int bs[3]);   // source-bin shape for kernel width w
size_t spread_smem_bytes(const N3Params& p);
int spread(const N3Params& p, const double* d_ptab, const SrcRec* d_src, const int32_t* d_item_bin, const int32_t* d_item_start,
           const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter, double* d_grid, cudaStream_t st);

// Clustered sources (N3Params::fine == 2): items are (key, start, count) slices of <= spread_runs_cap() sources with
// the same footprint (make_items over the per-footprint histogram); one warp per item, register accumulation.
int spread_runs_cap();
bool spread_runs_ok(int w, bool real_c);
int spread_runs(const N3Params& p, const double* d_ptab, const SrcRec* d_src, const int32_t* d_item_key,
                const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
                double* d_grid, cudaStream_t st);

// ---- interp.cu (A5-8) ------------------------------------------------------------------------------------
// v = complex double[nout_0][nout_1][nout_2][2], the band [lo, lo+nout) of the inner grid; writes G[k] (complex) for
// every sorted target.
size_t interp_smem_bytes(const N3Params& p);
void interp_bins(int w, bool f32, int bt[3]);   // target-bin shape for kernel width w (fp32 subgrids hold twice the cells)
int interp(const N3Params& p, const double* d_ptab, const double* d_v, const TgtRec* d_tgt, const int32_t* d_item_bin,
           const int32_t* d_item_start, const int32_t* d_item_count, const int32_t* d_n_items, int32_t* d_counter,
           double* d_G, cudaStream_t st);

// ---- nufft3_glue.cu: the HBM-bound one-pass kernels around spread / FFT / interp ---------------------------
constexpr int kBoundsBlocks = 296;
// (min[3], max[3]) of n points into d_out6; d_scratch holds kBoundsBlocks*6 doubles.
int bounds_minmax(const double* d_pts, int64_t n, double* d_out6, double* d_scratch, cudaStream_t st);
// A5-2/A5-3: bin key of every source + histogram; then scatter into bin order with grid coordinates and c'_j.
// mesh != nullptr: the sources are the atoms of the mesh, generated on the fly (atoms.cuh; d_x / d_w unused, d_rule = the
// rule's columns from rule_table_device).
struct MeshAtoms;
int source_keys(const N3Params& p, const double* d_x, int64_t J, int32_t* d_key, int32_t* d_hist, cudaStream_t st,
                const MeshAtoms* mesh = nullptr, const double* d_rule = nullptr);
// p.fine: keys are bin * cpb + sub-key, cpb = (bs0+1)(bs1+1)(bs2+1); after the scan of the fine histogram this
// extracts the per-bin offsets and counts that make_items wants: d_boff[b] = d_off[b cpb], d_bhist[b] = their differences.
inline int64_t source_subkeys(const N3Params& p) { return (int64_t)(p.bs[0] + 1) * (p.bs[1] + 1) * (p.bs[2] + 1); }
int source_bin_ranges(const N3Params& p, const int32_t* d_off, int64_t nbins, int64_t J, int32_t* d_bhist,
                      int32_t* d_boff, cudaStream_t st);
int source_scatter(const N3Params& p, const double* d_x, const double* d_w, int64_t J, const int32_t* d_key,
                   const int32_t* d_off, int32_t* d_cursor, SrcRec* d_out, cudaStream_t st,
                   const MeshAtoms* mesh = nullptr, const double* d_rule = nullptr);
// A5-7: same for the targets.
int target_keys(const N3Params& p, const double* d_xi, int64_t K, int32_t* d_key, int32_t* d_hist, cudaStream_t st);
int target_scatter(const N3Params& p, const double* d_xi, int64_t K, const int32_t* d_key, const int32_t* d_off,
                   int32_t* d_cursor, TgtRec* d_out, cudaStream_t st);
// Work items: every occupied bin is cut into slices of <= cap points.  d_items = int32[3][max_items] (bin, start,
// count); *d_n_items = number of items.  d_tmp holds nbins+1 int32.
int make_items(const int32_t* d_hist, const int32_t* d_off, int64_t nbins, int cap, int32_t* d_tmp, int32_t* d_items,
               int64_t max_items, int32_t* d_n_items, void* d_scan, size_t scan_bytes, cudaStream_t st);
// A5-5: dec[d][i] = (-1)^l / ((w/2) phihat(l w pi / n2_d)), l = i - nf_d/2 (applied by the first FFT pass, fft.cu).
int deconv_tables(const N3Params& p, const ChebTable& q, double* d_dec, cudaStream_t st);
// A5-9: nuhat_k = G_k e^{-i (xi_k-D).C} / prod_d (w/2) phihat((xi_kd-D_d) kap_d), in place on d_nuhat.
int post_deconv(const N3Params& p, const ChebTable& q, const double* d_xi, int64_t K, double* d_nuhat, cudaStream_t st);
// Type-1 tail (eq. 3.6): dec[d][m] = 1 / ((w/2) phihat(m w pi / n2_d)), m in [0, M/2]; then the FFT band
// v[M+1][M+1][M/2+1] (modes m0, m1, m2 >= 0) is unfolded by Hermitian symmetry into lattice order (nodes.cu
// lattice_kernel), deconvolved and multiplied by e^{-i xi.C}.
int lattice_tables(const N3Params& p, const ChebTable& q, int M, double* d_dec, cudaStream_t st);
int lattice_post(const N3Params& p, int M, double h, const double* d_dec, const double* d_v, double* d_nuhat,
                 cudaStream_t st);

}  // namespace sfd
