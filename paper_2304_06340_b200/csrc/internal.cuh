// internal.cuh -- launcher interfaces between the translation units of libsfd.so (the CUDA path).
// Every function returns an sfd_status and only enqueues work on `st` unless it says otherwise.
#pragma once
#include <vector>

#include "common.cuh"
#include "direct.cuh"

namespace sfd {

// ---- mesh.cu: A1/A2 icosahedral discretization --------------------------------------
int mesh_sizes(int level, int64_t* nV, int64_t* nF, size_t* work_bytes);
int mesh_icosphere(int level, double* d_V, int32_t* d_F, void* d_work, size_t work_bytes, cudaStream_t st);

// ---- nodes.cu: A3 atoms and the ball-shaped frequency quadrature --------------
struct FreqTables {
  std::vector<double> r, wr;         // Gauss-Legendre on [0,R]
  std::vector<double> mu, st, wmu;   // Gauss-Legendre in mu = cos(theta); st = sqrt(1-mu^2)
  std::vector<double> cph, sph;      // cos/sin of phi_c = 2 pi c / n_phi
  double wph;                        // 2 pi / n_phi
};
int freq_tables(const sfd_freq_quadrature* q, double R, FreqTables& t);
// n-point Gauss-Legendre rule on [-1,1] (ascending), long double Newton iteration (host)
void gauss_legendre_host(int n, std::vector<long double>& t, std::vector<long double>& wt);
size_t freq_tables_bytes(const sfd_freq_quadrature* q);
// radial shells [a0, a1) only (a1 < 0: all of them)
// half: only the nodes with xi_3 >= 0, weights doubled (nodes.cu freq_expand: exact for real measures, even n_phi)
int freq_expand(const sfd_freq_quadrature* q, const FreqTables& t, double* d_xi, double* d_W, void* d_work,
                size_t work_bytes, cudaStream_t st, int a0 = 0, int a1 = -1, bool half = false);
int64_t freq_half_count(const sfd_freq_quadrature* q, int a0, int a1);
int rule_table_host(int rule, double* lam, double* om);
int nodes(const double* d_V, int64_t nV, const int32_t* d_F, int64_t nF, int rule, double* d_x, double* d_w,
          cudaStream_t st);

// ---- scan.cu: exclusive prefix sum of int32 counts (used by the mesh ranks and the bin sorts) -----
size_t scan_workspace(int64_t n);
// out[i] = sum_{i'<i} in[i'] (in-place allowed); total (sum of all) is written to d_total if non-NULL.
int exclusive_scan_i32(const int32_t* d_in, int32_t* d_out, int64_t n, int32_t* d_total, void* d_work,
                       size_t work_bytes, cudaStream_t st);

// ---- reduce.cu: A6 fused target-side reduction (eq. 2.7, eq. 2.14) --------------------
size_t reduce_workspace(int64_t K);
// Enqueues the reduction; the result (I, already scaled by (2 pi)^-3) lands in d_result[0] (device double,
// inside the workspace: reduce_result_ptr).
// General form: I = pref * sum_k W_k |nuhat_k - sigmahat(|xi_k|)|^2 (1 + (scale |xi_k|)^2)^-s; pref < 0 means (2 pi)^-3.
int reduce_enqueue(const double* d_nuhat, const double* d_xi, const double* d_W, int64_t K, double s, void* d_work,
                   size_t work_bytes, cudaStream_t st, double** d_result, double scale = 1.0, double pref = -1.0,
                   const double* d_nuhat2 = nullptr);   // d_nuhat2: second operand instead of sigmahat
// The same on the paper's lattice (nodes and trapezoid weights recomputed from the index, not read): 16 B per node.
int reduce_lattice_enqueue(const double* d_nuhat, int M, double xi_max, double s, void* d_work, size_t work_bytes,
                           cudaStream_t st, double** d_result, double scale, double pref);
// nodes.cu: the paper's cube lattice: xi' = 2 pi xi_ijk, W = w_ijk h^3
int lattice_expand(int M, double xi_max, double* d_xi, double* d_W, cudaStream_t st);

// ---- exact.cu: direct summation of the exact triangle transform (eq. 2.19; S:8(f) NEXT-3) ---------
size_t exact_ft_workspace(int64_t nF);
int exact_ft(const double* d_V, int64_t nV, const int32_t* d_F, int64_t nF, const double* d_xi, int64_t K, double* d_out,
             void* d_work, size_t work_bytes, cudaStream_t st);

// ---- nufft3.cu: A5 three-dimensional type-3 nonuniform FFT -------------------------------
struct Nufft3Sizes {
  int w;               // kernel width in fine-grid cells
  double beta;         // ES kernel parameter: phi(z) = exp(beta (sqrt(1-z^2) - 1))
  int64_t nf[3];       // fine (spreading) grid
  int64_t n2[3];       // inner type-2 grid (sigma2 * nf)
  int64_t nout[3];     // kept part of the inner grid per axis (pruned FFT output)
  size_t work_bytes;   // total workspace
};
// real_only: size for real strengths only (targets known to be centred at the origin: about half the grids)
int nufft3_sizes(int64_t J, int64_t K, const double X[3], const double S[3], double eps, Nufft3Sizes* out,
                 bool real_only = false);
// What a caller may know about the extents, which replaces the reductions over all sources / all targets:
//   d_hull / n_hull: device points whose bounding box contains every source (the vertices of the mesh the atoms are
//     convex combinations of);  target_reach > 0: every target lies in [-target_reach, target_reach]^3 (target_ball: in
//     the ball of that radius -- the last FFT pass then skips the columns of the band outside the ball's projection).
struct ExtentHint {
  const double* d_hull = nullptr;
  int64_t n_hull = 0;
  double target_reach = 0.0;
  bool target_ball = false;   // with target_reach: the targets lie in the ball |xi| <= target_reach, not just the cube
};
// origin_centred: take the targets' box as symmetric about the origin whatever their extents say (the half rule of
// nodes.cu freq_expand: the strengths then stay real and the Hermitian half band is used)
int nufft3(const double* d_x, const double* d_w, int64_t J, const double* d_xi, int64_t K, double eps,
           double* d_nuhat, void* d_work, size_t work_bytes, cudaStream_t st, bool origin_centred = false,
           const ExtentHint* hint = nullptr);
int nufft3_release_cache();
// api.cu: the calling thread's grid precision (sfd_set_grid_precision): true = single-precision grids
bool grid_f32();
// Type-1 NUFFT onto the lattice xi = 2 pi h m, m in [-M/2, M/2]^3 (eq. 3.6, eq. 3.7), lattice order of
// lattice_expand.  *applicable = false (and nothing enqueued): the lattice is too coarse for the sources' extent or
// too long for the in-shared-memory FFT; the caller then runs the type-3 transform on the lattice nodes.
int nufft1_lattice_sizes(int64_t J, int M, double h, const double X[3], double eps, bool* applicable, size_t* bytes);
// mesh != nullptr: the sources are the atoms of that mesh (J = nF * rule), generated inside the sort kernels; d_x and
// d_w are not read.
// d_nuhat == nullptr with band != nullptr: stop after the FFT and describe its output instead -- the Hermitian half band
// v[M+1][M+1][M/2+1] (modes m0, m1, m2 >= 0, before deconvolution), the per-axis tables 1 / ((w/2) phihat) on |m| and the
// centre C of the sources -- for a consumer that folds deconvolution and phase into its own pass (reduce.cu).
struct Nufft1Band {
  const double* v = nullptr;     // complex128 (complex64 when f32), inside the workspace
  int f32 = 0;
  const double* dec = nullptr;   // [3][M/2+1]
  double C[3] = {0.0, 0.0, 0.0};
};
struct MeshAtoms;
int nufft1_lattice(const double* d_x, const double* d_w, int64_t J, int M, double h, double eps, double* d_nuhat,
                   void* d_work, size_t work_bytes, cudaStream_t st, bool* applicable, const ExtentHint* hint = nullptr,
                   const MeshAtoms* mesh = nullptr, Nufft1Band* band = nullptr);
// reduce.cu: I on the paper's lattice straight from that band: deconvolution, e^{-i xi.C}, sigmahat, weights and the
// sum in one pass over the half band (mirror modes contribute equal terms: counted twice), nuhat never materialised.
int reduce_lattice_band_enqueue(const Nufft1Band& band, int M, double xi_max, double s, void* d_work, size_t work_bytes,
                                cudaStream_t st, double** d_result, double scale, double pref);
// nodes.cu: the rule as four columns lam0[Q], lam1[Q], lam2[Q], om[Q] (4 * rule doubles) in device memory
int rule_table_device(int rule, double* d_tab, cudaStream_t st);

}  // namespace sfd
