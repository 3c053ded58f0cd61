/* sfd.h -- C ABI of the surface-Fourier-distance library (hand-written CUDA for sm_100a, one GPU).
 *
 * The hot path of Koga, "Computing weak distance between the 2-sphere and its nonsmooth
 * approximations" (arXiv 2304.06340).  "P:n" = /root/reference/PAPER.md line n.  The variant is the
 * one BASELINE.json fixes: Fourier kernel e^{-i xi.x}, Sobolev weight
 * (1+|xi|^2)^{-s} with s > 1/2, ball-shaped frequency quadrature, symmetric triangle rules.
 *
 * Conventions for every function
 *   - extern "C"; returns an int status: SFD_OK (0) or a negative sfd_status; never throws/aborts.
 *   - "d_" pointers are DEVICE pointers, "h_" pointers are HOST pointers.  All buffers are owned by
 *     the caller; the library keeps no pointer after the call returns except for work already
 *     enqueued on `stream`.  Outputs are fully overwritten, never accumulated into.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device-pointer
 *     calls only enqueue work unless the description says "synchronises".  The type-3 transform (eps > 0) runs part of its
 *     work (the target sort) on a second, non-blocking stream that the library creates once per host thread and device;
 *     that work is ordered after everything enqueued on `stream` before the call and before everything after it (event
 *     fork / join), so to the caller the call behaves as if all of it ran on `stream`.
 *   - Every call that needs scratch memory has a *_workspace query; d_work must be 256-byte aligned.
 *   - Arrays are C-contiguous fp64 / int32: points double[n][3], complex values double[n][2] = (re,im).
 *   - NULL pointer where one is required -> SFD_ERR_NULL; out-of-range scalar -> SFD_ERR_INVALID_ARG;
 *     n == 0 (no faces / sources / targets) is valid and yields empty or zero output.
 *   - sfd_last_error() returns a thread-local, human-readable description of the last failure.
 *   - Process-global state: host-side caches of quadrature / kernel / FFT tables (pure functions of their keys), and
 *     the device's stream-ordered memory pool, in which the host-buffer entry points keep their workspaces between
 *     calls (sfd_release_cache() trims it).
 */
#ifndef SFD_H_
#define SFD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  SFD_OK = 0,
  SFD_ERR_NULL = -1,
  SFD_ERR_INVALID_ARG = -2,
  SFD_ERR_BUFFER_TOO_SMALL = -3,
  SFD_ERR_WORKSPACE_TOO_SMALL = -4,
  SFD_ERR_CUDA = -5,
  SFD_ERR_RESERVED_6 = -6, /* never returned (was a cuFFT failure code before the inner FFT became the library's own) */
  SFD_ERR_UNSUPPORTED = -7
} sfd_status;

/* Symmetric triangle quadrature rules ("more symmetric rules are available on triangles");
 * the value is the number of nodes q per face. */
typedef enum { SFD_RULE_SYM6_DEG4 = 6, SFD_RULE_SYM12_DEG6 = 12,
               /* the paper's own rule: 8-point Gauss-Legendre applied twice as an iterated integral,
                * 64 nodes per face, exact for polynomials of total degree <= 14 */
               SFD_RULE_GL8X8 = 64 } sfd_rule;

/* Ball-shaped frequency quadrature: n_r-point Gauss-Legendre in r on [0,R] x n_theta-point
 * Gauss-Legendre in mu = cos(theta) on [-1,1] x n_phi-point periodic trapezoid in phi.
 * K = n_r*n_theta*n_phi nodes, index k = (a*n_theta + b)*n_phi + c (phi fastest, mu ascending),
 * xi_k = r_a (sqrt(1-mu_b^2) cos phi_c, sqrt(1-mu_b^2) sin phi_c, mu_b), phi_c = 2 pi c / n_phi,
 * W_k = w^r_a r_a^2 w^mu_b 2 pi / n_phi. */
typedef struct { int32_t n_r, n_theta, n_phi; } sfd_freq_quadrature;

typedef void* sfd_stream; /* cudaStream_t */

const char* sfd_last_error(void);
/* Library version string and the CUDA arch it was compiled for ("sm_100a"). */
const char* sfd_version(void);
/* Returns the memory kept in the device's stream-ordered pool to the driver.  Synchronises the device. */
int sfd_release_cache(void);

/* ---- A1/A2: icosahedral discretization T_level ------------------------------------
 * T_0 = icosahedron inscribed in S^2; each step adds the midpoint of every edge, projected onto
 * S^2, and splits each face into four.  nV = 10*4^level + 2, nF = 20*4^level.
 * Vertex/face numbering is the convention of DESIGN.md reading R4 (integer output is unique).
 * level in [0,10], else SFD_ERR_INVALID_ARG.  Any of nV, nF, work_bytes may be NULL. */
int sfd_mesh_icosphere_sizes(int level, int64_t* nV, int64_t* nF, size_t* work_bytes);
int sfd_mesh_icosphere(int level, double* d_vertices /*[nV][3]*/, int32_t* d_faces /*[nF][3]*/,
                       void* d_work, size_t work_bytes, sfd_stream stream);

/* ---- A3: triangle-quadrature atoms (eqs. 3.1-3.2) -----------------------------------
 * Converts the rule {(u_i,q_i)} on the standard simplex into {(L(u_i), q_i*gamma_A)} on each face:
 * x[f*q+i] = sum_m lambda_{i,m} p_m(f),  w[f*q+i] = omega_i * area(f).  Degenerate faces give zero
 * weights.  A face index outside [0,nV) can only be seen on the device: the face's atoms are written as NaN, a
 * device-side error word is set, and the NEXT SYNCHRONISING call of the library on this device (sfd_reduce*,
 * sfd_extents, sfd_weak_distance*, sfd_mesh_distance) returns SFD_ERR_INVALID_ARG and clears the word.  The calls that
 * take a mesh and synchronise themselves (sfd_weak_distance, sfd_mesh_distance, ...) report their own bad indices. */
int sfd_nodes(const double* d_vertices, int64_t nV, const int32_t* d_faces, int64_t nF, int rule,
              double* d_x /*[nF*q][3]*/, double* d_w /*[nF*q]*/, sfd_stream stream);
/* The rule itself (host): barycentric points h_lambda[q][3] and weights h_omega[q] summing to 1. */
int sfd_rule_table(int rule, double* h_lambda, double* h_omega);

/* ---- frequency quadrature (struct above) ------------------------------------------------
 * Host version: deterministic, no GPU needed.  Device version: uploads the three 1-D tables and
 * expands them with a kernel (d_xi [K][3], d_W [K]); n_r, n_theta, n_phi >= 1 and R > 0. */
int sfd_freq_nodes(const sfd_freq_quadrature* q, double R, double* h_xi /*[K][3]*/, double* h_W /*[K]*/);
int sfd_freq_nodes_workspace(const sfd_freq_quadrature* q, size_t* bytes);
int sfd_freq_nodes_device(const sfd_freq_quadrature* q, double R, double* d_xi /*[K][3]*/, double* d_W /*[K] or NULL*/,
                          void* d_work, size_t work_bytes, sfd_stream stream);

/* The nodes of the radial shells a in [a_begin, a_end) only: (a_end - a_begin) * n_theta * n_phi nodes, in the same
 * order as the full rule (node k of the full rule is node k - a_begin*n_theta*n_phi here).  The ball rule is a sum
 * over shells, so disjoint ranges partition the quadrature: this is how the targets are sharded over GPUs (DESIGN.md
 * "Multi-GPU"; partial sums I of sfd_reduce add up).  Same workspace as sfd_freq_nodes_device. */
int sfd_freq_nodes_device_range(const sfd_freq_quadrature* q, double R, int32_t a_begin, int32_t a_end,
                                double* d_xi, double* d_W, void* d_work, size_t work_bytes, sfd_stream stream);

/* ---- A5-1 as a call of its own: bounding box of n device points (two kernels, min/max per axis) ------------------
 * h_half[d] = (max_d - min_d)/2 (with the 1e-12 relative margin the type-3 transform applies itself), h_centre[d] =
 * (max_d + min_d)/2 (may be NULL): what sfd_surface_ft_workspace / sfd_surface_ft_lattice_workspace /
 * sfd_weak_distance_workspace take as X / S / x_extent.  n == 0 gives zeros.  A non-finite coordinate ->
 * SFD_ERR_INVALID_ARG.  Synchronises `stream`. */
int sfd_extents_workspace(size_t* bytes);
int sfd_extents(const double* d_pts /*[n][3]*/, int64_t n, double h_half[3], double h_centre[3] /*or NULL*/, void* d_work,
                size_t work_bytes, sfd_stream stream);

/* ---- A4/A5: Fourier transform of the atomic measure nu = sum_j w_j delta_{x_j} -----------------
 * nuhat_k = sum_{j<J} w_j exp(-i xi_k . x_j)   (eq. 2.8 applied to the atoms of P:152).
 *   eps == 0        : fp64 direct summation, error <= 1e-12 * sum|w_j| for |xi.x| <~ 2e3.
 *   0 < eps < 1     : 3-D type-3 nonuniform FFT at tolerance eps (>= 1e-14), error
 *                     <= 10 * eps * sum|w_j|.  Synchronises `stream` once (grid sizing).  The spreader adds the
 *                     bins' subgrids into the fine grid with fp64 reductions whose order is not fixed: the result
 *                     is reproducible to rounding (~1e-16 sum|w_j|) only, not bit for bit; the direct sum is
 *                     deterministic.
 * Workspace: query with the same (J, K, eps) and bounding half-widths X[d] >= max_j|x_jd - centre_d|,
 * S[d] >= max_k|xi_kd - centre_d| (ignored for eps == 0, may then be NULL).  If the data's actual
 * extents need more than work_bytes, the call fails with SFD_ERR_WORKSPACE_TOO_SMALL and writes
 * nothing. */
int sfd_surface_ft_workspace(int64_t J, int64_t K, const double X[3], const double S[3], double eps, size_t* bytes);
/* What the type-3 transform would use for these extents: kernel width w (cells), fine (spreading) grid nf[3] and
 * inner FFT grid n2[3].  Host only; any output may be NULL. */
int sfd_surface_ft_plan(int64_t J, int64_t K, const double X[3], const double S[3], double eps, int32_t* w,
                        int64_t nf[3], int64_t n2[3]);
int sfd_surface_ft(const double* d_x /*[J][3]*/, const double* d_w /*[J]*/, int64_t J,
                   const double* d_xi /*[K][3]*/, int64_t K, double eps, double* d_nuhat /*[K][2]*/,
                   void* d_work, size_t work_bytes, sfd_stream stream);

/* ---- A4 without a workspace: for callers that cannot allocate ------------------------------------
 * The fp64 direct sum (sfd_surface_ft with eps == 0: same kernels, same fixed summation order, bit-identical
 * result) for code that may not call cudaMalloc: under CUDA graph capture, in serving loops, in harnesses that forbid it.
 * The call allocates nothing, on the host or on the device, and takes no workspace: the partial sums of the direct sum's
 * source splits go to a static device array of SFD_STATIC_SCRATCH_BYTES (16 MiB) that every GPU which loads the library
 * holds until the process exits.  Device pointers d_x [J][3], d_w [J], d_xi [K][3], d_nuhat [K][2] (owned by the caller,
 * fully overwritten); enqueues on `stream`, does not synchronise.
 *   - Sizes whose partial sums do not fit (nsplit * K * 16 bytes; nsplit <= 32 is chosen from J, K and the SM count, 1 for
 *     large K) are rejected with SFD_ERR_UNSUPPORTED and a message naming the sizes; nothing is written.
 *     sfd_surface_ft_direct_static_scratch reports the bytes a (J, K) needs (host only; needs a CUDA device for the SM
 *     count, 148 SMs assumed otherwise); any K fits when that is 0.
 *   - The array is shared by every call on a device and keeps the last call's contents; every entry a call reads it has
 *     written itself, so nothing needs clearing.  Calls that OVERLAP on the GPU (other streams, graphs replayed
 *     concurrently) race on it and give wrong results: keep them on one stream or order them with events.
 *   - J == 0 gives zeros, K == 0 does nothing; NULL buffers -> SFD_ERR_NULL. */
#define SFD_STATIC_SCRATCH_BYTES (16u << 20)
int sfd_surface_ft_direct_static_scratch(int64_t J, int64_t K, size_t* bytes);
int sfd_surface_ft_direct_static(const double* d_x /*[J][3]*/, const double* d_w /*[J]*/, int64_t J,
                                 const double* d_xi /*[K][3]*/, int64_t K, double* d_nuhat /*[K][2]*/,
                                 sfd_stream stream);

/* ---- A6: fused target-side reduction (eq. 2.7 with P:55 eq. 2.5; eq. 2.14) ----------
 * I = (2 pi)^-3 sum_k W_k |nuhat_k - sigmahat(xi_k)|^2 (1+|xi_k|^2)^-s,  sigmahat = 4 pi sin|xi|/|xi|
 * (the unit sphere's transform).  Deterministic compensated fp64 sum.  s > 0.5, else
 * SFD_ERR_INVALID_ARG.  Writes I to *h_I; synchronises `stream`.  Workspace: sfd_reduce_workspace. */
int sfd_reduce_workspace(int64_t K, size_t* bytes);
int sfd_reduce(const double* d_nuhat /*[K][2]*/, const double* d_xi /*[K][3]*/, const double* d_W /*[K]*/,
               int64_t K, double s, void* d_work, size_t work_bytes, sfd_stream stream, double* h_I);

/* ---- whole path: mesh -> atoms -> nuhat on the ball quadrature -> sqrt(I) -----------------------
 * Distance in H^{-s} between the mesh's surface measure and the unit sphere's.  Runs A3,
 * the frequency quadrature, A4 (eps == 0) or A5 (eps > 0) and A6 on `stream`; synchronises; writes
 * sqrt(I) to *h_distance and I to *h_I (either may be NULL).  R > 0, s > 0.5.
 * The ball rule is symmetric under xi -> -xi when n_phi is even (Gauss-Legendre nodes in cos(theta) are symmetric and
 * phi + pi is a node), the surface measure is real, so nuhat(-xi) = conj nuhat(xi), and sigmahat is real and radial:
 * mirror nodes contribute equal terms to I.  The call therefore generates, transforms and reduces only the
 * sfd_weak_distance_targets(q) nodes with xi_3 >= 0, with doubled weights (a ring at cos(theta) = 0 keeps its own) --
 * the same I up to rounding, half the work.  An odd n_phi uses every node.
 * The workspace is sized for meshes whose bounding box has half-width <= x_extent on every axis (1.0 for an
 * icosphere; only used when eps > 0); a wider mesh fails with SFD_ERR_WORKSPACE_TOO_SMALL. */
int sfd_weak_distance_workspace(int64_t nF, int rule, const sfd_freq_quadrature* q, double R, double eps,
                                double x_extent, size_t* bytes);
int sfd_weak_distance(const double* d_vertices, int64_t nV, const int32_t* d_faces, int64_t nF, int rule,
                      double s, double R, const sfd_freq_quadrature* q, double eps, void* d_work,
                      size_t work_bytes, sfd_stream stream, double* h_distance, double* h_I);
/* Number of frequency nodes sfd_weak_distance evaluates for the rule q (host-only): n_r ceil(n_theta/2) n_phi when
 * n_phi is even, n_r n_theta n_phi otherwise. */
int sfd_weak_distance_targets(const sfd_freq_quadrature* q, int64_t* K_eval);

/* The same distance restricted to the radial shells a in [a_begin, a_end) of the rule (as sfd_freq_nodes_device_range):
 * the ball rule is a sum over shells, every nuhat_k is its own sum over the atoms, so disjoint ranges give
 * partial sums I_r that add up to I -- the unit of work of a multi-GPU run (one range per GPU, one all-reduce of the
 * result).  Same half rule, same fast paths as sfd_weak_distance; the transform's grids are
 * sized by the range's own largest radius r_{a_end-1}, so inner ranges are cheaper.  Nothing crosses to the host: the
 * partial sum is left in DEVICE memory as a compensated pair, d_partial[0] = sum, d_partial[1] = compensation,
 * I_r = d_partial[0] + d_partial[1] (already scaled by (2 pi)^-3); add pairs component-wise.  A face index outside
 * [0, nV) makes d_partial[0] NaN.  a_begin == a_end gives (0, 0).  Enqueues on `stream` after the one synchronisation
 * of the transform's sizing (eps > 0). */
int sfd_weak_distance_range_workspace(int64_t nF, int rule, const sfd_freq_quadrature* q, double R, int32_t a_begin,
                                      int32_t a_end, double eps, double x_extent, size_t* bytes);
int sfd_weak_distance_range(const double* d_vertices, int64_t nV, const int32_t* d_faces, int64_t nF, int rule, double s,
                            double R, const sfd_freq_quadrature* q, int32_t a_begin, int32_t a_end, double eps,
                            void* d_work, size_t work_bytes, sfd_stream stream, double* d_partial /*[2], device*/);

/* ---- the paper's own variant: cube lattice, trapezoidal rule, its norm convention ----
 * Lattice of P:156-166 eqs. 3.3-3.4: xi_ijk = (i,j,k) h, h = 2 xi_max / M, i,j,k = -M/2..M/2 (M even, 2..2046), with
 * trapezoid weights w_ijk h^3 (1 inside, 1/2 faces, 1/4 edges, 1/8 corners).  K = (M+1)^3, node index
 * ((i+M/2)(M+1) + (j+M/2))(M+1) + (k+M/2).  The paper's transform is e^{-2 pi i xi.x} (eq. 2.1); this library
 * evaluates e^{-i xi'.x}, so the nodes are written as xi' = 2 pi xi and can be passed to sfd_surface_ft as they are;
 * the weights stay in the paper's units (d xi). */
int sfd_lattice_nodes(int32_t M, double xi_max, double* h_xi /*[K][3]*/, double* h_W /*[K]*/);
int sfd_lattice_nodes_device(int32_t M, double xi_max, double* d_xi /*[K][3]*/, double* d_W /*[K] or NULL*/,
                             sfd_stream stream);
/* General form of A6: I = prefactor * sum_k W_k |nuhat_k - sigmahat(|xi_k|)|^2 (1 + (xi_scale |xi_k|)^2)^-s.
 * sfd_reduce is xi_scale = 1, prefactor = (2 pi)^-3; the paper's norm (eq. 2.7, exponent s_paper < -1/2) on
 * lattice nodes xi' = 2 pi xi is xi_scale = 1/(2 pi), s = -s_paper, prefactor = 1.  s > 0.5.  Synchronises. */
int sfd_reduce_ex(const double* d_nuhat, const double* d_xi, const double* d_W, int64_t K, double s, double xi_scale,
                  double prefactor, void* d_work, size_t work_bytes, sfd_stream stream, double* h_I);
/* sfd_reduce_ex on the lattice of sfd_lattice_nodes without reading it: nodes and trapezoid weights are recomputed from
 * the index with the same roundings, so the result equals sfd_reduce_ex on the expanded lattice bit for bit; 16 B of
 * traffic per node instead of 48.  d_nuhat complex128 [(M+1)^3] in lattice order; M even, 2..1624.  Synchronises. */
int sfd_reduce_lattice(const double* d_nuhat, int32_t M, double xi_max, double s, double xi_scale, double prefactor,
                       void* d_work, size_t work_bytes, sfd_stream stream, double* h_I);
/* nuhat on the lattice of sfd_lattice_nodes (same node order) -- the transform the paper itself runs (eq. 3.6:
 * type-1 NUFFT, nonuniform sources -> integer modes, after the rescaling x -> h x of P:188 eq. 3.7).  eps > 0: type-1
 * NUFFT (sort, spread, pruned FFT whose output band IS the lattice, deconvolution; no interpolation step); when the
 * lattice is too coarse for the sources' extent (2 pi h max|x - centre| close to pi: the periodic images would
 * overlap) or eps == 0, the lattice nodes are expanded in the workspace and the call runs sfd_surface_ft on them
 * (type-3 / direct sum).  X[3] in the workspace query: upper bounds of the half-extents of the sources per axis.
 * Device pointers; d_nuhat complex128 [K = (M+1)^3]; enqueues on `stream` after one synchronisation (the extents).
 * Errors as sfd_surface_ft. */
int sfd_surface_ft_lattice_workspace(int64_t J, int32_t M, double xi_max, const double X[3], double eps, size_t* bytes);
int sfd_surface_ft_lattice(const double* d_x, const double* d_w, int64_t J, int32_t M, double xi_max, double eps,
                           double* d_nuhat, void* d_work, size_t work_bytes, sfd_stream stream);
/* ||mu - sigma||_{H_s(R^3)} of P:65 eq. 2.7 for the mesh's surface measure mu against the unit sphere's, by the
 * paper's quadrature: atoms (rule 64 = the paper's) -> transform on the lattice (sfd_surface_ft_lattice: eps == 0
 * direct sum, eps > 0 type-1 NUFFT) -> trapezoidal rule.  s_paper < -1/2.
 * M even, 2..1624 (the reduction's 32-bit node index; the workspace query rejects larger M too).
 * Writes the norm to *h_norm and its square to *h_I.  Synchronises. */
int sfd_weak_distance_lattice_workspace(int64_t nF, int rule, int32_t M, double xi_max, double eps, double x_extent,
                                        size_t* bytes);
int sfd_weak_distance_lattice(const double* d_vertices, int64_t nV, const int32_t* d_faces, int64_t nF, int rule,
                              double s_paper, double xi_max, int32_t M, double eps, void* d_work, size_t work_bytes,
                              sfd_stream stream, double* h_norm, double* h_I);

/* ---- exact transform of the flat mesh -------------------------------------------------------
 * out_k = sum_f int_{Q_f} e^{-i xi_k.x} dS(x): the sum over the mesh's triangles of P:128 eq. 2.19 (e^{-i xi.x}
 * convention, gamma = 2 area), the O(N_S N_F) direct summation of the prior art, evaluated as a second
 * divided difference of exp so that no configuration -- xi orthogonal to an edge, xi along the normal, xi = 0, tiny
 * faces -- loses accuracy (P:140 names the cancellation of the literal formula): ~1e-15 sum_f area_f absolute, plus the
 * fp64 rounding of the phases xi.p.  No quadrature rule is involved; against sfd_nodes + sfd_surface_ft it isolates
 * the triangle rule's error.  Device pointers; d_out complex128 [K]; a face with a vertex index outside [0, nV)
 * poisons every output with NaN and is reported by the next synchronising call (as for sfd_nodes).  d_work: sfd_exact_ft_workspace(nF) bytes (80 B per face).
 * With few frequencies the faces are split over CTAs and the partial sums meet in fp64 reductions whose order is not
 * fixed (reproducible to rounding only).  Enqueues on `stream`. */
int sfd_exact_ft_workspace(int64_t nF, size_t* bytes);
int sfd_exact_ft(const double* d_vertices /*[nV][3]*/, int64_t nV, const int32_t* d_faces /*[nF][3]*/, int64_t nF,
                 const double* d_xi /*[K][3]*/, int64_t K, double* d_out /*[K][2]*/, void* d_work, size_t work_bytes,
                 sfd_stream stream);

/* ---- two meshes against each other ------------------------------------------------------------------
 * I = (2 pi)^-3 sum_k W_k |nuhat_a,k - nuhat_b,k|^2 (1+|xi_k|^2)^-s: the squared H^{-s} distance between two atomic
 * measures whose transforms on the same nodes are given (two calls of sfd_surface_ft).  Same workspace, determinism
 * and error behaviour as sfd_reduce.  Synchronises. */
int sfd_reduce_pair(const double* d_nuhat_a, const double* d_nuhat_b, const double* d_xi, const double* d_W, int64_t K,
                    double s, void* d_work, size_t work_bytes, sfd_stream stream, double* h_I);
/* Whole path for two meshes: "discretized surfaces are compared to each other by recomputing the Fourier transform
 * from their own data representations" (P:137 with a second linear combination of triangle transforms in place
 * of sigmahat).  Atoms of both meshes (same rule) -> nuhat_a, nuhat_b on the ball rule (q, R) -> sfd_reduce_pair ->
 * sqrt(I).  Both measures are real, so |nuhat_a - nuhat_b|^2 is even in xi and the half rule of sfd_weak_distance
 * applies unchanged.  x_extent bounds the half-width of BOTH meshes' bounding boxes.  An empty mesh is the zero
 * measure.  Synchronises. */
int sfd_mesh_distance_workspace(int64_t nF_a, int64_t nF_b, int rule, const sfd_freq_quadrature* q, double R, double eps,
                                double x_extent, size_t* bytes);
int sfd_mesh_distance(const double* d_vertices_a, int64_t nV_a, const int32_t* d_faces_a, int64_t nF_a,
                      const double* d_vertices_b, int64_t nV_b, const int32_t* d_faces_b, int64_t nF_b, int rule,
                      double s, double R, const sfd_freq_quadrature* q, double eps, void* d_work, size_t work_bytes,
                      sfd_stream stream, double* h_distance, double* h_I);

/* ---- host-buffer entry points (end-to-end: allocate, copy in, run, copy out, free) -------------
 * Same operations with HOST pointers; device memory comes from the stream-ordered CUDA pool of the
 * current device.  Synchronise. */
int sfd_surface_ft_host(const double* h_x, const double* h_w, int64_t J, const double* h_xi, int64_t K,
                        double eps, double* h_nuhat);
int sfd_weak_distance_host(const double* h_vertices, int64_t nV, const int32_t* h_faces, int64_t nF, int rule,
                           double s, double R, const sfd_freq_quadrature* q, double eps,
                           double* h_distance, double* h_I);

/* ---- single-precision grids -----------------------------------------------------------------
 * The paper ran its GPU NUFFT "in single precision" at eps_rel = 1e-7 because "shared memory is too small for practical
 * computations in the double-precision" (Fig. 4 caption P:242).  sfd_set_grid_precision(32) makes every
 * later transform of the CALLING THREAD keep its grids in single precision: the fine (spreading) grid, the
 * intermediates and the output band of the FFT passes in global memory, and the interpolation's shared-memory subgrid
 * (8-byte cells, twice the cells per bin; the gather accumulates its w planes in fp32).  Everything else -- atoms,
 * kernel evaluation, the spreader's shared-memory accumulation, the butterflies, phases, deconvolution factors, the
 * reduction -- stays fp64, so the error is the rounding of the stored grids (~6e-8 of their largest entries) on top of
 * the kernel's eps.  Accepted tolerances: eps >= 1e-6 for the type-3 transform, eps >= 1e-7 (the paper's) on the
 * lattice (type-1: no interpolation); a smaller eps > 0 returns SFD_ERR_INVALID_ARG while the switch is on.  eps == 0
 * (direct sum) is unaffected.  Error bar: 10 * max(eps, 1e-6) * sum|w_j|.  Workspace queries are precision-independent
 * (sized for fp64).  bits = 64 (the default) restores double precision.  Host-only; thread-local. */
int sfd_set_grid_precision(int bits);

/* ---- per-stage device timings of the last sfd_surface_ft / sfd_weak_distance call on this thread
 * (only recorded after sfd_set_profiling(1); adds event records and a sync).  Names are static
 * strings; returns the number of stages written (<= max). */
int sfd_set_profiling(int on);
int sfd_last_stage_times(const char** names, float* ms, int max);

/* Number of kernels of this library launched so far by the process. */
long long sfd_launch_count(void);

/* ---- environment switches (read at each call; for tests and A-B measurements, none changes a result beyond rounding) ----
 *   SFD_NO_OVERLAP=1         type-3 transform: the target sort stays on the caller's stream (no second stream)
 *   SFD_INTERP_NO_TMA=1      interpolation: subgrids staged by 16-byte asynchronous copies instead of TMA box copies
 *   SFD_DIRECT_PACKED=1      direct sum on the ball rule: rotation table packed behind the stages instead of 32 KB-aligned
 *   SFD_FFT_GENERIC=1        FFT passes: the generic kernel instead of the fixed-geometry ones
 *   SFD_DEBUG_POISON_BAND=1  FFT passes' output buffers filled with NaN first (a cell that is read without having been
 *                            stored then shows up as a NaN result) */

#ifdef __cplusplus
}
#endif
#endif /* SFD_H_ */
