// api.cu -- the C ABI of libsfd.so (include/sfd.h): argument checks, workspace carving, stage timing.  Every
// step of the path runs in the kernels of mesh.cu / nodes.cu / direct.cu / nufft3.cu / reduce.cu; there is no CPU
// fallback: without a CUDA device every compute call returns SFD_ERR_CUDA.
#include <cmath>
#include <cstring>

#include "atoms.cuh"
#include "internal.cuh"
#include "nufft3.cuh"

namespace sfd {

static thread_local char g_err[512] = "";
std::atomic<long long> g_launches{0};

// the device error word (common.cuh): one per device, zero-initialised with the module
__device__ int32_t g_dev_flags;
int32_t* device_flags() {
  void* p = nullptr;
  return cudaGetSymbolAddress(&p, g_dev_flags) == cudaSuccess ? static_cast<int32_t*>(p) : nullptr;
}

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

int num_sms() {
  static int sms = 0;
  if (sms == 0) {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
      sms = n;
    else
      return 148;  // B200; not cached so that a later successful query wins
  }
  return sms;
}

// ---- grid precision of the calling thread's transforms (sfd_set_grid_precision) ----------------------------------
static thread_local bool g_grid_f32 = false;
bool grid_f32() { return g_grid_f32; }

// ---- stage timing ---------------------------------------------------------------------------------
namespace {
constexpr int kMaxStages = 32;
struct Prof {
  bool on = false, active = false;
  int n = 0;
  cudaEvent_t ev[kMaxStages + 1] = {};
  const char* name[kMaxStages] = {};
  float ms[kMaxStages] = {};
  int n_done = 0;
};
thread_local Prof g_prof;
}  // namespace

void prof_begin(cudaStream_t st) {
  Prof& p = g_prof;
  if (!p.on) return;
  p.n = 0;
  p.active = true;
  if (!p.ev[0]) cudaEventCreate(&p.ev[0]);
  cudaEventRecord(p.ev[0], st);
}
void prof_mark(const char* name, cudaStream_t st) {
  Prof& p = g_prof;
  if (!p.on || !p.active || p.n >= kMaxStages) return;
  p.name[p.n] = name;
  ++p.n;
  if (!p.ev[p.n]) cudaEventCreate(&p.ev[p.n]);
  cudaEventRecord(p.ev[p.n], st);
}
void prof_end(cudaStream_t st) {
  Prof& p = g_prof;
  if (!p.on || !p.active) return;
  p.active = false;
  cudaStreamSynchronize(st);
  for (int i = 0; i < p.n; ++i) cudaEventElapsedTime(&p.ms[i], p.ev[i], p.ev[i + 1]);
  p.n_done = p.n;
}

namespace {
inline cudaStream_t as_stream(sfd_stream s) { return static_cast<cudaStream_t>(s); }

int check_quadrature(const sfd_freq_quadrature* q, double R) {
  SFD_REQUIRE(q, SFD_ERR_NULL, "frequency quadrature is NULL");
  SFD_REQUIRE(q->n_r >= 1 && q->n_theta >= 1 && q->n_phi >= 1, SFD_ERR_INVALID_ARG,
              "frequency quadrature sizes must be >= 1 (got %d,%d,%d)", q->n_r, q->n_theta, q->n_phi);
  SFD_REQUIRE(R > 0.0 && std::isfinite(R), SFD_ERR_INVALID_ARG, "R must be positive and finite");
  return SFD_OK;
}
// Reads back what reduce_final_kernel left in d_res (I, the device error word, the (sum, comp) pair) and synchronises.
int fetch_result(const char* who, cudaStream_t st, const double* d_res, double* I) {
  double h[2] = {0.0, 0.0};
  cudaError_t e = cudaMemcpyAsync(h, d_res, sizeof(h), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) {
    set_error("%s: %s", who, cudaGetErrorString(e));
    return SFD_ERR_CUDA;
  }
  SFD_REQUIRE(h[1] == 0.0, SFD_ERR_INVALID_ARG,
              "%s: a face index outside [0, nV) was met on the device (by this call or an earlier sfd_nodes / "
              "sfd_exact_ft / distance call on this device)", who);
  *I = h[0];
  return SFD_OK;
}

__global__ void copy_pair_kernel(const double* __restrict__ res, double* __restrict__ out) {
  out[0] = res[2];
  out[1] = res[3];
  // a bad face index met on the way poisons the partial sum, so that the caller's all-reduce cannot hide it
  if (res[1] != 0.0) out[0] = __longlong_as_double(0x7ff8000000000000LL);
}

int check_eps(double eps) {
  SFD_REQUIRE(eps == 0.0 || (eps >= 1e-14 && eps < 1.0), SFD_ERR_INVALID_ARG,
              "eps must be 0 (direct sum) or in [1e-14, 1), got %g", eps);
  return SFD_OK;
}
}  // namespace
}  // namespace sfd

using namespace sfd;

extern "C" {

const char* sfd_last_error(void) { return g_err; }
const char* sfd_version(void) { return "sfd 0.1 (sm_100a)"; }

int sfd_release_cache(void) {
  cudaDeviceSynchronize();
  int dev = 0;
  cudaMemPool_t pool;
  if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess)
    cudaMemPoolTrimTo(pool, 0);   // workspaces kept by the host-buffer entry points
  return nufft3_release_cache();
}

long long sfd_launch_count(void) { return g_launches.load(); }

int sfd_set_grid_precision(int bits) {
  SFD_REQUIRE(bits == 32 || bits == 64, SFD_ERR_INVALID_ARG, "grid precision must be 32 or 64 bits, got %d", bits);
  g_grid_f32 = bits == 32;
  return SFD_OK;
}

// ---- extents of a point set (A5-1 as a call of its own) ----------------------------------------------
int sfd_extents_workspace(size_t* bytes) {
  SFD_REQUIRE(bytes, SFD_ERR_NULL, "sfd_extents_workspace: bytes is NULL");
  *bytes = align_up(64) + align_up((size_t)kBoundsBlocks * 6 * sizeof(double));
  return SFD_OK;
}
int sfd_extents(const double* d_pts, int64_t n, double h_half[3], double h_centre[3], void* d_work, size_t work_bytes,
                sfd_stream stream) {
  SFD_REQUIRE(n >= 0, SFD_ERR_INVALID_ARG, "n must be >= 0");
  SFD_REQUIRE(h_half, SFD_ERR_NULL, "sfd_extents: h_half is NULL");
  if (n == 0) {
    for (int d = 0; d < 3; ++d) {
      h_half[d] = 0.0;
      if (h_centre) h_centre[d] = 0.0;
    }
    return SFD_OK;
  }
  size_t need = 0;
  sfd_extents_workspace(&need);
  SFD_REQUIRE(d_pts, SFD_ERR_NULL, "sfd_extents: d_pts is NULL");
  SFD_REQUIRE(d_work && work_bytes >= need, SFD_ERR_WORKSPACE_TOO_SMALL, "sfd_extents needs %zu workspace bytes, got %zu",
              need, work_bytes);
  cudaStream_t st = as_stream(stream);
  double* d_out = static_cast<double*>(d_work);
  SFD_TRY(bounds_minmax(d_pts, n, d_out, reinterpret_cast<double*>(static_cast<char*>(d_work) + 256), st));
  double hb[6];
  int32_t flag = 0;
  int32_t* d_flags = device_flags();
  SFD_CUDA_TRY(cudaMemcpyAsync(hb, d_out, sizeof(hb), cudaMemcpyDeviceToHost, st));
  if (d_flags) SFD_CUDA_TRY(cudaMemcpyAsync(&flag, d_flags, sizeof(flag), cudaMemcpyDeviceToHost, st));
  SFD_CUDA_TRY(cudaStreamSynchronize(st));
  if (flag) {
    SFD_CUDA_TRY(cudaMemsetAsync(d_flags, 0, sizeof(flag), st));
    SFD_REQUIRE(false, SFD_ERR_INVALID_ARG,
                "sfd_extents: a face index outside [0, nV) was met on the device by an earlier sfd_nodes / sfd_exact_ft call");
  }
  for (int d = 0; d < 3; ++d) {
    SFD_REQUIRE(std::isfinite(hb[d]) && std::isfinite(hb[3 + d]), SFD_ERR_INVALID_ARG, "sfd_extents: non-finite coordinate");
    h_half[d] = 0.5 * (hb[3 + d] - hb[d]) * (1.0 + 1e-12) + 1e-300;   // the margin nufft3() itself applies
    if (h_centre) h_centre[d] = 0.5 * (hb[d] + hb[3 + d]);
  }
  return SFD_OK;
}

int sfd_set_profiling(int on) {
  g_prof.on = on != 0;
  g_prof.n_done = 0;
  return SFD_OK;
}
int sfd_last_stage_times(const char** names, float* ms, int max) {
  int n = g_prof.n_done < max ? g_prof.n_done : max;
  for (int i = 0; i < n; ++i) {
    if (names) names[i] = g_prof.name[i];
    if (ms) ms[i] = g_prof.ms[i];
  }
  return n;
}

// ---- A1/A2 ----------------------------------------------------------------------------------------
int sfd_mesh_icosphere_sizes(int level, int64_t* nV, int64_t* nF, size_t* work_bytes) {
  return mesh_sizes(level, nV, nF, work_bytes);
}
int sfd_mesh_icosphere(int level, double* d_vertices, int32_t* d_faces, void* d_work, size_t work_bytes,
                       sfd_stream stream) {
  return mesh_icosphere(level, d_vertices, d_faces, d_work, work_bytes, as_stream(stream));
}

// ---- A3 -------------------------------------------------------------------------------------------
int sfd_nodes(const double* d_vertices, int64_t nV, const int32_t* d_faces, int64_t nF, int rule, double* d_x,
              double* d_w, sfd_stream stream) {
  return nodes(d_vertices, nV, d_faces, nF, rule, d_x, d_w, as_stream(stream));
}
int sfd_rule_table(int rule, double* h_lambda, double* h_omega) {
  SFD_REQUIRE(h_lambda && h_omega, SFD_ERR_NULL, "sfd_rule_table: NULL output");
  return rule_table_host(rule, h_lambda, h_omega);
}

// ---- frequency quadrature -------------------------------------------------------------------------
int sfd_freq_nodes(const sfd_freq_quadrature* q, double R, double* h_xi, double* h_W) {
  SFD_TRY(check_quadrature(q, R));
  SFD_REQUIRE(h_xi && h_W, SFD_ERR_NULL, "sfd_freq_nodes: NULL output");
  FreqTables t;
  SFD_TRY(freq_tables(q, R, t));
  for (int a = 0; a < q->n_r; ++a)
    for (int b = 0; b < q->n_theta; ++b)
      for (int c = 0; c < q->n_phi; ++c) {
        const int64_t k = ((int64_t)a * q->n_theta + b) * q->n_phi + c;
        // same roundings as freq_expand_kernel (each product rounds once)
        volatile double sc = t.st[b] * t.cph[c], ss = t.st[b] * t.sph[c];
        h_xi[3 * k + 0] = t.r[a] * sc;
        h_xi[3 * k + 1] = t.r[a] * ss;
        h_xi[3 * k + 2] = t.r[a] * t.mu[b];
        volatile double m1 = t.wr[a] * t.r[a];
        volatile double m2 = m1 * t.r[a];
        volatile double m3 = m2 * t.wmu[b];
        h_W[k] = m3 * t.wph;
      }
  return SFD_OK;
}
int sfd_freq_nodes_workspace(const sfd_freq_quadrature* q, size_t* bytes) {
  SFD_REQUIRE(q && bytes, SFD_ERR_NULL, "sfd_freq_nodes_workspace: NULL argument");
  SFD_TRY(check_quadrature(q, 1.0));
  *bytes = freq_tables_bytes(q);
  return SFD_OK;
}
int sfd_freq_nodes_device(const sfd_freq_quadrature* q, double R, double* d_xi, double* d_W, void* d_work,
                          size_t work_bytes, sfd_stream stream) {
  SFD_TRY(check_quadrature(q, R));
  SFD_REQUIRE(d_xi, SFD_ERR_NULL, "sfd_freq_nodes_device: NULL output");
  FreqTables t;
  SFD_TRY(freq_tables(q, R, t));
  return freq_expand(q, t, d_xi, d_W, d_work, work_bytes, as_stream(stream));
}

int sfd_freq_nodes_device_range(const sfd_freq_quadrature* q, double R, int32_t a_begin, int32_t a_end, double* d_xi,
                                double* d_W, void* d_work, size_t work_bytes, sfd_stream stream) {
  SFD_TRY(check_quadrature(q, R));
  SFD_REQUIRE(a_begin >= 0 && a_begin <= a_end && a_end <= q->n_r, SFD_ERR_INVALID_ARG,
              "radial range [%d,%d) outside [0,%d)", a_begin, a_end, q->n_r);
  if (a_begin == a_end) return SFD_OK;
  SFD_REQUIRE(d_xi, SFD_ERR_NULL, "sfd_freq_nodes_device_range: NULL output");
  FreqTables t;
  SFD_TRY(freq_tables(q, R, t));
  return freq_expand(q, t, d_xi, d_W, d_work, work_bytes, as_stream(stream), a_begin, a_end);
}

// ---- A4/A5 ----------------------------------------------------------------------------------------
int sfd_surface_ft_workspace(int64_t J, int64_t K, const double X[3], const double S[3], double eps, size_t* bytes) {
  SFD_REQUIRE(bytes, SFD_ERR_NULL, "sfd_surface_ft_workspace: bytes is NULL");
  SFD_REQUIRE(J >= 0 && K >= 0, SFD_ERR_INVALID_ARG, "J and K must be >= 0");
  SFD_TRY(check_eps(eps));
  if (eps == 0.0) {
    *bytes = (J == 0 || K == 0) ? 0 : direct_plan(J, K).work_bytes;
    return SFD_OK;
  }
  SFD_REQUIRE(X && S, SFD_ERR_NULL, "sfd_surface_ft_workspace: X and S are required when eps > 0");
  Nufft3Sizes sz;
  SFD_TRY(nufft3_sizes(J, K, X, S, eps, &sz));
  *bytes = sz.work_bytes;
  return SFD_OK;
}

int sfd_surface_ft_plan(int64_t J, int64_t K, const double X[3], const double S[3], double eps, int32_t* w,
                        int64_t nf[3], int64_t n2[3]) {
  SFD_REQUIRE(X && S, SFD_ERR_NULL, "sfd_surface_ft_plan: X and S are required");
  SFD_REQUIRE(J >= 0 && K >= 0, SFD_ERR_INVALID_ARG, "J and K must be >= 0");
  SFD_TRY(check_eps(eps));
  SFD_REQUIRE(eps > 0.0, SFD_ERR_INVALID_ARG, "sfd_surface_ft_plan: eps must be > 0 (the direct sum has no plan)");
  Nufft3Sizes sz;
  SFD_TRY(nufft3_sizes(J, K, X, S, eps, &sz));
  if (w) *w = sz.w;
  for (int d = 0; d < 3; ++d) {
    if (nf) nf[d] = sz.nf[d];
    if (n2) n2[d] = sz.n2[d];
  }
  return SFD_OK;
}

namespace {
int surface_ft_impl(const double* d_x, const double* d_w, int64_t J, const double* d_xi, int64_t K, double eps,
                    double* d_nuhat, void* d_work, size_t work_bytes, sfd_stream stream, bool origin_centred,
                    const ExtentHint* hint = nullptr) {
  SFD_REQUIRE(J >= 0 && K >= 0, SFD_ERR_INVALID_ARG, "J and K must be >= 0");
  SFD_TRY(check_eps(eps));
  if (K == 0) return SFD_OK;
  SFD_REQUIRE(d_xi && d_nuhat, SFD_ERR_NULL, "sfd_surface_ft: NULL target buffer");
  SFD_REQUIRE(J == 0 || (d_x && d_w), SFD_ERR_NULL, "sfd_surface_ft: NULL source buffer");
  cudaStream_t st = as_stream(stream);
  const bool own_prof = !g_prof.active;
  if (own_prof) prof_begin(st);
  int rc;
  if (eps == 0.0 || J == 0) {
    rc = direct_sum(d_x, d_w, J, d_xi, K, d_nuhat, d_work, work_bytes, st);
    prof_mark("direct_sum", st);
  } else {
    rc = nufft3(d_x, d_w, J, d_xi, K, eps, d_nuhat, d_work, work_bytes, st, origin_centred, hint);
  }
  if (own_prof) prof_end(st);
  return rc;
}
}  // namespace

int sfd_surface_ft(const double* d_x, const double* d_w, int64_t J, const double* d_xi, int64_t K, double eps,
                   double* d_nuhat, void* d_work, size_t work_bytes, sfd_stream stream) {
  return surface_ft_impl(d_x, d_w, J, d_xi, K, eps, d_nuhat, d_work, work_bytes, stream, false);
}

// ---- exact triangle transform (S:8(f) NEXT-3) -------------------------------------------------------
int sfd_exact_ft_workspace(int64_t nF, size_t* bytes) {
  SFD_REQUIRE(bytes, SFD_ERR_NULL, "sfd_exact_ft_workspace: bytes is NULL");
  SFD_REQUIRE(nF >= 0, SFD_ERR_INVALID_ARG, "nF must be >= 0");
  *bytes = exact_ft_workspace(nF);
  return SFD_OK;
}

int sfd_exact_ft(const double* d_vertices, int64_t nV, const int32_t* d_faces, int64_t nF, const double* d_xi, int64_t K,
                 double* d_out, void* d_work, size_t work_bytes, sfd_stream stream) {
  SFD_REQUIRE(nF >= 0 && K >= 0 && nV >= 0, SFD_ERR_INVALID_ARG, "nV, nF and K must be >= 0");
  if (K == 0) return SFD_OK;
  SFD_REQUIRE(d_xi && d_out, SFD_ERR_NULL, "sfd_exact_ft: NULL frequency or output buffer");
  SFD_REQUIRE(nF == 0 || (d_vertices && d_faces), SFD_ERR_NULL, "sfd_exact_ft: NULL mesh buffer");
  cudaStream_t st = as_stream(stream);
  const bool own_prof = !g_prof.active;
  if (own_prof) prof_begin(st);
  const int rc = exact_ft(d_vertices, nV, d_faces, nF, d_xi, K, d_out, d_work, work_bytes, st);
  prof_mark("exact_ft", st);
  if (own_prof) prof_end(st);
  return rc;
}

// ---- A6 -------------------------------------------------------------------------------------------
int sfd_reduce_workspace(int64_t K, size_t* bytes) {
  SFD_REQUIRE(bytes, SFD_ERR_NULL, "sfd_reduce_workspace: bytes is NULL");
  SFD_REQUIRE(K >= 0, SFD_ERR_INVALID_ARG, "K must be >= 0");
  *bytes = reduce_workspace(K);
  return SFD_OK;
}

int sfd_reduce(const double* d_nuhat, const double* d_xi, const double* d_W, int64_t K, double s, void* d_work,
               size_t work_bytes, sfd_stream stream, double* h_I) {
  SFD_REQUIRE(h_I, SFD_ERR_NULL, "sfd_reduce: h_I is NULL");
  cudaStream_t st = as_stream(stream);
  double* d_res = nullptr;
  SFD_TRY(reduce_enqueue(d_nuhat, d_xi, d_W, K, s, d_work, work_bytes, st, &d_res));
  return fetch_result("sfd_reduce", st, d_res, h_I);
}

// ---- whole path -----------------------------------------------------------------------------------
namespace {
struct DistLayout {
  int64_t J, K;
  size_t x, w, xi, W, nu, nu2, tab, red, ft, total;
  size_t ft_bytes, tab_bytes, red_bytes;
};
// Number of nodes the distance calls visit on the shells [a0, a1): the xi_3 >= 0 half when n_phi is even (R18).
int64_t visited_nodes(const sfd_freq_quadrature* q, int a0, int a1) {
  return (q->n_phi & 1) == 0 ? freq_half_count(q, a0, a1) : (int64_t)(a1 - a0) * q->n_theta * q->n_phi;
}
// J2 > 0: a second set of atoms (mesh against mesh) shares the buffers: x / w sized for the larger, two nuhat arrays.
int dist_layout(int64_t nF, int rule, const sfd_freq_quadrature* q, double reach, int a0, int a1, double eps, double x_extent,
                DistLayout* L, int64_t nF2 = 0) {
  SFD_REQUIRE(nF >= 0 && nF2 >= 0, SFD_ERR_INVALID_ARG, "nF must be >= 0");
  SFD_REQUIRE(rule == 6 || rule == 12 || rule == 64, SFD_ERR_INVALID_ARG, "unknown triangle rule %d (6, 12 or 64)", rule);
  SFD_TRY(check_quadrature(q, reach));
  SFD_REQUIRE(0 <= a0 && a0 <= a1 && a1 <= q->n_r, SFD_ERR_INVALID_ARG, "radial range [%d,%d) outside [0,%d)", a0, a1, q->n_r);
  SFD_TRY(check_eps(eps));
  L->J = std::max(nF, nF2) * rule;
  L->K = visited_nodes(q, a0, a1);
  const double X[3] = {x_extent, x_extent, x_extent}, S[3] = {reach, reach, reach};
  if (eps > 0.0) SFD_REQUIRE(x_extent > 0.0 && std::isfinite(x_extent), SFD_ERR_INVALID_ARG, "x_extent must be > 0");
  // the distance calls centre the targets' box at the origin: the strengths stay real (half the transform's grids)
  if (eps == 0.0 || L->J == 0 || L->K == 0) {
    SFD_TRY(sfd_surface_ft_workspace(L->J, L->K, X, S, 0.0, &L->ft_bytes));
    if (L->J > 0 && L->K > 0) L->ft_bytes = std::max(L->ft_bytes, direct_ball_work_bytes(L->J, L->K));
  } else {
    Nufft3Sizes sz;
    SFD_TRY(nufft3_sizes(L->J, L->K, X, S, eps, &sz, true));
    L->ft_bytes = sz.work_bytes;
  }
  L->tab_bytes = freq_tables_bytes(q);
  L->red_bytes = reduce_workspace(L->K);
  size_t o = 0;
  auto put = [&](size_t bytes) {
    const size_t at = o;
    o += align_up(bytes);
    return at;
  };
  L->x = put((size_t)L->J * 24);
  L->w = put((size_t)L->J * 8);
  L->xi = put((size_t)L->K * 24);
  L->W = put((size_t)L->K * 8);
  L->nu = put((size_t)L->K * 16);
  L->nu2 = put(nF2 > 0 ? (size_t)L->K * 16 : 0);
  L->tab = put(L->tab_bytes);
  L->red = put(L->red_bytes);
  L->ft = put(L->ft_bytes);
  L->total = o;
  return SFD_OK;
}

// The distance on the radial shells [a0, a1) of the rule: atoms -> nodes of those shells (half rule) -> transform ->
// reduction.  Leaves the result block of reduce_final_kernel (I, flag, sum, comp) at *d_res; does not read it back.
// Vb != nullptr: a second mesh takes the place of the unit sphere's closed form.
int distance_enqueue(const char* who, const double* d_V, int64_t nV, const int32_t* d_F, int64_t nF, const double* d_Vb,
                     int64_t nVb, const int32_t* d_Fb, int64_t nFb, int rule, double s, double R,
                     const sfd_freq_quadrature* q, int a0, int a1, double eps, void* d_work, size_t work_bytes,
                     sfd_stream stream, double** d_res) {
  SFD_REQUIRE(s > 0.5 && s < 1e6, SFD_ERR_INVALID_ARG, "Sobolev order s must exceed 1/2 (P:113), got %g", s);
  SFD_REQUIRE(nF == 0 || (d_V && d_F), SFD_ERR_NULL, "%s: NULL mesh buffer", who);
  SFD_REQUIRE(nFb == 0 || (d_Vb && d_Fb), SFD_ERR_NULL, "%s: NULL mesh buffer (second mesh)", who);
  const bool pair = d_Vb != nullptr;
  DistLayout L;
  // the workspace may have been sized with any x_extent: recompute the fixed part, give the rest to the transform
  SFD_TRY(dist_layout(nF, rule, q, R, a0, a1, 0.0, 1.0, &L, pair ? std::max<int64_t>(nFb, 1) : 0));
  SFD_TRY(check_eps(eps));
  SFD_REQUIRE(d_work && work_bytes >= L.ft, SFD_ERR_WORKSPACE_TOO_SMALL, "%s needs at least %zu workspace bytes, got %zu", who,
              L.total, work_bytes);
  cudaStream_t st = as_stream(stream);
  char* base = static_cast<char*>(d_work);
  double* x = reinterpret_cast<double*>(base + L.x);
  double* w = reinterpret_cast<double*>(base + L.w);
  double* xi = reinterpret_cast<double*>(base + L.xi);
  double* W = reinterpret_cast<double*>(base + L.W);
  double* nu = reinterpret_cast<double*>(base + L.nu);
  double* nu2 = reinterpret_cast<double*>(base + L.nu2);
  FreqTables t;
  SFD_TRY(freq_tables(q, R, t));
  // The ball rule is symmetric under xi -> -xi (even n_phi) and the measures are real: the nodes with xi_3 >= 0 carry
  // the whole sum with doubled weights (nodes.cu freq_expand), so only they are generated, transformed and reduced.
  const bool half = (q->n_phi & 1) == 0;
  const int64_t K = L.K;
  if (K == 0 || a0 == a1) {
    double* res = reinterpret_cast<double*>(base + L.red);
    SFD_CUDA_TRY(cudaMemsetAsync(res, 0, 4 * sizeof(double), st));
    *d_res = res;
    return SFD_OK;
  }
  SFD_TRY(freq_expand(q, t, xi, W, base + L.tab, L.tab_bytes, st, a0, a1, half));
  prof_mark("freq_nodes", st);
  for (int m = 0; m < (pair ? 2 : 1); ++m) {
    const double* V = m ? d_Vb : d_V;
    const int32_t* F = m ? d_Fb : d_F;
    const int64_t nv = m ? nVb : nV, nf = m ? nFb : nF;
    SFD_TRY(nodes(V, nv, F, nf, rule, x, w, st));
    prof_mark("nodes", st);
    // extents without a pass over the atoms and the nodes: the atoms lie in the hull of the vertices, the nodes of the
    // shells [a0, a1) in the ball of radius r_{a1-1} (Gauss-Legendre nodes ascend)
    ExtentHint hint;
    hint.d_hull = V;
    hint.n_hull = nv;
    hint.target_reach = t.r[a1 - 1];
    hint.target_ball = true;
    bool ball_done = false;
    if (eps == 0.0) {
      // the nodes are the ball rule's: the direct sum takes them from the rule's tables (one direction and four radii
      // per thread share the dot product dhat . x: direct.cu BALL); too small a rule falls through to the general kernel
      SFD_TRY(direct_sum_ball(x, w, nf * rule, reinterpret_cast<const double*>(base + L.tab), q->n_r, q->n_theta, q->n_phi,
                              a0, a1, half ? q->n_theta / 2 : 0, m ? nu2 : nu, base + L.ft, work_bytes - L.ft, st, &ball_done));
      if (ball_done) prof_mark("direct_sum", st);
    }
    if (!ball_done)
      SFD_TRY(surface_ft_impl(x, w, nf * rule, xi, K, eps, m ? nu2 : nu, base + L.ft, work_bytes - L.ft, stream, true, &hint));
  }
  SFD_TRY(reduce_enqueue(nu, xi, W, K, s, base + L.red, L.red_bytes, st, d_res, 1.0, -1.0, pair ? nu2 : nullptr));
  prof_mark("reduce", st);
  return SFD_OK;
}
}  // namespace

int sfd_weak_distance_workspace(int64_t nF, int rule, const sfd_freq_quadrature* q, double R, double eps,
                                double x_extent, size_t* bytes) {
  SFD_REQUIRE(bytes, SFD_ERR_NULL, "sfd_weak_distance_workspace: bytes is NULL");
  SFD_REQUIRE(q, SFD_ERR_NULL, "frequency quadrature is NULL");
  DistLayout L;
  SFD_TRY(dist_layout(nF, rule, q, R, 0, q->n_r, eps, x_extent, &L));
  *bytes = L.total;
  return SFD_OK;
}

int sfd_weak_distance_targets(const sfd_freq_quadrature* q, int64_t* K_eval) {
  SFD_REQUIRE(K_eval, SFD_ERR_NULL, "sfd_weak_distance_targets: K_eval is NULL");
  SFD_TRY(check_quadrature(q, 1.0));
  *K_eval = visited_nodes(q, 0, q->n_r);
  return SFD_OK;
}

int sfd_weak_distance(const double* d_vertices, int64_t nV, const int32_t* d_faces, int64_t nF, int rule, double s,
                      double R, const sfd_freq_quadrature* q, double eps, void* d_work, size_t work_bytes,
                      sfd_stream stream, double* h_distance, double* h_I) {
  SFD_REQUIRE(q, SFD_ERR_NULL, "frequency quadrature is NULL");
  cudaStream_t st = as_stream(stream);
  prof_begin(st);
  double* d_res = nullptr;
  int rc = distance_enqueue("sfd_weak_distance", d_vertices, nV, d_faces, nF, nullptr, 0, nullptr, 0, rule, s, R, q, 0,
                            q->n_r, eps, d_work, work_bytes, stream, &d_res);
  double I = 0.0;
  if (rc == SFD_OK) rc = fetch_result("sfd_weak_distance", st, d_res, &I);
  prof_end(st);
  if (rc != SFD_OK) return rc;
  if (h_I) *h_I = I;
  if (h_distance) *h_distance = std::sqrt(I);
  return SFD_OK;
}

// ---- a radial shard of the distance (multi-GPU: DESIGN.md "Multi-GPU") ---------------------------------------
int sfd_weak_distance_range_workspace(int64_t nF, int rule, const sfd_freq_quadrature* q, double R, int32_t a_begin,
                                      int32_t a_end, double eps, double x_extent, size_t* bytes) {
  SFD_REQUIRE(bytes, SFD_ERR_NULL, "sfd_weak_distance_range_workspace: bytes is NULL");
  SFD_REQUIRE(q, SFD_ERR_NULL, "frequency quadrature is NULL");
  SFD_TRY(check_quadrature(q, R));
  SFD_REQUIRE(0 <= a_begin && a_begin <= a_end && a_end <= q->n_r, SFD_ERR_INVALID_ARG,
              "radial range [%d,%d) outside [0,%d)", a_begin, a_end, q->n_r);
  // the transform's grids are sized by the shard's own reach r_{a_end-1} <= R
  double reach = R;
  if (a_end > a_begin) {
    FreqTables t;
    SFD_TRY(freq_tables(q, R, t));
    reach = t.r[a_end - 1];
  }
  DistLayout L;
  SFD_TRY(dist_layout(nF, rule, q, reach, a_begin, a_end, eps, x_extent, &L));
  *bytes = L.total;
  return SFD_OK;
}

int sfd_weak_distance_range(const double* d_vertices, int64_t nV, const int32_t* d_faces, int64_t nF, int rule, double s,
                            double R, const sfd_freq_quadrature* q, int32_t a_begin, int32_t a_end, double eps, void* d_work,
                            size_t work_bytes, sfd_stream stream, double* d_partial) {
  SFD_REQUIRE(q, SFD_ERR_NULL, "frequency quadrature is NULL");
  SFD_REQUIRE(d_partial, SFD_ERR_NULL, "sfd_weak_distance_range: d_partial is NULL");
  cudaStream_t st = as_stream(stream);
  prof_begin(st);
  double* d_res = nullptr;
  int rc = distance_enqueue("sfd_weak_distance_range", d_vertices, nV, d_faces, nF, nullptr, 0, nullptr, 0, rule, s, R, q,
                            a_begin, a_end, eps, d_work, work_bytes, stream, &d_res);
  if (rc == SFD_OK) {
    copy_pair_kernel<<<1, 1, 0, st>>>(d_res, d_partial);
    rc = launch_check("copy_pair_kernel");
  }
  prof_end(st);
  return rc;
}

// ---- mesh against mesh, whole path ---------------------------------------------------------------
int sfd_mesh_distance_workspace(int64_t nF_a, int64_t nF_b, int rule, const sfd_freq_quadrature* q, double R, double eps,
                                double x_extent, size_t* bytes) {
  SFD_REQUIRE(bytes, SFD_ERR_NULL, "sfd_mesh_distance_workspace: bytes is NULL");
  SFD_REQUIRE(q, SFD_ERR_NULL, "frequency quadrature is NULL");
  DistLayout L;
  SFD_TRY(dist_layout(nF_a, rule, q, R, 0, q->n_r, eps, x_extent, &L, std::max<int64_t>(nF_b, 1)));
  *bytes = L.total;
  return SFD_OK;
}

int sfd_mesh_distance(const double* d_vertices_a, int64_t nV_a, const int32_t* d_faces_a, int64_t nF_a,
                      const double* d_vertices_b, int64_t nV_b, const int32_t* d_faces_b, int64_t nF_b, int rule, double s,
                      double R, const sfd_freq_quadrature* q, double eps, void* d_work, size_t work_bytes, sfd_stream stream,
                      double* h_distance, double* h_I) {
  SFD_REQUIRE(q, SFD_ERR_NULL, "frequency quadrature is NULL");
  SFD_REQUIRE(nF_a >= 0 && nF_b >= 0, SFD_ERR_INVALID_ARG, "nF must be >= 0");
  // an empty second mesh is the zero measure, not "compare with the sphere": keep the pair path by passing a dummy pointer
  static const double kNoVertices[3] = {0.0, 0.0, 0.0};
  const double* Vb = d_vertices_b ? d_vertices_b : (nF_b == 0 ? kNoVertices : nullptr);
  SFD_REQUIRE(Vb, SFD_ERR_NULL, "sfd_mesh_distance: NULL mesh buffer (second mesh)");
  cudaStream_t st = as_stream(stream);
  prof_begin(st);
  double* d_res = nullptr;
  int rc = distance_enqueue("sfd_mesh_distance", d_vertices_a, nV_a, d_faces_a, nF_a, Vb, nV_b, d_faces_b, nF_b, rule, s, R, q,
                            0, q->n_r, eps, d_work, work_bytes, stream, &d_res);
  double I = 0.0;
  if (rc == SFD_OK) rc = fetch_result("sfd_mesh_distance", st, d_res, &I);
  prof_end(st);
  if (rc != SFD_OK) return rc;
  if (h_I) *h_I = I;
  if (h_distance) *h_distance = std::sqrt(I);
  return SFD_OK;
}

// ---- the paper's own variant: cube lattice + trapezoidal rule + its norm convention (S:8(f) NEXT-1/2) -----------
int sfd_lattice_nodes(int32_t M, double xi_max, double* h_xi, double* h_W) {
  SFD_REQUIRE(M >= 2 && (M & 1) == 0 && M <= 2046, SFD_ERR_INVALID_ARG, "lattice size M must be even, 2..2046 (got %d)", M);
  SFD_REQUIRE(xi_max > 0.0 && std::isfinite(xi_max), SFD_ERR_INVALID_ARG, "xi_max must be positive and finite");
  SFD_REQUIRE(h_xi && h_W, SFD_ERR_NULL, "sfd_lattice_nodes: NULL output");
  const int n = M + 1;
  const double two_pi = 6.283185307179586476925286766559;
  volatile double h = 2.0 * xi_max / M;
  for (int a = 0; a < n; ++a)
    for (int b = 0; b < n; ++b)
      for (int c = 0; c < n; ++c) {
        const int64_t k = ((int64_t)a * n + b) * n + c;
        const int idx[3] = {a - M / 2, b - M / 2, c - M / 2};
        volatile double wt = h * h;   // same roundings as lattice_kernel
        wt = wt * h;
        for (int d = 0; d < 3; ++d) {
          volatile double t = (double)idx[d] * h;
          h_xi[3 * k + d] = two_pi * t;
          if (idx[d] == -M / 2 || idx[d] == M / 2) wt = wt * 0.5;
        }
        h_W[k] = wt;
      }
  return SFD_OK;
}
int sfd_lattice_nodes_device(int32_t M, double xi_max, double* d_xi, double* d_W, sfd_stream stream) {
  return lattice_expand(M, xi_max, d_xi, d_W, as_stream(stream));
}

int sfd_reduce_ex(const double* d_nuhat, const double* d_xi, const double* d_W, int64_t K, double s, double xi_scale,
                  double prefactor, void* d_work, size_t work_bytes, sfd_stream stream, double* h_I) {
  SFD_REQUIRE(h_I, SFD_ERR_NULL, "sfd_reduce_ex: h_I is NULL");
  SFD_REQUIRE(xi_scale > 0.0 && std::isfinite(xi_scale) && prefactor > 0.0 && std::isfinite(prefactor),
              SFD_ERR_INVALID_ARG, "sfd_reduce_ex: xi_scale and prefactor must be positive and finite");
  cudaStream_t st = as_stream(stream);
  double* d_res = nullptr;
  SFD_TRY(reduce_enqueue(d_nuhat, d_xi, d_W, K, s, d_work, work_bytes, st, &d_res, xi_scale, prefactor));
  return fetch_result("sfd_reduce_ex", st, d_res, h_I);
}

namespace {
int check_lattice(int M, double xi_max) {
  SFD_REQUIRE(M >= 2 && (M & 1) == 0 && M <= 2046, SFD_ERR_INVALID_ARG, "lattice size M must be even, 2..2046 (got %d)", M);
  SFD_REQUIRE(xi_max > 0.0 && std::isfinite(xi_max), SFD_ERR_INVALID_ARG, "xi_max must be positive and finite");
  return SFD_OK;
}

// Workspace of the transform on the lattice when the expanded nodes are supplied by the caller.
int lattice_ft_bytes(int64_t J, int M, double xi_max, const double X[3], double eps, size_t* bytes) {
  const int64_t K = (int64_t)(M + 1) * (M + 1) * (M + 1);
  const double Sx = 6.283185307179586476925286766559 * xi_max;
  const double S[3] = {Sx, Sx, Sx};
  size_t t3 = 0, t1 = 0;
  bool ok = false;
  if (eps > 0.0 && J > 0) SFD_TRY(nufft1_lattice_sizes(J, M, 2.0 * xi_max / M, X, eps, &ok, &t1));
  if (ok) {
    *bytes = t1;
    return SFD_OK;
  }
  SFD_TRY(sfd_surface_ft_workspace(J, K, X, S, eps, &t3));
  *bytes = t3;
  return SFD_OK;
}

// nuhat on the lattice; d_xi_buf = room for the expanded nodes (24 K bytes), filled and used only by the type-3 /
// direct path.
int lattice_ft(const double* d_x, const double* d_w, int64_t J, int M, double xi_max, double eps, double* d_xi_buf,
               double* d_nuhat, void* d_work, size_t work_bytes, sfd_stream stream, const ExtentHint* hint = nullptr) {
  const int64_t K = (int64_t)(M + 1) * (M + 1) * (M + 1);
  cudaStream_t st = as_stream(stream);
  if (eps > 0.0 && J > 0) {
    const bool own_prof = !g_prof.active;
    if (own_prof) prof_begin(st);
    bool ok = false;
    const int rc = nufft1_lattice(d_x, d_w, J, M, 2.0 * xi_max / M, eps, d_nuhat, d_work, work_bytes, st, &ok, hint);
    if (own_prof) prof_end(st);
    if (rc != SFD_OK || ok) return rc;
  }
  SFD_TRY(lattice_expand(M, xi_max, d_xi_buf, nullptr, st));
  // the fallback is the type-3 transform, whose single-precision grids carry eps >= 1e-6 only: a tighter tolerance (the
  // lattice accepts 1e-7, the paper's) runs it with fp64 grids
  const bool f32 = g_grid_f32;
  if (eps < 1e-6) g_grid_f32 = false;
  const int rc = sfd_surface_ft(d_x, d_w, J, d_xi_buf, K, eps, d_nuhat, d_work, work_bytes, stream);
  g_grid_f32 = f32;
  return rc;
}
}  // namespace

int sfd_surface_ft_lattice_workspace(int64_t J, int32_t M, double xi_max, const double X[3], double eps, size_t* bytes) {
  SFD_REQUIRE(bytes && X, SFD_ERR_NULL, "sfd_surface_ft_lattice_workspace: NULL argument");
  SFD_REQUIRE(J >= 0, SFD_ERR_INVALID_ARG, "J must be >= 0");
  SFD_TRY(check_lattice(M, xi_max));
  SFD_TRY(check_eps(eps));
  const int64_t K = (int64_t)(M + 1) * (M + 1) * (M + 1);
  size_t b = 0;
  SFD_TRY(lattice_ft_bytes(J, M, xi_max, X, eps, &b));
  *bytes = align_up((size_t)K * 24) + b;   // room for the expanded nodes of the fallback
  return SFD_OK;
}

int sfd_surface_ft_lattice(const double* d_x, const double* d_w, int64_t J, int32_t M, double xi_max, double eps,
                           double* d_nuhat, void* d_work, size_t work_bytes, sfd_stream stream) {
  SFD_REQUIRE(J >= 0, SFD_ERR_INVALID_ARG, "J must be >= 0");
  SFD_TRY(check_lattice(M, xi_max));
  SFD_TRY(check_eps(eps));
  SFD_REQUIRE(d_nuhat, SFD_ERR_NULL, "sfd_surface_ft_lattice: NULL output");
  SFD_REQUIRE(J == 0 || (d_x && d_w), SFD_ERR_NULL, "sfd_surface_ft_lattice: NULL source buffer");
  const int64_t K = (int64_t)(M + 1) * (M + 1) * (M + 1);
  const size_t xi_bytes = align_up((size_t)K * 24);
  SFD_REQUIRE(d_work && work_bytes >= xi_bytes, SFD_ERR_WORKSPACE_TOO_SMALL,
              "sfd_surface_ft_lattice needs a workspace (sfd_surface_ft_lattice_workspace), got %zu bytes", work_bytes);
  char* base = static_cast<char*>(d_work);
  return lattice_ft(d_x, d_w, J, M, xi_max, eps, reinterpret_cast<double*>(base), d_nuhat, base + xi_bytes,
                    work_bytes - xi_bytes, stream);
}

int sfd_reduce_lattice(const double* d_nuhat, int32_t M, double xi_max, double s, double xi_scale, double prefactor,
                       void* d_work, size_t work_bytes, sfd_stream stream, double* h_I) {
  SFD_REQUIRE(h_I, SFD_ERR_NULL, "sfd_reduce_lattice: h_I is NULL");
  SFD_TRY(check_lattice(M, xi_max));
  SFD_REQUIRE(xi_scale > 0.0 && std::isfinite(xi_scale) && prefactor > 0.0 && std::isfinite(prefactor),
              SFD_ERR_INVALID_ARG, "sfd_reduce_lattice: xi_scale and prefactor must be positive and finite");
  cudaStream_t st = as_stream(stream);
  double* d_res = nullptr;
  SFD_TRY(reduce_lattice_enqueue(d_nuhat, M, xi_max, s, d_work, work_bytes, st, &d_res, xi_scale, prefactor));
  return fetch_result("sfd_reduce_lattice", st, d_res, h_I);
}

namespace {
int lattice_layout(int64_t nF, int rule, int M, double xi_max, double eps, double x_extent, DistLayout* L) {
  SFD_REQUIRE(nF >= 0, SFD_ERR_INVALID_ARG, "nF must be >= 0");
  SFD_REQUIRE(rule == 6 || rule == 12 || rule == 64, SFD_ERR_INVALID_ARG, "unknown triangle rule %d (6, 12 or 64)", rule);
  // the reduction over the lattice indexes its nodes with 32 bits: (M+1)^3 < 2^32 (the same limit as sfd_reduce_lattice),
  // checked here so that the workspace query and the call reject up front instead of after the transform
  SFD_REQUIRE(M >= 2 && (M & 1) == 0 && M <= 1624, SFD_ERR_INVALID_ARG, "lattice size M must be even, 2..1624 (got %d)", M);
  SFD_REQUIRE(xi_max > 0.0 && std::isfinite(xi_max), SFD_ERR_INVALID_ARG, "xi_max must be positive and finite");
  SFD_TRY(check_eps(eps));
  L->J = nF * rule;
  L->K = (int64_t)(M + 1) * (M + 1) * (M + 1);
  const double X[3] = {x_extent, x_extent, x_extent};
  if (eps > 0.0) SFD_REQUIRE(x_extent > 0.0 && std::isfinite(x_extent), SFD_ERR_INVALID_ARG, "x_extent must be > 0");
  SFD_TRY(lattice_ft_bytes(L->J, M, xi_max, X, eps, &L->ft_bytes));
  L->tab_bytes = 0;
  L->red_bytes = reduce_workspace(L->K);
  size_t o = 0;
  auto put = [&](size_t bytes) {
    const size_t at = o;
    o += align_up(bytes);
    return at;
  };
  L->x = put((size_t)L->J * 24);
  L->w = put((size_t)L->J * 8);
  L->xi = put((size_t)L->K * 24);
  L->W = put((size_t)L->K * 8);
  L->nu = put((size_t)L->K * 16);
  L->nu2 = L->nu;
  L->tab = put(256);
  L->red = put(L->red_bytes);
  L->ft = put(L->ft_bytes);
  L->total = o;
  return SFD_OK;
}
}  // namespace

int sfd_weak_distance_lattice_workspace(int64_t nF, int rule, int32_t M, double xi_max, double eps, double x_extent,
                                        size_t* bytes) {
  SFD_REQUIRE(bytes, SFD_ERR_NULL, "sfd_weak_distance_lattice_workspace: bytes is NULL");
  DistLayout L;
  SFD_TRY(lattice_layout(nF, rule, M, xi_max, eps, x_extent, &L));
  *bytes = L.total;
  return SFD_OK;
}

int sfd_weak_distance_lattice(const double* d_vertices, int64_t nV, const int32_t* d_faces, int64_t nF, int rule,
                              double s_paper, double xi_max, int32_t M, double eps, void* d_work, size_t work_bytes,
                              sfd_stream stream, double* h_norm, double* h_I) {
  SFD_REQUIRE(s_paper < -0.5 && s_paper > -1e6, SFD_ERR_INVALID_ARG,
              "the paper's Sobolev exponent s must be below -1/2 (P:113), got %g", s_paper);
  SFD_REQUIRE(nF == 0 || (d_vertices && d_faces), SFD_ERR_NULL, "sfd_weak_distance_lattice: NULL mesh buffer");
  DistLayout L;
  SFD_TRY(lattice_layout(nF, rule, M, xi_max, 0.0, 1.0, &L));
  SFD_TRY(check_eps(eps));
  SFD_REQUIRE(d_work && work_bytes >= L.ft, SFD_ERR_WORKSPACE_TOO_SMALL,
              "sfd_weak_distance_lattice needs at least %zu workspace bytes, got %zu", L.total, work_bytes);
  cudaStream_t st = as_stream(stream);
  char* base = static_cast<char*>(d_work);
  double* x = reinterpret_cast<double*>(base + L.x);
  double* w = reinterpret_cast<double*>(base + L.w);
  double* xi = reinterpret_cast<double*>(base + L.xi);
  double* nu = reinterpret_cast<double*>(base + L.nu);
  prof_begin(st);
  ExtentHint hint;   // the atoms lie in the hull of the vertices
  hint.d_hull = d_vertices;
  hint.n_hull = nV;
  int rc = SFD_OK;
  bool done = false;
  Nufft1Band band;
  if (eps > 0.0 && L.J > 0) {
    // the paper's transform, with the atoms generated inside its sort kernels ((x, w) are never materialised) and
    // stopped after the FFT: deconvolution and phase are folded into the reduction (nuhat is never materialised either)
    const MeshAtoms mesh{d_vertices, nV, d_faces, nF, rule};
    rc = nufft1_lattice(nullptr, nullptr, L.J, M, 2.0 * xi_max / M, eps, nullptr, base + L.ft, work_bytes - L.ft, st, &done,
                        &hint, &mesh, &band);
  }
  if (rc == SFD_OK && !done) {
    // direct sum, or a lattice too coarse for the type-1 transform: materialise the atoms; the lattice nodes are
    // expanded inside lattice_ft only if the transform needs them (the reduction recomputes them from the index)
    rc = nodes(d_vertices, nV, d_faces, nF, rule, x, w, st);
    prof_mark("nodes", st);
    if (rc == SFD_OK) rc = lattice_ft(x, w, L.J, M, xi_max, eps, xi, nu, base + L.ft, work_bytes - L.ft, stream, &hint);
  }
  double* d_res = nullptr;
  // the paper's norm (eq. 2.7) on nodes xi' = 2 pi xi: (1 + |xi|^2)^s = (1 + (|xi'|/2 pi)^2)^-(-s), weights in d xi
  const double inv_two_pi = 1.0 / 6.283185307179586476925286766559;
  if (rc == SFD_OK)
    rc = done ? reduce_lattice_band_enqueue(band, M, xi_max, -s_paper, base + L.red, L.red_bytes, st, &d_res, inv_two_pi, 1.0)
              : reduce_lattice_enqueue(nu, M, xi_max, -s_paper, base + L.red, L.red_bytes, st, &d_res, inv_two_pi, 1.0);
  prof_mark("reduce", st);
  double I = 0.0;
  if (rc == SFD_OK) rc = fetch_result("sfd_weak_distance_lattice", st, d_res, &I);
  prof_end(st);
  if (rc != SFD_OK) return rc;
  if (h_I) *h_I = I;
  if (h_norm) *h_norm = std::sqrt(I);
  return SFD_OK;
}

// ---- mesh against mesh ("discretized surfaces are compared to each other by recomputing the Fourier
// transform from their own data representations") ---------------------------------------------------------------
int sfd_reduce_pair(const double* d_nuhat_a, const double* d_nuhat_b, const double* d_xi, const double* d_W, int64_t K,
                    double s, void* d_work, size_t work_bytes, sfd_stream stream, double* h_I) {
  SFD_REQUIRE(h_I, SFD_ERR_NULL, "sfd_reduce_pair: h_I is NULL");
  SFD_REQUIRE(K == 0 || d_nuhat_b, SFD_ERR_NULL, "sfd_reduce_pair: NULL second operand");
  cudaStream_t st = as_stream(stream);
  double* d_res = nullptr;
  SFD_TRY(reduce_enqueue(d_nuhat_a, d_xi, d_W, K, s, d_work, work_bytes, st, &d_res, 1.0, -1.0, d_nuhat_b));
  return fetch_result("sfd_reduce_pair", st, d_res, h_I);
}

// ---- host-buffer entry points -----------------------------------------------------------------------
namespace {
struct HostCall {
  cudaStream_t st = nullptr;
  void* bufs[8] = {};
  int n = 0;
  int open() {
    // keep freed workspaces in the device's stream-ordered pool between calls (the default threshold of 0 hands
    // them back to the driver at every synchronisation, which costs tens of ms per call at GB sizes)
    static thread_local int pooled_dev = -1;
    int dev = 0;
    SFD_CUDA_TRY(cudaGetDevice(&dev));
    if (pooled_dev != dev) {
      cudaMemPool_t pool;
      SFD_CUDA_TRY(cudaDeviceGetDefaultMemPool(&pool, dev));
      unsigned long long keep = ~0ULL;
      SFD_CUDA_TRY(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
      pooled_dev = dev;
    }
    SFD_CUDA_TRY(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
    return SFD_OK;
  }
  int alloc(void** p, size_t bytes) {
    *p = nullptr;
    SFD_CUDA_TRY(cudaMallocAsync(p, bytes ? bytes : 256, st));
    bufs[n++] = *p;
    return SFD_OK;
  }
  ~HostCall() {
    if (!st) return;
    for (int i = 0; i < n; ++i) cudaFreeAsync(bufs[i], st);
    cudaStreamSynchronize(st);
    cudaStreamDestroy(st);
  }
};
void half_widths(const double* p, int64_t n, double out[3]) {
  for (int c = 0; c < 3; ++c) {
    double lo = 0.0, hi = 0.0;
    for (int64_t i = 0; i < n; ++i) {
      const double v = p[3 * i + c];
      if (i == 0 || v < lo) lo = v;
      if (i == 0 || v > hi) hi = v;
    }
    out[c] = 0.5 * (hi - lo) * (1.0 + 1e-12) + 1e-300;
  }
}
}  // namespace

int sfd_surface_ft_host(const double* h_x, const double* h_w, int64_t J, const double* h_xi, int64_t K, double eps,
                        double* h_nuhat) {
  SFD_REQUIRE(J >= 0 && K >= 0, SFD_ERR_INVALID_ARG, "J and K must be >= 0");
  SFD_TRY(check_eps(eps));
  if (K == 0) return SFD_OK;
  SFD_REQUIRE(h_xi && h_nuhat && (J == 0 || (h_x && h_w)), SFD_ERR_NULL, "sfd_surface_ft_host: NULL buffer");
  size_t wb = 0;
  double X[3], S[3];
  half_widths(h_x, J, X);
  half_widths(h_xi, K, S);
  SFD_TRY(sfd_surface_ft_workspace(J, K, X, S, J == 0 ? 0.0 : eps, &wb));
  HostCall hc;
  SFD_TRY(hc.open());
  void *dx, *dw, *dxi, *dnu, *dwork;
  SFD_TRY(hc.alloc(&dx, (size_t)J * 24));
  SFD_TRY(hc.alloc(&dw, (size_t)J * 8));
  SFD_TRY(hc.alloc(&dxi, (size_t)K * 24));
  SFD_TRY(hc.alloc(&dnu, (size_t)K * 16));
  SFD_TRY(hc.alloc(&dwork, wb));
  if (J > 0) {
    SFD_CUDA_TRY(cudaMemcpyAsync(dx, h_x, (size_t)J * 24, cudaMemcpyHostToDevice, hc.st));
    SFD_CUDA_TRY(cudaMemcpyAsync(dw, h_w, (size_t)J * 8, cudaMemcpyHostToDevice, hc.st));
  }
  SFD_CUDA_TRY(cudaMemcpyAsync(dxi, h_xi, (size_t)K * 24, cudaMemcpyHostToDevice, hc.st));
  SFD_TRY(sfd_surface_ft((double*)dx, (double*)dw, J, (double*)dxi, K, eps, (double*)dnu, dwork, wb, hc.st));
  SFD_CUDA_TRY(cudaMemcpyAsync(h_nuhat, dnu, (size_t)K * 16, cudaMemcpyDeviceToHost, hc.st));
  SFD_CUDA_TRY(cudaStreamSynchronize(hc.st));
  return SFD_OK;
}

int sfd_weak_distance_host(const double* h_vertices, int64_t nV, const int32_t* h_faces, int64_t nF, int rule, double s,
                           double R, const sfd_freq_quadrature* q, double eps, double* h_distance, double* h_I) {
  SFD_REQUIRE(nV >= 0 && nF >= 0, SFD_ERR_INVALID_ARG, "negative mesh size");
  SFD_REQUIRE(nF == 0 || (h_vertices && h_faces), SFD_ERR_NULL, "sfd_weak_distance_host: NULL mesh buffer");
  double X[3];
  half_widths(h_vertices, nV, X);
  const double ext = std::fmax(X[0], std::fmax(X[1], X[2]));
  size_t wb = 0;
  SFD_TRY(sfd_weak_distance_workspace(nF, rule, q, R, eps, ext, &wb));
  HostCall hc;
  SFD_TRY(hc.open());
  void *dV, *dF, *dwork;
  SFD_TRY(hc.alloc(&dV, (size_t)nV * 24));
  SFD_TRY(hc.alloc(&dF, (size_t)nF * 12));
  SFD_TRY(hc.alloc(&dwork, wb));
  if (nV > 0) SFD_CUDA_TRY(cudaMemcpyAsync(dV, h_vertices, (size_t)nV * 24, cudaMemcpyHostToDevice, hc.st));
  if (nF > 0) SFD_CUDA_TRY(cudaMemcpyAsync(dF, h_faces, (size_t)nF * 12, cudaMemcpyHostToDevice, hc.st));
  return sfd_weak_distance((double*)dV, nV, (int32_t*)dF, nF, rule, s, R, q, eps, dwork, wb, hc.st, h_distance, h_I);
}

}  // extern "C"
