// nodes.cu -- A3: triangle-quadrature atoms (eqs. 3.1-3.2) and the ball-shaped frequency quadrature
// of the CUDA path.  HBM-bound, one pass: 12 B + 72 B (cached) read and 32*q B written per face.
#include <cmath>
#include <map>
#include <mutex>
#include <tuple>
#include <vector>

#include "atoms.cuh"
#include "internal.cuh"

namespace sfd {
namespace {

// Symmetric rules in barycentric coordinates (weights sum to 1).  Orbit parameters solve the moment
// equations of degree 4 (6 points) and 6 (12 points); tests/test_binding_cpu.py re-checks exactness through
// sfd_rule_table.  Point order: DESIGN.md reading R6.
struct RuleTable {
  double lam[64][3];
  double om[64];
};
__constant__ RuleTable c_rule[3];   // 6-, 12- and 64-point rules

void legendre_rule(int n, std::vector<long double>& t, std::vector<long double>& wt);

void orbit3(double a, double w, double lam[][3], double* om) {
  const double b = 1.0 - 2.0 * a;
  const double p[3][3] = {{a, a, b}, {a, b, a}, {b, a, a}};
  for (int i = 0; i < 3; ++i) {
    for (int c = 0; c < 3; ++c) lam[i][c] = p[i][c];
    om[i] = w;
  }
}

void fill_rule(int q, RuleTable& t) {
  for (auto& r : t.lam) r[0] = r[1] = r[2] = 0.0;
  for (auto& o : t.om) o = 0.0;
  if (q == 64) {
    // The paper's own rule (N_P = 64 N_S): "the 8-point Gauss-Legendre rule is applied twice to the
    // right-hand side of (3.1) as an iterated integral" (reading R16): int_0^1 du1 int_0^{1-u1} du2, i.e.
    // u1 = a_i, u2 = (1 - a_i) a_j with a, g the 8-point rule on [0,1]; q_ij = g_i g_j (1 - a_i) sums to 1/2, so the
    // weights relative to the triangle's area are 2 q_ij.  Point i*8+j; barycentric (1-u1-u2, u1, u2).
    std::vector<long double> u, g;
    legendre_rule(8, u, g);
    for (int i = 0; i < 8; ++i)
      for (int j = 0; j < 8; ++j) {
        const long double ai = (1.0L + u[i]) / 2, aj = (1.0L + u[j]) / 2, gi = g[i] / 2, gj = g[j] / 2;
        const long double u1 = ai, u2 = (1.0L - ai) * aj;
        t.lam[8 * i + j][0] = (double)(1.0L - u1 - u2);
        t.lam[8 * i + j][1] = (double)u1;
        t.lam[8 * i + j][2] = (double)u2;
        t.om[8 * i + j] = (double)(2.0L * gi * gj * (1.0L - ai));
      }
  } else if (q == 6) {
    orbit3(0.445948490915964886318329, 0.223381589678011465695007, t.lam, t.om);
    orbit3(0.091576213509770743459571, 0.109951743655321867638326, t.lam + 3, t.om + 3);
  } else {
    orbit3(0.063089014491502228340332, 0.050844906370206816920937, t.lam, t.om);
    orbit3(0.249286745170910421291639, 0.116786275726379366025290, t.lam + 3, t.om + 3);
    const double a = 0.053145049844816947353250, b = 0.310352451033784405416608, c = 1.0 - a - b;
    const double w = 0.082851075618373575193553;
    const double p[6][3] = {{a, b, c}, {b, a, c}, {a, c, b}, {c, a, b}, {b, c, a}, {c, b, a}};
    for (int i = 0; i < 6; ++i) {
      for (int k = 0; k < 3; ++k) t.lam[6 + i][k] = p[i][k];
      t.om[6 + i] = w;
    }
  }
}

// One thread per atom j = f*q + i.  Each operation rounds once (no FMA contraction), so that the atoms are
// the same doubles on every build.  The coordinates go through shared memory so that the block's 3 x 256 doubles
// are stored contiguously (a thread's own three are 24 B apart from its neighbour's).
template <int Q>
__global__ void __launch_bounds__(256) nodes_kernel(const double* __restrict__ V, const int32_t* __restrict__ F,
                                                    int64_t nF, int64_t nV, double* __restrict__ x,
                                                    double* __restrict__ w, int32_t* __restrict__ flags) {
  __shared__ double sx[3 * 256];
  // the rule, one array per column: a warp's 32 atoms read 32 different rows, which the constant cache would serialise
  __shared__ double s_rule[4 * Q];
  {
    const RuleTable& R = c_rule[Q == 6 ? 0 : (Q == 12 ? 1 : 2)];
    for (int t = threadIdx.x; t < 4 * Q; t += 256) s_rule[t] = t / Q < 3 ? R.lam[t % Q][t / Q] : R.om[t % Q];
  }
  __syncthreads();
  const int64_t j0 = (int64_t)blockIdx.x * 256;
  const int64_t j = j0 + threadIdx.x;
  const int64_t J = nF * Q;
  if (j < J) {
    double wj;
    atom_eval(V, nV, F, j, Q, s_rule, sx[3 * threadIdx.x], sx[3 * threadIdx.x + 1], sx[3 * threadIdx.x + 2], wj, flags);
    w[j] = wj;
  }
  __syncthreads();
  const int64_t n = 3 * min((int64_t)256, J - j0);
  for (int t = threadIdx.x; t < n; t += 256) x[3 * j0 + t] = sx[t];
}

}  // namespace

// Gauss-Legendre nodes/weights on [-1,1], ascending, by Newton iteration on P_n evaluated with the
// Bonnet recurrence in long double; the derivative comes from (1-t^2) P_n' = n (P_{n-1} - t P_n).
namespace {
void legendre_rule(int n, std::vector<long double>& t, std::vector<long double>& wt) {
  const long double pi = 3.141592653589793238462643383279502884L;
  t.assign(n, 0.0L);
  wt.assign(n, 0.0L);
  for (int m = 0; m < (n + 1) / 2; ++m) {
    long double u = cosl(pi * (4 * m + 3) / (4 * n + 2));  // m-th largest root, Tricomi-like start
    long double pn = 0, pm = 0;
    for (int it = 0; it < 64; ++it) {
      pm = 1.0L;
      pn = u;
      for (int k = 1; k < n; ++k) {
        const long double nx = ((2 * k + 1) * u * pn - k * pm) / (k + 1);
        pm = pn;
        pn = nx;
      }
      const long double d = n * (pm - u * pn) / (1.0L - u * u);
      const long double step = pn / d;
      u -= step;
      if (fabsl(step) <= 4e-20L * (1.0L + fabsl(u))) break;
    }
    pm = 1.0L;
    pn = u;
    for (int k = 1; k < n; ++k) {
      const long double nx = ((2 * k + 1) * u * pn - k * pm) / (k + 1);
      pm = pn;
      pn = nx;
    }
    const long double d = n * (pm - u * pn) / (1.0L - u * u);
    const long double wgt = 2.0L / ((1.0L - u * u) * d * d);
    t[n - 1 - m] = u;
    t[m] = -u;
    wt[n - 1 - m] = wgt;
    wt[m] = wgt;
  }
  if (n & 1) t[n / 2] = 0.0L;
}

// Nodes of the radial shells [a0, a1) (a0 = 0, a1 = n_r: the whole rule); output index k - a0 n_th n_ph.
// half != 0: only the rings b >= n_th/2 (mu >= 0, the half-space xi_3 >= 0), weights doubled except on a ring that is
// its own mirror image (mu = 0, odd n_th) -- see freq_expand().  Output index ((a - a0) nb + (b - b0)) n_ph + c.
__global__ void __launch_bounds__(256) freq_expand_kernel(const double* __restrict__ tab, int n_r, int n_th, int n_ph,
                                                          int a0, int a1, int half, double wph, double* __restrict__ xi,
                                                          double* __restrict__ W) {
  const int b0 = half ? n_th / 2 : 0, nb = n_th - b0;
  const int64_t K = (int64_t)(a1 - a0) * nb * n_ph;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= K) return;
  const int c = (int)(k % n_ph);
  const int64_t ab = k / n_ph;
  const int b = b0 + (int)(ab % nb);
  const int a = a0 + (int)(ab / nb);
  const double* r = tab;
  const double* wr = r + n_r;
  const double* mu = wr + n_r;
  const double* st = mu + n_th;
  const double* wmu = st + n_th;
  const double* cph = wmu + n_th;
  const double* sph = cph + n_ph;
  const double ra = r[a];
  xi[3 * k + 0] = __dmul_rn(ra, __dmul_rn(st[b], cph[c]));
  xi[3 * k + 1] = __dmul_rn(ra, __dmul_rn(st[b], sph[c]));
  xi[3 * k + 2] = __dmul_rn(ra, mu[b]);
  if (W) {
    const double wk = __dmul_rn(__dmul_rn(__dmul_rn(__dmul_rn(wr[a], ra), ra), wmu[b]), wph);
    W[k] = (half && b != n_th - 1 - b) ? __dmul_rn(2.0, wk) : wk;
  }
}

}  // namespace

void gauss_legendre_host(int n, std::vector<long double>& t, std::vector<long double>& wt) { legendre_rule(n, t, wt); }

namespace {
// The paper's frequency quadrature (eqs. 3.3-3.4): lattice xi_ijk = (i,j,k) h, h = 2 xi_max / M,
// i,j,k = -M/2..M/2, trapezoid weights w_ijk h^3 (1, 1/2, 1/4, 1/8).  Nodes are written as xi' = 2 pi xi (reading R1).
__global__ void __launch_bounds__(256) lattice_kernel(int M, double h, double* __restrict__ xi, double* __restrict__ W) {
  const int n = M + 1;
  const int64_t K = (int64_t)n * n * n;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= K) return;
  const int c = (int)(k % n);
  const int64_t ab = k / n;
  const int b = (int)(ab % n), a = (int)(ab / n);
  const int idx[3] = {a - M / 2, b - M / 2, c - M / 2};
  const double two_pi = 6.283185307179586476925286766559;
  double wt = __dmul_rn(__dmul_rn(h, h), h);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    xi[3 * k + d] = __dmul_rn(two_pi, __dmul_rn((double)idx[d], h));
    if (idx[d] == -M / 2 || idx[d] == M / 2) wt = __dmul_rn(wt, 0.5);
  }
  if (W) W[k] = wt;
}
}  // namespace

int lattice_expand(int M, double xi_max, double* d_xi, double* d_W, cudaStream_t st) {
  SFD_REQUIRE(M >= 2 && (M & 1) == 0 && M <= 2046, SFD_ERR_INVALID_ARG, "lattice size M must be even, 2..2046 (got %d)", M);
  SFD_REQUIRE(xi_max > 0.0 && std::isfinite(xi_max), SFD_ERR_INVALID_ARG, "xi_max must be positive and finite");
  SFD_REQUIRE(d_xi, SFD_ERR_NULL, "lattice nodes: NULL output");
  const int64_t K = (int64_t)(M + 1) * (M + 1) * (M + 1);
  lattice_kernel<<<(unsigned)((K + 255) / 256), 256, 0, st>>>(M, 2.0 * xi_max / M, d_xi, d_W);
  return launch_check("lattice_kernel");
}

int freq_tables(const sfd_freq_quadrature* q, double R, FreqTables& t) {
  SFD_REQUIRE(q, SFD_ERR_NULL, "freq quadrature is NULL");
  SFD_REQUIRE(q->n_r >= 1 && q->n_theta >= 1 && q->n_phi >= 1, SFD_ERR_INVALID_ARG,
              "freq quadrature sizes must be >= 1 (got %d,%d,%d)", q->n_r, q->n_theta, q->n_phi);
  SFD_REQUIRE(R > 0.0 && std::isfinite(R), SFD_ERR_INVALID_ARG, "R must be positive and finite");
  // the Newton iterations cost ~1 ms of host time at 256 x 128 nodes: keep the last few rules (host-side cache,
  // thread-safe; the rules are a pure function of the key)
  static std::mutex mu;
  static std::map<std::tuple<int, int, int, double>, FreqTables> cache;
  const auto key = std::make_tuple(q->n_r, q->n_theta, q->n_phi, R);
  {
    std::lock_guard<std::mutex> lk(mu);
    auto it = cache.find(key);
    if (it != cache.end()) {
      t = it->second;
      return SFD_OK;
    }
  }
  const double pi = 3.14159265358979323846;
  std::vector<long double> u, wu;
  legendre_rule(q->n_r, u, wu);
  t.r.resize(q->n_r);
  t.wr.resize(q->n_r);
  const long double half = (long double)R / 2;
  for (int a = 0; a < q->n_r; ++a) {
    t.r[a] = (double)(half + half * u[a]);
    t.wr[a] = (double)(half * wu[a]);
  }
  legendre_rule(q->n_theta, u, wu);
  t.mu.resize(q->n_theta);
  t.st.resize(q->n_theta);
  t.wmu.resize(q->n_theta);
  for (int b = 0; b < q->n_theta; ++b) {
    t.mu[b] = (double)u[b];
    t.wmu[b] = (double)wu[b];
    t.st[b] = std::sqrt(1.0 - t.mu[b] * t.mu[b]);
  }
  t.cph.resize(q->n_phi);
  t.sph.resize(q->n_phi);
  for (int c = 0; c < q->n_phi; ++c) {
    const double ph = 2.0 * pi * c / q->n_phi;
    t.cph[c] = std::cos(ph);
    t.sph[c] = std::sin(ph);
  }
  t.wph = 2.0 * pi / q->n_phi;
  {
    std::lock_guard<std::mutex> lk(mu);
    if (cache.size() >= 16) cache.clear();
    cache[key] = t;
  }
  return SFD_OK;
}

size_t freq_tables_bytes(const sfd_freq_quadrature* q) {
  return align_up(sizeof(double) * (2 * (size_t)q->n_r + 3 * (size_t)q->n_theta + 2 * (size_t)q->n_phi));
}

// half: the rule is symmetric under xi -> -xi when n_phi is even (Gauss-Legendre in mu is symmetric, phi + pi is a
// node), and for a real measure nuhat(-xi) = conj nuhat(xi), sigmahat is real and radial, so the terms
// W_k |nuhat_k - sigmahat_k|^2 (1+|xi_k|^2)^-s of mirror nodes are equal: the sum over the half-space xi_3 >= 0 with
// doubled weights is the sum over the ball.  K_half = (a1 - a0) ceil(n_th / 2) n_ph nodes are written.
int64_t freq_half_count(const sfd_freq_quadrature* q, int a0, int a1) {
  return (int64_t)(a1 - a0) * (q->n_theta - q->n_theta / 2) * q->n_phi;
}

int freq_expand(const sfd_freq_quadrature* q, const FreqTables& t, double* d_xi, double* d_W, void* d_work,
                size_t work_bytes, cudaStream_t st, int a0, int a1, bool half) {
  if (a1 < 0) a1 = q->n_r;
  SFD_REQUIRE(0 <= a0 && a0 <= a1 && a1 <= q->n_r, SFD_ERR_INVALID_ARG, "radial range [%d,%d) outside [0,%d)", a0, a1,
              q->n_r);
  SFD_REQUIRE(!half || (q->n_phi & 1) == 0, SFD_ERR_INVALID_ARG, "the half rule needs an even n_phi (got %d)", q->n_phi);
  SFD_REQUIRE(work_bytes >= freq_tables_bytes(q) && d_work, SFD_ERR_WORKSPACE_TOO_SMALL,
              "frequency quadrature needs %zu workspace bytes, got %zu", freq_tables_bytes(q), work_bytes);
  std::vector<double> h;
  h.reserve(2 * t.r.size() + 3 * t.mu.size() + 2 * t.cph.size());
  for (const auto* v : {&t.r, &t.wr, &t.mu, &t.st, &t.wmu, &t.cph, &t.sph}) h.insert(h.end(), v->begin(), v->end());
  // pageable source: the runtime stages the copy before returning, so `h` may die at scope exit
  SFD_CUDA_TRY(cudaMemcpyAsync(d_work, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice, st));
  const int64_t K = half ? freq_half_count(q, a0, a1) : (int64_t)(a1 - a0) * q->n_theta * q->n_phi;
  if (K == 0) return SFD_OK;
  freq_expand_kernel<<<(unsigned)((K + 255) / 256), 256, 0, st>>>(static_cast<const double*>(d_work), q->n_r,
                                                                   q->n_theta, q->n_phi, a0, a1, half ? 1 : 0, t.wph, d_xi, d_W);
  return launch_check("freq_expand_kernel");
}

int rule_table_host(int rule, double* lam, double* om) {
  SFD_REQUIRE(rule == 6 || rule == 12 || rule == 64, SFD_ERR_INVALID_ARG, "unknown triangle rule %d (6, 12 or 64)", rule);
  RuleTable t;
  fill_rule(rule, t);
  for (int i = 0; i < rule; ++i) {
    for (int c = 0; c < 3; ++c) lam[3 * i + c] = t.lam[i][c];
    om[i] = t.om[i];
  }
  return SFD_OK;
}

// The rule as four columns lam0[Q], lam1[Q], lam2[Q], om[Q] in device memory (atoms.cuh atom_eval).
int rule_table_device(int rule, double* d_tab, cudaStream_t st) {
  SFD_REQUIRE(rule == 6 || rule == 12 || rule == 64, SFD_ERR_INVALID_ARG, "unknown triangle rule %d (6, 12 or 64)", rule);
  RuleTable t;
  fill_rule(rule, t);
  double h[4 * 64];
  for (int i = 0; i < rule; ++i) {
    for (int c = 0; c < 3; ++c) h[c * rule + i] = t.lam[i][c];
    h[3 * rule + i] = t.om[i];
  }
  // pageable source: staged by the runtime before the call returns
  SFD_CUDA_TRY(cudaMemcpyAsync(d_tab, h, sizeof(double) * 4 * rule, cudaMemcpyHostToDevice, st));
  return SFD_OK;
}

int nodes(const double* d_V, int64_t nV, const int32_t* d_F, int64_t nF, int rule, double* d_x, double* d_w,
          cudaStream_t st) {
  SFD_REQUIRE(rule == 6 || rule == 12 || rule == 64, SFD_ERR_INVALID_ARG, "unknown triangle rule %d (6, 12 or 64)", rule);
  SFD_REQUIRE(nF >= 0 && nV >= 0, SFD_ERR_INVALID_ARG, "negative mesh size");
  if (nF == 0) return SFD_OK;
  SFD_REQUIRE(d_V && d_F && d_x && d_w, SFD_ERR_NULL, "sfd_nodes: NULL buffer");
  static thread_local int uploaded_dev = -1;
  int dev = 0;
  SFD_CUDA_TRY(cudaGetDevice(&dev));
  if (uploaded_dev != dev) {
    static RuleTable t[3];
    fill_rule(6, t[0]);
    fill_rule(12, t[1]);
    fill_rule(64, t[2]);
    SFD_CUDA_TRY(cudaMemcpyToSymbol(c_rule, t, sizeof(t)));
    uploaded_dev = dev;
  }
  const int64_t J = nF * rule;
  const unsigned blocks = (unsigned)((J + 255) / 256);
  int32_t* flags = device_flags();
  if (rule == 6)
    nodes_kernel<6><<<blocks, 256, 0, st>>>(d_V, d_F, nF, nV, d_x, d_w, flags);
  else if (rule == 64)
    nodes_kernel<64><<<blocks, 256, 0, st>>>(d_V, d_F, nF, nV, d_x, d_w, flags);
  else
    nodes_kernel<12><<<blocks, 256, 0, st>>>(d_V, d_F, nF, nV, d_x, d_w, flags);
  return launch_check("nodes_kernel");
}

}  // namespace sfd
