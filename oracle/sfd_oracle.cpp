// sfd_oracle.cpp -- CPU ORACLE. TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, fp64 restatement of the hot path of Koga, "Computing weak distance between the
// 2-sphere and its nonsmooth approximations" (arXiv 2304.06340), written from PAPER.md ("P:n" =
// /root/reference/PAPER.md line n) in the variant BASELINE.json's north_star fixes (Fourier kernel
// e^{-i xi.x}, weight (1+|xi|^2)^{-s}, spherical-product frequency quadrature).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this file.  It shares no code, header, table or constant generator with
// paper_2304_06340_b200/ (the CUDA path) and includes nothing from it.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): every function below is pinned by something
// other than itself -- closed forms, invariants, mpmath/numpy library routines, brute force.
// No function here is "parity unpinned".
//
// Build: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -shared -fPIC (oracle/build_oracle.py).
// -ffp-contract=off: every operation below rounds once, exactly as written.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const double kPi = 3.14159265358979323846264338327950288;

// ---------------------------------------------------------------------------------------------
// Icosahedron T_0 ("the process begins with an icosahedron inscribed in S^2").  The paper
// delegates the mesh to an external generator; reading R4 fixes the convention:
// the three golden rectangles, faces found by enumeration i<j<k, oriented outward.
// ---------------------------------------------------------------------------------------------
void icosahedron(double* V, int32_t* F) {
  const double t = (1.0 + std::sqrt(5.0)) / 2.0;
  const double raw[12][3] = {{-1, t, 0}, {1, t, 0}, {-1, -t, 0}, {1, -t, 0}, {0, -1, t}, {0, 1, t},
                             {0, -1, -t}, {0, 1, -t}, {t, 0, -1}, {t, 0, 1}, {-t, 0, -1}, {-t, 0, 1}};
  const double nrm = std::sqrt(1.0 + t * t);
  for (int i = 0; i < 12; ++i)
    for (int c = 0; c < 3; ++c) V[3 * i + c] = raw[i][c] / nrm;
  int nf = 0;
  for (int i = 0; i < 12; ++i)
    for (int j = i + 1; j < 12; ++j)
      for (int k = j + 1; k < 12; ++k) {
        auto d2 = [&](int a, int b) {
          double s = 0;
          for (int c = 0; c < 3; ++c) s += (raw[a][c] - raw[b][c]) * (raw[a][c] - raw[b][c]);
          return s;
        };
        if (std::fabs(d2(i, j) - 4.0) > 1e-9 || std::fabs(d2(j, k) - 4.0) > 1e-9 ||
            std::fabs(d2(i, k) - 4.0) > 1e-9)
          continue;
        const double* a = raw[i];
        const double* b = raw[j];
        const double* c = raw[k];
        double det = a[0] * (b[1] * c[2] - b[2] * c[1]) - a[1] * (b[0] * c[2] - b[2] * c[0]) +
                     a[2] * (b[0] * c[1] - b[1] * c[0]);
        F[3 * nf + 0] = i;
        F[3 * nf + 1] = det > 0 ? j : k;
        F[3 * nf + 2] = det > 0 ? k : j;
        ++nf;
      }
}

// ---------------------------------------------------------------------------------------------
// One subdivision step T_{N-1} -> T_N ("an additional vertice is chosen to be the midpoint
// of each edge and connected to the others on the same triangle ... divides each face into four
// sub-triangles and the projection of those new vertices onto S^2").
// Vout must hold nV + E vertices (E = 3 nF / 2), Fout 4 nF faces.  Returns E.
// ---------------------------------------------------------------------------------------------
int64_t subdivide(const double* V, int64_t nV, const int32_t* F, int64_t nF, double* Vout,
                  int32_t* Fout) {
  std::vector<int64_t> keys;
  keys.reserve(3 * nF);
  auto key = [&](int32_t a, int32_t b) { return (int64_t)std::min(a, b) * nV + std::max(a, b); };
  for (int64_t f = 0; f < nF; ++f) {
    keys.push_back(key(F[3 * f + 0], F[3 * f + 1]));
    keys.push_back(key(F[3 * f + 1], F[3 * f + 2]));
    keys.push_back(key(F[3 * f + 2], F[3 * f + 0]));
  }
  std::sort(keys.begin(), keys.end());
  keys.erase(std::unique(keys.begin(), keys.end()), keys.end());
  const int64_t E = (int64_t)keys.size();
  std::memcpy(Vout, V, sizeof(double) * 3 * nV);
  for (int64_t e = 0; e < E; ++e) {
    const int64_t a = keys[e] / nV, b = keys[e] % nV;  // a < b
    const double mx = V[3 * a + 0] + V[3 * b + 0];
    const double my = V[3 * a + 1] + V[3 * b + 1];
    const double mz = V[3 * a + 2] + V[3 * b + 2];
    double s = mx * mx;
    s = s + my * my;
    s = s + mz * mz;
    const double n = std::sqrt(s);
    Vout[3 * (nV + e) + 0] = mx / n;
    Vout[3 * (nV + e) + 1] = my / n;
    Vout[3 * (nV + e) + 2] = mz / n;
  }
  auto mid = [&](int32_t a, int32_t b) {
    const int64_t k = key(a, b);
    return (int32_t)(nV + (std::lower_bound(keys.begin(), keys.end(), k) - keys.begin()));
  };
  for (int64_t f = 0; f < nF; ++f) {
    const int32_t i0 = F[3 * f], i1 = F[3 * f + 1], i2 = F[3 * f + 2];
    const int32_t m01 = mid(i0, i1), m12 = mid(i1, i2), m20 = mid(i2, i0);
    const int32_t ch[4][3] = {{i0, m01, m20}, {i1, m12, m01}, {i2, m20, m12}, {m01, m12, m20}};
    std::memcpy(Fout + 12 * f, ch, sizeof(ch));
  }
  return E;
}

// ---------------------------------------------------------------------------------------------
// Symmetric triangle rules in barycentric coordinates, weights summing to 1 ("more symmetric
// rules are available on triangles [27, 40]"; BASELINE.json fixes the 6-pt degree-4 and 12-pt
// degree-6 members).  Orbit parameters: the solutions of the moment equations, re-derived to
// 1e-15 by tests/test_oracle_pins.py::test_rule_exactness (never trusted as digits).
// ---------------------------------------------------------------------------------------------
void gauss_legendre_unit(int n, long double* x, long double* w);

int rule_table(int rule, double lam[][3], double* om) {
  if (rule == 64) {
    // The paper's own rule: "the 8-point Gauss-Legendre rule is applied twice to the right-hand side of
    // (3.1) as an iterated integral", 64 nodes per triangle (P:173 N_P = 64 N_S).  Reading (R16): the
    // iterated integral over Q_0^2 = {u1, u2 >= 0, u1 + u2 <= 1} (eq. 2.17) is int_0^1 du1 int_0^{1-u1} du2;
    // the inner interval is mapped to [0,1] by u2 = (1 - u1) t.  With (a_i, g_i) the 8-point rule on [0,1]:
    // u = (a_i, (1 - a_i) a_j), q_ij = g_i g_j (1 - a_i); sum q = 1/2 = |Q_0^2| and om = 2 q sums to 1.
    // L(u) = p0 + u1 (p1 - p0) + u2 (p2 - p0) (eq. 2.18) = barycentric (1 - u1 - u2, u1, u2).  Point i*8+j.
    long double t[8], g[8];
    gauss_legendre_unit(8, t, g);
    for (int i = 0; i < 8; ++i)
      for (int j = 0; j < 8; ++j) {
        const long double ai = (t[i] + 1.0L) / 2.0L, aj = (t[j] + 1.0L) / 2.0L;
        const long double u1 = ai, u2 = (1.0L - ai) * aj;
        lam[8 * i + j][0] = (double)(1.0L - u1 - u2);
        lam[8 * i + j][1] = (double)u1;
        lam[8 * i + j][2] = (double)u2;
        om[8 * i + j] = (double)(2.0L * (g[i] / 2.0L) * (g[j] / 2.0L) * (1.0L - ai));
      }
    return 64;
  }
  if (rule == 6) {
    const double a[2] = {0.4459484909159648863183293, 0.09157621350977074345957146};
    const double w[2] = {0.2233815896780114656950070, 0.1099517436553218676383263};
    for (int o = 0; o < 2; ++o) {
      const double b = 1.0 - 2.0 * a[o];
      const double p[3][3] = {{a[o], a[o], b}, {a[o], b, a[o]}, {b, a[o], a[o]}};
      for (int i = 0; i < 3; ++i) {
        for (int c = 0; c < 3; ++c) lam[3 * o + i][c] = p[i][c];
        om[3 * o + i] = w[o];
      }
    }
    return 6;
  }
  if (rule == 12) {
    const double a[2] = {0.0630890144915022283403316, 0.2492867451709104212916386};
    const double w[2] = {0.05084490637020681692093681, 0.1167862757263793660252896};
    for (int o = 0; o < 2; ++o) {
      const double b = 1.0 - 2.0 * a[o];
      const double p[3][3] = {{a[o], a[o], b}, {a[o], b, a[o]}, {b, a[o], a[o]}};
      for (int i = 0; i < 3; ++i) {
        for (int c = 0; c < 3; ++c) lam[3 * o + i][c] = p[i][c];
        om[3 * o + i] = w[o];
      }
    }
    const double A = 0.05314504984481694735324967, B = 0.3103524510337844054166077;
    const double C = 1.0 - A - B, W = 0.08285107561837357519355346;
    const double p[6][3] = {{A, B, C}, {B, A, C}, {A, C, B}, {C, A, B}, {B, C, A}, {C, B, A}};
    for (int i = 0; i < 6; ++i) {
      for (int c = 0; c < 3; ++c) lam[6 + i][c] = p[i][c];
      om[6 + i] = W;
    }
    return 12;
  }
  return -1;
}

// Gauss-Legendre on [-1,1], ascending nodes: Newton on the three-term recurrence in long double
// from the cos(pi (i - 1/4)/(n + 1/2)) guess (standard; P:154 cites an iteration-free variant).
void gauss_legendre_unit(int n, long double* x, long double* w) {
  const long double pi = 3.14159265358979323846264338327950288L;
  for (int i = 0; i < n; ++i) {
    long double z = std::cos(pi * ((long double)(i + 1) - 0.25L) / ((long double)n + 0.5L));
    long double dp = 0;
    for (int it = 0; it < 100; ++it) {
      long double p0 = 1.0L, p1 = z;
      for (int k = 2; k <= n; ++k) {
        const long double p2 = ((2 * k - 1) * z * p1 - (k - 1) * p0) / k;
        p0 = p1;
        p1 = p2;
      }
      if (n == 1) { p0 = 1.0L; p1 = z; }
      dp = n * (z * p1 - p0) / (z * z - 1.0L);
      const long double dz = p1 / dp;
      z -= dz;
      if (std::fabs(dz) < 1e-19L) break;
    }
    // recompute derivative at the converged node
    long double p0 = 1.0L, p1 = z;
    for (int k = 2; k <= n; ++k) {
      const long double p2 = ((2 * k - 1) * z * p1 - (k - 1) * p0) / k;
      p0 = p1;
      p1 = p2;
    }
    dp = n * (z * p1 - p0) / (z * z - 1.0L);
    x[n - 1 - i] = z;  // guess sequence is descending
    w[n - 1 - i] = 2.0L / ((1.0L - z * z) * dp * dp);
  }
}

}  // namespace

extern "C" {

// Sizes of T_N ("10 x 4^N + 2 vertices and 20 x 4^N triangles").
void orc_mesh_sizes(int level, int64_t* nV, int64_t* nF) {
  int64_t p = 1;
  for (int i = 0; i < level; ++i) p *= 4;
  *nV = 10 * p + 2;
  *nF = 20 * p;
}

// Icosphere T_level: vertices double[nV][3], faces int32[nF][3].
int orc_mesh_icosphere(int level, double* V, int32_t* F) {
  if (level < 0 || level > 10) return -2;
  std::vector<double> v(36);
  std::vector<int32_t> f(60);
  icosahedron(v.data(), f.data());
  int64_t nV = 12, nF = 20;
  for (int l = 0; l < level; ++l) {
    std::vector<double> v2(3 * (nV + 3 * nF / 2));
    std::vector<int32_t> f2(12 * nF);
    const int64_t E = subdivide(v.data(), nV, f.data(), nF, v2.data(), f2.data());
    nV += E;
    nF *= 4;
    v.swap(v2);
    f.swap(f2);
  }
  std::memcpy(V, v.data(), sizeof(double) * 3 * nV);
  std::memcpy(F, f.data(), sizeof(int32_t) * 3 * nF);
  return 0;
}

// One subdivision step on an arbitrary closed triangle mesh (exposed for the worked example pin).
int64_t orc_subdivide(const double* V, int64_t nV, const int32_t* F, int64_t nF, double* Vout,
                      int32_t* Fout) {
  return subdivide(V, nV, F, nF, Vout, Fout);
}

// Rule table: lam double[q][3] barycentric, om double[q] (sum 1).  Returns q or -1.
int orc_rule(int rule, double* lam, double* om) {
  double l[64][3], o[64];
  const int q = rule_table(rule, l, o);
  if (q < 0) return -1;
  std::memcpy(lam, l, sizeof(double) * 3 * q);
  std::memcpy(om, o, sizeof(double) * q);
  return q;
}

// Triangle-quadrature atoms (eqs. 3.1-3.2): node L(u_i) = sum_m lam_im p_m, weight
// q_i * gamma_A with sum_i q_i = 1/2 and gamma_A = 2 area  ==  om_i * area, sum_i om_i = 1.
// x double[nF*q][3], w double[nF*q], index j = f*q + i.
int orc_nodes(const double* V, int64_t nV, const int32_t* F, int64_t nF, int rule, double* x,
              double* w) {
  double lam[64][3], om[64];
  const int q = rule_table(rule, lam, om);
  if (q < 0) return -2;
  for (int64_t f = 0; f < nF; ++f) {
    const int32_t i0 = F[3 * f], i1 = F[3 * f + 1], i2 = F[3 * f + 2];
    if (i0 < 0 || i1 < 0 || i2 < 0 || i0 >= nV || i1 >= nV || i2 >= nV) return -2;
    const double* p0 = V + 3 * i0;
    const double* p1 = V + 3 * i1;
    const double* p2 = V + 3 * i2;
    const double e1[3] = {p1[0] - p0[0], p1[1] - p0[1], p1[2] - p0[2]};
    const double e2[3] = {p2[0] - p0[0], p2[1] - p0[1], p2[2] - p0[2]};
    const double cx = e1[1] * e2[2] - e1[2] * e2[1];
    const double cy = e1[2] * e2[0] - e1[0] * e2[2];
    const double cz = e1[0] * e2[1] - e1[1] * e2[0];
    const double area = 0.5 * std::sqrt(cx * cx + cy * cy + cz * cz);
    for (int i = 0; i < q; ++i) {
      const int64_t j = f * q + i;
      for (int c = 0; c < 3; ++c)
        x[3 * j + c] = lam[i][0] * p0[c] + lam[i][1] * p1[c] + lam[i][2] * p2[c];
      w[j] = om[i] * area;
    }
  }
  return 0;
}

// n-point Gauss-Legendre on [a,b], ascending nodes.
int orc_gauss_legendre(int n, double a, double b, double* x, double* w) {
  if (n < 1) return -2;
  std::vector<long double> xs(n), ws(n);
  gauss_legendre_unit(n, xs.data(), ws.data());
  const long double h = ((long double)b - (long double)a) / 2, c = ((long double)b + (long double)a) / 2;
  for (int i = 0; i < n; ++i) {
    x[i] = (double)(c + h * xs[i]);
    w[i] = (double)(h * ws[i]);
  }
  return 0;
}

// Ball-shaped frequency quadrature ("one may consider integrals over balls centered at the
// origin and construct numerical quadrature rules on them"; BASELINE.json configs): GL in r on
// [0,R] x GL in mu = cos(theta) on [-1,1] x periodic trapezoid in phi.  k = (a*n_th + b)*n_ph + c.
// xi double[K][3], W double[K] with W = w_r r^2 w_mu (2 pi / n_ph)   (d xi = r^2 dr dmu dphi).
int orc_freq_nodes(int n_r, int n_th, int n_ph, double R, double* xi, double* W) {
  if (n_r < 1 || n_th < 1 || n_ph < 1 || !(R > 0)) return -2;
  std::vector<double> r(n_r), wr(n_r), mu(n_th), wmu(n_th);
  orc_gauss_legendre(n_r, 0.0, R, r.data(), wr.data());
  orc_gauss_legendre(n_th, -1.0, 1.0, mu.data(), wmu.data());
  const double wph = 2.0 * kPi / n_ph;
  for (int a = 0; a < n_r; ++a)
    for (int b = 0; b < n_th; ++b) {
      const double st = std::sqrt(1.0 - mu[b] * mu[b]);
      for (int c = 0; c < n_ph; ++c) {
        const int64_t k = ((int64_t)a * n_th + b) * n_ph + c;
        const double ph = 2.0 * kPi * c / n_ph;
        xi[3 * k + 0] = r[a] * (st * std::cos(ph));
        xi[3 * k + 1] = r[a] * (st * std::sin(ph));
        xi[3 * k + 2] = r[a] * mu[b];
        W[k] = wr[a] * r[a] * r[a] * wmu[b] * wph;
      }
    }
  return 0;
}

// Fourier transform of the atomic measure nu = sum_j w_j delta_{x_j} (eq. 2.8 applied to
// P:152's Dirac approximation; kernel e^{-i xi.x}, reading R1):
//   nuhat_k = sum_j w_j (cos(xi_k.x_j) - i sin(xi_k.x_j)),  nuhat double[K][2].
// Plain direct summation, one target at a time, long double accumulator.
int orc_direct_sum(const double* x, const double* w, int64_t J, const double* xi, int64_t K,
                   double* nuhat) {
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < K; ++k) {
    long double re = 0, im = 0;
    const double a = xi[3 * k], b = xi[3 * k + 1], c = xi[3 * k + 2];
    for (int64_t j = 0; j < J; ++j) {
      const double th = a * x[3 * j] + b * x[3 * j + 1] + c * x[3 * j + 2];
      re += (long double)(w[j] * std::cos(th));
      im -= (long double)(w[j] * std::sin(th));
    }
    nuhat[2 * k] = (double)re;
    nuhat[2 * k + 1] = (double)im;
  }
  return 0;
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// sigma-hat of the unit sphere (eq. 2.14, 2 sin(2 pi |xi|)/|xi|, mapped to the e^{-i xi.x}
// convention: 4 pi sin r / r; series 4 pi (1 - r^2/6 + r^4/120) below r = 1e-4).
double orc_sigma_hat(double r) {
  if (r < 1e-4) return 4.0 * kPi * (1.0 - r * r / 6.0 + r * r * r * r / 120.0);
  return 4.0 * kPi * std::sin(r) / r;
}

// I = (2 pi)^-3 sum_k W_k |nuhat_k - sigmahat(xi_k)|^2 (1+|xi_k|^2)^{-s}   (eq. 2.7 with the
// Plancherel factor of P:55 eq. 2.5 in the e^{-i xi.x} convention; s > 0 is the order of H^{-s}).
double orc_reduce(const double* nuhat, const double* xi, const double* W, int64_t K, double s) {
  long double acc = 0;
  for (int64_t k = 0; k < K; ++k) {
    const double r2 = xi[3 * k] * xi[3 * k] + xi[3 * k + 1] * xi[3 * k + 1] + xi[3 * k + 2] * xi[3 * k + 2];
    const double r = std::sqrt(r2);
    const double dre = nuhat[2 * k] - orc_sigma_hat(r);
    const double dim = nuhat[2 * k + 1];
    acc += (long double)(W[k] * (dre * dre + dim * dim) * std::pow(1.0 + r2, -s));
  }
  return (double)(acc / (8.0L * 3.14159265358979323846264338327950288L * 3.14159265358979323846264338327950288L *
                         3.14159265358979323846264338327950288L));
}

// The paper's own frequency quadrature (eqs. 3.3-3.4): the cube D = [-xi_max, xi_max]^3 sampled on the
// lattice xi_ijk = (i h, j h, k h), h = 2 xi_max / M, i,j,k = -M/2..M/2 (M even), with the three-dimensional
// trapezoidal rule: weight w_ijk h^3, w = 1 inside, 1/2 on faces, 1/4 on edges, 1/8 at corners.  The paper's
// transform is e^{-2 pi i xi.x} (eq. 2.1); this code base evaluates e^{-i xi'.x}, so the nodes are returned as
// xi' = 2 pi xi (R1) while the weights stay in the paper's units (d xi).  Node index
// k = (a (M+1) + b)(M+1) + c with a,b,c = i + M/2 etc.  xi double[K][3], W double[K], K = (M+1)^3.
int orc_lattice_nodes(int M, double xi_max, double* xi, double* W) {
  if (M < 2 || (M & 1) || !(xi_max > 0)) return -2;
  const double h = 2.0 * xi_max / M;
  const int n = M + 1;
  for (int a = 0; a < n; ++a)
    for (int b = 0; b < n; ++b)
      for (int c = 0; c < n; ++c) {
        const int64_t k = ((int64_t)a * n + b) * n + c;
        const int idx[3] = {a - M / 2, b - M / 2, c - M / 2};
        double wt = h * h * h;
        for (int d = 0; d < 3; ++d) {
          xi[3 * k + d] = 2.0 * kPi * (idx[d] * h);
          if (idx[d] == -M / 2 || idx[d] == M / 2) wt *= 0.5;
        }
        W[k] = wt;
      }
  return 0;
}

// General form of the reduction: I = pref * sum_k W_k |nuhat_k - sigmahat(|xi_k|)|^2 (1 + (scale |xi_k|)^2)^{-s}.
// scale = 1, pref = (2 pi)^-3: orc_reduce.  The paper's norm (eq. 2.7, exponent s_paper < -1/2) on nodes given
// as xi' = 2 pi xi: scale = 1/(2 pi), s = -s_paper, pref = 1 (weights already in d xi).
double orc_reduce_ex(const double* nuhat, const double* xi, const double* W, int64_t K, double s, double scale,
                     double pref) {
  long double acc = 0;
  for (int64_t k = 0; k < K; ++k) {
    const double r2 = xi[3 * k] * xi[3 * k] + xi[3 * k + 1] * xi[3 * k + 1] + xi[3 * k + 2] * xi[3 * k + 2];
    const double r = std::sqrt(r2);
    const double dre = nuhat[2 * k] - orc_sigma_hat(r);
    const double dim = nuhat[2 * k + 1];
    acc += (long double)(W[k] * (dre * dre + dim * dim) * std::pow(1.0 + (scale * scale) * r2, -s));
  }
  return (double)(acc * (long double)pref);
}

// Two atomic measures against each other: I = (2 pi)^-3 sum_k W_k |a_k - b_k|^2 (1+|xi_k|^2)^{-s}.
double orc_reduce_pair(const double* a, const double* b, const double* xi, const double* W, int64_t K, double s) {
  long double acc = 0;
  for (int64_t k = 0; k < K; ++k) {
    const double r2 = xi[3 * k] * xi[3 * k] + xi[3 * k + 1] * xi[3 * k + 1] + xi[3 * k + 2] * xi[3 * k + 2];
    const double dre = a[2 * k] - b[2 * k], dim = a[2 * k + 1] - b[2 * k + 1];
    acc += (long double)(W[k] * (dre * dre + dim * dim) * std::pow(1.0 + r2, -s));
  }
  return (double)(acc / (8.0L * 3.14159265358979323846264338327950288L * 3.14159265358979323846264338327950288L *
                         3.14159265358979323846264338327950288L));
}

// sqrt(I) for a mesh against the unit sphere; also returns I.
int orc_weak_distance(const double* V, int64_t nV, const int32_t* F, int64_t nF, int rule, double s,
                      double R, int n_r, int n_th, int n_ph, double* dist, double* I) {
  double lam[64][3], om[64];
  const int q = rule_table(rule, lam, om);
  if (q < 0) return -2;
  const int64_t J = nF * q, K = (int64_t)n_r * n_th * n_ph;
  std::vector<double> x(3 * J), w(J), xi(3 * K), W(K), nu(2 * K);
  int rc = orc_nodes(V, nV, F, nF, rule, x.data(), w.data());
  if (rc) return rc;
  rc = orc_freq_nodes(n_r, n_th, n_ph, R, xi.data(), W.data());
  if (rc) return rc;
  orc_direct_sum(x.data(), w.data(), J, xi.data(), K, nu.data());
  *I = orc_reduce(nu.data(), xi.data(), W.data(), K, s);
  *dist = std::sqrt(*I);
  return 0;
}

}  // extern "C"
