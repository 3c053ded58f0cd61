// sfd_oracle_exact.cpp -- CPU ORACLE (part 2). TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Exact Fourier transform of the surface measure of a flat triangle mesh, the formula the prior-art codes sum
// directly (eq. 2.19, "several previous studies including [8, 38] employ the exact formula (2.19) and
// implement the direct summation in the frequency space"), in the e^{-i xi.x} convention of this repository
// (reading R1):
//
//   Q^(xi) = int_Q e^{-i xi.x} dS = 2A int_{Q_0} e^{-i(alpha_0 + u s + v t)} ds dt = 2A exp[z_0, z_1, z_2],
//   z_i = -i alpha_i,  alpha_i = xi.p_i,
//
// where exp[z_0,z_1,z_2] is the second divided difference of exp (Hermite-Genocchi: the integral of f'' over the
// simplex spanned by the nodes).  For distinct nodes it is sum_i e^{z_i} / prod_{j!=i} (z_i - z_j), which is
// eq. 2.19: -2A sum_i e^{-i alpha_i} / prod_{j!=i} (alpha_i - alpha_j)  (gamma = 2A, and (2 pi)^2 from the paper's
// e^{-2 pi i xi.x}).  The paper notes that "the closed form (2.19) suffers from large cancellation errors when a
// simplex is almost degenerate or when the vector xi is almost orthogonal to one of the edges"; the oracle
// therefore evaluates the divided difference by its textbook definitions, in binary128 (__float128, 113 bits --
// fp64 cannot carry eq. 2.19; this is the one place where the oracle leaves fp64, and says so):
//
//   * all three nodes within distance 1 of each other: the power series  exp[z_0,z_1,z_2] =
//     e^{z_0} sum_{n>=0} h_n(a, b) / (n+2)!,  a = z_1 - z_0, b = z_2 - z_0, h_n = sum_{i+j=n} a^i b^j
//     (the divided difference of z^m at (0,a,b) is the complete homogeneous polynomial h_{m-2}(a,b));
//   * otherwise the recursive definition  exp[z_a,z_b,z_c] = (exp[z_b,z_c] - exp[z_a,z_b]) / (z_c - z_a)  with
//     (a,c) the pair farthest apart (|z_c - z_a| > 1), and first divided differences
//     exp[x,y] = e^{x} phi_1(y - x),  phi_1(w) = (e^w - 1)/w  (its power series for |w| < 1/2).
//
// Pins (tests/test_exact_oracle_cpu.py): eq. 2.19 evaluated literally with mpmath at 60 digits on generic inputs, the
// 64-point rule + direct sum (exact to degree 14) at small |xi| h, the area at xi = 0, eq. 2.20, the degenerate
// directions (xi normal to the face / orthogonal to an edge) in closed form, the cube's product-of-sincs transform.
//
// Shares no code with paper_2304_06340_b200/.  Build: oracle/build_oracle.py (g++ ... -lquadmath).
#include <quadmath.h>

#include <cstdint>
#include <vector>

namespace {

typedef __float128 q128;

struct cq {
  q128 re, im;
};
inline cq operator+(cq a, cq b) { return {a.re + b.re, a.im + b.im}; }
inline cq operator-(cq a, cq b) { return {a.re - b.re, a.im - b.im}; }
inline cq operator*(cq a, cq b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
inline cq scale(cq a, q128 s) { return {a.re * s, a.im * s}; }
// e^{-i t}
inline cq expmi(q128 t) {
  q128 s, c;
  sincosq(t, &s, &c);
  return {c, -s};
}

// phi_1(-i d) = (e^{-i d} - 1) / (-i d)
cq phi1_mi(q128 d) {
  if (fabsq(d) < (q128)0.5) {
    // sum_{n>=0} (-i d)^n / (n+1)!
    cq term = {(q128)1.0, (q128)0.0}, acc = {(q128)0.0, (q128)0.0};
    for (int n = 0; n < 60; ++n) {
      acc = acc + scale(term, (q128)1.0);
      // term_{n+1} = term_n * (-i d) / (n+2)
      const cq t2 = {term.im * d, -term.re * d};
      term = scale(t2, (q128)1.0 / (q128)(n + 2));
    }
    return acc;
  }
  const cq e = expmi(d);
  // (e - 1) / (-i d) = i (e - 1) / d
  const cq num = {e.re - (q128)1.0, e.im};
  return {-num.im / d, num.re / d};
}

// exp[-i x, -i y] = e^{-i x} phi_1(-i (y - x))
cq dd1(q128 x, q128 y) { return expmi(x) * phi1_mi(y - x); }

// exp[-i a0, -i a1, -i a2]
cq dd2(q128 a0, q128 a1, q128 a2) {
  const q128 d01 = fabsq(a1 - a0), d02 = fabsq(a2 - a0), d12 = fabsq(a2 - a1);
  q128 dmax = d01 > d02 ? d01 : d02;
  if (d12 > dmax) dmax = d12;
  if (dmax <= (q128)1.0) {
    // e^{-i a0} sum_n h_n(a, b) / (n+2)!,  a = -i u, b = -i v  =>  h_n(a,b) = (-i)^n H_n(u,v)
    const q128 u = a1 - a0, v = a2 - a0;
    q128 H = (q128)1.0, vp = (q128)1.0, fact = (q128)2.0;   // H_0, v^0, 2!
    cq acc = {(q128)0.0, (q128)0.0};
    for (int n = 0; n < 70; ++n) {
      const q128 t = H / fact;
      switch (n & 3) {   // (-i)^n
        case 0: acc.re += t; break;
        case 1: acc.im -= t; break;
        case 2: acc.re -= t; break;
        default: acc.im += t; break;
      }
      vp *= v;
      H = u * H + vp;   // H_{n+1} = u H_n + v^{n+1}
      fact *= (q128)(n + 3);
    }
    return expmi(a0) * acc;
  }
  // farthest pair (a, c), middle b
  q128 xa, xb, xc;
  if (d02 >= d01 && d02 >= d12) {
    xa = a0; xb = a1; xc = a2;
  } else if (d01 >= d12) {
    xa = a0; xb = a2; xc = a1;
  } else {
    xa = a1; xb = a0; xc = a2;
  }
  const cq num = dd1(xb, xc) - dd1(xa, xb);
  // divide by z_c - z_a = -i (xc - xa):  num / (-i D) = i num / D
  const q128 D = xc - xa;
  return {-num.im / D, num.re / D};
}

}  // namespace

extern "C" {

// out[k] (complex128, interleaved) = sum_f 2 A_f exp[-i xi_k.p_0, -i xi_k.p_1, -i xi_k.p_2]  (eq. 2.19).
// Returns 0, or -1 for an out-of-range vertex index.
int orc_exact_ft(const double* V, int64_t nV, const int32_t* F, int64_t nF, const double* xi, int64_t K, double* out) {
  for (int64_t f = 0; f < nF; ++f)
    for (int c = 0; c < 3; ++c)
      if (F[3 * f + c] < 0 || F[3 * f + c] >= nV) return -1;
  std::vector<q128> area2(nF);
  for (int64_t f = 0; f < nF; ++f) {
    const double* p0 = V + 3 * (int64_t)F[3 * f];
    const double* p1 = V + 3 * (int64_t)F[3 * f + 1];
    const double* p2 = V + 3 * (int64_t)F[3 * f + 2];
    q128 e1[3], e2[3];
    for (int c = 0; c < 3; ++c) {
      e1[c] = (q128)p1[c] - (q128)p0[c];
      e2[c] = (q128)p2[c] - (q128)p0[c];
    }
    const q128 cx = e1[1] * e2[2] - e1[2] * e2[1], cy = e1[2] * e2[0] - e1[0] * e2[2], cz = e1[0] * e2[1] - e1[1] * e2[0];
    area2[f] = sqrtq(cx * cx + cy * cy + cz * cz);   // 2A = gamma of eq. 2.19
  }
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < K; ++k) {
    const q128 x0 = xi[3 * k], x1 = xi[3 * k + 1], x2 = xi[3 * k + 2];
    cq acc = {(q128)0.0, (q128)0.0};
    for (int64_t f = 0; f < nF; ++f) {
      q128 al[3];
      for (int i = 0; i < 3; ++i) {
        const double* p = V + 3 * (int64_t)F[3 * f + i];
        al[i] = x0 * (q128)p[0] + x1 * (q128)p[1] + x2 * (q128)p[2];
      }
      acc = acc + scale(dd2(al[0], al[1], al[2]), area2[f]);
    }
    out[2 * k] = (double)acc.re;
    out[2 * k + 1] = (double)acc.im;
  }
  return 0;
}

}  // extern "C"
