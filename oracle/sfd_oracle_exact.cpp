// sfd_oracle_exact.cpp -- CPU ORACLE (part 2). TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Exact Fourier transform of the surface measure of a flat triangle mesh, the formula the prior-art codes sum
// directly (eq. 2.19; "several previous studies including [8, 38] employ the exact formula (2.19) and
// implement the direct summation in the frequency space"), in the e^{-i xi.x} convention of this repository
// (reading R1: gamma = 2A, and the (2 pi)^2 of the paper's e^{-2 pi i xi.x} disappears):
//
//   Q^(xi) = int_Q e^{-i xi.x} dS = -2A sum_{i=0}^{2} e^{-i alpha_i} / prod_{j != i} (alpha_i - alpha_j),   alpha_i = xi.p_i.
//
// This file evaluates exactly that expression, term by term as printed, and nothing else.  The paper warns that it
// "suffers from large cancellation errors when a simplex is almost degenerate or when the vector xi is almost
// orthogonal to one of the edges": the three quotients are O(1/d^2) for node distance d while their sum is O(1).
// The oracle therefore (i) works in binary128 (__float128, 113 bits; fp64 cannot carry the formula -- the one place
// where the oracle leaves fp64), which leaves ~1e-34 / d^2 of absolute error, and (ii) does NOT evaluate a pair (face,
// frequency) whose smallest |alpha_i - alpha_j| is below kSep * max(1, max|alpha_i|): such pairs are skipped and reported
// to the caller, and oracle/sfd_oracle.py evaluates the same printed formula for them with as many digits as the
// cancellation needs (mpmath), or -- when two or three alpha coincide exactly, where the printed formula is 0/0 --
// its limit, the divided difference with repeated nodes.  With kSep = 1e-5 the error of every pair evaluated here is
// below 1e-34 * 1e10 * (a few) = 1e-23 relative to the face's area.
//
// There is no series, no recursion and no branch on the size of |xi| h here: the CUDA kernel (csrc/exact.cu) has those,
// and the oracle must not share its structure.
//
// Pins (tests/test_exact_oracle_cpu.py): the same formula typed again in mpmath at 80-120 digits on generic and nearly
// degenerate inputs, the 64-point rule + direct sum (exact to degree 14) at small |xi| h, the area at xi = 0, eq. 2.20,
// the degenerate directions in closed form, the cube's product-of-sincs transform.
//
// Shares no code with paper_2304_06340_b200/.  Build: oracle/build_oracle.py (g++ ... -lquadmath).
#include <quadmath.h>

#include <cstdint>
#include <vector>

namespace {

typedef __float128 q128;
const q128 kSep = (q128)1e-5;   // (the fp64 literal: an exact threshold is not needed)

}  // namespace

extern "C" {

// out[k] (complex128, interleaved) = sum over the faces f of eq. 2.19, EXCEPT the pairs (k, f) whose alpha are too
// close for binary128 (above): those are written to skipped[2 n] = k, skipped[2 n + 1] = f and left out of the sum.
// Returns 0; -1 for an out-of-range vertex index; -2 if more than `cap` pairs had to be skipped (*n_skipped = the number).
int orc_exact_ft(const double* V, int64_t nV, const int32_t* F, int64_t nF, const double* xi, int64_t K, double* out,
                 int64_t* skipped, int64_t cap, int64_t* n_skipped) {
  for (int64_t f = 0; f < nF; ++f)
    for (int c = 0; c < 3; ++c)
      if (F[3 * f + c] < 0 || F[3 * f + c] >= nV) return -1;
  std::vector<q128> area2(nF);   // 2A = gamma of eq. 2.19
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
    area2[f] = sqrtq(cx * cx + cy * cy + cz * cz);
  }
  int64_t n_skip = 0;
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < K; ++k) {
    const q128 x0 = xi[3 * k], x1 = xi[3 * k + 1], x2 = xi[3 * k + 2];
    q128 re = (q128)0.0, im = (q128)0.0;
    for (int64_t f = 0; f < nF; ++f) {
      q128 al[3];
      for (int i = 0; i < 3; ++i) {
        const double* p = V + 3 * (int64_t)F[3 * f + i];
        al[i] = x0 * (q128)p[0] + x1 * (q128)p[1] + x2 * (q128)p[2];
      }
      q128 dmin = fabsq(al[0] - al[1]), amax = (q128)1.0;
      if (fabsq(al[1] - al[2]) < dmin) dmin = fabsq(al[1] - al[2]);
      if (fabsq(al[2] - al[0]) < dmin) dmin = fabsq(al[2] - al[0]);
      for (int i = 0; i < 3; ++i)
        if (fabsq(al[i]) > amax) amax = fabsq(al[i]);
      if (!(dmin > kSep * amax)) {
        int64_t at;
#pragma omp atomic capture
        at = n_skip++;
        if (at < cap) {
          skipped[2 * at] = k;
          skipped[2 * at + 1] = f;
        }
        continue;
      }
      // -2A sum_i e^{-i alpha_i} / prod_{j != i} (alpha_i - alpha_j)
      q128 sre = (q128)0.0, sim = (q128)0.0;
      for (int i = 0; i < 3; ++i) {
        q128 den = (q128)1.0;
        for (int j = 0; j < 3; ++j)
          if (j != i) den *= al[i] - al[j];
        q128 s, c;
        sincosq(al[i], &s, &c);
        sre += c / den;    // e^{-i alpha} = cos alpha - i sin alpha
        sim -= s / den;
      }
      re -= area2[f] * sre;
      im -= area2[f] * sim;
    }
    out[2 * k] = (double)re;
    out[2 * k + 1] = (double)im;
  }
  *n_skipped = n_skip;
  return n_skip > cap ? -2 : 0;
}

}  // extern "C"
