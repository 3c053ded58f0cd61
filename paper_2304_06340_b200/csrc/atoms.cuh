// atoms.cuh -- one atom of the triangle quadrature (eqs. 3.1-3.2): node L(u_i) = sum_m lam_im p_m, weight
// om_i * area.  Shared by nodes.cu (sfd_nodes) and by the source kernels of the transforms when they generate the
// atoms from the mesh instead of reading them (nufft3_glue.cu), so that both give the same doubles: every operation
// rounds once, in this order (no FMA contraction).
#pragma once
#include "common.cuh"

namespace sfd {

// A mesh + rule as a source of atoms j = f * rule + i (host-side description).
struct MeshAtoms {
  const double* d_V;
  int64_t nV;
  const int32_t* d_F;
  int64_t nF;
  int rule;
};

// rule = the four columns lam0[q], lam1[q], lam2[q], om[q] of the rule (4 x Q doubles, in shared or global memory)
__device__ __forceinline__ void atom_eval(const double* __restrict__ V, int64_t nV, const int32_t* __restrict__ F, int64_t j,
                                          int Q, const double* __restrict__ rule, double& x0, double& x1, double& x2,
                                          double& w, int32_t* flags = nullptr) {
  const int64_t f = j / Q;
  const int i = (int)(j - f * Q);
  const int32_t i0 = F[3 * f], i1 = F[3 * f + 1], i2 = F[3 * f + 2];
  if (i0 < 0 || i1 < 0 || i2 < 0 || i0 >= nV || i1 >= nV || i2 >= nV) {
    x0 = x1 = x2 = w = __longlong_as_double(0x7ff8000000000000LL);   // a face with a bad index poisons its atoms
    if (flags) atomicOr(flags, kFlagBadIndex);                       // ... and is reported at the next synchronising call
    return;
  }
  double p0[3], p1[3], p2[3], e1[3], e2[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    p0[c] = V[3 * (int64_t)i0 + c];
    p1[c] = V[3 * (int64_t)i1 + c];
    p2[c] = V[3 * (int64_t)i2 + c];
    e1[c] = __dsub_rn(p1[c], p0[c]);
    e2[c] = __dsub_rn(p2[c], p0[c]);
  }
  const double cx = __dsub_rn(__dmul_rn(e1[1], e2[2]), __dmul_rn(e1[2], e2[1]));
  const double cy = __dsub_rn(__dmul_rn(e1[2], e2[0]), __dmul_rn(e1[0], e2[2]));
  const double cz = __dsub_rn(__dmul_rn(e1[0], e2[1]), __dmul_rn(e1[1], e2[0]));
  const double n2 = __dadd_rn(__dadd_rn(__dmul_rn(cx, cx), __dmul_rn(cy, cy)), __dmul_rn(cz, cz));
  const double area = __dmul_rn(0.5, __dsqrt_rn(n2));
  const double l0 = rule[i], l1 = rule[Q + i], l2 = rule[2 * Q + i];
  x0 = __dadd_rn(__dadd_rn(__dmul_rn(l0, p0[0]), __dmul_rn(l1, p1[0])), __dmul_rn(l2, p2[0]));
  x1 = __dadd_rn(__dadd_rn(__dmul_rn(l0, p0[1]), __dmul_rn(l1, p1[1])), __dmul_rn(l2, p2[1]));
  x2 = __dadd_rn(__dadd_rn(__dmul_rn(l0, p0[2]), __dmul_rn(l1, p1[2])), __dmul_rn(l2, p2[2]));
  w = __dmul_rn(rule[3 * Q + i], area);
}

}  // namespace sfd
