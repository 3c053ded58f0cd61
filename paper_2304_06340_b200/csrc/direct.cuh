// direct.cuh -- launcher interface of the fp64 direct-summation kernel (direct.cu).
#pragma once
#include "common.cuh"

namespace sfd {

struct DirectPlan {
  int T;                // targets per thread
  int64_t blocks_k;     // CTAs along the target axis
  int nsplit;           // CTAs along the source axis (partials combined in a fixed order)
  int64_t j_per_split;  // sources per split (multiple of the tile)
  size_t work_bytes;    // workspace for the partial sums (0 when nsplit == 1)
};

DirectPlan direct_plan(int64_t J, int64_t K);

// nuhat[k] = sum_j w_j exp(-i xi_k . x_j); d_work must hold direct_plan(J,K).work_bytes.
int direct_sum(const double* d_x, const double* d_w, int64_t J, const double* d_xi, int64_t K, double* d_nuhat,
               void* d_work, size_t work_bytes, cudaStream_t st);

}  // namespace sfd
