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

DirectPlan direct_plan(int64_t J, int64_t K, int T_force = 0);

// nuhat[k] = sum_j w_j exp(-i xi_k . x_j); d_work must hold direct_plan(J,K).work_bytes.
int direct_sum(const double* d_x, const double* d_w, int64_t J, const double* d_xi, int64_t K, double* d_nuhat,
               void* d_work, size_t work_bytes, cudaStream_t st);

size_t direct_ball_work_bytes(int64_t J, int64_t K);   // workspace of direct_sum_ball (may exceed direct_sum's)
// The same on the nodes of the ball rule taken from its 1-D tables (direct.cu BALL): *used = false when not applicable.
int direct_sum_ball(const double* d_x, const double* d_w, int64_t J, const double* d_tables, int n_r, int n_th, int n_ph,
                    int a0, int a1, int b0, double* d_nuhat, void* d_work, size_t work_bytes, cudaStream_t st, bool* used);

}  // namespace sfd
