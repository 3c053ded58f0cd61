// mesh.cu -- A1/A2: icosahedral discretization T_N of S^2 on the device: "an additional vertice is
// chosen to be the midpoint of each edge ... divides each face into four sub-triangles and the projection of
// those new vertices onto S^2", 10*4^N+2 vertices and 20*4^N faces.
//
// Numbering (reading R4): the midpoint of the undirected edge {a<b} gets id nV + rank of the key
// a*nV+b among all edge keys.  On a closed, consistently oriented mesh every undirected edge occurs exactly once
// as a directed face edge u->v with u<v, so no sort is needed: rank = (#edges whose smaller end is < a) +
// (#up-neighbours of a that are < b).  Integer-exact and independent of thread order: a count of up-neighbours
// per vertex (atomic append, order irrelevant), one exclusive scan, and a <=6-element comparison per edge.
// Vertex arithmetic rounds once per operation (no FMA contraction) so that vertices are the same doubles
// everywhere.
#include <cmath>

#include "internal.cuh"

namespace sfd {
namespace {

constexpr int kMaxUp = 6;  // valence of an icosphere vertex is 5 or 6

// T_0: the three golden rectangles, scaled to the unit sphere; faces oriented outward.
const int32_t kIcoFaces[20][3] = {{0, 5, 1},  {0, 1, 7},   {0, 11, 5}, {0, 7, 10}, {0, 10, 11}, {1, 5, 9},  {1, 8, 7},
                                  {1, 9, 8},  {2, 3, 4},   {2, 6, 3},  {2, 4, 11}, {2, 10, 6},  {2, 11, 10}, {3, 9, 4},
                                  {3, 6, 8},  {3, 8, 9},   {4, 9, 5},  {4, 5, 11}, {6, 7, 8},   {6, 10, 7}};

void icosahedron_vertices(double* v) {
  const double g = (1.0 + std::sqrt(5.0)) / 2.0;
  const double len = std::sqrt(1.0 + g * g);
  const double s[12][3] = {{-1, g, 0}, {1, g, 0}, {-1, -g, 0}, {1, -g, 0}, {0, -1, g}, {0, 1, g},
                           {0, -1, -g}, {0, 1, -g}, {g, 0, -1}, {g, 0, 1}, {-g, 0, -1}, {-g, 0, 1}};
  for (int i = 0; i < 12; ++i)
    for (int c = 0; c < 3; ++c) v[3 * i + c] = s[i][c] / len;
}

__global__ void __launch_bounds__(256) up_neighbours_kernel(const int32_t* __restrict__ F, int64_t nF,
                                                            int32_t* __restrict__ cnt, int32_t* __restrict__ upn) {
  const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= nF) return;
  const int32_t i[3] = {F[3 * f], F[3 * f + 1], F[3 * f + 2]};
#pragma unroll
  for (int e = 0; e < 3; ++e) {
    const int32_t a = i[e], b = i[(e + 1) % 3];
    if (a < b) {
      const int slot = atomicAdd(&cnt[a], 1);
      if (slot < kMaxUp) upn[(int64_t)a * kMaxUp + slot] = b;
    }
  }
}

__device__ __forceinline__ int32_t midpoint_id(int32_t a, int32_t b, int32_t nV, const int32_t* __restrict__ cnt,
                                               const int32_t* __restrict__ off, const int32_t* __restrict__ upn) {
  const int32_t lo = min(a, b), hi = max(a, b);
  const int c = min(cnt[lo], kMaxUp);
  int r = off[lo];
  for (int s = 0; s < c; ++s) r += upn[(int64_t)lo * kMaxUp + s] < hi ? 1 : 0;
  return nV + r;
}

__global__ void __launch_bounds__(256) split_faces_kernel(const int32_t* __restrict__ F, int64_t nF, int32_t nV,
                                                          const int32_t* __restrict__ cnt, const int32_t* __restrict__ off,
                                                          const int32_t* __restrict__ upn, int32_t* __restrict__ Fout,
                                                          double* __restrict__ V) {
  const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= nF) return;
  const int32_t i0 = F[3 * f], i1 = F[3 * f + 1], i2 = F[3 * f + 2];
  const int32_t m01 = midpoint_id(i0, i1, nV, cnt, off, upn);
  const int32_t m12 = midpoint_id(i1, i2, nV, cnt, off, upn);
  const int32_t m20 = midpoint_id(i2, i0, nV, cnt, off, upn);
  int32_t* o = Fout + 12 * f;
  o[0] = i0;  o[1] = m01;  o[2] = m20;
  o[3] = i1;  o[4] = m12;  o[5] = m01;
  o[6] = i2;  o[7] = m20;  o[8] = m12;
  o[9] = m01; o[10] = m12; o[11] = m20;
  // the face that sees the edge as u->v with u<v writes the projected midpoint (A2)
  const int32_t ea[3] = {i0, i1, i2}, eb[3] = {i1, i2, i0}, em[3] = {m01, m12, m20};
#pragma unroll
  for (int e = 0; e < 3; ++e) {
    if (ea[e] < eb[e]) {
      const double* p = V + 3 * (int64_t)ea[e];
      const double* q = V + 3 * (int64_t)eb[e];
      const double mx = __dadd_rn(p[0], q[0]), my = __dadd_rn(p[1], q[1]), mz = __dadd_rn(p[2], q[2]);
      double s = __dmul_rn(mx, mx);
      s = __dadd_rn(s, __dmul_rn(my, my));
      s = __dadd_rn(s, __dmul_rn(mz, mz));
      const double n = __dsqrt_rn(s);
      double* out = V + 3 * (int64_t)em[e];
      out[0] = __ddiv_rn(mx, n);
      out[1] = __ddiv_rn(my, n);
      out[2] = __ddiv_rn(mz, n);
    }
  }
}

int64_t pow4(int level) { return (int64_t)1 << (2 * level); }

struct MeshWork {
  size_t faces, cnt, off, upn, scan, total;
};
MeshWork mesh_work(int level) {
  MeshWork m{};
  if (level == 0) return m;
  const int64_t nVp = 10 * pow4(level - 1) + 2, nFp = 20 * pow4(level - 1);
  m.faces = align_up((size_t)nFp * 12);
  m.cnt = align_up((size_t)nVp * 4);
  m.off = align_up((size_t)nVp * 4);
  m.upn = align_up((size_t)nVp * kMaxUp * 4);
  m.scan = align_up(scan_workspace(nVp));
  m.total = m.faces + m.cnt + m.off + m.upn + m.scan;
  return m;
}

}  // namespace

int mesh_sizes(int level, int64_t* nV, int64_t* nF, size_t* work_bytes) {
  SFD_REQUIRE(level >= 0 && level <= 10, SFD_ERR_INVALID_ARG, "icosphere level %d outside [0,10]", level);
  if (nV) *nV = 10 * pow4(level) + 2;
  if (nF) *nF = 20 * pow4(level);
  if (work_bytes) *work_bytes = mesh_work(level).total;
  return SFD_OK;
}

int mesh_icosphere(int level, double* d_V, int32_t* d_F, void* d_work, size_t work_bytes, cudaStream_t st) {
  SFD_REQUIRE(level >= 0 && level <= 10, SFD_ERR_INVALID_ARG, "icosphere level %d outside [0,10]", level);
  SFD_REQUIRE(d_V && d_F, SFD_ERR_NULL, "sfd_mesh_icosphere: NULL output buffer");
  const MeshWork mw = mesh_work(level);
  SFD_REQUIRE(work_bytes >= mw.total && (mw.total == 0 || d_work), SFD_ERR_WORKSPACE_TOO_SMALL,
              "icosphere level %d needs %zu workspace bytes, got %zu", level, mw.total, work_bytes);
  static double v0[36];
  static bool have_v0 = false;
  if (!have_v0) {
    icosahedron_vertices(v0);
    have_v0 = true;
  }
  char* w = static_cast<char*>(d_work);
  int32_t* faces_alt = reinterpret_cast<int32_t*>(w);
  int32_t* cnt = reinterpret_cast<int32_t*>(w + mw.faces);
  int32_t* off = reinterpret_cast<int32_t*>(w + mw.faces + mw.cnt);
  int32_t* upn = reinterpret_cast<int32_t*>(w + mw.faces + mw.cnt + mw.off);
  void* scan_w = w + mw.faces + mw.cnt + mw.off + mw.upn;
  // faces ping-pong between d_F and the workspace so that the last step writes d_F
  int32_t* cur = (level % 2 == 0) ? d_F : faces_alt;
  int32_t* nxt = (level % 2 == 0) ? faces_alt : d_F;
  SFD_CUDA_TRY(cudaMemcpyAsync(d_V, v0, sizeof(v0), cudaMemcpyHostToDevice, st));
  SFD_CUDA_TRY(cudaMemcpyAsync(cur, kIcoFaces, sizeof(kIcoFaces), cudaMemcpyHostToDevice, st));
  int64_t nV = 12, nF = 20;
  for (int l = 0; l < level; ++l) {
    SFD_CUDA_TRY(cudaMemsetAsync(cnt, 0, (size_t)nV * 4, st));
    const unsigned blocks = (unsigned)((nF + 255) / 256);
    up_neighbours_kernel<<<blocks, 256, 0, st>>>(cur, nF, cnt, upn);
    SFD_TRY(launch_check("up_neighbours_kernel"));
    SFD_TRY(exclusive_scan_i32(cnt, off, nV, nullptr, scan_w, mw.scan, st));
    split_faces_kernel<<<blocks, 256, 0, st>>>(cur, nF, (int32_t)nV, cnt, off, upn, nxt, d_V);
    SFD_TRY(launch_check("split_faces_kernel"));
    nV += 3 * nF / 2;
    nF *= 4;
    int32_t* t = cur;
    cur = nxt;
    nxt = t;
  }
  return SFD_OK;
}

}  // namespace sfd
