// fft.cu -- A5-5 + A5-6: deconvolution and the inner uniform FFT of the type-3 NUFFT, pruned.
//
// The inner type-2 step needs v[m] = sum_l b~[l] exp(-2 pi i l.m / n2) where b~ (the deconvolved fine grid) is
// non-zero only on the central nf = n2/2 modes of every axis and v is needed only on the band of n2/2 + w + O(1)
// cells per axis that the targets touch (SURVEY.md 8(a) "Consequences" (i)).  A full n2^3 transform (what the
// paper's library does on the lattice, "fastest GPU version ... provided by CUDA Toolkit") would read and write
// 8x more data than that, and at BASELINE.json config 5 (n2 = 2700) would not fit 180 GB.  Here the 3-D transform
// is three passes of 1-D transforms, each over the rows that are non-zero on input and cut to the band on output:
//     A (axis 2): nf0*nf1 rows  -> [nf0][nf1][nout2]      (also multiplies by the deconvolution factors, A5-5)
//     B (axis 1): nf0*nout2 rows -> [nf0][nout1][nout2]
//     C (axis 0): nout1*nout2 rows -> [nout0][nout1][nout2]
// Each row transform runs entirely in shared memory: a tile of `tb` rows is loaded with coalesced 16-byte accesses
// (along the axis for pass A, across the rows for B and C), zero-padded to n2, transformed in place by a
// decimation-in-frequency mixed-radix (4,2,3,5) FFT -- consecutive threads work on the same butterfly of
// consecutive rows, so every shared-memory access is a contiguous run (row pitch tb+1: the transposing load of pass
// A is conflict-free too) -- and the band is written out through the digit-reversal table.  HBM traffic per pass is
// one read of the input rows and one write of the band: ~16x less than padded library transforms at config 3.
#include <algorithm>
#include <cstdlib>
#include <map>
#include <mutex>
#include <vector>

#include "fft.cuh"

namespace sfd {
namespace {


__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
  return make_double2(__fma_rn(a.x, b.x, -a.y * b.y), __fma_rn(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ double2 mul_mi(double2 a) { return make_double2(a.y, -a.x); }   // a * (-i)
__device__ __forceinline__ double2 mul_pi(double2 a) { return make_double2(-a.y, a.x); }   // a * (+i)

// Global-memory elements of a pass: fp64, or single precision when FftPass::f32 (the arithmetic and the shared-memory
// rows stay fp64 either way).  `i` counts elements of the array's own type.
__device__ __forceinline__ double ld_real(const void* base, int64_t i, int f32) {
  return f32 ? (double)__ldcs(static_cast<const float*>(base) + i) : __ldcs(static_cast<const double*>(base) + i);
}
__device__ __forceinline__ double2 ld_cplx_cs(const void* base, int64_t i, int f32) {
  if (f32) {
    const float2 v = __ldcs(static_cast<const float2*>(base) + i);
    return make_double2((double)v.x, (double)v.y);
  }
  return __ldcs(static_cast<const double2*>(base) + i);
}
__device__ __forceinline__ double2 ld_cplx_cg(const void* base, int64_t i, int f32) {
  if (f32) {
    const float2 v = __ldcg(static_cast<const float2*>(base) + i);
    return make_double2((double)v.x, (double)v.y);
  }
  return __ldcg(static_cast<const double2*>(base) + i);
}
__device__ __forceinline__ void st_cplx(double2* base, int64_t i, double2 v, int f32) {
  if (f32) reinterpret_cast<float2*>(base)[i] = make_float2((float)v.x, (float)v.y);
  else base[i] = v;
}

// ---- radix-R butterflies on register arrays: x <- DFT_R(x), forward sign, natural output order -------------------
template <int R>
__device__ __forceinline__ void bfly(double2 (&x)[R]);
template <>
__device__ __forceinline__ void bfly<1>(double2 (&)[1]) {}
template <>
__device__ __forceinline__ void bfly<2>(double2 (&x)[2]) {
  const double2 a = x[0], b = x[1];
  x[0] = cadd(a, b);
  x[1] = csub(a, b);
}
template <>
__device__ __forceinline__ void bfly<3>(double2 (&x)[3]) {
  const double2 x0 = x[0], x1 = x[1], x2 = x[2];
  const double2 t1 = cadd(x1, x2);
  const double2 t2 = make_double2(x0.x - 0.5 * t1.x, x0.y - 0.5 * t1.y);
  const double h = 0.86602540378443864676;
  const double2 t3 = make_double2(h * (x1.x - x2.x), h * (x1.y - x2.y));
  x[0] = cadd(x0, t1);
  x[1] = cadd(t2, mul_mi(t3));
  x[2] = cadd(t2, mul_pi(t3));
}
template <>
__device__ __forceinline__ void bfly<4>(double2 (&x)[4]) {
  const double2 t0 = cadd(x[0], x[2]), t1 = csub(x[0], x[2]), t2 = cadd(x[1], x[3]), t3 = csub(x[1], x[3]);
  x[0] = cadd(t0, t2);
  x[1] = cadd(t1, mul_mi(t3));
  x[2] = csub(t0, t2);
  x[3] = cadd(t1, mul_pi(t3));
}
template <>
__device__ __forceinline__ void bfly<5>(double2 (&x)[5]) {
  const double2 x0 = x[0], x1 = x[1], x2 = x[2], x3 = x[3], x4 = x[4];
  const double c1 = 0.30901699437494742410, c2 = -0.80901699437494742410;
  const double s1 = 0.95105651629515357212, s2 = 0.58778525229247312917;
  const double2 t1 = cadd(x1, x4), t2 = cadd(x2, x3), t3 = csub(x1, x4), t4 = csub(x2, x3);
  const double2 a1 = make_double2(x0.x + c1 * t1.x + c2 * t2.x, x0.y + c1 * t1.y + c2 * t2.y);
  const double2 a2 = make_double2(x0.x + c2 * t1.x + c1 * t2.x, x0.y + c2 * t1.y + c1 * t2.y);
  const double2 b1 = make_double2(s1 * t3.x + s2 * t4.x, s1 * t3.y + s2 * t4.y);
  const double2 b2 = make_double2(s2 * t3.x - s1 * t4.x, s2 * t3.y - s1 * t4.y);
  x[0] = make_double2(x0.x + t1.x + t2.x, x0.y + t1.y + t2.y);
  x[1] = cadd(a1, mul_mi(b1));
  x[2] = cadd(a2, mul_mi(b2));
  x[3] = cadd(a2, mul_pi(b2));
  x[4] = cadd(a1, mul_pi(b1));
}

template <>
__device__ __forceinline__ void bfly<7>(double2 (&x)[7]) {
  // X_k = x0 + sum_j t_j cos(2 pi j k / 7) - i sum_j d_j sin(2 pi j k / 7),  t_j = x_j + x_{7-j}, d_j = x_j - x_{7-j}
  const double c1 = 0.62348980185873353053, c2 = -0.22252093395631440429, c3 = -0.90096886790241912624;
  const double s1 = 0.78183148246802980871, s2 = 0.97492791218182360702, s3 = 0.43388373911755812048;
  const double2 x0 = x[0];
  const double2 t1 = cadd(x[1], x[6]), t2 = cadd(x[2], x[5]), t3 = cadd(x[3], x[4]);
  const double2 d1 = csub(x[1], x[6]), d2 = csub(x[2], x[5]), d3 = csub(x[3], x[4]);
  const double2 a1 = make_double2(x0.x + c1 * t1.x + c2 * t2.x + c3 * t3.x, x0.y + c1 * t1.y + c2 * t2.y + c3 * t3.y);
  const double2 a2 = make_double2(x0.x + c2 * t1.x + c3 * t2.x + c1 * t3.x, x0.y + c2 * t1.y + c3 * t2.y + c1 * t3.y);
  const double2 a3 = make_double2(x0.x + c3 * t1.x + c1 * t2.x + c2 * t3.x, x0.y + c3 * t1.y + c1 * t2.y + c2 * t3.y);
  const double2 b1 = make_double2(s1 * d1.x + s2 * d2.x + s3 * d3.x, s1 * d1.y + s2 * d2.y + s3 * d3.y);
  const double2 b2 = make_double2(s2 * d1.x - s3 * d2.x - s1 * d3.x, s2 * d1.y - s3 * d2.y - s1 * d3.y);
  const double2 b3 = make_double2(s3 * d1.x - s1 * d2.x + s2 * d3.x, s3 * d1.y - s1 * d2.y + s2 * d3.y);
  x[0] = make_double2(x0.x + t1.x + t2.x + t3.x, x0.y + t1.y + t2.y + t3.y);
  x[1] = cadd(a1, mul_mi(b1));
  x[2] = cadd(a2, mul_mi(b2));
  x[3] = cadd(a3, mul_mi(b3));
  x[4] = cadd(a3, mul_pi(b3));
  x[5] = cadd(a2, mul_pi(b2));
  x[6] = cadd(a1, mul_pi(b1));
}

// One decimation-in-frequency stage of radix R.  A thread owns butterfly bf of CG consecutive rows of the tile: the
// index arithmetic and the R-1 twiddle loads are paid once per thread and amortised over CG butterflies, whose
// chains are independent (instruction-level parallelism on top of the warps).  Lanes run over (bf, column group) with
// the group fastest; with the odd row pitch tbp every 8 lanes of an LDS/STS.128 fall into distinct bank groups.
template <int R, int CG>
__device__ __forceinline__ void dif_stage(double2* __restrict__ a, const double2* __restrict__ tw, int N, int L,
                                          unsigned magic, int cgsh, int tbp, int tid, int nthreads) {
  const int Ls = L / R;
  const int tstep = N / L;
  const int nitems = (N / R) << cgsh;
  const int st = Ls * tbp;
  for (int idx = tid; idx < nitems; idx += nthreads) {
    const int bf = idx >> cgsh, cg = idx & ((1 << cgsh) - 1);
    const int b = Ls == 1 ? bf : (int)__umulhi((unsigned)bf, magic);   // bf / Ls (exact: bf * Ls < 2^32)
    const int j = bf - b * Ls;
    double2* base = a + (b * L + j) * tbp + cg * CG;
    double2 w[R];
#pragma unroll
    for (int p = 1; p < R; ++p) w[p] = tw[p * j * tstep];
#pragma unroll
    for (int c = 0; c < CG; ++c) {
      double2 x[R];
#pragma unroll
      for (int q = 0; q < R; ++q) x[q] = base[q * st + c];
      bfly<R>(x);
      base[c] = x[0];
#pragma unroll
      for (int p = 1; p < R; ++p) base[p * st + c] = cmul(x[p], w[p]);
    }
  }
}

// Two consecutive decimation-in-frequency stages (radices R1 then R2; R2 = 1: a single stage) fused in registers:
// a thread owns the R1 R2 elements b L + j' + q1 L/R1 + q2 L/(R1 R2) of one row, which stage s (radix R1 over q1, twiddle
// w_L^{(j' + q2 Lq) p1}) and stage s+1 (radix R2 over q2 inside block (b, p1), twiddle w_{L/R1}^{j' p2}) map onto
// themselves: one shared-memory round trip instead of two.
template <int R1, int R2>
__device__ __forceinline__ void fused_stages(double2* __restrict__ a, const double2* __restrict__ tw, int N, int L,
                                             unsigned magic, int tb, int tbp, int tsh, int tid, int nthreads) {
  constexpr int R = R1 * R2;
  const int Lq = L / R;              // j' range
  const int L1 = L / R1;             // stride of q1
  const int tstep = N / L;           // twiddle index step of stage s; stage s+1 uses tstep * R1
  const int ngroups = N / R;
  for (int idx = tid; idx < (ngroups << tsh); idx += nthreads) {
    const int g = idx >> tsh, col = idx & (tb - 1);
    const int b = Lq == 1 ? g : (int)__umulhi((unsigned)g, magic);   // g / Lq
    const int jp = g - b * Lq;
    double2* base = a + (b * L + jp) * tbp + col;
    double2 v[R1][R2];
#pragma unroll
    for (int q1 = 0; q1 < R1; ++q1)
#pragma unroll
      for (int q2 = 0; q2 < R2; ++q2) v[q1][q2] = base[(q1 * L1 + q2 * Lq) * tbp];
    // stage s
#pragma unroll
    for (int q2 = 0; q2 < R2; ++q2) {
      double2 x[R1];
#pragma unroll
      for (int q1 = 0; q1 < R1; ++q1) x[q1] = v[q1][q2];
      bfly<R1>(x);
      const int tj = (jp + q2 * Lq) * tstep;
      v[0][q2] = x[0];
#pragma unroll
      for (int p1 = 1; p1 < R1; ++p1) v[p1][q2] = cmul(x[p1], tw[p1 * tj]);
    }
    // stage s+1
    if (R2 > 1) {
      const int tj2 = jp * tstep * R1;
#pragma unroll
      for (int p1 = 0; p1 < R1; ++p1) {
        double2 x[R2];
#pragma unroll
        for (int q2 = 0; q2 < R2; ++q2) x[q2] = v[p1][q2];
        bfly<R2>(x);
        v[p1][0] = x[0];
#pragma unroll
        for (int p2 = 1; p2 < R2; ++p2) v[p1][p2] = cmul(x[p2], tw[p2 * tj2]);
      }
    }
#pragma unroll
    for (int p1 = 0; p1 < R1; ++p1)
#pragma unroll
      for (int p2 = 0; p2 < R2; ++p2) base[(p1 * L1 + p2 * Lq) * tbp] = v[p1][p2];
  }
}

// FftPass::ball: normalised squared distance of column `lo` from the axis of the ellipsoid the consumer reads.
__device__ __forceinline__ double ball_q(const FftPass& P, int64_t lo) {
  const int64_t ia = P.ball == 1 ? lo / P.ball_nb : 0;
  const double da = ((double)ia - P.ball_ca) * P.ball_ira;
  const double db = ((double)(lo - ia * (P.ball == 1 ? P.ball_nb : 0)) - P.ball_cb) * P.ball_irb;
  return da * da + db * db;
}

// =====================================================================================================================
// Fixed-geometry pruned passes.  For the transform lengths the type-3 planner emits on BASELINE.json's configurations
// (n2 = 360, 672, 720, 1344, 1440, 2700) with exactly the central half of the inputs non-zero (n_in = N/2: sigma = 2), the
// pass is compiled for the length: N = G1 G2 G3 with three register-resident groups G = A B <= 16 (radix A then radix B
// fused, as in fused_stages), every stride, twiddle step and loop bound a compile-time constant.  Against the generic
// kernel above this removes the zero-padding and the separate load phase (group 1 reads its inputs straight from global
// memory -- with A1 = 4 the elements q1 = 1, 2 of every radix-4 butterfly lie in the zero half, so only q1 = 0, 3 are
// loaded and the butterfly costs 4 complex additions), the separate store phase of the strided passes (group 3 writes the
// band straight from registers: in those passes every output element is its own 16 TB-byte segment whatever the order),
// the trivial twiddles of the last stage, and the run-time index arithmetic (~58 of 124 instructions per point in the
// generic kernel, profiles/r1j_fft_phases.md).  Shared-memory round trips per point: 2 (4 accesses) instead of 4-5.
template <int N_, int A1_, int B1_, int A2_, int B2_, int A3_, int B3_, int TB_, int T_, int CTAS_, bool PADDED_ = true>
struct FixedPlan {
  static constexpr int N = N_, A1 = A1_, B1 = B1_, A2 = A2_, B2 = B2_, A3 = A3_, B3 = B3_, TB = TB_, T = T_, CTAS = CTAS_;
  static constexpr int G1 = A1 * B1, G2 = A2 * B2, G3 = A3 * B3;
  // Contiguous passes (lanes run along the axis, a column is N consecutive cells): every block of L2 = N / G1 positions
  // is followed by PAD cells with L2 + PAD = G3 (mod 8), so that (i) the lanes of group 2 -- G3 consecutive positions,
  // then the next block -- and (ii) eight consecutive frequencies of the digit-reversed store -- positions N/4 and
  // N/(4 B1) apart -- fall into different 16-byte bank groups (unpadded: 2-way and 4-way conflicts, 35 % of pass A's
  // shared-memory wavefronts at N = 672, profiles/r2b_fft.md).
  static constexpr int L2 = N / G1;
  // (PADDED_ = false where the padding would push two CTAs' shared memory from the 196 KB to the 228 KB carve-out and
  // the L1 from 60 to 28 KB: N = 720 measured 0.768 ms without, 0.793 ms with)
  static constexpr int PAD = PADDED_ ? ((G3 - L2) % 8 + 8) % 8 : 0;
  static constexpr int NP = N + G1 * PAD;   // cells of a padded column
  static_assert(G1 * G2 * G3 == N && A1 == 4 && N % 4 == 0, "plan must factor N with a leading radix 4");
  static_assert((TB & (TB - 1)) == 0, "tile height must be a power of two");
};

// One fused group = a radix-G DFT (G = A B) in registers followed by its outer twiddles, v[q1][q2] -> v[p1][p2]:
//   radix A over q1;  inner constants c[p1][q2] = e^{-2 pi i p1 q2 / G} (p1, q2 >= 1; FftPass::cst, i.e. the kernel's
//   parameter bank: compile-time indices make them immediate operands of the DFMA / DMUL);  radix B over q2;
//   outer twiddles w^{p1 jp tstep} (row p1-1 of ta) and w^{p2 jp tstep A} (row p2-1 of tb), both in SHARED memory, laid out
//   [row][jp] so that the lanes of a warp -- consecutive jp -- read consecutive 16-byte entries (pointers already point at
//   column jp; `stride` = row length).  The product form w^{p1 (jp + q2 Lq)} = w^{p1 jp} c[p1][q2] keeps the tables at
//   (A + B - 2) Lq entries per group (22 KB for N = 2700) instead of N: small enough to sit beside two resident CTAs' data.
//   History: indexing the one table exp(-2 pi i k / N) by the products made every lane of a load touch its own cache line
//   and the L1 the busiest unit of the pass (79 %); per-stage tables read through the L1 missed 80 % of the time
//   (profiles/r2b_fft.md).
// LAST: the last group (jp = 0) has no outer twiddles.
template <int A, int B, bool LAST>
__device__ __forceinline__ void group_twiddle_b(double2 (&v)[A][B], const double2* __restrict__ cst,
                                                const double2* __restrict__ ta, const double2* __restrict__ tb, int stride) {
  // on entry v[p1][q2] holds the radix-A outputs (before any twiddle)
#pragma unroll
  for (int p1 = 1; p1 < A; ++p1)
#pragma unroll
    for (int q2 = 1; q2 < B; ++q2) v[p1][q2] = cmul(v[p1][q2], cst[(p1 - 1) * (B - 1) + (q2 - 1)]);
  if (B > 1) {
#pragma unroll
    for (int p1 = 0; p1 < A; ++p1) {
      double2 x[B];
#pragma unroll
      for (int q2 = 0; q2 < B; ++q2) x[q2] = v[p1][q2];
      bfly<B>(x);
#pragma unroll
      for (int p2 = 0; p2 < B; ++p2) v[p1][p2] = x[p2];
    }
  }
  if (!LAST) {
#pragma unroll
    for (int p1 = 1; p1 < A; ++p1) {
      const double2 t = ta[(p1 - 1) * stride];
#pragma unroll
      for (int p2 = 0; p2 < B; ++p2) v[p1][p2] = cmul(v[p1][p2], t);
    }
#pragma unroll
    for (int p2 = 1; p2 < B; ++p2) {
      const double2 t = tb[(p2 - 1) * stride];
#pragma unroll
      for (int p1 = 0; p1 < A; ++p1) v[p1][p2] = cmul(v[p1][p2], t);
    }
  }
}
template <int A, int B, bool LAST>
__device__ __forceinline__ void group_dft(double2 (&v)[A][B], const double2* __restrict__ cst, const double2* __restrict__ ta,
                                          const double2* __restrict__ tb, int stride) {
#pragma unroll
  for (int q2 = 0; q2 < B; ++q2) {
    double2 x[A];
#pragma unroll
    for (int q1 = 0; q1 < A; ++q1) x[q1] = v[q1][q2];
    bfly<A>(x);
#pragma unroll
    for (int p1 = 0; p1 < A; ++p1) v[p1][q2] = x[p1];
  }
  group_twiddle_b<A, B, LAST>(v, cst, ta, tb, stride);
}

// Layout of the outer-twiddle tables of a fixed plan (complex128 entries; one array per axis in global memory, copied
// to shared memory once per CTA).
template <class PL>
struct FixedTw {
  static constexpr int Lq1 = PL::N / PL::G1, Lq2 = PL::G3;
  static constexpr int off1a = 0;                                   // [A1-1][Lq1]: w^{p1 jp}
  static constexpr int off1b = off1a + (PL::A1 - 1) * Lq1;          // [B1-1][Lq1]: w^{A1 p2 jp}
  static constexpr int off2a = off1b + (PL::B1 - 1) * Lq1;          // [A2-1][Lq2]: w^{p1 jp G1}
  static constexpr int off2b = off2a + (PL::A2 - 1) * Lq2;          // [B2-1][Lq2]: w^{p2 jp G1 A2}
  static constexpr int total = off2b + (PL::B2 - 1) * Lq2;
};

// MODE 0: contiguous axis, real input, two rows packed per column (pass A, real strengths); 1: contiguous axis, complex
// input (pass A, complex strengths); 2: strided complex (passes B, C).  Persistent CTAs (PL::CTAS per SM) walk the tiles
// of TB columns.  Shared memory: the twiddle tables, then N * TB complex128 of data, element (pos, col) at pos * TB + col
// in the strided passes (lanes run over the tile's columns first, like the global accesses) and at col * N + pos in the
// contiguous ones (lanes run along the axis).
template <class PL, int MODE, bool F32>
__global__ void __launch_bounds__(PL::T, PL::CTAS) fft_fixed_kernel(const __grid_constant__ FftPass P, const void* __restrict__ in_raw,
                                                                    double2* __restrict__ out, int64_t n_tiles, int RUN) {
  constexpr int N = PL::N, TB = PL::TB, T = PL::T;
  constexpr int A1 = PL::A1, B1 = PL::B1, A2 = PL::A2, B2 = PL::B2, A3 = PL::A3, B3 = PL::B3;
  constexpr int G1 = PL::G1, G2 = PL::G2, G3 = PL::G3;
  constexpr bool STRIDED = MODE == 2;
  constexpr int PACK = MODE == 0 ? 2 : 1;
  using FT = FixedTw<PL>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2* stw = reinterpret_cast<double2*>(smem_raw);
  double2* a = stw + FT::total;
  __shared__ int s_mm[2 * TB];   // strided passes: the range of outputs [mm0, mm1) every column of the tile has to store
  const int tid = threadIdx.x;
  // element `pos` (in block blk = pos / L2) of column col
  auto at = [](int pos, int blk, int col) { return STRIDED ? pos * TB + col : col * PL::NP + pos + blk * PL::PAD; };
  for (int i = tid; i < FT::total; i += T) stw[i] = P.ftw[i];
  (void)G1;
  __syncthreads();   // the twiddle tables are in place

  constexpr int64_t rows_per_tile = (int64_t)TB * PACK;
  const int64_t tiles_per_hi = (P.n_lo + rows_per_tile - 1) / rows_per_tile;
  // Tiles are handed out in RUNS of consecutive tiles from a device counter (zeroed with the tables), so that the tiles in
  // flight stay a contiguous window like the hardware's own block order: a tile touches TB * 16 bytes of every 128-byte
  // line of the strided arrays, and the rest of the line is wanted by its neighbours while it is still in the L2 (with a
  // fixed stride per CTA, or with streaming loads, the strided passes read 3.8x their input from DRAM:
  // profiles/r2b_fft.md).
  __shared__ int s_run;
  for (;;) {
    if (tid == 0) s_run = atomicAdd(P.counter, 1);
    __syncthreads();
    const int64_t run = s_run;
    __syncthreads();   // (a run whose tiles are all skipped has no other barrier before s_run is written again)
    if (run * RUN >= n_tiles) break;
   for (int64_t tile = run * RUN; tile < min(n_tiles, (run + 1) * RUN); ++tile) {
    const int64_t hi = tile / tiles_per_hi;
    const int64_t lo0 = (tile - hi * tiles_per_hi) * rows_per_tile;
    const int nrow = (int)min(rows_per_tile, P.n_lo - lo0);
    const int ncol = (nrow + PACK - 1) / PACK;
    if (STRIDED) {
      if (P.ball) {   // uniform in the block
        bool needed = false;
        for (int c = 0; c < ncol; ++c) needed = needed || ball_q(P, lo0 + c) <= 1.0;
        if (!needed) continue;
      }
      if (tid < TB) {
        int mm0 = 0, mm1 = tid < ncol ? P.nout : 0;
        if (P.ball && tid < ncol) {
          const double q = ball_q(P, lo0 + tid);
          if (q > 1.0) {
            mm1 = 0;
          } else {
            const double rad = P.ball_rt * sqrt(1.0 - q) + 1.0;
            mm0 = max(0, (int)floor(P.ball_ct - rad));
            mm1 = min(P.nout, (int)ceil(P.ball_ct + rad) + 1);
          }
        }
        s_mm[2 * tid] = mm0;
        s_mm[2 * tid + 1] = mm1;
      }
    }

    // ---- group 1: inputs from global memory.  Input i <-> mode l = i - N/4 <-> position l mod N: positions [0, N/4)
    // hold i = pos + N/4, positions [3N/4, N) hold i = pos - 3N/4, the rest is zero: of the radix-4 butterfly (elements
    // r + q1 N/4, r < N/4) only q1 = 0 (h = in[r + N/4]) and q1 = 3 (l = in[r]) exist:  X_p = h + i^p l.
    constexpr int Lq1 = N / G1;
    bool nz = STRIDED;
    const double fhi = (MODE != 2 && P.dec_hi) ? P.dec_hi[hi] : 1.0;
    // Strided passes, fp64 arrays: every thread first issues the loads of ALL its group-1 tasks as 16-byte asynchronous
    // copies straight into the tile, each input at the position it has in the column (h at r, l at r + 3N/4) -- the task
    // that reads them is the only one that writes positions congruent to jp modulo Lq1, so the tile is its own staging
    // buffer and no barrier is needed, only the thread's own wait.  All loads of the tile are then in flight at once
    // instead of one round of 2 B1 register loads per task with a DRAM round trip each.
    constexpr bool ASYNC_IN = MODE == 2 && !F32;
    if (ASYNC_IN) {
      for (int idx = tid; idx < Lq1 * TB; idx += T) {
        const int col = idx % TB, jp = idx / TB;
        const bool live = col < ncol;
        const int64_t src = hi * P.in_hi + lo0 + (live ? col : 0);
        const double2* inb = static_cast<const double2*>(in_raw);
        const int nbytes = live ? 16 : 0;   // src-size 0: zero fill
#pragma unroll
        for (int q2 = 0; q2 < B1; ++q2) {
          const int r = jp + q2 * Lq1;
          const unsigned dh = (unsigned)__cvta_generic_to_shared(&a[at(r, 0, col)]);
          const unsigned dl = (unsigned)__cvta_generic_to_shared(&a[at(r + 3 * (N / 4), 0, col)]);
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dh), "l"(inb + src + (int64_t)(r + N / 4) * P.in_el), "r"(nbytes) : "memory");
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dl), "l"(inb + src + (int64_t)r * P.in_el), "r"(nbytes) : "memory");
        }
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    for (int idx = tid; idx < Lq1 * TB; idx += T) {
      const int col = STRIDED ? idx % TB : idx / Lq1;
      const int jp = STRIDED ? idx / TB : idx % Lq1;
      double2 xl[B1], xh[B1];
      if (ASYNC_IN) {
#pragma unroll
        for (int q2 = 0; q2 < B1; ++q2) {
          const int r = jp + q2 * Lq1;
          xh[q2] = a[at(r, 0, col)];
          xl[q2] = a[at(r + 3 * (N / 4), 0, col)];
        }
      } else if (MODE == 2) {
        const bool live = col < ncol;
        const int64_t src = hi * P.in_hi + lo0 + (live ? col : 0);
#pragma unroll
        for (int q2 = 0; q2 < B1; ++q2) {
          const int r = jp + q2 * Lq1;
          // L2-only loads with the normal retention: a tile uses TB * 16 bytes of every 128-byte line and the rest of
          // the line is wanted by the next tiles of the run (streaming loads mark the line evict-first: 3.8x re-reads)
          xl[q2] = live ? ld_cplx_cg(in_raw, src + (int64_t)r * P.in_el, F32) : make_double2(0.0, 0.0);
          xh[q2] = live ? ld_cplx_cg(in_raw, src + (int64_t)(r + N / 4) * P.in_el, F32) : make_double2(0.0, 0.0);
        }
      } else if (MODE == 1) {
        const bool live = col < ncol;
        const int64_t src = hi * P.in_hi + (lo0 + (live ? col : 0)) * P.in_lo;
        const double f0 = P.dec_axis ? fhi * P.dec_lo[lo0 + (live ? col : 0)] : 1.0;
#pragma unroll
        for (int q2 = 0; q2 < B1; ++q2) {
          const int r = jp + q2 * Lq1;
          const double fl = P.dec_axis ? f0 * P.dec_axis[r] : 1.0, fh = P.dec_axis ? f0 * P.dec_axis[r + N / 4] : 1.0;
          const double2 l = live ? ld_cplx_cs(in_raw, src + r, F32) : make_double2(0.0, 0.0);
          const double2 h = live ? ld_cplx_cs(in_raw, src + r + N / 4, F32) : make_double2(0.0, 0.0);
          xl[q2] = make_double2(l.x * fl, l.y * fl);
          xh[q2] = make_double2(h.x * fh, h.y * fh);
          nz |= (l.x != 0.0) | (l.y != 0.0) | (h.x != 0.0) | (h.y != 0.0);
        }
      } else {
        const bool live = col < ncol, two = 2 * col + 1 < nrow;
        const int64_t r0 = lo0 + 2 * (live ? col : 0);
        const int64_t src0 = hi * P.in_hi + r0 * P.in_lo;
        const int64_t src1 = src0 + (two ? P.in_lo : 0);
        const double f0 = live ? (P.dec_axis ? fhi * P.dec_lo[r0] : 1.0) : 0.0;
        const double f1 = two ? (P.dec_axis ? fhi * P.dec_lo[r0 + 1] : 1.0) : 0.0;
        double la[B1], lb[B1], ha[B1], hb[B1], fl[B1], fh[B1];
#pragma unroll
        for (int q2 = 0; q2 < B1; ++q2) {
          const int r = jp + q2 * Lq1;
          la[q2] = ld_real(in_raw, src0 + r, F32);
          lb[q2] = ld_real(in_raw, src1 + r, F32);
          ha[q2] = ld_real(in_raw, src0 + r + N / 4, F32);
          hb[q2] = ld_real(in_raw, src1 + r + N / 4, F32);
          fl[q2] = P.dec_axis ? P.dec_axis[r] : 1.0;
          fh[q2] = P.dec_axis ? P.dec_axis[r + N / 4] : 1.0;
        }
#pragma unroll
        for (int q2 = 0; q2 < B1; ++q2) {
          nz |= live & ((la[q2] != 0.0) | (lb[q2] != 0.0) | (ha[q2] != 0.0) | (hb[q2] != 0.0));
          xl[q2] = make_double2(la[q2] * (fl[q2] * f0), lb[q2] * (fl[q2] * f1));
          xh[q2] = make_double2(ha[q2] * (fh[q2] * f0), hb[q2] * (fh[q2] * f1));
        }
      }
      double2 v[A1][B1];
#pragma unroll
      for (int q2 = 0; q2 < B1; ++q2) {
        const double2 h = xh[q2], l = xl[q2];
        v[0][q2] = cadd(h, l);
        v[1][q2] = make_double2(h.x - l.y, h.y + l.x);   // h + i l
        v[2][q2] = csub(h, l);
        v[3][q2] = make_double2(h.x + l.y, h.y - l.x);   // h - i l
      }
      group_twiddle_b<A1, B1, false>(v, P.cst[0], stw + FT::off1a + jp, stw + FT::off1b + jp, Lq1);
#pragma unroll
      for (int p1 = 0; p1 < A1; ++p1)
#pragma unroll
        for (int p2 = 0; p2 < B1; ++p2) a[at(jp + p1 * (N / A1) + p2 * Lq1, p1 * B1 + p2, col)] = v[p1][p2];
    }
    // The sources lie on a shell: a third of the rows of the first pass (those outside the shell's projection) are
    // entirely zero, and so is their transform: store zeros, skip the other two groups.
    const bool all_zero = __syncthreads_or(nz) == 0;
    if (!STRIDED && all_zero) {
      for (int row = 0; row < nrow; ++row) {
        const int64_t o = hi * P.out_hi + (lo0 + row) * P.out_lo;
        for (int mm = tid; mm < P.nout; mm += T) st_cplx(out, o + mm, make_double2(0.0, 0.0), F32);
      }
      continue;   // (the next tile's group 1 writes shared memory nobody reads any more: every thread is past the barrier)
    }

    // ---- group 2: blocks of L2 = N / G1 points, twiddle step G1
    {
      constexpr int L2 = N / G1, Lq2 = L2 / G2;
      for (int idx = tid; idx < (N / G2) * TB; idx += T) {
        const int col = STRIDED ? idx % TB : idx / (N / G2);
        const int g = STRIDED ? idx / TB : idx % (N / G2);
        const int b = g / Lq2, jp = g - b * Lq2;
        const int base = b * L2 + jp;
        double2 v[A2][B2];
#pragma unroll
        for (int q1 = 0; q1 < A2; ++q1)
#pragma unroll
          for (int q2 = 0; q2 < B2; ++q2) v[q1][q2] = a[at(base + q1 * (L2 / A2) + q2 * Lq2, b, col)];
        group_dft<A2, B2, false>(v, P.cst[1], stw + FT::off2a + jp, stw + FT::off2b + jp, Lq2);
#pragma unroll
        for (int p1 = 0; p1 < A2; ++p1)
#pragma unroll
          for (int p2 = 0; p2 < B2; ++p2) a[at(base + p1 * (L2 / A2) + p2 * Lq2, b, col)] = v[p1][p2];
      }
    }
    __syncthreads();

    // ---- group 3: blocks of G3 points (no outer twiddles); output (p1, p2) of block b is frequency
    // klow[b] + (N / G3)(p1 + A3 p2)
    for (int idx = tid; idx < (N / G3) * TB; idx += T) {
      const int col = STRIDED ? idx % TB : idx / (N / G3);
      const int b = STRIDED ? idx / TB : idx % (N / G3);
      double2 v[A3][B3];
#pragma unroll
      for (int q1 = 0; q1 < A3; ++q1)
#pragma unroll
        for (int q2 = 0; q2 < B3; ++q2) v[q1][q2] = a[at(b * G3 + q1 * B3 + q2, b / G2, col)];
      group_dft<A3, B3, true>(v, P.cst[2], nullptr, nullptr, 0);
      if (STRIDED) {
        const int mm0 = s_mm[2 * col], mm1 = s_mm[2 * col + 1];
        if (mm1 > mm0) {
          const int64_t o = hi * P.out_hi + lo0 + col;
          const int mm = __ldg(&P.klow[b]) - P.lo;   // output index of frequency klow[b]; the band may wrap around N
#pragma unroll
          for (int p2 = 0; p2 < B3; ++p2)
#pragma unroll
            for (int p1 = 0; p1 < A3; ++p1) {
              int m = mm + (N / G3) * (p1 + A3 * p2);
              m = m < 0 ? m + N : (m >= N ? m - N : m);
              if (m >= mm0 && m < mm1) st_cplx(out, o + (int64_t)m * P.out_el, v[p1][p2], F32);   // (partial lines meet in the L2)
            }
        }
      } else {
#pragma unroll
        for (int p1 = 0; p1 < A3; ++p1)
#pragma unroll
          for (int p2 = 0; p2 < B3; ++p2) a[at(b * G3 + p1 * B3 + p2, b / G2, col)] = v[p1][p2];
      }
    }
    __syncthreads();
    if (STRIDED) continue;

    // ---- contiguous passes: the band goes out along the axis, through the digit-reversal table.  One loop over all
    // (column, output) pairs of the tile: with a loop per column only nout of the T threads had work (47 % at n2 = 672).
    {
      const int nout = P.nout, total = ncol * nout;
      const float inv_nout = 1.0f / (float)nout;
      for (int idx = tid; idx < total; idx += T) {
        // idx / nout: the half-cell offset keeps the rounded quotient on the right side of every multiple of nout
        // (idx < 2^15, nout < 2^12: the float error is far below 0.5 / nout)
        const int col = (int)(((float)idx + 0.5f) * inv_nout);
        const int mm = idx - col * nout;
        const int64_t o0 = hi * P.out_hi + (lo0 + PACK * col) * P.out_lo;
        int m = P.lo + mm;
        m = m < 0 ? m + N : (m >= N ? m - N : m);
        const int pz = __ldg(&P.rev[m]);
        const double2 z = a[at(pz, pz / PL::L2, col)];
        if (MODE == 0) {
          const bool two = 2 * col + 1 < nrow;
          const int pc = __ldg(&P.rev[m == 0 ? 0 : N - m]);
          const double2 zc = a[at(pc, pc / PL::L2, col)];
          st_cplx(out, o0 + mm, make_double2(0.5 * (z.x + zc.x), 0.5 * (z.y - zc.y)), F32);
          if (two) st_cplx(out, o0 + P.out_lo + mm, make_double2(0.5 * (z.y + zc.y), 0.5 * (zc.x - z.x)), F32);
        } else {
          st_cplx(out, o0 + mm, z, F32);
        }
      }
    }
    __syncthreads();
   }
  }
}

// The lengths with a fixed plan and their factor sequence (A1, B1, A2, B2, A3, B3).
bool fixed_plan_factors(int N, int f[6]) {
  static const int plans[][7] = {{360, 4, 2, 3, 3, 5, 1},  {672, 4, 2, 4, 3, 7, 1},  {720, 4, 2, 2, 5, 3, 3},
                                 {1344, 4, 4, 4, 3, 7, 1}, {1440, 4, 4, 2, 5, 3, 3}, {2700, 4, 3, 3, 5, 3, 5}};
  for (const auto& pl : plans)
    if (pl[0] == N) {
      for (int i = 0; i < 6; ++i) f[i] = pl[1 + i];
      return true;
    }
  return false;
}

// One pass; see FftPass (fft.cuh).  Shared memory: a[N][tbp] complex128.  THREADS = 512 with two CTAs per SM, or
// 1024 with one (long transforms): 32 warps per SM either way -- the stages are bound by dependent FP64 chains and
// the shared-memory pipe, so occupancy is what buys throughput (profiles/r1c_after_rewrites.md, r1j_fft_phases.md).
// R7: the length has a factor 7 (a separate instantiation: the radix-7 butterfly's register pressure costs the other
// lengths ~5 % when it shares their kernel).
template <bool REAL_IN, bool CONTIG, int THREADS, int CG, bool FUSED, bool R7>
__global__ void __launch_bounds__(THREADS, (FUSED ? 512 : 1024) / THREADS)
fft_pass_kernel(FftPass P, const void* __restrict__ in_raw, double2* __restrict__ out) {
  constexpr int kFftThreads = THREADS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2* a = reinterpret_cast<double2*>(smem_raw);
  const int N = P.N, tb = P.tb, tbp = P.tbp, tid = threadIdx.x;
  // PACK (real input only): a column of the tile carries two real rows, 2c as the real and 2c+1 as the imaginary
  // part; their transforms are separated at the store, A[m] = (Z[m] + conj Z[-m])/2, B[m] = (Z[m] - conj Z[-m])/(2i)
  constexpr int PACK = REAL_IN ? 2 : 1;
  const int64_t rows_per_tile = (int64_t)tb * PACK;
  const int64_t tiles_per_hi = (P.n_lo + rows_per_tile - 1) / rows_per_tile;
  const int64_t hi = blockIdx.x / tiles_per_hi;
  const int64_t lo0 = (blockIdx.x - hi * tiles_per_hi) * rows_per_tile;
  const int nrow = (int)min(rows_per_tile, P.n_lo - lo0);   // rows of this tile
  const int ncol = (nrow + PACK - 1) / PACK;
  if (!CONTIG && P.ball) {   // uniform in the block: every thread tests the tile's few columns
    bool needed = false;
    for (int c = 0; c < ncol; ++c) needed = needed || ball_q(P, lo0 + c) <= 1.0;
    if (!needed) return;
  }
  const int tsh = P.tb_shift;
  const double2* __restrict__ tw = P.tw;

  // ---- load: input i <-> mode l = i - n_in/2 goes to position l mod N of the padded row; the rest is zero.
  // Addressing is kept out of the inner loops (the first version spent 70 % of its instructions on 64-bit index
  // arithmetic here and in the store): threads form a (ty, col) grid with col fastest in the strided passes, a
  // (warp = column, lane = element) grid in the contiguous one; pointers advance by constant strides; four
  // independent loads per thread are in flight before the first store.
  const int half_in = P.n_in / 2;
  const double fhi = P.dec_hi ? P.dec_hi[hi] : 1.0;
  const int n_pad = N - P.n_in;          // zero positions: [n_in - half_in, N - half_in)
  bool nz = false;                       // did this thread load anything non-zero?
  const int pad0 = P.n_in - half_in;
  if (CONTIG) {
    // warp grid (column, segment): with fewer columns than warps every column is shared by nseg warps, each taking
    // every nseg-th group of 32 elements, so all warps load whatever the tile height is
    const int lane = tid & 31, wrp = tid >> 5, nw = kFftThreads / 32;
    const int nseg = nw >= tb ? nw / tb : 1;
    const int cstep = nw >= tb ? tb : nw;            // columns advance by this per outer iteration
    const int seg = nw >= tb ? wrp / tb : 0;
    const int lstep = 32 * nseg;                     // element stride of one warp inside a row
    for (int col = nw >= tb ? wrp % tb : wrp; col < tb && seg < nseg; col += cstep) {
      for (int j = lane + 32 * seg; j < n_pad; j += lstep) a[(pad0 + j) * tbp + col] = make_double2(0.0, 0.0);
      if (col >= ncol) {
        for (int i = lane + 32 * seg; i < P.n_in; i += lstep) {
          const int l = i - half_in;
          a[(l < 0 ? l + N : l) * tbp + col] = make_double2(0.0, 0.0);
        }
        continue;
      }
      if (REAL_IN) {
        const int64_t r0 = lo0 + 2 * col;
        const bool two = 2 * col + 1 < nrow;
        const int64_t src0 = hi * P.in_hi + r0 * P.in_lo;
        const int64_t src1 = src0 + (two ? P.in_lo : 0);
        const double f0 = P.dec_axis ? fhi * P.dec_lo[r0] : 1.0;
        const double f1 = two ? (P.dec_axis ? fhi * P.dec_lo[r0 + 1] : 1.0) : 0.0;
        for (int i0 = lane + 32 * seg; i0 < P.n_in; i0 += 4 * lstep) {
          double va[4], vb[4], fa[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int i = i0 + lstep * u;
            const bool ok = i < P.n_in;
            va[u] = ok ? ld_real(in_raw, src0 + i, P.f32) : 0.0;
            vb[u] = ok ? ld_real(in_raw, src1 + i, P.f32) : 0.0;
            fa[u] = (ok && P.dec_axis) ? P.dec_axis[i] : 1.0;
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int i = i0 + lstep * u;
            if (i < P.n_in) {
              const int l = i - half_in;
              a[(l < 0 ? l + N : l) * tbp + col] = make_double2(va[u] * (fa[u] * f0), vb[u] * (fa[u] * f1));
              nz |= (va[u] != 0.0) | (vb[u] != 0.0);
            }
          }
        }
      } else {
        const int64_t src = hi * P.in_hi + (lo0 + col) * P.in_lo;
        const double f0 = P.dec_axis ? fhi * P.dec_lo[lo0 + col] : 1.0;
        for (int i0 = lane + 32 * seg; i0 < P.n_in; i0 += 4 * lstep) {
          double2 v[4];
          double fa[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int i = i0 + lstep * u;
            const bool ok = i < P.n_in;
            v[u] = ok ? ld_cplx_cs(in_raw, src + i, P.f32) : make_double2(0.0, 0.0);
            fa[u] = (ok && P.dec_axis) ? P.dec_axis[i] * f0 : 1.0;
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int i = i0 + lstep * u;
            if (i < P.n_in) {
              const int l = i - half_in;
              a[(l < 0 ? l + N : l) * tbp + col] = make_double2(v[u].x * fa[u], v[u].y * fa[u]);
              nz |= (v[u].x != 0.0) | (v[u].y != 0.0);
            }
          }
        }
      }
    }
  } else {
    // strided passes (complex input, no deconvolution factors): in_lo = 1, rows in_el apart
    const int col = tid & (tb - 1), ty = tid >> tsh, nty = kFftThreads >> tsh;
    for (int j = ty; j < n_pad; j += nty) a[(pad0 + j) * tbp + col] = make_double2(0.0, 0.0);
    // 16-byte asynchronous copies (LDGSTS) straight into the padded rows: every thread issues all of its elements
    // back to back and waits once -- the pass is bound by memory latency, so what counts is bytes in flight
    const bool live = col < ncol;
    if (P.f32) {   // single-precision input: converted on the way in (no asynchronous copy can do that)
      const int64_t src32 = hi * P.in_hi + lo0 + (live ? col : 0);
      for (int i = ty; i < P.n_in; i += nty) {
        const int l = i - half_in;
        a[(l < 0 ? l + N : l) * tbp + col] = live ? ld_cplx_cg(in_raw, src32 + (int64_t)i * P.in_el, 1) : make_double2(0.0, 0.0);
      }
    }
    const double2* src = static_cast<const double2*>(in_raw) + hi * P.in_hi + lo0 + (live ? col : 0) + (int64_t)ty * P.in_el;
    const int64_t step = (int64_t)nty * P.in_el;
    for (int i = ty; i < (P.f32 ? 0 : P.n_in); i += nty) {
      const int l = i - half_in;
      const unsigned dst = (unsigned)__cvta_generic_to_shared(a + (l < 0 ? l + N : l) * tbp + col);
      const int nbytes = live ? 16 : 0;   // src-size 0: zero-fill (columns beyond the edge of the array)
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(nbytes) : "memory");
      src += step;
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    nz = true;   // (no zero-tile detection in the strided passes)
  }
  // The sources lie on a shell: a third of the rows of the first pass (those outside the shell's projection) and the
  // outer planes of the second are entirely zero, and so is their transform: skip the stages, store zeros.
  const bool all_zero = __syncthreads_or(nz) == 0;

  // ---- in-place decimation-in-frequency stages
  int L = N;
  for (int s = 0; s < (all_zero ? 0 : P.npair); ++s) {
    const int code = P.pair[s];
    const unsigned mg = P.magic[s];
#define SFD_FFT_STAGE(R_) \
  case R_ * 8 + 1: dif_stage<R_, CG>(a, tw, N, L, mg, P.cg_shift, tbp, tid, kFftThreads); L /= R_; break;
#define SFD_FFT_PAIR(R1_, R2_) \
  case R1_ * 8 + R2_: fused_stages<R1_, R2_>(a, tw, N, L, mg, tb, tbp, tsh, tid, kFftThreads); L /= R1_ * R2_; break;
    if (FUSED) {
      switch (code) {
        SFD_FFT_PAIR(4, 4) SFD_FFT_PAIR(4, 2) SFD_FFT_PAIR(4, 3) SFD_FFT_PAIR(2, 3) SFD_FFT_PAIR(2, 5) SFD_FFT_PAIR(3, 3)
        SFD_FFT_PAIR(3, 5) SFD_FFT_PAIR(2, 2) SFD_FFT_PAIR(4, 1) SFD_FFT_PAIR(2, 1) SFD_FFT_PAIR(3, 1) SFD_FFT_PAIR(5, 1)
      }
      if (R7) {
        switch (code) { SFD_FFT_PAIR(2, 7) SFD_FFT_PAIR(7, 1) }
      }
    } else {
      switch (code) {
        SFD_FFT_STAGE(4) SFD_FFT_STAGE(2) SFD_FFT_STAGE(3) SFD_FFT_STAGE(5)
      }
      if (R7) {
        switch (code) { SFD_FFT_STAGE(7) }
      }
    }
#undef SFD_FFT_PAIR
#undef SFD_FFT_STAGE
    __syncthreads();
  }

  // ---- store the band m in [lo, lo + nout) through the digit-reversal table
  if (CONTIG) {
    const int lane = tid & 31, wrp = tid >> 5, nw = kFftThreads / 32;
    const int nseg = nw >= tb ? nw / tb : 1;
    const int cstep = nw >= tb ? tb : nw;
    const int seg = nw >= tb ? wrp / tb : 0;
    const int lstep = 32 * nseg;
    for (int col = nw >= tb ? wrp % tb : wrp; col < ncol && seg < nseg; col += cstep) {
      if (REAL_IN) {
        const bool two = 2 * col + 1 < nrow;
        const int64_t o0 = hi * P.out_hi + (lo0 + 2 * col) * P.out_lo;
        const int64_t o1 = o0 + P.out_lo;
        for (int mm = lane + 32 * seg; mm < P.nout; mm += lstep) {
          int m = P.lo + mm;
          m = m < 0 ? m + N : (m >= N ? m - N : m);
          const double2 z = a[P.rev[m] * tbp + col], zc = a[P.rev[m == 0 ? 0 : N - m] * tbp + col];
          st_cplx(out, o0 + mm, make_double2(0.5 * (z.x + zc.x), 0.5 * (z.y - zc.y)), P.f32);
          if (two) st_cplx(out, o1 + mm, make_double2(0.5 * (z.y + zc.y), 0.5 * (zc.x - z.x)), P.f32);
        }
      } else {
        const int64_t o0 = hi * P.out_hi + (lo0 + col) * P.out_lo;
        for (int mm = lane + 32 * seg; mm < P.nout; mm += lstep) {
          int m = P.lo + mm;
          m = m < 0 ? m + N : (m >= N ? m - N : m);
          st_cplx(out, o0 + mm, a[P.rev[m] * tbp + col], P.f32);
        }
      }
    }
  } else {
    const int col = tid & (tb - 1), ty = tid >> tsh, nty = kFftThreads >> tsh;
    if (col < ncol) {
      int mm0 = 0, mm1 = P.nout;   // the outputs this column has to store
      if (P.ball) {
        const double q = ball_q(P, lo0 + col);
        if (q > 1.0) {
          mm1 = 0;
        } else {
          const double rad = P.ball_rt * sqrt(1.0 - q) + 1.0;
          mm0 = max(0, (int)floor(P.ball_ct - rad));
          mm1 = min(P.nout, (int)ceil(P.ball_ct + rad) + 1);
        }
      }
      const int first = mm0 + ((ty - mm0) % nty + nty) % nty;   // smallest mm >= mm0 congruent to ty modulo nty
      int64_t o = hi * P.out_hi + lo0 + col + (int64_t)first * P.out_el;
      const int64_t step = (int64_t)nty * P.out_el;
      for (int mm = first; mm < mm1; mm += nty) {
        int m = P.lo + mm;
        m = m < 0 ? m + N : (m >= N ? m - N : m);
        st_cplx(out, o, a[P.rev[m] * tbp + col], P.f32);
        o += step;
      }
    }
  }
}

// ---- host tables, cached per transform length ----------------------------------------------------------------
struct HostTables {
  std::vector<double> tw;     // N complex: exp(-2 pi i t / N)
  std::vector<int32_t> rev;   // position of output frequency k after the DIF stages
  std::vector<int32_t> klow;  // fixed-geometry plans: klow[b] = frequency stored at position b * G3 (G3 = last group)
  std::vector<double> ftw;    // fixed-geometry plans: outer-twiddle tables (FixedTw), complex
  double cst[3][9][2] = {};   // fixed-geometry plans: inner constants of the three groups
  int nfac;
  int fac[16];      // single radices in execution order
  int npair;
  int pair[16];     // the same sequence grouped into fused pairs: code R1 * 8 + R2 (R2 = 1: single)
};
std::mutex g_mu;
std::map<int, HostTables> g_tables;

const HostTables& tables_for(int N) {
  std::lock_guard<std::mutex> lk(g_mu);
  auto it = g_tables.find(N);
  if (it != g_tables.end()) return it->second;
  HostTables t;
  // radices 4s, 2, 3s, 5s, 7s, then ordered so that consecutive stages pair up into register-resident radix-(R1 R2)
  // butterflies with R1 R2 <= 16: take the first remaining factor and the largest other one that fits
  // (2700 -> (4,3)(3,5)(3,5); 1440 -> (4,4)(2,5)(3,3); 720 -> (4,4)(3,5)(3); 360 -> (4,3)(2,5)(3))
  std::vector<int> rest;
  int n = N;
  while (n % 4 == 0) { rest.push_back(4); n /= 4; }
  while (n % 2 == 0) { rest.push_back(2); n /= 2; }
  while (n % 3 == 0) { rest.push_back(3); n /= 3; }
  while (n % 5 == 0) { rest.push_back(5); n /= 5; }
  while (n % 7 == 0) { rest.push_back(7); n /= 7; }
  t.nfac = 0;
  t.npair = 0;
  int fx[6];
  const bool fixed = fixed_plan_factors(N, fx);
  if (fixed) {   // the fixed-geometry kernels and the generic one share the factor order (and so the reversal table)
    rest.clear();
    for (int g = 0; g < 3; ++g) {
      t.fac[t.nfac++] = fx[2 * g];
      if (fx[2 * g + 1] > 1) t.fac[t.nfac++] = fx[2 * g + 1];
      t.pair[t.npair++] = fx[2 * g] * 8 + fx[2 * g + 1];
    }
  }
  while (!rest.empty()) {
    const int r1 = rest.front();
    rest.erase(rest.begin());
    int best = -1;
    for (size_t i = 0; i < rest.size(); ++i)
      if (r1 * rest[i] <= 16 && (best < 0 || rest[i] > rest[best])) best = (int)i;
    int r2 = 1;
    if (best >= 0) {
      r2 = rest[best];
      rest.erase(rest.begin() + best);
    }
    t.fac[t.nfac++] = r1;
    if (r2 > 1) t.fac[t.nfac++] = r2;
    t.pair[t.npair++] = r1 * 8 + r2;
  }
  t.tw.resize(2 * (size_t)N);
  const long double two_pi = 6.283185307179586476925286766559005768L;
  for (int k = 0; k < N; ++k) {
    const long double ang = two_pi * k / N;
    t.tw[2 * k] = (double)cosl(ang);
    t.tw[2 * k + 1] = (double)(-sinl(ang));
  }
  t.rev.resize(N);
  for (int k = 0; k < N; ++k) {
    int kk = k, M = N, pos = 0;
    for (int s = 0; s < t.nfac; ++s) {
      const int p = kk % t.fac[s];
      kk /= t.fac[s];
      M /= t.fac[s];
      pos += p * M;
    }
    t.rev[k] = pos;
  }
  t.klow.assign(N, 0);
  if (fixed) {
    const int A1 = fx[0], B1 = fx[1], A2 = fx[2], B2 = fx[3], A3 = fx[4], B3 = fx[5];
    const int G1 = A1 * B1, G3 = A3 * B3, Lq1 = N / G1, Lq2 = G3;
    for (int k = 0; k < N / G3; ++k) t.klow[t.rev[k] / G3] = k;
    auto put = [&](long long idx) {   // exp(-2 pi i idx / N), the index reduced first so that every entry is exact to an ulp
      idx %= N;
      t.ftw.push_back(t.tw[2 * idx]);
      t.ftw.push_back(t.tw[2 * idx + 1]);
    };
    for (int p1 = 1; p1 < A1; ++p1)
      for (int jp = 0; jp < Lq1; ++jp) put((long long)p1 * jp);
    for (int p2 = 1; p2 < B1; ++p2)
      for (int jp = 0; jp < Lq1; ++jp) put((long long)p2 * jp * A1);
    for (int p1 = 1; p1 < A2; ++p1)
      for (int jp = 0; jp < Lq2; ++jp) put((long long)p1 * jp * G1);
    for (int p2 = 1; p2 < B2; ++p2)
      for (int jp = 0; jp < Lq2; ++jp) put((long long)p2 * jp * G1 * A2);
    // inner constants of the three groups: e^{-2 pi i p1 q2 / (A B)} = entry p1 q2 N / (A B) of the twiddle table
    for (int g = 0; g < 3; ++g) {
      const int A = fx[2 * g], B = fx[2 * g + 1];
      for (int p1 = 1; p1 < A; ++p1)
        for (int q2 = 1; q2 < B; ++q2) {
          const long long idx = ((long long)p1 * q2 * (N / (A * B))) % N;
          t.cst[g][(p1 - 1) * (B - 1) + (q2 - 1)][0] = t.tw[2 * idx];
          t.cst[g][(p1 - 1) * (B - 1) + (q2 - 1)][1] = t.tw[2 * idx + 1];
        }
    }
    (void)A3;
    (void)B3;
  }
  return g_tables.emplace(N, std::move(t)).first->second;
}

}  // namespace

bool fft_length_ok(int N) {
  int n = N;
  while (n % 2 == 0) n /= 2;
  while (n % 3 == 0) n /= 3;
  while (n % 5 == 0) n /= 5;
  while (n % 7 == 0) n /= 7;
  return n == 1 && N >= 2;
}

size_t fft_tables_bytes(const int n2[3]) {
  size_t b = 0;
  // twiddles, reversal table, klow, and the per-stage tables of a fixed plan (< 1.25 N entries)
  for (int d = 0; d < 3; ++d)
    b += align_up((size_t)n2[d] * 16) + 2 * align_up((size_t)n2[d] * 4) + align_up((size_t)n2[d] * 20 + 4096);
  return b + 256;   // + the passes' tile counters
}

// Rows per tile (a power of two) and row pitch.  Prefer tiles that let two CTAs share an SM (one CTA's loads and
// stores overlap the other's butterflies).  The pitch is odd (conflict-free transposing load of the contiguous-axis
// pass, conflict-free column-group lanes) except for long transforms in the strided passes, where 4 unpadded rows
// are what still fits twice (their lanes run over consecutive rows: contiguous either way).
int fft_tile(int N, int contig, int* tbp) {
  int pick = 0, pitch = 0;
  auto fits = [&](int tb, int pt, size_t cap) { return (size_t)N * pt * 16 <= cap; };
  const size_t half = (size_t)112 * 1024, full = (size_t)224 * 1024;
  if (fits(8, 9, half)) pick = 8, pitch = 9;                       // column groups of 2, 2-4 CTAs per SM
  // long transforms: two CTAs per SM matter more than the conflict-free transposing load (even pitch)
  if (!pick && fits(4, contig ? 5 : 4, half)) pick = 4, pitch = contig ? 5 : 4;
  if (!pick && fits(4, 4, half)) pick = 4, pitch = 4;
  if (!pick && fits(2, contig ? 3 : 2, half)) pick = 2, pitch = contig ? 3 : 2;
  if (!pick && fits(2, 2, half)) pick = 2, pitch = 2;
  for (int tb = 8; tb >= 1 && !pick; tb >>= 1)                     // one CTA per SM
    if (fits(tb, contig ? (tb | 1) : tb, full)) pick = tb, pitch = contig ? (tb | 1) : tb;
  if (tbp) *tbp = pitch;
  return pick;
}

int fft_upload_tables(const int n2[3], void* d_tables, FftTables* out, cudaStream_t st) {
  char* base = static_cast<char*>(d_tables);
  size_t o = 256;
  out->counters = reinterpret_cast<int32_t*>(base);   // one tile counter per pass, zero until its pass runs
  SFD_CUDA_TRY(cudaMemsetAsync(base, 0, 256, st));
  for (int d = 0; d < 3; ++d) {
    SFD_REQUIRE(fft_length_ok(n2[d]) && fft_tile(n2[d], 1, nullptr) > 0, SFD_ERR_UNSUPPORTED, "FFT length %d is not supported", n2[d]);
    const HostTables& t = tables_for(n2[d]);
    out->tw[d] = reinterpret_cast<double2*>(base + o);
    SFD_CUDA_TRY(cudaMemcpyAsync(base + o, t.tw.data(), (size_t)n2[d] * 16, cudaMemcpyHostToDevice, st));
    o += align_up((size_t)n2[d] * 16);
    out->rev[d] = reinterpret_cast<int32_t*>(base + o);
    SFD_CUDA_TRY(cudaMemcpyAsync(base + o, t.rev.data(), (size_t)n2[d] * 4, cudaMemcpyHostToDevice, st));
    o += align_up((size_t)n2[d] * 4);
    out->klow[d] = reinterpret_cast<int32_t*>(base + o);
    SFD_CUDA_TRY(cudaMemcpyAsync(base + o, t.klow.data(), (size_t)n2[d] * 4, cudaMemcpyHostToDevice, st));
    o += align_up((size_t)n2[d] * 4);
    out->ftw[d] = reinterpret_cast<double2*>(base + o);
    SFD_REQUIRE(t.ftw.size() * 8 <= (size_t)n2[d] * 20 + 4096, SFD_ERR_UNSUPPORTED, "fixed-plan twiddle tables do not fit");
    if (!t.ftw.empty()) SFD_CUDA_TRY(cudaMemcpyAsync(base + o, t.ftw.data(), t.ftw.size() * 8, cudaMemcpyHostToDevice, st));
    o += align_up((size_t)n2[d] * 20 + 4096);
    for (int g = 0; g < 3; ++g)
      for (int i = 0; i < 9; ++i) out->cst[d][g][i] = make_double2(t.cst[g][i][0], t.cst[g][i][1]);
    out->nfac[d] = t.nfac;
    for (int s = 0; s < t.nfac; ++s) out->fac[d][s] = t.fac[s];
    out->npair[d] = t.npair;
    for (int s = 0; s < t.npair; ++s) out->pair[d][s] = t.pair[s];
  }
  return SFD_OK;
}

namespace {
// Launch of a fixed-geometry pass (above) when the length has a plan and exactly the central half of the inputs is
// non-zero; returns false when the generic kernel has to run.
template <class PL>
int launch_fixed(const FftPass& P, const void* d_in, double* d_out, cudaStream_t st) {
  const int mode = P.contig ? (P.real_in ? 0 : 1) : 2;
  const int64_t rows_per_tile = (int64_t)PL::TB * (mode == 0 ? 2 : 1);
  const int64_t tiles = P.n_hi * ((P.n_lo + rows_per_tile - 1) / rows_per_tile);
  if (tiles == 0) return SFD_OK;
  const size_t smem = ((size_t)(mode == 2 ? PL::N : PL::NP) * PL::TB + FixedTw<PL>::total) * 16;
  SFD_REQUIRE(tiles < 0x7fffffffLL && P.counter, SFD_ERR_UNSUPPORTED, "FFT pass has too many tiles");
  unsigned grid = (unsigned)std::min<int64_t>(tiles, (int64_t)PL::CTAS * num_sms());   // persistent CTAs
  // tiles per run: two 64-byte tiles share a 128-byte line (measured at config 5: run 1 / 2 / 4 -> 49.6 / 47.1 / 50.1 ms)
  const int run = (mode == 2 && PL::TB <= 4) ? 2 : 1;
  auto go = [&](auto kern) -> int {
    SFD_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<grid, PL::T, smem, st>>>(P, d_in, reinterpret_cast<double2*>(d_out), tiles, run);
    return SFD_OK;
  };
  if (P.f32) {   // single-precision arrays: instantiations of their own, so that the fp64 ones carry no branch
    if (mode == 0) SFD_TRY(go(fft_fixed_kernel<PL, 0, true>));
    else if (mode == 1) SFD_TRY(go(fft_fixed_kernel<PL, 1, true>));
    else SFD_TRY(go(fft_fixed_kernel<PL, 2, true>));
  } else {
    if (mode == 0) SFD_TRY(go(fft_fixed_kernel<PL, 0, false>));
    else if (mode == 1) SFD_TRY(go(fft_fixed_kernel<PL, 1, false>));
    else SFD_TRY(go(fft_fixed_kernel<PL, 2, false>));
  }
  return launch_check("fft_fixed_kernel");
}
bool try_fixed(const FftPass& P, const void* d_in, double* d_out, cudaStream_t st, int* rc) {
  if (P.n_in * 2 != P.N) return false;
  if (P.contig ? (P.in_el != 1 || P.out_el != 1) : (P.real_in || P.dec_axis || P.in_lo != 1 || P.out_lo != 1)) return false;
  switch (P.N) {   //                       N    A1 B1 A2 B2 A3 B3  TB   T  CTAs/SM
    case 360:  *rc = launch_fixed<FixedPlan<360,  4, 2, 3, 3, 5, 1, 8, 128, 4>>(P, d_in, d_out, st); return true;
    // How many columns a tile has and how many CTAs share an SM is measured per length and per kind of pass
    // (profiles/r2b_fft.md).  The warps of a CTA go through a tile's phases together -- all load, all compute, all store,
    // a barrier between -- so what keeps the SM's pipes busy is the number of CTAs in different phases, not the number of
    // warps: the contiguous pass, whose global accesses run along the axis whatever the tile, takes ONE column (two
    // packed real rows) per tile in as many CTAs as fit; the strided passes need TB * 16-byte segments of the other axis.
    // 672 / 720: groups of at most 12 / 10 points fit 80 registers.
    case 672:
      if (P.contig) *rc = launch_fixed<FixedPlan<672,  4, 2, 4, 3, 7, 1, 1, 96, 8>>(P, d_in, d_out, st);
      else *rc = launch_fixed<FixedPlan<672,  4, 2, 4, 3, 7, 1, 4, 192, 4>>(P, d_in, d_out, st);
      return true;
    case 720:
      if (P.contig) *rc = launch_fixed<FixedPlan<720,  4, 2, 2, 5, 3, 3, 1, 96, 8>>(P, d_in, d_out, st);
      else *rc = launch_fixed<FixedPlan<720,  4, 2, 2, 5, 3, 3, 8, 384, 2, false>>(P, d_in, d_out, st);
      return true;
    case 1344:
      if (P.contig) *rc = launch_fixed<FixedPlan<1344, 4, 4, 4, 3, 7, 1, 1, 96, 6>>(P, d_in, d_out, st);
      else *rc = launch_fixed<FixedPlan<1344, 4, 4, 4, 3, 7, 1, 4, 256, 2>>(P, d_in, d_out, st);
      return true;
    case 1440:
      if (P.contig) *rc = launch_fixed<FixedPlan<1440, 4, 4, 2, 5, 3, 3, 1, 96, 6>>(P, d_in, d_out, st);
      else *rc = launch_fixed<FixedPlan<1440, 4, 4, 2, 5, 3, 3, 4, 256, 2>>(P, d_in, d_out, st);
      return true;
    // 2700, strided: one 512-thread CTA per SM with 4 columns (64-byte segments) beats two CTAs with 2 columns each
    // (54.6 -> 47.1 ms at config 5: the strided passes' DRAM over-fetch halves); at 1344 the same trade loses (5.0 -> 5.6 ms)
    case 2700:
      if (P.contig) *rc = launch_fixed<FixedPlan<2700, 4, 3, 3, 5, 3, 5, 1, 192, 3>>(P, d_in, d_out, st);
      else *rc = launch_fixed<FixedPlan<2700, 4, 3, 3, 5, 3, 5, 4, 512, 1>>(P, d_in, d_out, st);
      return true;
  }
  return false;
}
}  // namespace

int fft_pass(FftPass P, const FftTables& T, int axis, const void* d_in, double* d_out, cudaStream_t st) {
  P.tw = T.tw[axis];
  P.rev = T.rev[axis];
  P.klow = T.klow[axis];
  P.ftw = T.ftw[axis];
  P.counter = T.counters + axis;
  for (int g = 0; g < 3; ++g)
    for (int i = 0; i < 9; ++i) P.cst[g][i] = T.cst[axis][g][i];
  {
    int rc = SFD_OK;
    const char* generic = std::getenv("SFD_FFT_GENERIC");   // debugging / A-B measurements: force the generic kernel
    if (!(generic && generic[0] == '1') && try_fixed(P, d_in, d_out, st, &rc)) return rc;
  }
  P.nfac = T.nfac[axis];
  for (int s = 0; s < P.nfac; ++s) P.fac[s] = T.fac[axis][s];
  P.tb = fft_tile(P.N, P.contig, &P.tbp);
  P.tb_shift = 0;
  while ((1 << P.tb_shift) < P.tb) ++P.tb_shift;
  // Long transforms (one CTA per SM either way) run two stages per shared-memory round trip in registers (128
  // registers, 16 warps): measured 13-19 % faster at N = 1440 / 2700; the short ones are faster with single stages
  // at 32 warps and column groups (profiles/r1c_after_rewrites.md).
  const bool fused = (size_t)P.N * 9 * 16 > (size_t)112 * 1024;
  {
    int L = P.N;
    P.npair = 0;
    auto push = [&](int r1, int r2) {
      const int Lq = L / (r1 * r2);
      P.pair[P.npair] = r1 * 8 + r2;
      P.magic[P.npair] = Lq > 1 ? (unsigned)(0x100000000ULL / (unsigned long long)Lq + 1ULL) : 0u;
      ++P.npair;
      L = Lq;
    };
    if (fused)
      for (int s = 0; s < T.npair[axis]; ++s) push(T.pair[axis][s] / 8, T.pair[axis][s] % 8);
    else
      for (int s = 0; s < P.nfac; ++s) push(P.fac[s], 1);
  }
  const int64_t rows_per_tile = (int64_t)P.tb * (P.real_in ? 2 : 1);   // real rows are packed in pairs
  const int64_t tiles = P.n_hi * ((P.n_lo + rows_per_tile - 1) / rows_per_tile);
  if (tiles == 0) return SFD_OK;
  SFD_REQUIRE(tiles < 0x7fffffffLL, SFD_ERR_UNSUPPORTED, "FFT pass has too many tiles");
  const size_t smem = (size_t)P.N * P.tbp * 16;
  // column group CG = 2 rows per thread; threads per CTA sized to the butterflies of a stage (N/5 .. N/2 per row) and
  // to the CTAs that fit an SM: 32 warps per SM in every case
  // (measured: the column groups pay off for the short transforms that fit 2-4 CTAs per SM, not for the long ones)
  const int cg = (!fused && P.tb == 8 && smem <= (size_t)112 * 1024) ? 2 : 1;
  P.cg_shift = 0;
  while ((cg << P.cg_shift) < P.tb) ++P.cg_shift;
  const int per_sm = (int)std::min<size_t>(4, (size_t)(226 * 1024) / (smem + 1024));
  int threads = per_sm >= 4 ? 256 : (per_sm >= 2 ? 512 : 1024);
  if (fused) threads = per_sm >= 2 ? 256 : 512;   // 128 registers per thread: 16 warps per SM
  auto go = [&](auto kern) -> int {
    SFD_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024));
    kern<<<(unsigned)tiles, threads, smem, st>>>(P, d_in, reinterpret_cast<double2*>(d_out));
    return SFD_OK;
  };
  // kernel variants: (real, contiguous) = pass A with real strengths; (complex, contiguous) = pass A otherwise;
  // (complex, strided) = passes B and C
  const bool r7 = P.N % 7 == 0;
#define SFD_FFT_T7(REAL_, CONTIG_, R7_)                                                                          \
  (fused ? (threads == 256 ? go(fft_pass_kernel<REAL_, CONTIG_, 256, 1, true, R7_>)                              \
                           : go(fft_pass_kernel<REAL_, CONTIG_, 512, 1, true, R7_>))                             \
         : (threads == 256 ? (cg == 2 ? go(fft_pass_kernel<REAL_, CONTIG_, 256, 2, false, R7_>)                  \
                                      : go(fft_pass_kernel<REAL_, CONTIG_, 256, 1, false, R7_>))                 \
            : threads == 512 ? (cg == 2 ? go(fft_pass_kernel<REAL_, CONTIG_, 512, 2, false, R7_>)                \
                                        : go(fft_pass_kernel<REAL_, CONTIG_, 512, 1, false, R7_>))               \
                             : go(fft_pass_kernel<REAL_, CONTIG_, 1024, 1, false, R7_>)))
#define SFD_FFT_T(REAL_, CONTIG_) (r7 ? SFD_FFT_T7(REAL_, CONTIG_, true) : SFD_FFT_T7(REAL_, CONTIG_, false))
  SFD_REQUIRE(P.contig || (!P.real_in && !P.dec_axis && P.in_lo == 1 && P.out_lo == 1), SFD_ERR_INVALID_ARG,
              "strided FFT passes take complex input with unit row stride and no deconvolution factors");
  SFD_REQUIRE(!P.contig || (P.in_el == 1 && P.out_el == 1), SFD_ERR_INVALID_ARG,
              "the contiguous FFT pass needs unit element stride");
  if (P.contig && P.real_in)
    SFD_TRY(SFD_FFT_T(true, true));
  else if (P.contig)
    SFD_TRY(SFD_FFT_T(false, true));
  else
    SFD_TRY(SFD_FFT_T(false, false));
#undef SFD_FFT_T
#undef SFD_FFT_T7
  return launch_check("fft_pass_kernel");
}

}  // namespace sfd
