// fft.cuh -- interface of the pruned in-shared-memory FFT passes (fft.cu; A5-5/A5-6 of the type-3 NUFFT).
#pragma once
#include "common.cuh"

namespace sfd {

// Device tables per axis: twiddles exp(-2 pi i t / N), digit-reversal positions, radix list (4s, 2, 3s, 5s).
struct FftTables {
  const double2* tw[3];
  const int32_t* rev[3];
  const int32_t* klow[3];   // fixed-geometry kernels: frequency of the first output of the last group's block b
  const double2* ftw[3];    // fixed-geometry kernels: outer-twiddle tables
  int32_t* counters;        // fixed-geometry kernels: one zeroed tile counter per axis (each pass runs once per upload)
  double2 cst[3][3][9];     // fixed-geometry kernels: inner constants e^{-2 pi i p1 q2 / G} of the three groups, per axis
  int nfac[3];
  int fac[3][16];
  int npair[3];
  int pair[3][16];   // fused stage pairs, code R1 * 8 + R2
};

// One pass of 1-D transforms of length N over a 2-level set of rows ("columns" c = (hi, lo)).
//   input  element (hi, lo, i), i in [0, n_in):  in [hi*in_hi  + lo*in_lo  + i*in_el]    <-> mode l = i - n_in/2
//   output element (hi, lo, m), m in [lo, lo+nout): out[hi*out_hi + lo*out_lo + (m-lo)*out_el]
//   out(m) = sum_l in(l) exp(-2 pi i l m / N)
// contig = 1: the transform axis is the contiguous one (in_el = out_el = 1; loads and stores run along the axis);
// contig = 0: `lo` is the contiguous index (in_lo = out_lo = 1; loads and stores run across the tile's rows).
// dec_axis/dec_hi/dec_lo (all or none): the input is multiplied by dec_axis[i] * dec_hi[hi] * dec_lo[lo].
struct FftPass {
  int N, n_in, lo, nout;
  int64_t n_hi, n_lo;
  int64_t in_hi, in_lo, in_el, out_hi, out_lo, out_el;
  int contig, real_in;
  int f32;   // 1: input and output arrays are single precision (float / float2); arithmetic and shared memory stay fp64
  const double *dec_axis, *dec_hi, *dec_lo;
  // ball != 0 (strided passes): the consumer reads the output only inside an ellipsoid (the targets of the ball rule).
  // With q = ((a - ball_ca) ball_ira)^2 + ((b - ball_cb) ball_irb)^2 of a column -- ball == 1: lo = a * ball_nb + b (both
  // other axes are frequencies: the last pass); ball == 2: b = lo only (ball_ira = 0: the third axis is still spatial) --
  // a column stores only the outputs |mm - ball_ct| <= ball_rt sqrt(1 - q) (+1), none when q > 1, and a tile none of
  // whose columns has q <= 1 is skipped.  The rest of the output is left untouched.
  int ball, ball_nb;
  double ball_ca, ball_cb, ball_ira, ball_irb, ball_ct, ball_rt;
  // filled in by fft_pass():
  int tb, tbp, tb_shift, cg_shift, nfac, fac[16];   // cg_shift: log2(column groups per tile)
  int npair, pair[16];  // fused stage pairs: code = R1 * 8 + R2 (R2 = 1: single stage)
  unsigned magic[16];   // floor(2^32 / Lq) + 1 per pair: g / Lq = umulhi(g, magic)
  const double2* tw;
  const int32_t* rev;
  const int32_t* klow;
  const double2* ftw;
  int32_t* counter;
  double2 cst[3][9];
};

bool fft_length_ok(int N);
int fft_tile(int N, int contig, int* tbp);             // rows per tile (0: does not fit shared memory) and pitch
size_t fft_tables_bytes(const int n2[3]);
int fft_upload_tables(const int n2[3], void* d_tables, FftTables* out, cudaStream_t st);
int fft_pass(FftPass P, const FftTables& T, int axis, const void* d_in, double* d_out, cudaStream_t st);

}  // namespace sfd
