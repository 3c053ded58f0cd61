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
#include <map>
#include <mutex>
#include <vector>

#include "fft.cuh"

namespace sfd {
namespace {

constexpr int kFftThreads = 512;

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
  return make_double2(__fma_rn(a.x, b.x, -a.y * b.y), __fma_rn(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ double2 mul_mi(double2 a) { return make_double2(a.y, -a.x); }   // a * (-i)
__device__ __forceinline__ double2 mul_pi(double2 a) { return make_double2(-a.y, a.x); }   // a * (+i)

// One pass; see FftPass (fft.cuh).  Shared memory: a[N][tbp] complex128, tbp = tb | 1.
template <bool REAL_IN>
__global__ void __launch_bounds__(kFftThreads) fft_pass_kernel(FftPass P, const void* __restrict__ in_raw,
                                                              double2* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2* a = reinterpret_cast<double2*>(smem_raw);
  const int N = P.N, tb = P.tb, tbp = P.tbp, tid = threadIdx.x;
  const int64_t tiles_per_hi = (P.n_lo + tb - 1) / tb;
  const int64_t hi = blockIdx.x / tiles_per_hi;
  const int64_t lo0 = (blockIdx.x - hi * tiles_per_hi) * tb;
  const int ncol = (int)min((int64_t)tb, P.n_lo - lo0);
  const int tsh = P.tb_shift;
  const double2* __restrict__ tw = P.tw;

  // ---- load: position j of the padded row holds mode l = j (j < N/2) or j - N; input index i = l + n_in/2
  const int half_in = P.n_in / 2;
  const double fhi = P.dec_hi ? P.dec_hi[hi] : 1.0;
  for (int idx = tid; idx < N * tb; idx += kFftThreads) {
    int j, col;
    if (P.contig) {
      col = idx / N;
      j = idx - col * N;
    } else {
      j = idx >> tsh;
      col = idx & (tb - 1);
    }
    const int l = j < N / 2 ? j : j - N;
    const int i = l + half_in;
    double2 val = make_double2(0.0, 0.0);
    if (col < ncol && i >= 0 && i < P.n_in) {
      const int64_t g = hi * P.in_hi + (lo0 + col) * P.in_lo + (int64_t)i * P.in_el;
      if (REAL_IN)
        val.x = static_cast<const double*>(in_raw)[g];
      else
        val = static_cast<const double2*>(in_raw)[g];
      if (P.dec_axis) {
        const double f = P.dec_axis[i] * fhi * P.dec_lo[lo0 + col];
        val.x *= f;
        val.y *= f;
      }
    }
    a[j * tbp + col] = val;
  }
  __syncthreads();

  // ---- in-place decimation-in-frequency stages
  int L = N;
  for (int s = 0; s < P.nfac; ++s) {
    const int r = P.fac[s];
    const int Ls = L / r;
    const int tstep = N / L;
    const int nbf = N / r;
    for (int idx = tid; idx < (nbf << tsh); idx += kFftThreads) {
      const int bf = idx >> tsh, col = idx & (tb - 1);
      const int b = Ls == 1 ? bf : (int)__umulhi((unsigned)bf, P.magic[s]);   // bf / Ls (exact: bf < 2^16)
      const int j = bf - b * Ls;
      double2* x = a + (b * L + j) * tbp + col;
      const int st = Ls * tbp;
      const int tj = j * tstep;
      if (r == 4) {
        const double2 x0 = x[0], x1 = x[st], x2 = x[2 * st], x3 = x[3 * st];
        const double2 t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), t3 = csub(x1, x3);
        x[0] = cadd(t0, t2);
        x[st] = cmul(cadd(t1, mul_mi(t3)), tw[tj]);
        x[2 * st] = cmul(csub(t0, t2), tw[2 * tj]);
        x[3 * st] = cmul(cadd(t1, mul_pi(t3)), tw[3 * tj]);
      } else if (r == 2) {
        const double2 x0 = x[0], x1 = x[st];
        x[0] = cadd(x0, x1);
        x[st] = cmul(csub(x0, x1), tw[tj]);
      } else if (r == 3) {
        const double2 x0 = x[0], x1 = x[st], x2 = x[2 * st];
        const double2 t1 = cadd(x1, x2);
        const double2 t2 = make_double2(x0.x - 0.5 * t1.x, x0.y - 0.5 * t1.y);
        const double h = 0.86602540378443864676;
        const double2 t3 = make_double2(h * (x1.x - x2.x), h * (x1.y - x2.y));
        x[0] = cadd(x0, t1);
        x[st] = cmul(cadd(t2, mul_mi(t3)), tw[tj]);
        x[2 * st] = cmul(cadd(t2, mul_pi(t3)), tw[2 * tj]);
      } else {  // r == 5
        const double2 x0 = x[0], x1 = x[st], x2 = x[2 * st], x3 = x[3 * st], x4 = x[4 * st];
        const double c1 = 0.30901699437494742410, c2 = -0.80901699437494742410;
        const double s1 = 0.95105651629515357212, s2 = 0.58778525229247312917;
        const double2 t1 = cadd(x1, x4), t2 = cadd(x2, x3), t3 = csub(x1, x4), t4 = csub(x2, x3);
        const double2 a1 = make_double2(x0.x + c1 * t1.x + c2 * t2.x, x0.y + c1 * t1.y + c2 * t2.y);
        const double2 a2 = make_double2(x0.x + c2 * t1.x + c1 * t2.x, x0.y + c2 * t1.y + c1 * t2.y);
        const double2 b1 = make_double2(s1 * t3.x + s2 * t4.x, s1 * t3.y + s2 * t4.y);
        const double2 b2 = make_double2(s2 * t3.x - s1 * t4.x, s2 * t3.y - s1 * t4.y);
        x[0] = make_double2(x0.x + t1.x + t2.x, x0.y + t1.y + t2.y);
        x[st] = cmul(cadd(a1, mul_mi(b1)), tw[tj]);
        x[2 * st] = cmul(cadd(a2, mul_mi(b2)), tw[2 * tj]);
        x[3 * st] = cmul(cadd(a2, mul_pi(b2)), tw[3 * tj]);
        x[4 * st] = cmul(cadd(a1, mul_pi(b1)), tw[4 * tj]);
      }
    }
    __syncthreads();
    L = Ls;
  }

  // ---- store the band m in [lo, lo + nout) through the digit-reversal table
  for (int idx = tid; idx < P.nout * tb; idx += kFftThreads) {
    int mm, col;
    if (P.contig) {
      col = idx / P.nout;
      mm = idx - col * P.nout;
    } else {
      mm = idx >> tsh;
      col = idx & (tb - 1);
    }
    if (col >= ncol) continue;
    int m = P.lo + mm;
    m = m < 0 ? m + N : (m >= N ? m - N : m);
    out[hi * P.out_hi + (lo0 + col) * P.out_lo + (int64_t)mm * P.out_el] = a[P.rev[m] * tbp + col];
  }
}

// ---- host tables, cached per transform length ----------------------------------------------------------------
struct HostTables {
  std::vector<double> tw;     // N complex: exp(-2 pi i t / N)
  std::vector<int32_t> rev;   // position of output frequency k after the DIF stages
  int nfac;
  int fac[16];
};
std::mutex g_mu;
std::map<int, HostTables> g_tables;

const HostTables& tables_for(int N) {
  std::lock_guard<std::mutex> lk(g_mu);
  auto it = g_tables.find(N);
  if (it != g_tables.end()) return it->second;
  HostTables t;
  t.nfac = 0;
  int n = N;
  while (n % 4 == 0) { t.fac[t.nfac++] = 4; n /= 4; }
  while (n % 2 == 0) { t.fac[t.nfac++] = 2; n /= 2; }
  while (n % 3 == 0) { t.fac[t.nfac++] = 3; n /= 3; }
  while (n % 5 == 0) { t.fac[t.nfac++] = 5; n /= 5; }
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
  return g_tables.emplace(N, std::move(t)).first->second;
}

}  // namespace

bool fft_length_ok(int N) {
  int n = N;
  while (n % 2 == 0) n /= 2;
  while (n % 3 == 0) n /= 3;
  while (n % 5 == 0) n /= 5;
  return n == 1 && N >= 2;
}

size_t fft_tables_bytes(const int n2[3]) {
  size_t b = 0;
  for (int d = 0; d < 3; ++d) b += align_up((size_t)n2[d] * 16) + align_up((size_t)n2[d] * 4);
  return b;
}

// Rows per tile (a power of two) and row pitch.  Two CTAs per SM whenever at least 4 rows fit in half the shared
// memory (one CTA's loads and stores overlap the other's butterflies), else one CTA per SM.  Only the transposing
// load of the contiguous-axis pass needs the odd pitch.
int fft_tile(int N, int contig, int* tbp) {
  auto pitch = [&](int tb) { return contig ? (tb | 1) : tb; };
  int pick = 0;
  for (int tb = 8; tb >= 4 && !pick; tb >>= 1)
    if ((size_t)N * pitch(tb) * 16 <= (size_t)112 * 1024) pick = tb;
  for (int tb = 8; tb >= 1 && !pick; tb >>= 1)
    if ((size_t)N * pitch(tb) * 16 <= (size_t)224 * 1024) pick = tb;
  if (tbp) *tbp = pick ? pitch(pick) : 0;
  return pick;
}

int fft_upload_tables(const int n2[3], void* d_tables, FftTables* out, cudaStream_t st) {
  char* base = static_cast<char*>(d_tables);
  size_t o = 0;
  for (int d = 0; d < 3; ++d) {
    SFD_REQUIRE(fft_length_ok(n2[d]) && fft_tile(n2[d], 1, nullptr) > 0, SFD_ERR_UNSUPPORTED, "FFT length %d is not supported", n2[d]);
    const HostTables& t = tables_for(n2[d]);
    out->tw[d] = reinterpret_cast<double2*>(base + o);
    SFD_CUDA_TRY(cudaMemcpyAsync(base + o, t.tw.data(), (size_t)n2[d] * 16, cudaMemcpyHostToDevice, st));
    o += align_up((size_t)n2[d] * 16);
    out->rev[d] = reinterpret_cast<int32_t*>(base + o);
    SFD_CUDA_TRY(cudaMemcpyAsync(base + o, t.rev.data(), (size_t)n2[d] * 4, cudaMemcpyHostToDevice, st));
    o += align_up((size_t)n2[d] * 4);
    out->nfac[d] = t.nfac;
    for (int s = 0; s < t.nfac; ++s) out->fac[d][s] = t.fac[s];
  }
  return SFD_OK;
}

int fft_pass(FftPass P, const FftTables& T, int axis, const void* d_in, double* d_out, cudaStream_t st) {
  P.tw = T.tw[axis];
  P.rev = T.rev[axis];
  P.nfac = T.nfac[axis];
  for (int s = 0; s < P.nfac; ++s) P.fac[s] = T.fac[axis][s];
  P.tb = fft_tile(P.N, P.contig, &P.tbp);
  P.tb_shift = 0;
  while ((1 << P.tb_shift) < P.tb) ++P.tb_shift;
  {
    int L = P.N;
    for (int s = 0; s < P.nfac; ++s) {
      const int Ls = L / P.fac[s];
      P.magic[s] = Ls > 1 ? (unsigned)(0x100000000ULL / (unsigned long long)Ls + 1ULL) : 0u;
      L = Ls;
    }
  }
  const int64_t tiles = P.n_hi * ((P.n_lo + P.tb - 1) / P.tb);
  if (tiles == 0) return SFD_OK;
  SFD_REQUIRE(tiles < 0x7fffffffLL, SFD_ERR_UNSUPPORTED, "FFT pass has too many tiles");
  const size_t smem = (size_t)P.N * P.tbp * 16;
  static bool attr[2] = {false, false};
  if (!attr[P.real_in]) {
    if (P.real_in)
      SFD_CUDA_TRY(cudaFuncSetAttribute(fft_pass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024));
    else
      SFD_CUDA_TRY(cudaFuncSetAttribute(fft_pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024));
    attr[P.real_in] = true;
  }
  if (P.real_in)
    fft_pass_kernel<true><<<(unsigned)tiles, kFftThreads, smem, st>>>(P, d_in, reinterpret_cast<double2*>(d_out));
  else
    fft_pass_kernel<false><<<(unsigned)tiles, kFftThreads, smem, st>>>(P, d_in, reinterpret_cast<double2*>(d_out));
  return launch_check("fft_pass_kernel");
}

}  // namespace sfd
