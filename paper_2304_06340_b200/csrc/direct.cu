// direct.cu -- A4: fp64 direct summation nuhat_k = sum_j w_j exp(-i xi_k . x_j)  (eq. 2.8
// applied to the atoms of P:152).  FP64-pipe bound: 17 FP64 instructions per pair (phase 3, reduction 3, table +
// short monic polynomials 5, rotate and accumulate 6); 15.3 in the ball-rule variant (BALL below).
//
// Layout: one CTA = 128 threads x T targets held in registers (xi and the two accumulators); the sources
// stream through shared memory in tiles of kTile atoms, double-buffered with 1-D bulk TMA copies
// (cp.async.bulk + mbarrier) issued by one elected thread; every thread reads the same source at the same
// time (shared-memory broadcast, no bank conflicts).  For small K the source range is split over
// gridDim.y and the partial sums are combined in a fixed order by a second kernel (deterministic).
#include <algorithm>
#include <cstdlib>
#include <type_traits>

#include "common.cuh"
#include "direct.cuh"

namespace sfd {
namespace {

constexpr int kThreads = 128;
constexpr int kTile = 256;  // atoms per stage: 256*32 B = 8 KB; two stages (+ the 32 KB table: 48 KB per CTA, 4 CTAs per SM)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// exp(-i theta) for the inner loop, table + short polynomials.  The targets are pre-scaled by kTab/(2 pi) once per
// thread, so the phase arrives in units of 1/kTab of a turn: tq = n + f with n = rint(tq) (the 1.5*2^52 trick: three
// exact additions) and |f| <= 1/2, i.e. a residual angle of at most pi/256.  The table holds (cos, sin)(2 pi k / kTab)
// for the whole turn, so there is no quadrant logic at all; sin and cos of the residual need 3 coefficients each
// (Chebyshev-node fits at 60 digits, max error 1.2e-18 and 2.3e-16: tests/test_kernel_constants_cpu.py); one complex rotation joins the two.  17 FP64-pipe
// instructions per pair (phase 3, reduction 3, f^2 1, sin 3, cos 2, rotate + accumulate 6 -- 2 per source fold the polynomials' leading coefficients into the weight) against 21 plus a 10-instruction
// integer fix-up for the polynomial-only version: measured 1.31x faster (profiles/r1e_direct_sum_table.md), because
// every non-FP64 instruction costs an issue cycle next to a 2-cycle DFMA.
// The table is replicated kRep = 8 times in shared memory, entry (k, lane & 7) at index k*8 + (lane & 7): the 8 lanes
// of each LDS.128 phase then read 8 different 16-byte bank groups whatever their k -- conflict-free by construction.
constexpr int kTab = 256;
constexpr int kRep = 8;
static_assert(kRep * sizeof(double2) == 128, "the inner loop addresses table entry q at byte 128 q");
// The two polynomials are kept monic, S(z) = S2 ((z + As) z + Bs) and C(z) = C2 ((z + Ac) z + Bc), with the leading
// coefficients folded into the source's weight once per source: every step then reads at most two registers and one
// constant (a DFMA on three registers issues every 3 clocks instead of 2, profiles/r1b_direct_sum.md).
__constant__ double c_sc[8] = {
    -33201.10767024445654340395, 330692250.2493696703277053, 7.4219134520576935249e-11,   // As, Bs, S2: sin(a f) = f S(f^2)
    -19920.70833352124336730809, 66138595.24347913412699348, 1.5119764735229900432e-8,    // Ac, Bc, C2: cos(a f) = C(f^2)
    6755399441055744.0,                                                               // 1.5 * 2^52
    40.743665431525205956834243423364};                                               // kTab / (2 pi)

struct __align__(16) Stage {
  double x[kTile * 3];
  double w[kTile];
};

// BALL: the targets are nodes of the ball rule, xi_k = r_a dhat_m with k = (a - a0) n_dir + m (nodes.cu
// freq_expand_kernel; `xi` then points at the rule's 1-D tables).  A thread holds ONE direction and T radii: the dot
// product g = dhat . x_j is shared by its T pairs and the phase of a pair, r_a g, is never formed on its own: it enters
// the rounding addition and the residual f as the product of a DFMA -- 15 + 5/T FP64 instructions per pair instead of 17
// (8 + 2/T DFMA, 4 + 3/T DMUL, 3 DADD); five of them read three registers (the four accumulations and f) and issue every
// 3 clocks instead of 2 (profiles/r1b), the polynomial steps read two and a constant.  Measured at config 2: 37.0 clocks
// per warp and pair = 2 x 15.3 + 5.1 + 1.3 (four non-FP64 instructions: shift, mask, add, LDS.128).
// blockIdx.y runs over groups of T radii and blockIdx.z over the source splits.
// radii per thread of the ball-rule variant.  Measured at config 2 (direct_sum stage): general kernel 20.54 ms; ball
// variant with 4 / 8 / 12 / 16 radii per thread 19.05 / 17.76 / 18.09 / 16.86 ms (63 / 94 / 126 / 168 registers, 4 / 4 / 3 / 3
// CTAs per SM): the shared dot product and the per-source loads are amortised over more pairs
constexpr int kBallT = 16;
struct BallRule {
  int n_r, n_th, n_ph;   // sizes of the rule's tables: r[n_r] wr[n_r] mu[n_th] st[n_th] wmu[n_th] cph[n_ph] sph[n_ph]
  int a0, na;            // radial shells [a0, a0 + na)
  int b0, nb;            // rings [b0, b0 + nb) (the half rule: b0 = n_th / 2)
};

template <int T, bool BALL>
__global__ void __launch_bounds__(kThreads) direct_sum_kernel(const double* __restrict__ x, const double* __restrict__ w,
                                                             int64_t J, const double* __restrict__ xi, int64_t K,
                                                             double* __restrict__ out, int64_t j_per_split, int use_tma,
                                                             BallRule ball) {
  extern __shared__ __align__(16) unsigned char smem_raw[];   // 48.1 KB: beyond the static limit
  Stage* stage = reinterpret_cast<Stage*>(smem_raw);
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 2 * sizeof(Stage));
  // The table sits right after the stages and the barriers -- or, when the launch left room for it (kSmemAligned), at
  // the next shared-memory address that is a multiple of its 32 KB: the address of entry q is then a single LOP3,
  // ((q << 7) & 0x7f80) | (table + 16 (lane & 7)), instead of a mask and an addition (every non-FP64 instruction costs
  // the inner loop about a clock per pair: 16.03 -> 15.57 ms at config 2).  Decided here, uniformly for the CTA.
  const uint32_t smem_base = smem_u32(smem_raw), tab_lo = smem_base + 2 * (uint32_t)sizeof(Stage) + 16;
  uint32_t dyn_bytes;
  asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn_bytes));
  constexpr uint32_t kTabBytes = sizeof(double2) * kTab * kRep;
  const uint32_t tab_hi = (tab_lo + kTabBytes - 1) & ~(kTabBytes - 1);
  const bool aligned = BALL && tab_hi + kTabBytes <= smem_base + dyn_bytes;
  const uint32_t tab_sa = aligned ? tab_hi : tab_lo;
  double2* tab = reinterpret_cast<double2*>(smem_raw + (tab_sa - smem_base));
  const int tid = threadIdx.x;
  // (cos, sin)(2 pi k / kTab), replicated: entry (k, r) at k*kRep + r
  for (int i = tid; i < kTab * kRep; i += kThreads) {
    double sv, cv;
    sincospi((double)(i / kRep) * (2.0 / kTab), &sv, &cv);
    tab[i] = make_double2(cv, sv);
  }
  const uint32_t lane_sa = tab_sa + (uint32_t)(tid & (kRep - 1)) * 16;   // this lane's copy of entry 0
  const int64_t k0 = (int64_t)blockIdx.x * (kThreads * T);
  const int64_t jb = (int64_t)(BALL ? blockIdx.z : blockIdx.y) * j_per_split;
  const int64_t je = min(J, jb + j_per_split);
  const int ntiles = (int)((je - jb + kTile - 1) / kTile);

  double a0[T], a1[T], a2[T], re[T], im[T];
  const int n_dir = BALL ? ball.nb * ball.n_ph : 0;
  const int m_dir = BALL ? min((int)(blockIdx.x * kThreads + tid), n_dir - 1) : 0;   // this thread's direction
#pragma unroll
  for (int t = 0; t < T; ++t) {
    if (BALL) {
      const double* tr = xi;                       // r
      const double* tmu = xi + 2 * ball.n_r;       // mu, st, wmu, cph, sph
      const double* tst = tmu + ball.n_th;
      const double* tcp = tst + 2 * ball.n_th;
      const double* tsp = tcp + ball.n_ph;
      const int b = ball.b0 + m_dir / ball.n_ph, c = m_dir % ball.n_ph;
      // a0[0..2] = dhat in units of 1/kTab of a turn per unit radius (t == 0 only); a1[t] = the t-th radius
      if (t == 0) {
        a0[0] = __dmul_rn(tst[b], tcp[c]) * c_sc[7];
        a0[T > 1 ? 1 : 0] = __dmul_rn(tst[b], tsp[c]) * c_sc[7];
        a0[T > 2 ? 2 : 0] = tmu[b] * c_sc[7];
      }
      a1[t] = tr[ball.a0 + min((int)blockIdx.y * T + t, ball.na - 1)];
      a2[t] = 0.0;
    } else {
      const int64_t k = min(k0 + t * kThreads + tid, K - 1);
      a0[t] = xi[3 * k] * c_sc[7];   // phases in units of 1/kTab of a turn
      a1[t] = xi[3 * k + 1] * c_sc[7];
      a2[t] = xi[3 * k + 2] * c_sc[7];
    }
    re[t] = 0.0;
    im[t] = 0.0;
  }

  if (tid == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // a tile goes by TMA when it is full (sizes and addresses are then multiples of 16 B)
  auto issue = [&](int t) {
    const int64_t j0 = jb + (int64_t)t * kTile;
    Stage& s = stage[t & 1];
    mbar_expect_tx(&bar[t & 1], kTile * 32);
    bulk_g2s(s.x, x + 3 * j0, kTile * 24, &bar[t & 1]);
    bulk_g2s(s.w, w + j0, kTile * 8, &bar[t & 1]);
  };
  auto tile_n = [&](int t) { return (int)min((int64_t)kTile, je - (jb + (int64_t)t * kTile)); };

  if (tid == 0 && ntiles > 0 && use_tma && tile_n(0) == kTile) issue(0);

  auto run = [&](auto aligned_tag) {
  constexpr bool ALIGNED = decltype(aligned_tag)::value;
  for (int t = 0; t < ntiles; ++t) {
    const int n = tile_n(t);
    Stage& s = stage[t & 1];
    const bool tma = use_tma && n == kTile;
    if (tid == 0 && t + 1 < ntiles && use_tma && tile_n(t + 1) == kTile) issue(t + 1);
    if (tma) {
      mbar_wait(&bar[t & 1], (t >> 1) & 1);
    } else {
      const int64_t j0 = jb + (int64_t)t * kTile;
      for (int i = tid; i < 3 * n; i += kThreads) s.x[i] = x[3 * j0 + i];
      for (int i = tid; i < n; i += kThreads) s.w[i] = w[j0 + i];
      __syncthreads();
    }
#pragma unroll 2
    for (int j = 0; j < n; ++j) {
      const double x0 = s.x[3 * j], x1 = s.x[3 * j + 1], x2 = s.x[3 * j + 2], wj = s.w[j];
      const double wcj = wj * c_sc[5], wsj = wj * c_sc[2];   // w_j C2, w_j S2
      const double g = BALL ? __fma_rn(a0[0], x0, __fma_rn(a0[T > 1 ? 1 : 0], x1, a0[T > 2 ? 2 : 0] * x2)) : 0.0;
#pragma unroll
      for (int u = 0; u < T; ++u) {
        // BALL: the product r_a g goes into both additions unrounded (one instruction fewer, f exact)
        const double tq = BALL ? 0.0 : __fma_rn(a0[u], x0, __fma_rn(a1[u], x1, a2[u] * x2));
        const double nm = BALL ? __fma_rn(a1[u], g, c_sc[6]) : __dadd_rn(tq, c_sc[6]);
        const int q = __double2loint(nm);
        const double nn = __dsub_rn(nm, c_sc[6]);
        const double f = BALL ? __fma_rn(a1[u], g, -nn) : __dsub_rn(tq, nn);
        const double z = f * f;
        const double qs = __fma_rn(__dadd_rn(z, c_sc[0]), z, c_sc[1]);
        const double qc = __fma_rn(__dadd_rn(z, c_sc[3]), z, c_sc[4]);
        // table entry (q mod kTab, lane & 7) by its byte offset: 128 q + 16 (lane & 7)
        const uint32_t qoff = (uint32_t)(q << 7) & (uint32_t)((kTab - 1) << 7);
        const uint32_t ea = ALIGNED ? (qoff | lane_sa) : qoff + lane_sa;
        double2 e;   // read-only after the barrier above: no memory clobber needed
        asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(e.x), "=d"(e.y) : "r"(ea));
        // w e^{+i theta} = w (e.x + i e.y)(cr + i sr); the sign of the imaginary part is flipped at the store
        const double wc = wcj * qc, ws = wsj * (f * qs);
        re[u] = __fma_rn(e.x, wc, re[u]);
        im[u] = __fma_rn(e.y, wc, im[u]);
        re[u] = __fma_rn(-e.y, ws, re[u]);
        im[u] = __fma_rn(e.x, ws, im[u]);
      }
    }
    __syncthreads();  // everyone is done with this stage before it is refilled
  }
  };
  if (BALL && aligned) run(std::true_type{});
  else run(std::false_type{});

  double* o = out + (size_t)(BALL ? blockIdx.z : blockIdx.y) * (size_t)K * 2;
#pragma unroll
  for (int t = 0; t < T; ++t) {
    if (BALL) {
      const int ia = (int)blockIdx.y * T + t;
      const int m = (int)(blockIdx.x * kThreads + tid);
      if (ia < ball.na && m < n_dir) reinterpret_cast<double2*>(o)[(int64_t)ia * n_dir + m] = make_double2(re[t], -im[t]);
    } else {
      const int64_t k = k0 + t * kThreads + tid;
      if (k < K) reinterpret_cast<double2*>(o)[k] = make_double2(re[t], -im[t]);
    }
  }
}

__global__ void combine_splits_kernel(const double* __restrict__ part, int nsplit, int64_t n2, double* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n2) return;
  double acc = 0.0;
  for (int s = 0; s < nsplit; ++s) acc += part[(size_t)s * n2 + i];
  out[i] = acc;
}

constexpr size_t kSmemBytes = 2 * sizeof(Stage) + sizeof(double2) * kTab * kRep + 16;   // stages, table, 2 mbarriers
// The ball-rule variant (3 CTAs per SM by its registers) asks for enough to hold the table at a multiple of 32 KB: the
// dynamic segment starts 1 KB into the CTA's window (the system-reserved part), so the table can sit at 32 KB ... 64 KB.
// The kernel checks what it got and falls back to the packed layout otherwise.
constexpr size_t kSmemAligned = 64 * 1024 - 1024;

// Resident CTAs per SM of direct_sum_kernel<T> (shared memory binds: 4 with the current build); queried from the
// runtime once, with that number as the fallback when there is no device (workspace queries on a CPU box).
int ctas_per_sm(int T) {
  static int cache[kBallT + 1] = {};
  if (T == kBallT) {   // the ball-rule variant: 168 registers, 3 CTAs per SM
    if (cache[T] == 0) {
      int n = 0;
      cudaFuncSetAttribute(direct_sum_kernel<kBallT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemAligned);
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, direct_sum_kernel<kBallT, true>, kThreads, kSmemAligned) != cudaSuccess ||
          n <= 0) {
        cudaGetLastError();
        return 3;
      }
      cache[T] = n;
    }
    return cache[T];
  }
  if (cache[T] == 0) {
    int n = 0;
    cudaError_t e = cudaErrorUnknown;
    cudaFuncSetAttribute(direct_sum_kernel<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
    cudaFuncSetAttribute(direct_sum_kernel<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
    cudaFuncSetAttribute(direct_sum_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
    if (T == 4) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, direct_sum_kernel<4, false>, kThreads, kSmemBytes);
    if (T == 2) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, direct_sum_kernel<2, false>, kThreads, kSmemBytes);
    if (T == 1) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, direct_sum_kernel<1, false>, kThreads, kSmemBytes);
    if (e != cudaSuccess || n <= 0) {
      cudaGetLastError();
      return 4;
    }
    cache[T] = n;
  }
  return cache[T];
}

}  // namespace

DirectPlan direct_plan(int64_t J, int64_t K, int T_force) {
  DirectPlan p;
  const int64_t sms = num_sms();
  p.T = K >= sms * kThreads * 4 * 2 ? 4 : (K >= sms * kThreads * 2 * 2 ? 2 : 1);
  if (T_force > 0) p.T = T_force;
  p.blocks_k = (K + (int64_t)kThreads * p.T - 1) / ((int64_t)kThreads * p.T);
  // The CTAs are equal pieces of work and the SMs hold `slots` of them at a time: blocks_k * nsplit CTAs run in
  // ceil(blocks_k * nsplit / slots) waves, the last one partly empty.  Split the sources over gridDim.y so that
  // (a) every slot has work when K is small and (b) the last wave is nearly full (config 2: 2048 CTAs on 888 slots
  // are 2.31 waves, 77 % efficient; split in 3 they are 6.92 waves, 98.8 %).
  const int64_t slots = sms * ctas_per_sm(p.T);
  const int64_t tiles = std::max<int64_t>(1, (J + kTile - 1) / kTile);
  const int64_t max_split = std::min<int64_t>(tiles, 32);
  int64_t best = 1;
  double best_eff = 0.0;
  for (int64_t n = 1; n <= max_split; ++n) {
    const int64_t tiles_per = (tiles + n - 1) / n;
    const int64_t n_eff = (tiles + tiles_per - 1) / tiles_per;   // splits that actually get sources
    if (n_eff != n) continue;
    const double waves = (double)(p.blocks_k * n) / (double)slots;
    // uneven source split: the longest split sets the pace
    const double eff = waves / std::ceil(waves) * ((double)tiles / (double)(tiles_per * n));
    if (eff > best_eff + 0.02) {   // a further split must pay for its extra partial-sum traffic
      best_eff = eff;
      best = n;
    }
    if (best_eff >= 0.97) break;
  }
  const int64_t tiles_per = (tiles + best - 1) / best;
  p.j_per_split = tiles_per * kTile;
  p.nsplit = (int)std::max<int64_t>(1, (J + p.j_per_split - 1) / p.j_per_split);
  p.work_bytes = p.nsplit > 1 ? align_up((size_t)p.nsplit * (size_t)K * 16) : 0;
  return p;
}

int direct_sum(const double* d_x, const double* d_w, int64_t J, const double* d_xi, int64_t K, double* d_nuhat,
               void* d_work, size_t work_bytes, cudaStream_t st) {
  if (K == 0) return SFD_OK;
  if (J == 0) {
    SFD_CUDA_TRY(cudaMemsetAsync(d_nuhat, 0, (size_t)K * 16, st));
    return SFD_OK;
  }
  const DirectPlan p = direct_plan(J, K);
  {  // > 48 KB of dynamic shared memory needs the opt-in (per device; cheap to repeat)
    static thread_local int attr_dev = -1;
    int dev = 0;
    SFD_CUDA_TRY(cudaGetDevice(&dev));
    if (attr_dev != dev) {
      SFD_CUDA_TRY(cudaFuncSetAttribute(direct_sum_kernel<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes));
      SFD_CUDA_TRY(cudaFuncSetAttribute(direct_sum_kernel<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes));
      SFD_CUDA_TRY(cudaFuncSetAttribute(direct_sum_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes));
      attr_dev = dev;
    }
  }
  SFD_REQUIRE(work_bytes >= p.work_bytes && (p.work_bytes == 0 || d_work), SFD_ERR_WORKSPACE_TOO_SMALL,
              "direct sum needs %zu workspace bytes, got %zu", p.work_bytes, work_bytes);
  SFD_REQUIRE(p.blocks_k <= 0x7fffffffLL, SFD_ERR_INVALID_ARG, "K too large");
  const int use_tma = ((reinterpret_cast<uintptr_t>(d_x) | reinterpret_cast<uintptr_t>(d_w)) & 15) == 0;
  double* out = p.nsplit > 1 ? static_cast<double*>(d_work) : d_nuhat;
  dim3 grid((unsigned)p.blocks_k, (unsigned)p.nsplit);
  switch (p.T) {
    case 4: direct_sum_kernel<4, false><<<grid, kThreads, kSmemBytes, st>>>(d_x, d_w, J, d_xi, K, out, p.j_per_split, use_tma, BallRule{}); break;
    case 2: direct_sum_kernel<2, false><<<grid, kThreads, kSmemBytes, st>>>(d_x, d_w, J, d_xi, K, out, p.j_per_split, use_tma, BallRule{}); break;
    default: direct_sum_kernel<1, false><<<grid, kThreads, kSmemBytes, st>>>(d_x, d_w, J, d_xi, K, out, p.j_per_split, use_tma, BallRule{}); break;
  }
  SFD_TRY(launch_check("direct_sum_kernel"));
  if (p.nsplit > 1) {
    const int64_t n2 = 2 * K;
    combine_splits_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>(out, p.nsplit, n2, d_nuhat);
    SFD_TRY(launch_check("combine_splits_kernel"));
  }
  return SFD_OK;
}

size_t direct_ball_work_bytes(int64_t J, int64_t K) { return direct_plan(J, K, kBallT).work_bytes; }

// The same sum on the nodes of the ball rule (shells [a0, a1), rings [b0, n_theta) -- b0 = n_theta / 2 is the half rule),
// taken from the rule's 1-D tables in device memory (layout of nodes.cu freq_expand) instead of from the expanded nodes:
// one direction and four radii per thread (BALL above).  *used = false (nothing enqueued) when the rule is too small
// for that shape; the caller then runs direct_sum() on the expanded nodes.  Same workspace as direct_sum(J, K).
int direct_sum_ball(const double* d_x, const double* d_w, int64_t J, const double* d_tables, int n_r, int n_th, int n_ph,
                    int a0, int a1, int b0, double* d_nuhat, void* d_work, size_t work_bytes, cudaStream_t st, bool* used) {
  *used = false;
  const int na = a1 - a0, nb = n_th - b0;
  const int64_t n_dir = (int64_t)nb * n_ph, K = (int64_t)na * n_dir;
  if (J == 0 || K == 0 || na < kBallT || n_dir < kThreads) return SFD_OK;
  if (n_dir > 0x7fffffffLL / 4) return SFD_OK;
  const DirectPlan p = direct_plan(J, K, kBallT);
  {
    static thread_local int attr_dev = -1;
    int dev = 0;
    SFD_CUDA_TRY(cudaGetDevice(&dev));
    if (attr_dev != dev) {
      SFD_CUDA_TRY(cudaFuncSetAttribute(direct_sum_kernel<kBallT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemAligned));
      attr_dev = dev;
    }
  }
  SFD_REQUIRE(work_bytes >= p.work_bytes && (p.work_bytes == 0 || d_work), SFD_ERR_WORKSPACE_TOO_SMALL,
              "direct sum needs %zu workspace bytes, got %zu", p.work_bytes, work_bytes);
  const int use_tma = ((reinterpret_cast<uintptr_t>(d_x) | reinterpret_cast<uintptr_t>(d_w)) & 15) == 0;
  double* out = p.nsplit > 1 ? static_cast<double*>(d_work) : d_nuhat;
  const BallRule ball{n_r, n_th, n_ph, a0, na, b0, nb};
  dim3 grid((unsigned)((n_dir + kThreads - 1) / kThreads), (unsigned)((na + kBallT - 1) / kBallT), (unsigned)p.nsplit);
  SFD_REQUIRE(grid.y <= 65535 && grid.z <= 65535, SFD_ERR_UNSUPPORTED, "direct_sum_ball: rule too large");
  // SFD_DIRECT_PACKED=1 (tests): launch without the room for the aligned table, i.e. run the kernel's packed-layout loop
  const char* packed = std::getenv("SFD_DIRECT_PACKED");
  const size_t smem = packed && packed[0] == '1' ? kSmemBytes : kSmemAligned;
  direct_sum_kernel<kBallT, true><<<grid, kThreads, smem, st>>>(d_x, d_w, J, d_tables, K, out, p.j_per_split, use_tma, ball);
  SFD_TRY(launch_check("direct_sum_kernel"));
  if (p.nsplit > 1) {
    const int64_t n2 = 2 * K;
    combine_splits_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>(out, p.nsplit, n2, d_nuhat);
    SFD_TRY(launch_check("combine_splits_kernel"));
  }
  *used = true;
  return SFD_OK;
}

}  // namespace sfd
