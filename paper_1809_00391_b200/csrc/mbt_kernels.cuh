// mbt_kernels.cuh -- CUDA kernels (sm_100a) of the longitudinal multi-bunch tracker.
//
// One turn = two launches:
//   k_pass  the fused particle pass (S0 kick of the previous turn, S7 moments, S1 RF, S2 radiation,
//           S3 drift, S4 binning), one read and one write of the SoA fp64 particle store;
//   k_wake  per bunch: counts -> charges, S5 Toeplitz short-range convolution, S6 source phasors, and (the default,
//           one CTA per bunch) the bunch's own phasor gathered from the sources of the bunches ahead and the history
//           ring, as soon as those are flagged ready; where a bunch is split over several CTAs the last CTA to finish
//           runs the S6 in-turn phasor scan over the fill pattern instead.
// The long-range part of the wake is kept as ONE complex number per (bunch, resonator) and expanded onto the
// bins when a CTA of the next pass stages the bunch's wake grid in shared memory.
//
// Step numbers and citations: include/mbt.h.  DESIGN.md has the data layout and the roofline of each kernel.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "mbt_math.cuh"

namespace mbt {

constexpr int kPassThreads = 256;
constexpr int kWakeThreads = 256;
static_assert(kWakeThreads == kPassThreads, "the one-launch turn runs wake_body in a pass CTA");
constexpr int kMaxCav = 8;
constexpr int kMaxLR = 8;
constexpr int kDefaultNPair = 0;  // pairs per thread and iteration of the pass: 1, 2, or 0 = chosen from the workload at create

struct cplx {
  double re, im;
};
__host__ __device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return cplx{fma(a.re, b.re, -(a.im * b.im)), fma(a.re, b.im, a.im * b.re)};
}
__host__ __device__ __forceinline__ cplx cadd(cplx a, cplx b) { return cplx{a.re + b.re, a.im + b.im}; }
// a*b + c
__host__ __device__ __forceinline__ cplx cfma(cplx a, cplx b, cplx c) {
  return cplx{fma(a.re, b.re, fma(-a.im, b.im, c.re)), fma(a.re, b.im, fma(a.im, b.re, c.im))};
}

// device-resident control words (so that a captured CUDA graph replays without parameter updates)
struct Ctrl {
  uint32_t turn;          // completed turns
  uint32_t ticket[2];     // CTAs that have closed their bunch in the turn of this parity (last-CTA-done election; two
                          // slots: the first CTAs of a turn's wake kernel may overlap the last ones of the turn before)
  uint32_t kick_pending;  // 1: the wake of turn `turn` has not been applied to delta yet
  uint32_t kick_base;     // the turn at which no kick was pending last (create, mbt_set_particles, a getter's flush)
  uint32_t pad[3];
};

// gather cell k of a wake grid V[0..nb) (D12): linear gather: the particle with rint(t) = k sits between the centres
// of bins k-1 and k, v(f) = mid + f dif, f = t - k in [-1/2, 1/2], mid = (V[k-1] + V[k]) / 2, dif = V[k] - V[k-1],
// with V[-1] := V[0], V[nb] := V[nb-1]; nearest grid point: mid = V[k], dif = 0.  Cell nb+1 is zero.
struct WakeCell {
  double mid, dif;
};
struct CellF {  // the same cell of the complex table F_r
  cplx mid, dif;
};

struct Args {
  // particle store: tau[M][ld], delta[M][ld], ld even; pair p of bunch b = particles (2p, 2p+1)
  double *tau, *delta;
  int64_t ld;
  uint32_t Np;       // particles per bunch
  uint32_t ppb;      // pairs per bunch = ld / 2
  int32_t M;
  int64_t total_pairs;
  uint32_t tile_pairs;  // pairs per CTA of the pass (a multiple of kPassThreads * NPAIR)
  // S1
  int32_t n_cav;
  double cav_amp[kMaxCav];  // V_c / E0
  double cav_w[kMaxCav];    // m_c * omega_rf
  double cav_ph[kMaxCav];
  double loss;              // U0 / E0
  // S2
  int32_t rad;
  double one_minus_DE, A_q;
  PhiloxKeys keys;
  // S3
  double drift;  // alpha_c * T0
  // S4 / S0
  int32_t nb;
  int32_t gather;
  const double *lo_hist;  // [M] start of the window the current histogram / wake was built on (S0 reads it)
  const double *lo_next;  // [M] start of the window this pass bins with (S4); equal to lo_hist unless window_mode 1 (D31)
  double invDelta, nb_d, invE0;
  // wake state
  const double *Vsr;    // [M][nb]   short-range wake of the last turn [V]
  const cplx *P;        // [M][R]    long-range phasor seen by bunch b
  const cplx *F;        // [R][nb]   C_r exp(lambda_r c_j)
  const WakeCell *cellSR;   // [M][nb+2] gather cells of the short-range wake of the last turn (k_wake)
  const CellF *cellF;       // [R][nb+2] gather cells of F_r: cell(V_SR + sum_r Re[F_r P_r]) = cellSR + sum_r Re[cellF_r P_r]
  int32_t R;            // long-range resonators
  uint32_t *hist;       // [M][nb]   accumulating counts of the pass in flight
  double *mom_acc;      // [M][4]    sum tau, sum delta, sum tau^2, sum delta^2
  unsigned long long *nout_acc;  // [M]
  Ctrl *ctrl;
  const LogTabEntry *logtab;  // [128] device copy of the log table
  MathTab mt;
  // one-launch turn (mbt_tuning.turn_mode 2): the last CTA of a bunch to finish builds that bunch's wake (wake_body)
  int32_t fused;              // 1: this launch is a whole turn; its predecessor in the stream is the pass before it
  int32_t b0;                 // global index of the handle's first bunch (Philox counter word; 0 unless sharded)
  // per-bunch start (two-launch turn, one k_wake CTA per bunch): a pass CTA waits for ITS bunch's wake, not for the grid
  int32_t flag_wait;
  int32_t count_done;           // 1: count this CTA in bunch_done[b] when it has flushed (the wake kernel's CTA of the bunch waits for it)
  const uint32_t *bunch_ready;  // [M] turn whose wake of bunch b is complete (k_wake, release)
  uint32_t *tile_turn;          // [M][tiles] completed turns of the tile: written by the tile's own CTA, read by its next one
  uint32_t *bunch_done;       // [M] pass CTAs of the bunch that have flushed their counts and moment sums
};

// Particle staging: a CTA owns kStages shared-memory stages of kPassThreads*NPAIR pairs (tau block, then delta
// block), filled by cp.async.bulk (TMA, global -> shared) kStages-1 iterations ahead of their use.  full[stage]
// completes when both blocks have landed (expect_tx); empty[stage] completes when all warps have read the stage
// (one arrival per warp).  Thread 0 is the producer.  Bytes in flight are bounded by shared memory, not registers.
#ifndef MBT_STAGES
#define MBT_STAGES 4
#endif
constexpr int kStages = MBT_STAGES;
__host__ __device__ inline size_t pass_stage_bytes(int npair) {
  return (size_t)kStages * 2 * kPassThreads * npair * 16;
}
__host__ __device__ inline size_t pass_smem_bytes(int nb, int npair) {
  return pass_stage_bytes(npair) + (size_t)(nb + 2) * sizeof(WakeCell) + (size_t)(nb + 1) * sizeof(uint32_t) +
         128 * sizeof(LogTabEntry) + 16;
}

// ---- programmatic dependent launch (PTX griddepcontrol; no-ops in a kernel launched without the attribute).  The pass and
// k_wake of a turn are launched as a chain of programmatic dependents: a kernel may become resident while its
// predecessor is still running, does what does not depend on it, and waits before it touches the predecessor's output.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ---- mbarrier / bulk-copy primitives (PTX; SASS: SYNCS / UBLKCP)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ double2 lds_double2(uint32_t addr) {  // volatile: the stage is rewritten by the async proxy
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void stg_double4(void *p, double a, double b, double c, double d) {  // STG.E.256 (sm_100)
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "MBT_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra MBT_DONE;\n"
      "bra MBT_WAIT;\n"
      "MBT_DONE:\n"
      "}" ::"r"(bar),
      "r"(parity)
      : "memory");
}

// 0 <= t < nb decided on the high word of t: nb < 2^21 is an integer, so the low word of (double)nb is zero and
// t >= nb  <=>  hi(t) >= hi(nb) for t >= +0; a negative t (sign bit) or a NaN compares above hi(nb) as unsigned.
// t = -0.0 cannot occur: a window start of 0 is stored as -0.0, so that (-0.0) - lo = +0.0 (in the window, bin 0,
// as the oracle's t >= 0 decides) and every other difference is unchanged.
__device__ __forceinline__ bool in_window(double t, uint32_t hi_nb) { return (uint32_t)__double2hiint(t) < hi_nb; }

// ------------------------------------------------------------------ wake
struct WakeArgs {
  int32_t M, nb, R, K;
  int32_t S;               // CTAs per bunch (grid.y): the outputs of the convolution are dealt out over them
  uint32_t *rd_cnt, *wr_cnt;  // [M] splits that have read the counts / written their share of V_SR (S > 1)
  uint32_t Np;
  int32_t mode;            // 0: full turn (S5, S6, bump the turn counter); 1: finalise counts and moments only
  const double *qm;        // [M]      macro-particle charge Q_b / N_p
  const double *w;         // [nb]     short-range table w_k = W(k Delta); nullptr: none
  const cplx *Esrc;        // [R][nb]  exp(-lambda_r c_k)
  const cplx *g_step;      // [M][R]   exp(lambda_r (s_{j+1}-s_j) T_rf), j < M-1
  const cplx *g_tail;      // [M][R]   exp(lambda_r (s_{M-1}-s_j) T_rf)
  const cplx *g_hist;      // [K][R]   exp(lambda_r (k T0 - (s_{M-1}-s_0) T_rf)), k = 1..K
  uint32_t *hist;          // [M][nb]  in: counts of this turn; out: zero
  uint32_t *hist_last;     // [M][nb]  out: counts of this turn
  double *Vsr;             // [M][nb]
  WakeCell *cellSR;        // [M][nb+2] gather cells of Vsr (what the pass stages)
  int32_t gather;          // 1 linear, 0 nearest grid point
  // bunch-following window (D31); window_mode 0: the arrays below keep their initial values
  int32_t window_mode, s_max;
  double tau_lo, Delta;
  int32_t *s_hist, *s_next;   // [M] window shift in bins: of this turn's histogram / of the next binning
  double *lo_hist, *lo_next;  // [M] tau_lo + s Delta (0 stored as -0.0, see in_window())
  const cplx *shift_src;      // [R][2 s_max + 1] exp(-lambda_r s Delta), s = -s_max..s_max
  const cplx *shift_wit;      // [R][2 s_max + 1] exp(+lambda_r s Delta)
  cplx *a_cur;             // [M][R]   source phasors of this turn
  cplx *ring_a;            // [K+1][M][R] slot n % (K+1)
  cplx *ring_A;            // [K+1][R]    per-turn aggregates, slot n % (K+1)
  cplx *P;                 // [M][R]
  double *mom_acc;         // [M][4]  in: sums gathered by the pass; out: zero
  unsigned long long *nout_acc;  // [M]
  double *mom_last;        // [M][6]
  double *mom_log;         // [cap][M][6] or nullptr
  int64_t log_cap;
  Ctrl *ctrl;
  uint32_t smem_wake_bytes, smem_pass_bytes;  // dynamic shared memory of a k_wake launch / of a pass launch (one-launch turn)
  // one-launch turn: per-bunch phasor gather instead of the scan (wake_body<false, true>)
  int32_t bunch_wait, tiles;  // 1: a CTA waits for the `tiles` pass CTAs of ITS bunch (bunch_done) instead of the pass's grid
  uint32_t *bunch_done;       // [M] (the pass counts, this kernel's CTA of the bunch resets)
  int32_t part;               // 0: the whole wake; sharded handle: 1 = up to the gather cells, 2 = phasor gather and close
  int32_t Mg, b0;             // bunches of the whole fill and index of this handle's first one (Mg = M, b0 = 0 unless sharded)
  cplx *xbuf;                 // sharded: [Mg padded][R] exchange buffer of the turn's source phasors (else nullptr)
  int32_t gather_P;           // k_wake with one CTA per bunch: per-bunch phasor gather (all CTAs resident) instead of the scan
  int32_t h, slots;           // harmonic number; slots of ring_a / ring_A (K + 1, at least 2)
  const int32_t *bucket;      // [M]
  const cplx *gd;             // [R][h] exp(lambda_r d T_rf), d = 0 .. h-1 (bucket distance)
  uint32_t *a_ready;          // [M][R] turn whose source phasor a[b][r] is in ring_a (release / acquire)
  uint32_t *bunch_ready;      // [M]    turn whose wake (cells, phasor P, windows, cleared counts) of bunch b is complete
  uint32_t *agg_ready;        // [1]    turn whose aggregate A_n is in ring_A
};

// L2 load of a complex number written earlier in this kernel by another CTA (never through a stale L1 line)
__device__ __forceinline__ cplx __ldcg_cplx(const cplx *p) {
  const double2 v = __ldcg(reinterpret_cast<const double2 *>(p));
  return cplx{v.x, v.y};
}

// flags written by one CTA and awaited by another of the same (or the next) launch
__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t *p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_u32(uint32_t *p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// turn numbers are compared modulo 2^32
__device__ __forceinline__ void wait_turn(const uint32_t *flag, uint32_t n) {
  while ((int32_t)(ld_acquire_u32(flag) - n) < 0) {
  }
}

// affine map x -> g x + c over the complex numbers; (first o second)(x) = second(first(x))
struct Affine {
  cplx g, c;
};
__device__ __forceinline__ Affine compose(const Affine &first, const Affine &second) {
  return Affine{cmul(first.g, second.g), cfma(first.c, second.g, second.c)};
}

// Shared memory of wake_body: charges, V_SR, and the wake table with sixteen zeros in front and eight behind (the sliding
// window of the register-blocked convolution runs off both ends).  The scan of the turn's last CTA stages its operands
// (48 bytes per bunch and resonator) in the same memory if they fit into what the launch provides (`smem_bytes`).
// Up to this many bins the one CTA of a bunch convolves on the fp64 tensor path (wake_first).  Measured, same session, us
// per turn: c1 (200 bins) 9.81 -> 9.27; c3 (500 bins) 18.9 -> 20.2 -- a column group's accumulator is a chain of n_b / 32
// dependent DMMAs, and their latency, not their number, is what a single CTA pays -- so the limit sits between.
constexpr int kDmmaMaxBins = 320;
__host__ __device__ inline size_t wake_part_bytes(int nb) {  // per-warp partial sums of the tensor-core convolution
  return nb <= kDmmaMaxBins ? (size_t)(kWakeThreads / 32) * 64 * ((nb + 63) / 64) * sizeof(double) + 16 : 0;
}
__host__ __device__ inline size_t wake_smem_bytes(int nb, int M) {
  return (size_t)(3 * nb + 24) * sizeof(double) + (size_t)M * sizeof(int32_t) + wake_part_bytes(nb);
}
// D += A B, A 8x4 (row-major: lane holds A[lane >> 2][lane & 3]), B 4x8 (lane holds B[lane & 3][lane >> 2]),
// D 8x8 (lane holds D[lane >> 2][2 (lane & 3) + {0, 1}]), all fp64 (SASS: DMMA)
__device__ __forceinline__ void dmma_8x8x4(double &d0, double &d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__host__ __device__ inline size_t scan_smem_bytes(int M, int R) { return (size_t)M * (size_t)R * 3 * sizeof(cplx); }

// The wake of bunch b (and, for the CTA that finishes last, the closing of the turn).  Called by every thread of a CTA of
// kWakeThreads threads: by k_wake (SPLIT: the S = gridDim.y CTAs of a bunch share its convolution), and by the last pass
// CTA of a bunch in the one-launch turn (SPLIT = false).  smem_d: smem_bytes >= wake_smem_bytes(nb) of shared memory.
// Counts and moment sums were accumulated with atomics by other CTAs, possibly of this same launch: they are read
// through L2 (__ldcg), never through an L1 line that a neighbouring bunch's reader may have pulled in earlier.
//
// Everything here is latency: a bunch's wake is ~1e5 multiply-adds, but a dependent trip to L2 costs most of a
// microsecond, and this code runs ONCE per CTA, so its instruction fetches miss too -- a first version with every loop
// over resonators and scan elements unrolled (200 KB of SASS) ran slower than the loops it replaced.  Hence: compact loops,
// few dependent trips to memory, a register-blocked convolution that uses every thread.
template <bool SPLIT, bool FUSED>
__device__ __forceinline__ bool wake_first(const WakeArgs &A, const int b, const int split, double *smem_d, const uint32_t smem_bytes) {
  constexpr int NW = kWakeThreads / 32;
  const int nb = A.nb;
  double *sq = smem_d;               // [nb] charge per bin
  double *sv = smem_d + nb;          // [nb] V_SR of this bunch
  double *sw = smem_d + 2 * nb + 16;  // [-16, nb + 8) wake table, zero outside [0, nb)
  int32_t *sB = reinterpret_cast<int32_t *>(smem_d + 3 * nb + 24);  // [M] buckets (FUSED)
  __shared__ bool s_last;
  __shared__ unsigned long long s_cnt[NW][2];

  const int tid = threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5;
  const int S = SPLIT ? A.S : 1;  // few bunches: S CTAs share a bunch (split 0 also does the per-bunch work)
  // completed turns; the turn being closed is n_done + 1.  One CTA per bunch: from the bunch's own flag (what this bunch's
  // CTA of the turn before published -- the control word may still be waiting for that turn's closing CTA)
  const uint32_t n_done = FUSED ? __ldcg(&A.bunch_ready[b]) : A.ctrl->turn;
  const uint32_t n = n_done + 1u;

  // counts -> charges; keep a copy of the counts; clear the accumulator for the next pass.  The loads of a round (counts,
  // table, and -- if it fits -- the source factors exp(-lambda_r c_k) of all resonators, into shared memory) have no
  // global store between them, so that they are all in flight together: one trip to L2.
  const double qm = A.qm[b];
  const bool follow = A.mode == 0 && A.window_mode == 1;
  const int32_t s_used = follow ? A.s_next[b] : 0;   // the window the pass binned this turn with
  unsigned long long n_in = 0ull, m1 = 0ull;         // sum c_k, sum k c_k
  const bool sources = A.mode == 0 && split == 0 && A.R > 0;
  const cplx *pE = A.Esrc;  // [R][nb] as the source sums read it: staged behind the buckets if the launch's memory holds it
  if (sources && wake_smem_bytes(nb, A.Mg) + (size_t)A.R * nb * sizeof(cplx) + 16 <= (size_t)smem_bytes) {
    cplx *sE = reinterpret_cast<cplx *>(((reinterpret_cast<uintptr_t>(sB + A.Mg) + 15) & ~(uintptr_t)15) + wake_part_bytes(nb));
    const int nE = A.R * nb;
#pragma unroll 4
    for (int i = tid; i < nE; i += kWakeThreads) sE[i] = A.Esrc[i];
    pE = sE;
  }
#pragma unroll 2
  for (int j = tid; j < nb; j += kWakeThreads) {
    const uint32_t c = __ldcg(&A.hist[(size_t)b * nb + j]);
    if (A.mode == 0) sw[j] = A.w ? A.w[j] : 0.0;
    sq[j] = qm * (double)c;
    reinterpret_cast<uint32_t *>(sv)[j] = c;
    n_in += c;
    m1 += (unsigned long long)j * c;
  }
  for (int j = tid; j < nb; j += kWakeThreads) {  // the stores, from the thread's own shared-memory copy
    const uint32_t c = reinterpret_cast<const uint32_t *>(sv)[j];
    if (split == 0) A.hist_last[(size_t)b * nb + j] = c;
    if (S == 1) A.hist[(size_t)b * nb + j] = 0u;
  }
  if (tid < 24) sw[tid < 16 ? tid - 16 : nb + tid - 16] = 0.0;
  if (FUSED && A.mode == 0 && A.R > 0)
    for (int j = tid; j < A.Mg; j += kWakeThreads) sB[j] = A.bucket[j];
  if (S > 1) {  // the last split to have read the counts clears them (nobody waits for anybody)
    __syncthreads();
    if (tid == 0) s_last = (atomicAdd(&A.rd_cnt[b], 1u) == (uint32_t)(S - 1));
    __syncthreads();
    if (s_last) {
      for (int j = tid; j < nb; j += kWakeThreads) A.hist[(size_t)b * nb + j] = 0u;
      if (tid == 0) A.rd_cnt[b] = 0u;
    }
  }
  if (follow && split == 0) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      n_in += __shfl_down_sync(0xffffffffu, n_in, o);
      m1 += __shfl_down_sync(0xffffffffu, m1, o);
    }
    if (lane == 0) { s_cnt[warp][0] = n_in; s_cnt[warp][1] = m1; }
  }
  __syncthreads();
  if (follow && split == 0 && tid == 0) {
    // D31: the window moves by rint(centroid in bins - nb/2) whole bins (half up), exact integer arithmetic
    long long N = 0, S1 = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) { N += (long long)s_cnt[w][0]; S1 += (long long)s_cnt[w][1]; }
    long long step = 0;
    if (N > 0) {
      const long long num = 2 * S1 + (2 - (long long)nb) * N, den = 2 * N;
      step = num / den;
      if (num % den != 0 && num < 0) step -= 1;
    }
    long long s_new = (long long)s_used + step;
    s_new = s_new > A.s_max ? A.s_max : (s_new < -(long long)A.s_max ? -(long long)A.s_max : s_new);
    double lo_h = __dadd_rn(A.tau_lo, __dmul_rn((double)s_used, A.Delta));
    double lo_n = __dadd_rn(A.tau_lo, __dmul_rn((double)s_new, A.Delta));
    if (lo_h == 0.0) lo_h = -0.0;
    if (lo_n == 0.0) lo_n = -0.0;
    A.s_hist[b] = s_used;
    A.lo_hist[b] = lo_h;
    A.s_next[b] = (int32_t)s_new;
    A.lo_next[b] = lo_n;
  }
  // S7: close the moments the pass gathered (state after turn n_done's kick): by the last thread of the CTA, beside
  // the convolution of the others
  if (split == 0 && tid == kWakeThreads - 1) {
    const double N = (double)A.Np;
    const double s1 = __ldcg(&A.mom_acc[b * 4 + 0]), s2 = __ldcg(&A.mom_acc[b * 4 + 1]);
    const double s11 = __ldcg(&A.mom_acc[b * 4 + 2]), s22 = __ldcg(&A.mom_acc[b * 4 + 3]);
    const double no = (double)__ldcg(&A.nout_acc[b]);
    const double iN = 1.0 / N;
    const double mt = s1 * iN, md = s2 * iN;
    const double vt = fmax(s11 * iN - mt * mt, 0.0), vd = fmax(s22 * iN - md * md, 0.0);
    double m[6] = {N - no, no, mt, md, sqrt(vt), sqrt(vd)};
#pragma unroll
    for (int k = 0; k < 6; ++k) A.mom_last[b * 6 + k] = m[k];
    if (A.mom_log && n_done >= 1u && (int64_t)n_done <= A.log_cap) {
#pragma unroll
      for (int k = 0; k < 6; ++k) A.mom_log[((size_t)(n_done - 1u) * A.M + b) * 6 + k] = m[k];
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) A.mom_acc[b * 4 + k] = 0.0;
    A.nout_acc[b] = 0ull;
  }
  if (A.mode != 0) return false;

  // S6 sources: a[b][r] = sum_k q[k] exp(-lambda_r c_k).  One warp per resonator, counted from the LAST warp down (the
  // first warps carry the convolution's heaviest tasks); shuffles only, no block barrier.
  for (int r = NW - 1 - warp; r < A.R && split == 0; r += NW) {
    double are = 0.0, aim = 0.0;
#pragma unroll 4
    for (int k = lane; k < nb; k += 32) {
      const cplx e = pE[(size_t)r * nb + k];
      are = fma(sq[k], e.re, are);
      aim = fma(sq[k], e.im, aim);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      are += __shfl_xor_sync(0xffffffffu, are, o);
      aim += __shfl_xor_sync(0xffffffffu, aim, o);
    }
    if (lane == 0) {
      cplx a{are, aim};
      if (follow) a = cmul(a, A.shift_src[(size_t)r * (2 * A.s_max + 1) + (s_used + A.s_max)]);  // bin centres at their own window
      A.a_cur[(size_t)b * A.R + r] = a;
      A.ring_a[((size_t)(n % (uint32_t)A.slots) * A.Mg + (A.b0 + b)) * A.R + r] = a;  // rows by the GLOBAL bunch index
      if (A.xbuf) A.xbuf[(size_t)(A.b0 + b) * A.R + r] = a;                          // sharded: this rank's rows of the exchange
      if (FUSED) st_release_u32(&A.a_ready[(size_t)(A.b0 + b) * A.R + r], n);        // later bunches' gathers wait for it
    }
  }

  // S5: V_SR[j] = sum_{k<=j} w[j-k] q[k], register-blocked.  Outputs come in blocks of NO = 8 consecutive bins; block pi
  // is paired with block J-1-pi so that every pair has nb + 8 (+-8) terms; a pair is dealt to SEG lanes of one warp, lane
  // g taking the g-th segment of each block's k-range with the NO table values it needs in a sliding register window
  // (per k: two shared-memory loads and NO independent DFMAs -- 2 bytes of shared-memory traffic per multiply-add, where
  // one output per thread moves 16; the load/store unit, not the fp64 pipe, bounds this loop); a shuffle reduction over
  // the SEG lanes closes the sums.  SEG is the largest power of two that keeps all threads of the bunch's S CTAs busy;
  // segment lengths are odd, so that the lanes of a pair fall into different banks.
  if (A.w && !SPLIT && nb <= kDmmaMaxBins) {
    // One CTA per bunch, up to kDmmaMaxBins bins: the convolution as a dense fp64 contraction on the tensor path (north_star (3)).
    // With j = 8a + alpha, k = 8(a - d) + beta:  V[alpha][a] = sum_d sum_beta W_d[alpha][beta] Q_d[beta][a],
    // W_d[alpha][beta] = w[8d + alpha - beta] (an 8x8 Toeplitz block, zero outside the table: causality is the zero
    // padding in front of it), Q_d[beta][a] = q[8(a - d) + beta]: for every block diagonal d an (8x8)(8 x n_b/8) product,
    // n_b^2 / 2 multiply-adds in all, none wasted.  mma.m8n8k4 tiles: 8 columns a per tile (a column group g), two k-steps
    // of four beta.  Warp w takes the diagonals d = w mod 8 for ALL column groups (equal work; the A fragment of a
    // diagonal serves every group), an accumulator pair per group and k-step (independent chains); the eight partial
    // results are added in shared memory in warp order (reproducible).  ~30 DMMA per warp where the DFMA loop issued 640 per thread.
    const int G = (nb + 63) >> 6;
    double *part = reinterpret_cast<double *>((reinterpret_cast<uintptr_t>(sB + A.Mg) + 15) & ~(uintptr_t)15);  // [NW][64 G]
    const int al = lane >> 2, k4 = lane & 3;
    // column groups four at a time, the two k-steps on accumulators of their own: 8 independent DMMA chains in flight
    for (int g0 = 0; g0 < G; g0 += 4) {
      double c[4][2][2];
#pragma unroll
      for (int g = 0; g < 4; ++g) c[g][0][0] = c[g][0][1] = c[g][1][0] = c[g][1][1] = 0.0;
      for (int d = warp; 8 * d < nb + 7 && d <= 8 * (g0 + 3) + 7; d += NW) {
#pragma unroll
        for (int ks = 0; ks < 2; ++ks) {
          const int beta = 4 * ks + k4;
          const int wi = 8 * d + al - beta;                    // >= -7: the zeros in front of the table
          const double av = wi < nb ? sw[wi] : 0.0;
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            if (g0 + g < G && 8 * (g0 + g) + 7 >= d) {         // warp-uniform
              const int a = 8 * (g0 + g) + al;
              const int qi = 8 * (a - d) + beta;
              const double bv = (a >= d && qi < nb) ? sq[qi] : 0.0;
              dmma_8x8x4(c[g][ks][0], c[g][ks][1], av, bv);
            }
          }
        }
      }
#pragma unroll
      for (int g = 0; g < 4; ++g)
        if (g0 + g < G) {
          part[(size_t)warp * 64 * G + (8 * (g0 + g) + 2 * k4) * 8 + al] = c[g][0][0] + c[g][1][0];
          part[(size_t)warp * 64 * G + (8 * (g0 + g) + 2 * k4 + 1) * 8 + al] = c[g][0][1] + c[g][1][1];
        }
    }
    __syncthreads();
    for (int j = tid; j < nb; j += kWakeThreads) {
      double v = 0.0;
#pragma unroll
      for (int w = 0; w < NW; ++w) v += part[(size_t)w * 64 * G + j];
      A.Vsr[(size_t)b * nb + j] = v;
      sv[j] = v;
    }
  } else if (A.w) {
    constexpr int NO = 8;
    const int J = (nb + NO - 1) / NO, pairs = (J + 1) >> 1;
    const int nthreads = S * kWakeThreads;
    int seg = 1, lg = 0;
    while (seg < 32 && 2 * seg * pairs <= nthreads) { seg <<= 1; ++lg; }
    const int tasks = pairs << lg;
    const int g = tid & (seg - 1);
    for (int base = 0; base < tasks; base += nthreads) {  // uniform over the CTA: the shuffles need every lane
      const int task = base + split * kWakeThreads + tid;
      const bool act = task < tasks;
      const int pi = act ? (task >> lg) : 0;
#pragma unroll 1
      for (int h = 0; h < 2; ++h) {
        const int jb = h ? J - 1 - pi : pi;
        const int j0 = NO * jb;
        const bool skip = h && jb == pi;                      // the middle block of an odd J is its own partner
        const int kend = (act && !skip) ? min(j0 + NO, nb) : 0;  // k in [0, kend)
        const int len = ((kend + seg - 1) >> lg) | 1;
        const int ka = min(g * len, kend), kb = min(ka + len, kend);
        const double *wp = sw + (j0 - ka);  // wp[i] = w[j0 + i - ka]
        double w[NO], a[NO];
#pragma unroll
        for (int i = 0; i < NO; ++i) { w[i] = wp[i]; a[i] = 0.0; }
        // NO values of k per round: all 2 NO loads first, then NO x NO multiply-adds on static register indices (the
        // window slides by renaming, not by moves); beyond kb the charges are taken as zero
#pragma unroll 1
        for (int k = ka; k < kb; k += NO) {
          double q[NO], nw[NO];
#pragma unroll
          for (int t = 0; t < NO; ++t) {
            q[t] = (k + t < kb) ? sq[k + t] : 0.0;
            nw[t] = wp[-1 - t];  // w[j0 - k - 1 - t]
          }
#pragma unroll
          for (int t = 0; t < NO; ++t)
#pragma unroll
            for (int i = 0; i < NO; ++i) a[i] = fma(i >= t ? w[i - t] : nw[t - i - 1], q[t], a[i]);
#pragma unroll
          for (int i = 0; i < NO; ++i) w[i] = nw[NO - 1 - i];
          wp -= NO;
        }
        for (int o = seg >> 1; o > 0; o >>= 1) {
#pragma unroll
          for (int i = 0; i < NO; ++i) a[i] += __shfl_xor_sync(0xffffffffu, a[i], o);
        }
        if (act && g == 0 && !skip) {
#pragma unroll
          for (int i = 0; i < NO; ++i) {
            const int j = j0 + i;
            if (j < nb) {
              A.Vsr[(size_t)b * nb + j] = a[i];
              if (!SPLIT) sv[j] = a[i];
            }
          }
        }
      }
    }
  } else {
    for (int j = split * kWakeThreads + tid; j < nb; j += S * kWakeThreads) { A.Vsr[(size_t)b * nb + j] = 0.0; sv[j] = 0.0; }
  }
  if (S > 1) {  // the last split to finish gathers the bunch's V_SR and goes on alone
    __syncthreads();
    if (tid == 0) {
      __threadfence();
      s_last = (atomicAdd(&A.wr_cnt[b], 1u) == (uint32_t)(S - 1));
    }
    __syncthreads();
    if (!s_last) return false;
    __threadfence();
    if (tid == 0) A.wr_cnt[b] = 0u;
    for (int j = tid; j < nb; j += kWakeThreads) sv[j] = __ldcg(&A.Vsr[(size_t)b * nb + j]);
  }
  __syncthreads();
  for (int k = tid; k < nb + 2; k += kWakeThreads) {
    WakeCell c{0.0, 0.0};
    if (A.gather == 1) {
      if (k <= nb) {
        const double lo = sv[k > 0 ? k - 1 : 0], hi = sv[k < nb ? k : nb - 1];
        c.mid = 0.5 * (lo + hi);
        c.dif = hi - lo;
      }
    } else if (k < nb) {
      c.mid = sv[k];
    }
    A.cellSR[(size_t)b * (nb + 2) + k] = c;
  }
  return true;
}

// The second half of a bunch's wake: the phasor P[b] and the closing of the turn.  FUSED (one CTA per bunch): the
// per-bunch gather; else the last-CTA scan.  Needs the buckets in shared memory (FUSED; staged by wake_first, or by
// wake_body for a sharded handle's second phase).
template <bool FUSED>
__device__ __forceinline__ void wake_second(const WakeArgs &A, const int b, double *smem_d, const uint32_t smem_bytes) {
  constexpr int NW = kWakeThreads / 32;
  const int nb = A.nb;
  int32_t *sB = reinterpret_cast<int32_t *>(smem_d + 3 * nb + 24);  // [Mg] buckets (FUSED)
  __shared__ bool s_last;
  const int tid = threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5;
  const uint32_t n = (FUSED ? __ldcg(&A.bunch_ready[b]) : A.ctrl->turn) + 1u;  // the turn being closed
  const bool follow = A.mode == 0 && A.window_mode == 1;
  const int32_t s_used = follow ? A.s_hist[b] : 0;  // the window this turn's counts were taken on (set by wake_first)
  const int M = A.M, R = A.R, K = A.K;
  if constexpr (FUSED) {
    // S6, one-launch turn: the phasor bunch b sees, gathered by the bunch's own closing CTA as the pairwise sum itself --
    //   P[b][r] = gd_r[s_b - s_0] sum_{k=1..min(K,n-1)} A_{n-k}[r] g_hist[k][r] + sum_{j<b} a_j[r] gd_r[s_b - s_j],
    // gd_r[d] = exp(lambda_r d T_rf) a host table over the bucket distance (every factor decays).  The sources a_j of the
    // bunches ahead are awaited one by one (flags a_ready, set by their closing CTAs: CTAs of a lower index, dispatched
    // earlier, so they are resident or done -- the wait cannot deadlock); no CTA waits for the whole grid, and the scan of
    // the two-launch turn, which ran alone on the device after the last bunch, is gone.  A resonator is dealt to
    // NW / R warps (fixed order of summation: deterministic).
    __shared__ cplx s_part[NW];
    if (R > 0) {
      const int nq = NW / R;                 // warps per resonator (R <= NW)
      const int r = warp % R, q = warp / R;  // warps >= nq R idle
      const int Kh = (int)min((uint32_t)K, n - 1u);
      const int bg = A.b0 + b;               // global index of the bunch: the bunches ahead are 0 .. bg-1, on any rank
      const int n_el = bg + Kh;
      const int sb = sB[bg];
      cplx acc{0.0, 0.0};
      if (q < nq) {
        const cplx *gdr = A.gd + (size_t)r * A.h;
        const cplx g0 = gdr[sb - sB[0]];
#pragma unroll 2
        for (int e = q * 32 + lane; e < n_el; e += 32 * nq) {
          if (e < bg) {
            wait_turn(&A.a_ready[(size_t)e * R + r], n);
            acc = cfma(__ldcg_cplx(&A.ring_a[((size_t)(n % (uint32_t)A.slots) * A.Mg + e) * R + r]), gdr[sb - sB[e]], acc);
          } else {
            const int k = e - bg + 1;
            wait_turn(A.agg_ready, n - 1u);
            acc = cfma(__ldcg_cplx(&A.ring_A[(size_t)((n - (uint32_t)k) % (uint32_t)A.slots) * R + r]),
                       cmul(A.g_hist[(size_t)(k - 1) * R + r], g0), acc);
          }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          acc.re += __shfl_xor_sync(0xffffffffu, acc.re, o);
          acc.im += __shfl_xor_sync(0xffffffffu, acc.im, o);
        }
      }
      if (lane == 0) s_part[warp] = acc;
      __syncthreads();
      if (tid < R) {
        cplx Pb{0.0, 0.0};
        for (int w = tid; w < nq * R; w += R) { Pb.re += s_part[w].re; Pb.im += s_part[w].im; }
        // the phasor as bunch b's own window sees it: the pass expands Re[cellF_r P], cellF built on the unshifted grid
        A.P[(size_t)b * R + tid] = follow ? cmul(Pb, A.shift_wit[(size_t)tid * (2 * A.s_max + 1) + (s_used + A.s_max)]) : Pb;
      }
    }
    // the bunch is complete: publish it, take a ticket; the CTA that closes the last bunch closes the turn
    __syncthreads();
    if (tid == 0) {
      __threadfence();
      st_release_u32(&A.bunch_ready[b], n);
      s_last = (atomicAdd(&A.ctrl->ticket[n & 1u], 1u) == (uint32_t)(M - 1));
      // All M tickets of turn n are taken: the counter goes back to zero at once, before anything this CTA publishes can
      // let turn n + 2 (the next user of this word) advance -- not after the release of agg_ready, as it used to.
      if (s_last) A.ctrl->ticket[n & 1u] = 0u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // A_n[r] = sum_j a_j[r] exp(lambda_r (s_{M-1} - s_j) T_rf): the aggregate later turns' seeds are built from
    if (R > 0) {
      const int nq = NW / R, r = warp % R, q = warp / R;
      cplx acc{0.0, 0.0};
      if (q < nq) {
#pragma unroll 2
        for (int j = q * 32 + lane; j < A.Mg; j += 32 * nq)
          acc = cfma(__ldcg_cplx(&A.ring_a[((size_t)(n % (uint32_t)A.slots) * A.Mg + j) * R + r]), A.g_tail[(size_t)j * R + r], acc);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          acc.re += __shfl_xor_sync(0xffffffffu, acc.re, o);
          acc.im += __shfl_xor_sync(0xffffffffu, acc.im, o);
        }
      }
      if (lane == 0) s_part[warp] = acc;
      __syncthreads();
      if (tid < R) {
        cplx An{0.0, 0.0};
        for (int w = tid; w < nq * R; w += R) { An.re += s_part[w].re; An.im += s_part[w].im; }
        A.ring_A[(size_t)(n % (uint32_t)A.slots) * R + tid] = An;
      }
    }
    __syncthreads();
    if (tid == 0) {
      __threadfence();
      st_release_u32(A.agg_ready, n);
      A.ctrl->kick_pending = 1u;
      A.ctrl->turn = n;
    }
  } else {
  // last-CTA-done election: the CTA that sees every other CTA's ticket closes the turn.  Barrier, then ONE thread's
  // fence and ticket (the pattern of a cooperative grid barrier: the barrier orders the CTA's writes before the fence).
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    s_last = (atomicAdd(&A.ctrl->ticket[n & 1u], 1u) == (uint32_t)(A.M - 1));
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();

  // S6: P_0 = G_n (history seed), P_{j+1} = (P_j + a_j) g_j -- an inclusive scan of affine maps over the fill
  // pattern; every factor is exp(lambda * positive time), |g| < 1.  One WARP per resonator, all resonators at once,
  // shuffles only (no block barrier inside): this tail runs alone on the device, so its latency is the turn's.  Its
  // operands -- a, g_step, g_tail of every bunch and resonator -- are first staged in shared memory by ALL threads (one
  // trip to L2 instead of one per four bunches of a lane's run) if the launch's shared memory holds them.
  const int total = M * R;
  const cplx *pa = A.a_cur, *pgs = A.g_step, *pgt = A.g_tail;
  const bool staged = scan_smem_bytes(M, R) <= (size_t)smem_bytes;
  if (staged) {
    cplx *sa = reinterpret_cast<cplx *>(smem_d), *sgs = sa + total, *sgt = sgs + total;
#pragma unroll 2
    for (int i = tid; i < total; i += kWakeThreads) {
      sa[i] = __ldcg_cplx(&A.a_cur[i]);
      sgs[i] = A.g_step[i];
      sgt[i] = A.g_tail[i];
    }
    pa = sa; pgs = sgs; pgt = sgt;
    __syncthreads();
  }
  const int run = (M + 31) / 32;  // consecutive bunches per lane
  for (int r = warp; r < R; r += NW) {
    // G_n = sum_{k=1..min(K,n-1)} A_{n-k} exp(lambda (k T0 - span)): lanes take k = lane+1, lane+33, ...
    cplx G{0.0, 0.0};
    for (int k = lane + 1; k <= K && (int64_t)n - k >= 1; k += 32)
      G = cfma(__ldcg_cplx(&A.ring_A[(size_t)((n - (uint32_t)k) % (uint32_t)A.slots) * R + r]), A.g_hist[(size_t)(k - 1) * R + r], G);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      G.re += __shfl_xor_sync(0xffffffffu, G.re, o);
      G.im += __shfl_xor_sync(0xffffffffu, G.im, o);
    }
    // lane-local composite of its run of bunches, and this turn's own aggregate.  The run is walked four bunches
    // at a time with all of a chunk's loads issued before its arithmetic.
    const int j_lo = lane * run, j_hi = min(j_lo + run, M);
    Affine loc{cplx{1.0, 0.0}, cplx{0.0, 0.0}};
    cplx own{0.0, 0.0};
    for (int j0 = j_lo; j0 < j_hi; j0 += 4) {
      cplx a[4], gt[4], gs[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int j = min(j0 + u, M - 1);
        a[u] = staged ? pa[(size_t)j * R + r] : __ldcg_cplx(&pa[(size_t)j * R + r]);
        gt[u] = pgt[(size_t)j * R + r];
        gs[u] = pgs[(size_t)j * R + r];
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int j = j0 + u;
        if (j < j_hi) {
          own = cfma(a[u], gt[u], own);
          if (j + 1 < M) loc = compose(loc, Affine{gs[u], cmul(a[u], gs[u])});
        }
      }
    }
    // inclusive warp scan of the lane composites (Kogge-Stone on shuffles), then the exclusive prefix applied to G
    Affine inc = loc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      Affine up;
      up.g.re = __shfl_up_sync(0xffffffffu, inc.g.re, o); up.g.im = __shfl_up_sync(0xffffffffu, inc.g.im, o);
      up.c.re = __shfl_up_sync(0xffffffffu, inc.c.re, o); up.c.im = __shfl_up_sync(0xffffffffu, inc.c.im, o);
      if (lane >= o) inc = compose(up, inc);
    }
    Affine pre;
    pre.g.re = __shfl_up_sync(0xffffffffu, inc.g.re, 1); pre.g.im = __shfl_up_sync(0xffffffffu, inc.g.im, 1);
    pre.c.re = __shfl_up_sync(0xffffffffu, inc.c.re, 1); pre.c.im = __shfl_up_sync(0xffffffffu, inc.c.im, 1);
    cplx Pj = (lane > 0) ? cfma(pre.g, G, pre.c) : G;
    for (int j0 = j_lo; j0 < j_hi; j0 += 4) {
      cplx a[4], gs[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int j = min(j0 + u, M - 1);
        a[u] = staged ? pa[(size_t)j * R + r] : __ldcg_cplx(&pa[(size_t)j * R + r]);
        gs[u] = pgs[(size_t)j * R + r];
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int j = j0 + u;
        if (j < j_hi) {
          // the phasor as bunch j's own window sees it: the pass expands Re[cellF_r P], cellF built on the unshifted grid
          A.P[(size_t)j * R + r] = follow ? cmul(Pj, A.shift_wit[(size_t)r * (2 * A.s_max + 1) + (__ldcg(&A.s_hist[j]) + A.s_max)]) : Pj;
          if (j + 1 < M) Pj = cmul(cadd(Pj, a[u]), gs[u]);
        }
      }
    }
    // A_n = sum_j a_j exp(lambda (s_{M-1}-s_j) T_rf)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      own.re += __shfl_xor_sync(0xffffffffu, own.re, o);
      own.im += __shfl_xor_sync(0xffffffffu, own.im, o);
    }
    if (lane == 0) A.ring_A[(size_t)(n % (uint32_t)A.slots) * R + r] = own;
  }
  __syncthreads();
  if (tid == 0) {
    A.ctrl->ticket[n & 1u] = 0u;
    A.ctrl->kick_pending = 1u;
    A.ctrl->turn = n;
  }
  }  // !FUSED
}


// The wake of bunch b: wake_first, then wake_second.  A sharded handle (mbt_params.shard) runs the two halves as two
// launches around the exchange of the source phasors: part 1 stops after the gather cells (the sources of the other
// ranks' bunches are not here yet), part 2 starts at the phasor gather.
template <bool SPLIT, bool FUSED>
__device__ __forceinline__ void wake_body(const WakeArgs &A, const int b, const int split, double *smem_d, const uint32_t smem_bytes) {
  if (FUSED && A.part == 2) {
    int32_t *sB = reinterpret_cast<int32_t *>(smem_d + 3 * A.nb + 24);
    for (int j = threadIdx.x; j < A.Mg; j += kWakeThreads) sB[j] = A.bucket[j];
    __syncthreads();
  } else {
    if (!wake_first<SPLIT, FUSED>(A, b, split, smem_d, smem_bytes)) return;
    if (FUSED && A.part == 1) return;
  }
  wake_second<FUSED>(A, b, smem_d, smem_bytes);
}

__global__ void __launch_bounds__(kWakeThreads, 3) k_wake(const __grid_constant__ WakeArgs A) {
  extern __shared__ double smem_wake[];
  // The pass of this turn is complete (counts, moment sums) -- or, with bunch_wait (one CTA per bunch, launched as a
  // programmatic dependent of the pass): the pass CTAs of THIS bunch are.  CTAs that become resident during the pass's last
  // wave then build the wakes of the bunches that are long complete, and the next pass -- whose CTAs wait for their own
  // bunch's wake -- finds them ready when it starts.
  if (A.bunch_wait) {
    if (threadIdx.x == 0) {
      while (ld_acquire_u32(&A.bunch_done[blockIdx.x]) < (uint32_t)A.tiles) {
      }
      A.bunch_done[blockIdx.x] = 0u;
    }
    __syncthreads();
  } else {
    griddep_wait();
  }
  griddep_launch_dependents();  // the next pass may become resident: it stages what does not depend on this kernel
  if (A.S > 1) wake_body<true, false>(A, (int)blockIdx.x, (int)blockIdx.y, smem_wake, A.smem_wake_bytes);
  else if (A.gather_P) wake_body<false, true>(A, (int)blockIdx.x, 0, smem_wake, A.smem_wake_bytes);
  else wake_body<false, false>(A, (int)blockIdx.x, 0, smem_wake, A.smem_wake_bytes);
}
// out of line in the pass, so that its registers are not the hot loop's
__device__ __noinline__ void wake_bunch_fused(const WakeArgs &A, int b, double *smem_d) {
  wake_body<false, true>(A, b, 0, smem_d, A.smem_pass_bytes);
}


// One iteration of the fused pass on registers, for the NPAIR pairs (2 NPAIR particles) a thread owns: S0 S7 | S1 S2 S3 |
// S4.  t2, d2: the pairs as loaded (tau, delta); tau, del: the particles after the iteration (the caller stores them).
// p: the thread's first pair in the bunch, p1: end of the tile; sW: the bunch's gather cells, sL: the log table, sH: the
// CTA's counts (bin nb is a sink).  Shared by the streaming pass (k_pass) and the chip-resident one (k_resident).
template <bool MAP, bool RAD, int GATHER, int NCAV, int NPAIR, bool FULL>
__device__ __forceinline__ void advance_pairs(const Args &A, const double2 (&t2)[NPAIR], const double2 (&d2)[NPAIR],
                                              double (&tau)[2 * NPAIR], double (&del)[2 * NPAIR], const uint32_t p, const uint32_t p1,
                                              const int b, const uint32_t n, const double lo_old, const double lo_new,
                                              const uint32_t hi_nb, const int nb, const WakeCell *sW, const LogTabEntry *sL,
                                              uint32_t *sH, double &st, double &sd, double &stt, double &sdd, uint32_t &nout) {
  constexpr int NP = 2 * NPAIR;
  double z[NP];
  bool live[NP];
  BmState bm[NPAIR];
  uint32_t xs[4] = {0u, 0u, 0u, 0u};
#pragma unroll
  for (int q = 0; q < NPAIR; ++q) {
    const uint32_t pq = p + q;
    tau[2 * q] = t2[q].x; tau[2 * q + 1] = t2[q].y;
    del[2 * q] = d2[q].x; del[2 * q + 1] = d2[q].y;
    live[2 * q] = FULL || (pq < p1 && 2u * pq < A.Np);  // past the end of the tile: stale stage contents, ignored;
    live[2 * q + 1] = FULL || (live[2 * q] && (2u * pq + 1u < A.Np));  // the slots from N_p up to ld are padding
    z[2 * q] = z[2 * q + 1] = 0.0;
    if (MAP && RAD) {
      // one Philox block serves FOUR consecutive particles (D8): counter (particle >> 2, bunch, turn, tag 0);
      // its words (x0, x1) give the Box-Muller pair of particles 4j, 4j+1, (x2, x3) that of 4j+2, 4j+3; the even
      // particle of a pair takes z_c, the odd one z_s.  A thread that owns the whole quad (NPAIR = 2) calls it once.
      if (q == 0 || NPAIR == 1) philox4x32_10(pq >> 1, (uint32_t)(b + A.b0), n, 0u, A.keys, xs[0], xs[1], xs[2], xs[3]);
      const bool hi_half = (NPAIR == 2) ? (q == 1) : ((pq & 1u) != 0u);  // with NPAIR = 2 the thread's first pair is even
      const double u1 = uniform32(A.mt, hi_half ? xs[2] : xs[0]), u2 = uniform32(A.mt, hi_half ? xs[3] : xs[1]);
      if (NCAV > 0) bm[q] = box_muller_head(A.mt, sL, u1, u2, A.A_q);  // polynomials: lock step with S1's
      else box_muller_fast(A.mt, sL, u1, u2, A.A_q, z[2 * q], z[2 * q + 1]);
    }
  }
  // S0: kick of the previous turn's wake.  t exactly as the binning computed it (one subtraction, one
  // multiplication, no contraction), so the in-window decision is the one that deposited the particle.
  // In-window test 0 <= t < nb on the high word of t alone (in_window()): an integer compare, off the fp64 pipe.
  double t[NP];
  bool in[NP];
#pragma unroll
  for (int i = 0; i < NP; ++i) {
    t[i] = __dmul_rn(__dsub_rn(tau[i], lo_old), A.invDelta);
    in[i] = live[i] && in_window(t[i], hi_nb);
    int kk;
    double f;
    if (GATHER == 1) {
      const double km = t[i] + MBT_MAGIC;
      kk = __double2loint(km);
      f = t[i] - (km - MBT_MAGIC);
    } else {
      kk = __double2int_rd(t[i]);
      f = 0.0;
    }
    kk = in[i] ? kk : nb + 1;
    const WakeCell c = sW[kk];
    del[i] = fma(-fma(f, c.dif, c.mid), A.invE0, del[i]);
    if (!in[i] && live[i]) nout += 1u;
  }
  // S7: moments of the state after the kick
#pragma unroll
  for (int i = 0; i < NP; ++i)
    if (live[i]) {
      st += tau[i];
      sd += del[i];
      stt = fma(tau[i], tau[i], stt);
      sdd = fma(del[i], del[i], sdd);
    }
  if (MAP) {
    // S1: RF cavities.  The phase is formed as the oracle forms it (product rounded, then the sum).  All fast sines
    // of the iteration are evaluated first, in ONE basic block together with the Box-Muller above, so that the
    // independent polynomial chains interleave (DFMA latency is 8 cycles); a particle long lost from the bucket
    // (|y| >= 2^16, or not finite) is then patched with the library sine in a single cold branch.
    if (NCAV > 0) {
      constexpr int NS = (NCAV > 0 ? NCAV : 1) * NP;
      constexpr int NB = RAD ? NPAIR : 0;
      SinState ss[NS];
      constexpr int NB1 = NB > 0 ? NB : 1;
      double zz[NS], pp[NS], f2[NB1], ps[NB1], pc[NB1];
      uint32_t worst = 0u;
#pragma unroll
      for (int c = 0; c < NCAV; ++c)
#pragma unroll
        for (int i = 0; i < NP; ++i) {
          const double y = __dadd_rn(__dmul_rn(A.cav_w[c], tau[i]), A.cav_ph[c]);
          ss[c * NP + i] = sin_rf_head(A.mt, y);
          zz[c * NP + i] = ss[c * NP + i].z;
          worst = max(worst, (uint32_t)__double2hiint(y) & 0x7FFFFFFFu);
        }
#pragma unroll
      for (int q = 0; q < NB; ++q) f2[q] = bm[q].f2;
      horner7_lockstep<NS, NB>(A.mt, zz, pp, f2, ps, pc);
      double sn[NCAV > 0 ? NCAV : 1][NP];
#pragma unroll
      for (int c = 0; c < NCAV; ++c)
#pragma unroll
        for (int i = 0; i < NP; ++i) sn[c][i] = sin_rf_tail(ss[c * NP + i], pp[c * NP + i]);
      if (RAD) {
#pragma unroll
        for (int q = 0; q < NB; ++q) box_muller_tail(A.mt, bm[q], ps[q], pc[q], z[2 * q], z[2 * q + 1]);
      }
      if (__builtin_expect(worst >= 0x40F00000u, 0)) {  // some |y| >= 65536, inf or NaN
#pragma unroll
        for (int c = 0; c < NCAV; ++c)
#pragma unroll
          for (int i = 0; i < NP; ++i) {
            const double y = __dadd_rn(__dmul_rn(A.cav_w[c], tau[i]), A.cav_ph[c]);
            if (!(fabs(y) < 65536.0)) sn[c][i] = sin_rf_slow(y);
          }
      }
#pragma unroll
      for (int c = 0; c < NCAV; ++c)
#pragma unroll
        for (int i = 0; i < NP; ++i) del[i] = fma(A.cav_amp[c], sn[c][i], del[i]);
    } else {
#pragma unroll 1
      for (int c = 0; c < A.n_cav; ++c) {
        const double cw = A.cav_w[c], cp = A.cav_ph[c], ca = A.cav_amp[c];
#pragma unroll
        for (int i = 0; i < NP; ++i) {
          const double y = __dadd_rn(__dmul_rn(cw, tau[i]), cp);
          double sv = sin_rf_fast(A.mt, y);
          if (__builtin_expect(!(fabs(y) < 65536.0), 0)) sv = sin_rf_slow(y);
          del[i] = fma(ca, sv, del[i]);
        }
      }
    }
#pragma unroll
    for (int i = 0; i < NP; ++i) {
      del[i] -= A.loss;
      if (RAD) del[i] = fma(del[i], A.one_minus_DE, z[i]);  // S2 (z already scaled by sigma_delta sqrt(2 D_E))
      tau[i] = fma(A.drift, del[i], tau[i]);                // S3
      t[i] = __dmul_rn(__dsub_rn(tau[i], lo_new), A.invDelta);  // S4
      in[i] = live[i] && in_window(t[i], hi_nb);
    }
  }
  // S4: deposit.  Branch-free: a particle outside the window (or a padding slot) counts into the spare bin nb.
#pragma unroll
  for (int i = 0; i < NP; ++i) atomicAdd(&sH[in[i] ? __double2int_rd(t[i]) : nb], 1u);
}

// ------------------------------------------------------------------ fused particle pass
// MAP = true : S0 S7 | S1 S2 S3 | S4      (a tracked turn)
// MAP = false: S0 S7 |          | S4      (flush of the pending kick before the state is observed)
// RAD: radiation on; GATHER: 1 linear, 0 nearest grid point; NCAV: 1 or 2 cavities unrolled, 0 = loop over n_cav.
// NPAIR pairs (2 NPAIR particles) are advanced together per thread and iteration, in lock step and without
// branches, so that every coefficient load serves all of them and their dependency chains interleave.
//
// Wake gather (S0, D12): with kk = rint(t) the particle sits between the centres of bins kk-1 and kk, at
// f = t - kk in [-1/2, 1/2] from their midpoint: v = mid[kk] + f dif[kk], mid = (V[kk-1]+V[kk])/2,
// dif = V[kk]-V[kk-1], with V[-1] := V[0] and V[nb] := V[nb-1] (constant outer half bins).  Cell nb+1 is zero and
// serves every particle outside the window (no kick, D11), which keeps the step branch-free.
template <bool MAP, bool RAD, int GATHER, int NCAV, int NPAIR>
__global__ void __launch_bounds__(kPassThreads, NPAIR == 1 ? 3 : 2) k_pass(const __grid_constant__ Args A,
                                                                             const __grid_constant__ WakeArgs Wk) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int NP = 2 * NPAIR;                       // particles per thread and iteration
  constexpr uint32_t STRIDE = kPassThreads * NPAIR;   // pairs per CTA and iteration (one stage)
  constexpr uint32_t STAGE_BYTES = 2 * STRIDE * 16;   // tau block + delta block
  constexpr int NWARP = kPassThreads / 32;
  unsigned char *sStage = smem_raw;                   // [stage]{double2 tau[STRIDE]; double2 delta[STRIDE]}
  WakeCell *sW = reinterpret_cast<WakeCell *>(smem_raw + kStages * STAGE_BYTES);  // [nb+2]
  LogTabEntry *sL = reinterpret_cast<LogTabEntry *>(sW + (A.nb + 2));          // [128]
  uint32_t *sH = reinterpret_cast<uint32_t *>(sL + 128);                        // [nb + 1], bin nb is a sink
  __shared__ double s_red[NWARP][4];
  __shared__ uint32_t s_nout[NWARP];
  __shared__ __align__(8) uint64_t s_bar[2 * kStages];  // full[kStages], then empty[kStages]

  const int tid = threadIdx.x;
  const int lane = tid & 31;
  const int nb = A.nb;
  const uint32_t hi_nb = (uint32_t)__double2hiint(A.nb_d);
  if (tid < kStages) {
    mbar_init(smem_u32(&s_bar[tid]), 1u);
    mbar_init(smem_u32(&s_bar[kStages + tid]), (uint32_t)NWARP);
  }
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  if (MAP && RAD)
    for (int i = tid; i < 128; i += kPassThreads) sL[i] = A.logtab[i];
  __syncthreads();
  const uint32_t stage0 = smem_u32(sStage), full0 = smem_u32(&s_bar[0]), empty0 = full0 + kStages * 8u;

  // one CTA = one tile of one bunch: pairs [p0, p1) of bunch b (grid = tiles per bunch x bunches).  Many small
  // CTAs in address order, placed by the hardware scheduler, stream HBM measurably faster than one resident wave of
  // persistent CTAs with a fixed range each (6.7 vs 5.5 TB/s for a bare read-modify-write of this store).
  {
    const int b = (int)blockIdx.y;
    const uint32_t p0 = blockIdx.x * A.tile_pairs;
    const uint32_t p1 = (A.ppb - p0 < A.tile_pairs) ? A.ppb : p0 + A.tile_pairs;

    // chunk k of the tile = pairs [p0 + k STRIDE, + STRIDE) clipped to p1; it lives in stage k % kStages
    const uint32_t n_it = (p1 - p0 + STRIDE - 1u) / STRIDE;
    const double2 *gT = reinterpret_cast<const double2 *>(A.tau + (size_t)b * A.ld);
    const double2 *gD = reinterpret_cast<const double2 *>(A.delta + (size_t)b * A.ld);
    auto issue = [&](uint32_t k) {  // producer thread: fill the stage of chunk k once every warp has released it
      const uint32_t c = k, stage = c % kStages;
      if (c >= (uint32_t)kStages) mbar_wait(empty0 + stage * 8u, ((c / kStages) + 1u) & 1u);
      const uint32_t pc = p0 + k * STRIDE;
      const uint32_t bytes = ((p1 - pc < STRIDE) ? p1 - pc : STRIDE) * 16u;
      const uint32_t bar = full0 + stage * 8u, dst = stage0 + stage * STAGE_BYTES;
      mbar_expect_tx(bar, 2u * bytes);
      bulk_g2s(dst, gT + pc, bytes, bar);
      bulk_g2s(dst + STRIDE * 16u, gD + pc, bytes, bar);
    };
    const bool fused = MAP && A.fused != 0;
    if (tid == 0 && !fused)
      for (uint32_t k = 0; k + 1u < (uint32_t)kStages && k < n_it; ++k) issue(k);

    // Everything above is independent of the wake kernel before this pass (barriers, log table, the first particle
    // stages: the particles were last written by the pass before it, which that wake kernel waited for); its output --
    // the control words, the gather cells, the phasors, the windows -- is read from here on.  In the one-launch turn the
    // predecessor is the pass before, which wrote the particles: the first stages are issued after the wait.
    griddep_launch_dependents();  // the kernel after this pass may become resident; it waits for this grid itself
    // What this CTA needs of the wake kernel before it is the wake of ITS bunch: with one k_wake CTA per bunch
    // (flag_wait) it waits for bunch_ready[b] instead of the whole grid -- the CTAs of the first bunches stream while the
    // wakes of the last ones, and the closing of the turn, are still under way.  The turn number cannot then come from
    // the control word (the closing CTA may not have bumped it yet): the tile's own CTA of the pass before left it in
    // tile_turn (that pass is complete: the wake kernel in between waited for it).  A wait that reads a stale flag just
    // keeps waiting; everything the wake kernel wrote is read through L2 below (__ldcg), never through an L1 line.
    __shared__ uint32_t s_turn;
    const bool by_flag = MAP && A.flag_wait != 0;
    if (by_flag) {
      if (tid == 0) {
        const uint32_t done = __ldcg(&A.tile_turn[(size_t)b * gridDim.x + blockIdx.x]);
        wait_turn(&A.bunch_ready[b], done);
        s_turn = done;
      }
      __syncthreads();
    } else {
      griddep_wait();
    }
    if (tid == 0 && fused)
      for (uint32_t k = 0; k + 1u < (uint32_t)kStages && k < n_it; ++k) issue(k);
    const uint32_t n_done = by_flag ? s_turn : A.ctrl->turn;
    const uint32_t n = n_done + 1u;  // the turn this pass tracks (Philox counter word, D24)
    const bool have_kick = by_flag ? (n_done != A.ctrl->kick_base) : (A.ctrl->kick_pending != 0u);
    // window of the wake being applied (S0) and window this pass bins with (S4); the flush pass re-bins on the former
    const double lo_old = __ldcg(&A.lo_hist[b]);
    const double lo_new = MAP ? __ldcg(&A.lo_next[b]) : lo_old;

    // stage the gather cells of bunch b's wake: cellSR + sum_r Re[cellF_r P[b][r]] (S6 expansion); clear the counts.
    // All loads of a cell -- its short-range part and, for up to four resonators, the table cell and the phasor -- are
    // issued before the first of them is used: one trip to L2 per cell, where a loop over the resonators made 1 + R_lr
    // dependent ones (c4: 3 per CTA prologue, 4.9 waves of CTAs per pass).
    for (int k = tid; k < nb + 2; k += kPassThreads) {
      WakeCell c{0.0, 0.0};
      if (have_kick) {
        constexpr int RU = 4;
        CellF f[RU];
        cplx pb[RU];
        {
          const double2 v = __ldcg(reinterpret_cast<const double2 *>(&A.cellSR[(size_t)b * (nb + 2) + k]));
          c.mid = v.x; c.dif = v.y;
        }
#pragma unroll
        for (int r = 0; r < RU; ++r)
          if (r < A.R) {
            f[r] = A.cellF[(size_t)r * (nb + 2) + k];
            pb[r] = __ldcg_cplx(&A.P[(size_t)b * A.R + r]);
          }
#pragma unroll
        for (int r = 0; r < RU; ++r)
          if (r < A.R) {
            c.mid += fma(f[r].mid.re, pb[r].re, -(f[r].mid.im * pb[r].im));
            c.dif += fma(f[r].dif.re, pb[r].re, -(f[r].dif.im * pb[r].im));
          }
#pragma unroll 1
        for (int r = RU; r < A.R; ++r) {
          const CellF fr = A.cellF[(size_t)r * (nb + 2) + k];
          const cplx pr = __ldcg_cplx(&A.P[(size_t)b * A.R + r]);
          c.mid += fma(fr.mid.re, pr.re, -(fr.mid.im * pr.im));
          c.dif += fma(fr.dif.re, pr.re, -(fr.dif.im * pr.im));
        }
      }
      sW[k] = c;
      if (k < nb) sH[k] = 0u;
    }
    __syncthreads();

    double st = 0.0, sd = 0.0, stt = 0.0, sdd = 0.0;
    uint32_t nout = 0u;
    // a thread owns NPAIR consecutive pairs (NPAIR = 2: one quad of four particles, 32 bytes per array, one 256-bit
    // store); one running pointer per thread: tau at T[q], delta at the constant byte distance d_off
    uint32_t p = p0 + (uint32_t)tid * NPAIR;
    double2 *T = reinterpret_cast<double2 *>(A.tau + (size_t)b * A.ld) + p;
    const ptrdiff_t d_off = reinterpret_cast<const char *>(A.delta) - reinterpret_cast<const char *>(A.tau);
#define MBT_D(ptr) reinterpret_cast<double2 *>(reinterpret_cast<char *>(ptr) + d_off)
    // chunk this thread will issue next (lane 0 of warp w issues the chunks c = w mod NWARP, c >= kStages - 1:
    // the producer role rotates over the warps, so no warp carries it on its critical path); ~0: none
    uint32_t next_issue = ~0u;
    if (lane == 0) {
      uint32_t c = (uint32_t)(tid >> 5);
      while (c + 1u < (uint32_t)kStages) c += NWARP;
      if (c < n_it) next_issue = c;
    }
    // a full tile has no ragged end and no padding slot: the `live` logic drops out of its loop
    const bool full_tile = (p1 - p0 == n_it * STRIDE) && !(A.Np != 2u * A.ppb && p1 == A.ppb);
    auto run = [&](auto full_tag) {
    constexpr bool FULL = decltype(full_tag)::value;
    // running shared-memory addresses of the stage in use: full barrier (empty barrier kStages * 8 bytes above it)
    // and this thread's slot; they wrap every kStages iterations, where the mbarrier parity flips
    uint32_t bar_a = full0, slot_a = stage0 + (uint32_t)tid * (16u * NPAIR), parity = 0u, until_wrap = kStages;
    for (uint32_t k = 0; k < n_it; ++k) {
      mbar_wait(bar_a, parity);
      double2 t2[NPAIR], d2[NPAIR];
#pragma unroll
      for (int q = 0; q < NPAIR; ++q) {
        t2[q] = lds_double2(slot_a + q * 16u);
        d2[q] = lds_double2(slot_a + (STRIDE + q) * 16u);
      }
      __syncwarp();  // every lane of the warp has read the stage
      if (lane == 0) mbar_arrive(bar_a + kStages * 8u);
      if (k + (uint32_t)kStages - 1u == next_issue) {
        issue(next_issue);
        next_issue = (next_issue + NWARP < n_it) ? next_issue + NWARP : ~0u;
      }
      bar_a += 8u;
      slot_a += STAGE_BYTES;
      if (--until_wrap == 0u) {
        until_wrap = kStages;
        bar_a = full0;
        slot_a -= kStages * STAGE_BYTES;
        parity ^= 1u;
      }

      double tau[NP], del[NP];
      advance_pairs<MAP, RAD, GATHER, NCAV, NPAIR, FULL>(A, t2, d2, tau, del, p, p1, b, n, lo_old, lo_new, hi_nb, nb, sW, sL, sH, st,
                                                        sd, stt, sdd, nout);
      if (FULL || p < p1) {  // p and p1 are even when NPAIR = 2: the thread's pairs are inside the tile together
        if (NPAIR == 2) {
          if (MAP) stg_double4(T, tau[0], tau[1], tau[NP - 2], tau[NP - 1]);
          stg_double4(MBT_D(T), del[0], del[1], del[NP - 2], del[NP - 1]);
        } else {
          if (MAP) T[0] = make_double2(tau[0], tau[1]);
          *MBT_D(T) = make_double2(del[0], del[1]);
        }
      }
      p += STRIDE;
      T += STRIDE;
    }
    };  // run
    if (full_tile) run(std::true_type{}); else run(std::false_type{});
#undef MBT_D

    // S7: warp shuffles, then one atomic per CTA and bunch
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      st += __shfl_down_sync(0xffffffffu, st, o);
      sd += __shfl_down_sync(0xffffffffu, sd, o);
      stt += __shfl_down_sync(0xffffffffu, stt, o);
      sdd += __shfl_down_sync(0xffffffffu, sdd, o);
      nout += __shfl_down_sync(0xffffffffu, nout, o);
    }
    if ((tid & 31) == 0) {
      s_red[tid >> 5][0] = st; s_red[tid >> 5][1] = sd; s_red[tid >> 5][2] = stt; s_red[tid >> 5][3] = sdd;
      s_nout[tid >> 5] = nout;
    }
    __syncthreads();  // also: all shared-memory counts of this segment are in
    if (tid < 4) {
      double s = 0.0;
#pragma unroll
      for (int w = 0; w < kPassThreads / 32; ++w) s += s_red[w][tid];
      atomicAdd(&A.mom_acc[(size_t)b * 4 + tid], s);
    } else if (tid == 4) {
      uint32_t s = 0u;
#pragma unroll
      for (int w = 0; w < kPassThreads / 32; ++w) s += s_nout[w];
      if (s) atomicAdd(&A.nout_acc[b], (unsigned long long)s);
    }
    // S4: flush the CTA's counts into the bunch histogram (integer, order-independent)
    for (int j = tid; j < nb; j += kPassThreads) {
      const uint32_t c = sH[j];
      if (c) atomicAdd(&A.hist[(size_t)b * nb + j], c);
    }
    if (MAP) {
      if (tid == 0 && A.tile_turn) A.tile_turn[(size_t)b * gridDim.x + blockIdx.x] = n;
      if (!fused && !A.count_done) return;
      // One-launch turn: the CTA that completes bunch b (every other CTA of the bunch has flushed its counts and sums:
      // barrier, one thread's fence, then the counter) builds the bunch's wake while other bunches still stream -- S5, the
      // S6 source, the gather cells, the closing of S7, and the phasor P[b] gathered from the sources of the bunches ahead
      // (wake_body<false, true>) -- in the shared memory of the particle stages, which are drained; the CTA that completes
      // the last bunch adds up the turn's aggregate and bumps the turn.  Who may touch what, when: hist[b], mom_acc[b],
      // cellSR[b], Vsr[b], P[b] and the windows of bunch b are written here only after ALL pass CTAs of bunch b are done
      // with them (they read the cells and P[b] in their prologue); ring_A and the control words only after all CTAs of
      // the grid are (the grid-wide ticket in wake_body); the next launch reads all of it after its griddepcontrol.wait,
      // i.e. after this grid has completed.
      __shared__ bool s_mine;
      __syncthreads();
      if (!fused) {  // two-launch turn, wake kernel starting per bunch: release this CTA's counts and sums, count it, done
        if (tid == 0) {
          __threadfence();
          atomicAdd(&A.bunch_done[b], 1u);  // result unused: a reduction, nobody waits for its round trip
        }
        return;
      }
      if (tid == 0) {
        __threadfence();
        s_mine = (atomicAdd(&A.bunch_done[b], 1u) == gridDim.x - 1u);
        if (s_mine) A.bunch_done[b] = 0u;
      }
      __syncthreads();
      if (!s_mine) return;
      __threadfence();
      wake_bunch_fused(Wk, b, reinterpret_cast<double *>(smem_raw));
    }
  }
}

// ------------------------------------------------------------------ small kernels
// wake potential on the bins for mbt_get_wake: total = sr + lr, lr[b][j] = sum_r Re[F_r[j] P[b][r]]
__global__ void k_eval_wake(int M, int nb, int R, const double *Vsr, const cplx *P, const cplx *F, double *total,
                            double *sr, double *lr) {
  const int b = blockIdx.x;
  for (int j = threadIdx.x; j < nb; j += blockDim.x) {
    const double s = Vsr[(size_t)b * nb + j];
    double l = 0.0;
    for (int r = 0; r < R; ++r) {
      const cplx f = F[(size_t)r * nb + j];
      const cplx pb = P[(size_t)b * R + r];
      l += fma(f.re, pb.re, -(f.im * pb.im));
    }
    total[(size_t)b * nb + j] = s + l;
    sr[(size_t)b * nb + j] = s;
    lr[(size_t)b * nb + j] = l;
  }
}

// initial distribution (D20): Philox stream tag 1, counter (i, b, 0, 1); tau = sigma_tau0 z_c, delta = sigma_delta0 z_s
__global__ void k_init(double *tau, double *delta, int64_t ld, uint32_t Np, int M, int b0, PhiloxKeys keys, double s_tau,
                       double s_delta) {
  const int b = blockIdx.y;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < (uint32_t)ld; i += gridDim.x * blockDim.x) {
    double t = 0.0, d = 0.0;
    if (i < Np) {
      uint32_t x0, x1, x2, x3;
      philox4x32_10(i, (uint32_t)(b + b0), 0u, 1u, keys, x0, x1, x2, x3);
      double zc, zs;
      box_muller_accurate(uniform52(x0, x1), uniform52(x2, x3), zc, zs);
      t = s_tau * zc;
      d = s_delta * zs;
    }
    tau[(size_t)b * ld + i] = t;
    delta[(size_t)b * ld + i] = d;
  }
}

// packed [M][Np] <-> strided [M][ld]
__global__ void k_pack(const double *src, int64_t ld, uint32_t Np, double *dst) {
  const int b = blockIdx.y;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < Np; i += gridDim.x * blockDim.x)
    dst[(size_t)b * Np + i] = src[(size_t)b * ld + i];
}
__global__ void k_unpack(const double *src, int64_t ld, uint32_t Np, double *dst) {
  const int b = blockIdx.y;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < (uint32_t)ld; i += gridDim.x * blockDim.x)
    dst[(size_t)b * ld + i] = (i < Np) ? src[(size_t)b * Np + i] : 0.0;
}

// per-turn aggregates A_{n'} = sum_j a[j][n'] g_tail[j] from an uploaded source-phasor history
__global__ void k_aggregate_history(int M, int R, int K, const cplx *ring_a, const cplx *g_tail, cplx *ring_A) {
  const int slot = blockIdx.x;  // 0..K
  const int r = threadIdx.x;
  if (r >= R) return;
  cplx acc{0.0, 0.0};
  for (int j = 0; j < M; ++j) acc = cfma(ring_a[((size_t)slot * M + j) * R + r], g_tail[(size_t)j * R + r], acc);
  ring_A[(size_t)slot * R + r] = acc;
}

// set the turn counter; every flag of the one-launch turn says "complete through `turn`"
__global__ void k_set_ctrl(Ctrl *c, uint32_t turn, uint32_t pending, uint32_t *a_ready, int n_a, uint32_t *bunch_ready, int M,
                           uint32_t *agg_ready, uint32_t *bunch_done, uint32_t *tile_turn, int n_tiles) {
  for (int i = threadIdx.x; i < n_tiles; i += blockDim.x) tile_turn[i] = turn;
  for (int i = threadIdx.x; i < n_a; i += blockDim.x) a_ready[i] = turn;
  for (int i = threadIdx.x; i < M; i += blockDim.x) { bunch_ready[i] = turn; bunch_done[i] = 0u; }
  if (threadIdx.x == 0) {
    *agg_ready = turn;
    c->turn = turn;
    c->ticket[0] = c->ticket[1] = 0u;
    c->kick_pending = pending;
    c->kick_base = turn;
  }
}
__global__ void k_clear_pending(Ctrl *c) {
  c->kick_pending = 0u;
  c->kick_base = c->turn;
}

// Sharded handle, after the all-gather of the exchange buffer: the source phasors of ALL bunches of the turn being closed
// go into the history ring (so that every rank holds the whole history), and their flags are raised, so that the phasor
// gather of the second half of the wake finds them like sources of its own launch.
__global__ void k_shard_scatter(const cplx *xbuf, int n_rows, int R, int Mg, int slots, const Ctrl *ctrl, cplx *ring_a, uint32_t *a_ready) {
  const uint32_t n = ctrl->turn + 1u;
  cplx *dst = ring_a + (size_t)(n % (uint32_t)slots) * Mg * R;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_rows * R; i += gridDim.x * blockDim.x) {
    dst[i] = xbuf[i];
    a_ready[i] = n;
  }
}

__global__ void k_philox_selftest(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, PhiloxKeys keys, uint32_t *out) {
  uint32_t x0, x1, x2, x3;
  philox4x32_10(c0, c1, c2, c3, keys, x0, x1, x2, x3);
  out[0] = x0; out[1] = x1; out[2] = x2; out[3] = x3;
}
__global__ void k_normal_selftest(int64_t n, const uint32_t *ctr, PhiloxKeys keys, const LogTabEntry *logtab, MathTab mt,
                                  double *out) {
  __shared__ LogTabEntry sL[128];
  for (int i = threadIdx.x; i < 128; i += blockDim.x) sL[i] = logtab[i];
  __syncthreads();
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    uint32_t x0, x1, x2, x3;
    philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], keys, x0, x1, x2, x3);
    box_muller_fast(mt, sL, uniform32(mt, x0), uniform32(mt, x1), 1.0, out[4 * i], out[4 * i + 1]);
    box_muller_fast(mt, sL, uniform32(mt, x2), uniform32(mt, x3), 1.0, out[4 * i + 2], out[4 * i + 3]);
  }
}

}  // namespace mbt
