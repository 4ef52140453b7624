// mbt_resident.cuh -- the chip-resident turn loop for workloads whose particle store fits in the shared memory of the chip
// (BASELINE c1, c2, c3: 0.16 / 16 / 4.8 MB against 148 x ~200 KB).
//
// The streaming path (k_pass + k_wake per turn) spends a turn of such a workload on launch and dependency latency: two
// dependent launches, every CTA re-reading its particles, cells and tables from L2.  Here ONE cooperative launch tracks
// all n_turns of an mbt_track call: a CTA loads its slice of one bunch into shared memory once, and per turn
//     stages the bunch's gather cells, advances its particles in place (advance_pairs, the streaming pass's own loop body:
//     the same arithmetic, the same Philox counters -- results are bit-identical to the streaming path), flushes counts
//     and moment sums;  GRID BARRIER;  the first S CTAs of a bunch run wake_body (the wake kernel's own code: S5, S6, S7,
//     the closing of the turn);  GRID BARRIER.
// HBM and L2 are touched by the particles only at entry and exit.  The grid barrier is a monotonic arrival counter and a
// generation word in global memory (release / acquire); the launch is cooperative, so all CTAs are resident and a
// waiting CTA cannot starve the ones it waits for.
#pragma once
#include "mbt_kernels.cuh"

namespace mbt {

struct ResArgs {
  int32_t n_turns;
  int32_t ctas_per_bunch;  // grid = M * ctas_per_bunch CTAs
  uint32_t tile_pairs;     // pairs per CTA (even)
  uint32_t wake_off;       // byte offset of wake_body's shared memory within the dynamic shared memory
  uint32_t wake_bytes;     // ... and its size
  uint32_t *bar;           // [2] arrival count, generation (zero at launch)
};

__host__ __device__ inline size_t resident_smem_bytes(uint32_t tile_pairs, int nb, size_t wake_bytes) {
  size_t n = (size_t)tile_pairs * 32;                                   // tau block, delta block
  n += (size_t)(nb + 2) * sizeof(WakeCell) + 128 * sizeof(LogTabEntry); // cells, log table
  n += ((size_t)(nb + 1) * sizeof(uint32_t) + 15) & ~(size_t)15;        // counts
  return n + wake_bytes + 16;
}

// all CTAs of the (cooperative) grid; `gen` counts the barriers this CTA has passed
__device__ __forceinline__ void grid_barrier(uint32_t *bar, uint32_t &gen, const uint32_t n_ctas) {
  __syncthreads();
  if (threadIdx.x == 0) {
    gen += 1u;
    __threadfence();
    if (atomicAdd(&bar[0], 1u) + 1u == n_ctas * gen) st_release_u32(&bar[1], gen);  // the last arrival opens the barrier
    while ((int32_t)(ld_acquire_u32(&bar[1]) - gen) < 0) {
    }
    __threadfence();
  }
  __syncthreads();
}

template <bool RAD, int GATHER, int NCAV>
__global__ void __launch_bounds__(kPassThreads, 2) k_resident(const __grid_constant__ Args A, const __grid_constant__ WakeArgs Wk,
                                                             const __grid_constant__ ResArgs Rs) {
  constexpr int NPAIR = 2;
  constexpr int NP = 2 * NPAIR;
  constexpr uint32_t STRIDE = kPassThreads * NPAIR;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int tid = threadIdx.x, nb = A.nb;
  const int b = (int)(blockIdx.x / (uint32_t)Rs.ctas_per_bunch), x = (int)(blockIdx.x % (uint32_t)Rs.ctas_per_bunch);
  const uint32_t tile = Rs.tile_pairs;
  double2 *sT = reinterpret_cast<double2 *>(smem_raw);  // [tile] tau pairs
  double2 *sD = sT + tile;                              // [tile] delta pairs
  WakeCell *sW = reinterpret_cast<WakeCell *>(sD + tile);
  LogTabEntry *sL = reinterpret_cast<LogTabEntry *>(sW + (nb + 2));
  uint32_t *sH = reinterpret_cast<uint32_t *>(sL + 128);
  double *sWake = reinterpret_cast<double *>(smem_raw + Rs.wake_off);
  __shared__ double s_red[kPassThreads / 32][4];
  __shared__ uint32_t s_nout[kPassThreads / 32];

  const uint32_t hi_nb = (uint32_t)__double2hiint(A.nb_d);
  const uint32_t p0 = min((uint32_t)x * tile, A.ppb);
  const uint32_t p1 = min(p0 + tile, A.ppb);
  const uint32_t n_it = (p1 - p0 + STRIDE - 1u) / STRIDE;
  double2 *gT = reinterpret_cast<double2 *>(A.tau + (size_t)b * A.ld);
  double2 *gD = reinterpret_cast<double2 *>(A.delta + (size_t)b * A.ld);

  // entry: this CTA's slice of the bunch into shared memory; the log table
  for (uint32_t i = tid; i < tile; i += kPassThreads) {
    const bool ok = p0 + i < p1;
    sT[i] = ok ? gT[p0 + i] : make_double2(0.0, 0.0);
    sD[i] = ok ? gD[p0 + i] : make_double2(0.0, 0.0);
  }
  if (RAD)
    for (int i = tid; i < 128; i += kPassThreads) sL[i] = A.logtab[i];
  uint32_t gen = 0u;
  const uint32_t n_ctas = gridDim.x;

  for (int turn = 0; turn < Rs.n_turns; ++turn) {
    // what the wake of the turn before left (after the barrier that closed it): turn number, kick, windows, cells, phasors
    const uint32_t n = __ldcg(&A.ctrl->turn) + 1u;
    const bool have_kick = __ldcg(&A.ctrl->kick_pending) != 0u;
    const double lo_old = __ldcg(&A.lo_hist[b]);
    const double lo_new = __ldcg(&A.lo_next[b]);
    for (int k = tid; k < nb + 2; k += kPassThreads) {
      WakeCell c{0.0, 0.0};
      if (have_kick) {
        const double2 v = __ldcg(reinterpret_cast<const double2 *>(&A.cellSR[(size_t)b * (nb + 2) + k]));
        c.mid = v.x; c.dif = v.y;
#pragma unroll 1
        for (int r = 0; r < A.R; ++r) {
          const CellF f = A.cellF[(size_t)r * (nb + 2) + k];
          const cplx pb = __ldcg_cplx(&A.P[(size_t)b * A.R + r]);
          c.mid += fma(f.mid.re, pb.re, -(f.mid.im * pb.im));
          c.dif += fma(f.dif.re, pb.re, -(f.dif.im * pb.im));
        }
      }
      sW[k] = c;
    }
    for (int k = tid; k < nb + 1; k += kPassThreads) sH[k] = 0u;
    __syncthreads();

    // the pass over the resident slice, in place
    double st = 0.0, sd = 0.0, stt = 0.0, sdd = 0.0;
    uint32_t nout = 0u;
    uint32_t p = p0 + (uint32_t)tid * NPAIR;
    for (uint32_t k = 0; k < n_it; ++k, p += STRIDE) {
      const uint32_t i = (uint32_t)tid * NPAIR + k * STRIDE;  // slot in the slice
      double2 t2[NPAIR], d2[NPAIR];
#pragma unroll
      for (int q = 0; q < NPAIR; ++q) {
        t2[q] = (i + q < tile) ? sT[i + q] : make_double2(0.0, 0.0);
        d2[q] = (i + q < tile) ? sD[i + q] : make_double2(0.0, 0.0);
      }
      double tau[NP], del[NP];
      advance_pairs<true, RAD, GATHER, NCAV, NPAIR, false>(A, t2, d2, tau, del, p, p1, b, n, lo_old, lo_new, hi_nb, nb, sW, sL, sH,
                                                         st, sd, stt, sdd, nout);
      if (p < p1) {
#pragma unroll
        for (int q = 0; q < NPAIR; ++q)
          if (i + q < tile) {
            sT[i + q] = make_double2(tau[2 * q], tau[2 * q + 1]);
            sD[i + q] = make_double2(del[2 * q], del[2 * q + 1]);
          }
      }
    }
    // S7 sums and S4 counts of this CTA into the bunch's accumulators (as the streaming pass does)
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
    __syncthreads();
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
    for (int j = tid; j < nb; j += kPassThreads) {
      const uint32_t c = sH[j];
      if (c) atomicAdd(&A.hist[(size_t)b * nb + j], c);
    }
    grid_barrier(Rs.bar, gen, n_ctas);  // every bunch's counts and sums are complete

    // the wake of the turn: the wake kernel's own code, by the first S CTAs of every bunch
    if (x < Wk.S) {
      if (Wk.S > 1) wake_body<true, false>(Wk, b, x, sWake, Rs.wake_bytes);
      else if (Wk.gather_P) wake_body<false, true>(Wk, b, 0, sWake, Rs.wake_bytes);
      else wake_body<false, false>(Wk, b, 0, sWake, Rs.wake_bytes);
    }
    grid_barrier(Rs.bar, gen, n_ctas);  // cells, phasors, windows, the turn counter: ready for the next turn
  }

  // exit: the slice back to the store
  for (uint32_t i = tid; i < tile; i += kPassThreads)
    if (p0 + i < p1) {
      gT[p0 + i] = sT[i];
      gD[p0 + i] = sD[i];
    }
}

// after a resident run: the flags of the streaming path say "complete through `turn`" (the kick state is the control word's)
__global__ void k_sync_flags(const Ctrl *c, uint32_t *a_ready, int n_a, uint32_t *bunch_ready, int M, uint32_t *agg_ready,
                             uint32_t *tile_turn, int n_tiles) {
  const uint32_t turn = c->turn;
  for (int i = threadIdx.x; i < n_tiles; i += blockDim.x) tile_turn[i] = turn;
  for (int i = threadIdx.x; i < n_a; i += blockDim.x) a_ready[i] = turn;
  for (int i = threadIdx.x; i < M; i += blockDim.x) bunch_ready[i] = turn;
  if (threadIdx.x == 0) *agg_ready = turn;
}

}  // namespace mbt
