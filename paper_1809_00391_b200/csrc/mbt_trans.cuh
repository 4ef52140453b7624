// mbt_trans.cuh -- transverse planes (P:l.73-92 Eqs.(3)-(5), l.100-111 Eq.(6b); DESIGN.md
// readings T1..T8), fused with the longitudinal path: a handle with the planes enabled runs, per turn,
//
//   k_pass6    one pass over the 6-D SoA store (96 B per particle-turn): both kicks of turn n-1, the longitudinal
//              map and the betatron map / excitation of turn n, counts and dipole sums of turn n
//   k_wake     longitudinal wake of turn n                                        (mbt_kernels.cuh, unchanged)
//   k_wake_tr  per bunch: K[j] = sum_{k<j} (Q_b/N_p) S[k] W_perp((j-k) Delta) for both planes, gather cells, bunch
//              centroids (per-turn log; source ring of the resistive wall), scale of the next turn's dipole sums
//   k_rw       long-range resistive-wall kick per bunch (readings W1..W5), if enabled
//
// k_wake_tr and k_rw run on a side stream beside k_wake (they read only what the pass wrote; the next pass joins both),
// and, like the longitudinal kick, the transverse kick of the last tracked turn stays pending until the next pass or
// a getter's flush pass (k_pass6<false>) applies it.
#pragma once
#include "mbt_kernels.cuh"

namespace mbt {

struct Plane {
  double t_frac;  // nu - floor(nu): the betatron phase in turns, Psi / (2 pi) = nu (1 + xi delta), is used mod 1
  double t_xi;    // nu xi
  double alpha, beta, gamma, eta, etap;
  double exc_u, exc_up;  // sigma_u sqrt(D_exc), sigma_up sqrt(D_exc)
};

// Dipole sums in fixed point.  Shared memory has no native fp64 (nor 64-bit integer) atomic add -- both compile to a
// compare-and-swap loop, measured at 6 ps per particle for two sums against 0.5 ps for the integer histogram -- so a
// particle's offset is deposited as a 64-bit integer v = rint(u 2^kFixBits / X_max) split over two native 32-bit
// atomics: the low word's returned old value tells the one thread whose addition wraps it, and that thread adds the
// carry to the high word (1.7 ps per particle for both planes, measured).  X_max = 2^E >= 64 rms(u) comes from the
// bunch's <u^2> of the turn before; a particle with |u| >= X_max (none in a Gaussian bunch) adds its offset in fp64
// to a global table instead, so the sum is right for any input.  Integer sums do not depend on the order of
// addition: S is reproducible bit for bit from run to run.  Rounding: 2^-kFixBits X_max per particle.
constexpr int kFixBitsMax = 44;
#ifndef MBT_LOCK6
#define MBT_LOCK6 2  // particles whose angle polynomials run in lock step in k_pass6 (1 or 2; 2 measured 2 % faster at c4)
#endif
struct FixScale {
  double inv_lsb;    // 2^fix_bits / X_max (a power of two: the scaling is exact)
  double lsb;        // X_max / 2^fix_bits
  uint32_t xmax_hi;  // high word of X_max; |u| < X_max  <=>  (hi(u) & 0x7fffffff) < xmax_hi
  uint32_t pad;
};

struct Args6 {
  Args L;                      // the longitudinal pass's arguments (mbt_kernels.cuh), same meaning
  double *x, *xp, *y, *yp;     // [M][ld]
  Plane px, py;
  const WakeCell *cellX, *cellY;  // [M][nb+2] gather cells of the kick tables K_x, K_y of the last turn (k_wake_tr)
  unsigned long long *Sfix;    // [M][2][nb+1] dipole sums of the turn in flight, fixed point (two's complement);
                               //              entry nb: the particles outside the window (for the bunch centroid)
  double *Sov;                 // [M][2][nb+1] ... of the particles beyond X_max
  const double *rw;            // [M][2] long-range resistive-wall kick of the last turn [V] (zeros without it)
  const FixScale *fix;         // [M][2]
  double *acc2;                // [M][2] sum u^2 of the mapped state (the next turn's scale)
  uint32_t *turn_tr;           // the turn this pass tracks, for k_wake_tr / k_rw: they run beside k_wake, which bumps
                               // ctrl->turn, so they must not read that word
  uint32_t *bunch_done_tr;     // [M] second completion count (the transverse side of k_wake6 resets it), or nullptr
  const uint32_t *tr_ready;    // [M] turn whose transverse kick tables of bunch b are complete (k_wake_tr), or nullptr
  const uint32_t *rw_ready;    // [M] ... whose resistive-wall kick is (k_rw), or nullptr (no resistive wall / grid-wide waits)
  uint32_t tile_pairs;         // pairs per CTA
  int32_t stages;              // shared-memory stages of the particle stream (2..kMaxStages6)
};

// Particle staging as in k_pass: `stages` shared-memory stages of kPassThreads pairs x six arrays (24 KB each), filled
// by cp.async.bulk stages-1 iterations ahead; full[stage] completes on the bytes, empty[stage] on one arrival per warp.
constexpr int kMaxStages6 = 4;
constexpr uint32_t kBlock6 = kPassThreads * 16u;   // bytes of one array's block in a stage
constexpr uint32_t kStage6 = 6u * kBlock6;
__host__ __device__ inline size_t pass6_smem_bytes(int nb, int stages) {
  return (size_t)stages * kStage6 + (size_t)(nb + 2) * 3 * sizeof(WakeCell) + 128 * sizeof(LogTabEntry) +
         (size_t)(nb + 1) * 5 * sizeof(uint32_t) + 16;
}

// sin, cos of 2 pi t: q = rint(2 t), f = t - q/2 in [-1/4, 1/4] (exact), polynomials of mbt_math.cuh, sign (-1)^q
__device__ __forceinline__ void sincos_turns(const MathTab &C, double t, double &sn, double &cs) {
  const double qm = fma(t, 2.0, MBT_MAGIC);
  const int q = __double2loint(qm);
  const double f = fma(qm - MBT_MAGIC, -0.5, t), f2 = f * f;
  const double ps = MBT_POLY7(C.sinf, MBT_SINF_I4, MBT_SINF_I5, f2), pc = MBT_POLY7(C.cosf, MBT_COSF_I4, MBT_COSF_I5, f2);
  sn = flip_sign_if_odd(f * fma(f2, ps, C.two_pi), q);
  cs = flip_sign_if_odd(fma(f2, pc, 1.0), q);
}

// Eqs. (3), (4) for one plane (readings T2, T3).  The oracle rounds Psi = 2 pi nu (1 + xi delta) at |Psi| ~ 100 rad
// (2e-14 rad); here the phase is reduced exactly in turns first, so the two differ by that rounding (<< 1e-12).
__device__ __forceinline__ void betatron_map(const MathTab &C, const Plane &p, double &u, double &up, double d) {
  double sn, cs;
  sincos_turns(C, fma(p.t_xi, d, p.t_frac), sn, cs);
  const double ub = fma(-p.eta, d, u), upb = fma(-p.etap, d, up);
  const double un = fma(fma(p.alpha, sn, cs), ub, (p.beta * sn) * upb);
  const double upn = fma(fma(-p.alpha, sn, cs), upb, -((p.gamma * sn) * ub));
  u = fma(p.eta, d, un);
  up = fma(p.etap, d, upn);
}

// the same in two halves around the polynomial evaluation, so that the caller can run the chains of several angles in
// lock step (horner7_lockstep): head = phase reduction, tail = sin / cos and the matrix of Eq. (4)
struct AngState {
  double f, f2;
  int q;
};
__device__ __forceinline__ AngState turns_head(double t) {
  const double qm = fma(t, 2.0, MBT_MAGIC);
  AngState S;
  S.q = __double2loint(qm);
  S.f = fma(qm - MBT_MAGIC, -0.5, t);
  S.f2 = S.f * S.f;
  return S;
}
__device__ __forceinline__ void betatron_tail(const MathTab &C, const Plane &p, const AngState &S, double ps, double pc, double &u,
                                              double &up, double d) {
  const double sn = flip_sign_if_odd(S.f * fma(S.f2, ps, C.two_pi), S.q);
  const double cs = flip_sign_if_odd(fma(S.f2, pc, 1.0), S.q);
  const double ub = fma(-p.eta, d, u), upb = fma(-p.etap, d, up);
  const double un = fma(fma(p.alpha, sn, cs), ub, (p.beta * sn) * upb);
  const double upn = fma(fma(-p.alpha, sn, cs), upb, -((p.gamma * sn) * ub));
  u = fma(p.eta, d, un);
  up = fma(p.etap, d, upn);
}

// num / den for den near 1: MUFU.RCP64H seed (2^-22), two Newton steps, one residual correction (<= 1 ulp)
__device__ __forceinline__ double div_near_one(double num, double den) {
  double r = rcp_approx_f64(den);
  r = fma(r, fma(-den, r, 1.0), r);
  r = fma(r, fma(-den, r, 1.0), r);
  const double q = num * r;
  return fma(fma(-den, q, num), r, q);
}

// Fused 6-D pass (readings T1..T8 on top of the longitudinal S0..S7):
//   head : kicks of turn n-1 -- longitudinal (S0) and transverse (Eq. 6b), gathered at the same bin position; S7
//   MAP  : S1 S2 S3 of turn n, Eqs. (3), (4) with the turn's delta, Eq. (5) lines 2-3, then S4: counts and dipole sums
// One pair of particles per thread and iteration, 96 bytes per particle-turn.  MAP = false is the flush pass.
template <bool MAP, bool RAD, int GATHER, int NCAV>
__global__ void __launch_bounds__(kPassThreads, 2) k_pass6(const __grid_constant__ Args6 A6) {
  const Args &A = A6.L;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int nb = A.nb;
  const uint32_t nst = (uint32_t)A6.stages;
  WakeCell *sW = reinterpret_cast<WakeCell *>(smem_raw + (size_t)nst * kStage6);  // [nb+2] longitudinal
  WakeCell *sX = sW + (nb + 2), *sY = sX + (nb + 2);           // [nb+2] each
  LogTabEntry *sL = reinterpret_cast<LogTabEntry *>(sY + (nb + 2));  // [128]
  uint32_t *sH = reinterpret_cast<uint32_t *>(sL + 128);       // [nb+1] counts, bin nb is a sink
  uint32_t *sLo = sH + (nb + 1), *sHi = sLo + 2 * (nb + 1);    // [2][nb+1] each: low / high words of the dipole sums
  __shared__ double s_red[kPassThreads / 32][6];
  __shared__ uint32_t s_nout[kPassThreads / 32];
  __shared__ __align__(8) uint64_t s_bar[2 * kMaxStages6];  // full[], then empty[]
  constexpr uint32_t NWARP = kPassThreads / 32;

  const int tid = threadIdx.x, b = (int)blockIdx.y, lane = tid & 31;
  if (tid < (int)nst) {
    mbar_init(smem_u32(&s_bar[tid]), 1u);
    mbar_init(smem_u32(&s_bar[kMaxStages6 + tid]), NWARP);
  }
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  const uint32_t hi_nb = (uint32_t)__double2hiint(A.nb_d);
  const uint32_t p0 = blockIdx.x * A6.tile_pairs;
  const uint32_t p1 = (A.ppb - p0 < A6.tile_pairs) ? A.ppb : p0 + A6.tile_pairs;
  const size_t base = (size_t)b * A.ld;
  const uint32_t n_it = (p1 - p0 + kPassThreads - 1u) / kPassThreads;
  const uint32_t stage0 = smem_u32(smem_raw), full0 = smem_u32(&s_bar[0]), empty0 = smem_u32(&s_bar[kMaxStages6]);
  const double *gsrc[6] = {A.tau + base, A.delta + base, A6.x + base, A6.xp + base, A6.y + base, A6.yp + base};
  auto issue = [&](uint32_t k) {  // fill the stage of chunk k once every warp has released it
    const uint32_t stage = k % nst;
    if (k >= nst) mbar_wait(empty0 + stage * 8u, ((k / nst) + 1u) & 1u);
    const uint32_t pc = p0 + k * kPassThreads;
    const uint32_t bytes = ((p1 - pc < (uint32_t)kPassThreads) ? p1 - pc : (uint32_t)kPassThreads) * 16u;
    const uint32_t bar = full0 + stage * 8u, dst = stage0 + stage * kStage6;
    mbar_expect_tx(bar, 6u * bytes);
#pragma unroll
    for (int a = 0; a < 6; ++a) bulk_g2s(dst + a * kBlock6, gsrc[a] + 2u * (size_t)pc, bytes, bar);
  };
  __syncthreads();  // barriers initialised
  if (tid == 0)
    for (uint32_t k = 0; k + 1u < nst && k < n_it; ++k) issue(k);
  // Sequencing as in k_pass: with flag_wait the kernels of a 6-D turn are a chain of programmatic
  // dependents on one stream, and this CTA waits for the wakes of ITS bunch -- longitudinal (bunch_ready), transverse
  // (tr_ready) and resistive wall (rw_ready) -- instead of the grids before it; the turn number comes from the tile's own
  // CTA of the pass before.  (The particle stages above were written by that pass, which is complete: the wake kernels
  // between it and this launch let their dependents in only after they had seen their bunch's pass CTAs counted.)
  __shared__ uint32_t s_turn;
  const bool by_flag = MAP && A.flag_wait != 0;
  griddep_launch_dependents();
  if (by_flag) {
    if (tid == 0) {
      const uint32_t done = __ldcg(&A.tile_turn[(size_t)b * gridDim.x + blockIdx.x]);
      wait_turn(&A.bunch_ready[b], done);
      wait_turn(&A6.tr_ready[b], done);
      if (A6.rw_ready) wait_turn(&A6.rw_ready[b], done);
      s_turn = done;
    }
    __syncthreads();
  }
  const uint32_t n_done = by_flag ? s_turn : A.ctrl->turn;
  const uint32_t n = n_done + 1u;
  const bool have_kick = by_flag ? (n_done != A.ctrl->kick_base) : (A.ctrl->kick_pending != 0u);
  if (MAP && tid == 0 && blockIdx.x == 0 && b == 0) *A6.turn_tr = n;
  const double lo_old = __ldcg(&A.lo_hist[b]);
  const double lo_new = MAP ? __ldcg(&A.lo_next[b]) : lo_old;
  FixScale fx, fy;  // (written by k_wake_tr of the turn before: through L2)
  fx.inv_lsb = __ldcg(&A6.fix[2 * b].inv_lsb); fx.lsb = __ldcg(&A6.fix[2 * b].lsb); fx.xmax_hi = __ldcg(&A6.fix[2 * b].xmax_hi); fx.pad = 0u;
  fy.inv_lsb = __ldcg(&A6.fix[2 * b + 1].inv_lsb); fy.lsb = __ldcg(&A6.fix[2 * b + 1].lsb); fy.xmax_hi = __ldcg(&A6.fix[2 * b + 1].xmax_hi); fy.pad = 0u;

  if (MAP && RAD)
    for (int i = tid; i < 128; i += kPassThreads) sL[i] = A.logtab[i];
  for (int k = tid; k < nb + 2; k += kPassThreads) {
    WakeCell c{0.0, 0.0}, cx{0.0, 0.0}, cy{0.0, 0.0};
    if (have_kick) {
      {
        const double2 v = __ldcg(reinterpret_cast<const double2 *>(&A.cellSR[(size_t)b * (nb + 2) + k]));
        c.mid = v.x; c.dif = v.y;
      }
#pragma unroll 1
      for (int r = 0; r < A.R; ++r) {
        const CellF f = A.cellF[(size_t)r * (nb + 2) + k];
        const cplx pb = __ldcg_cplx(&A.P[(size_t)b * A.R + r]);
        c.mid += fma(f.mid.re, pb.re, -(f.mid.im * pb.im));
        c.dif += fma(f.dif.re, pb.re, -(f.dif.im * pb.im));
      }
      {
        const double2 vx = __ldcg(reinterpret_cast<const double2 *>(&A6.cellX[(size_t)b * (nb + 2) + k]));
        const double2 vy = __ldcg(reinterpret_cast<const double2 *>(&A6.cellY[(size_t)b * (nb + 2) + k]));
        cx.mid = vx.x; cx.dif = vx.y; cy.mid = vy.x; cy.dif = vy.y;
      }
      cx.mid += __ldcg(&A6.rw[2 * b]);      // the resistive-wall kick is the same for every particle of the bunch (W4),
      cy.mid += __ldcg(&A6.rw[2 * b + 1]);  // cell nb+1 (outside the window) included
    }
    sW[k] = c; sX[k] = cx; sY[k] = cy;
  }
  for (int k = tid; k < 5 * (nb + 1); k += kPassThreads) sH[k] = 0u;
  __syncthreads();

  double st = 0.0, sd = 0.0, stt = 0.0, sdd = 0.0, sxx = 0.0, syy = 0.0;
  uint32_t nout = 0u;
  // the producer role rotates over the warps: lane 0 of warp w issues the chunks c = w mod NWARP, c >= nst - 1
  uint32_t next_issue = ~0u;
  if (lane == 0) {
    uint32_t c = (uint32_t)(tid >> 5);
    while (c + 1u < nst) c += NWARP;
    if (c < n_it) next_issue = c;
  }
  uint32_t stage = 0u, parity = 0u, p = p0 + (uint32_t)tid;
  for (uint32_t k = 0; k < n_it; ++k, p += kPassThreads) {
    const bool active = p < p1;  // the last chunk of a tile may be ragged
    mbar_wait(full0 + stage * 8u, parity);
    const uint32_t slot = stage0 + stage * kStage6 + (uint32_t)tid * 16u;
    double2 t2 = make_double2(0.0, 0.0), d2 = t2, x2 = t2, xp2 = t2, y2 = t2, yp2 = t2;
    if (active) {
      t2 = lds_double2(slot); d2 = lds_double2(slot + kBlock6); x2 = lds_double2(slot + 2u * kBlock6);
      xp2 = lds_double2(slot + 3u * kBlock6); y2 = lds_double2(slot + 4u * kBlock6); yp2 = lds_double2(slot + 5u * kBlock6);
    }
    __syncwarp();  // every lane of the warp has read the stage
    if (lane == 0) mbar_arrive(empty0 + stage * 8u);
    if (k + nst - 1u == next_issue) {
      issue(next_issue);
      next_issue = (next_issue + NWARP < n_it) ? next_issue + NWARP : ~0u;
    }
    if (++stage == nst) { stage = 0u; parity ^= 1u; }
    if (!active) continue;
    const size_t o = base + 2u * (size_t)p;
    double tau[2] = {t2.x, t2.y}, del[2] = {d2.x, d2.y};
    double x[2] = {x2.x, x2.y}, xp[2] = {xp2.x, xp2.y}, y[2] = {y2.x, y2.y}, yp[2] = {yp2.x, yp2.y};
    const bool live[2] = {2u * p < A.Np, 2u * p + 1u < A.Np};  // the slots from N_p up to ld are padding
    double t[2];
    bool in[2];
    // kicks of the previous turn (S0, Eq. 6b): t as the binning computed it
#pragma unroll
    for (int i = 0; i < 2; ++i) {
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
      const WakeCell c = sW[kk], cx = sX[kk], cy = sY[kk];
      del[i] = fma(-fma(f, c.dif, c.mid), A.invE0, del[i]);
      xp[i] = fma(fma(f, cx.dif, cx.mid), A.invE0, xp[i]);
      yp[i] = fma(fma(f, cy.dif, cy.mid), A.invE0, yp[i]);
      if (!in[i] && live[i]) nout += 1u;
      if (live[i]) {  // S7
        st += tau[i];
        sd += del[i];
        stt = fma(tau[i], tau[i], stt);
        sdd = fma(del[i], del[i], sdd);
      }
    }
    if (MAP) {
      double z[2] = {0.0, 0.0};
      if (RAD) {  // D8: the Philox block of the quad (p >> 1); its half (p & 1) is this pair's Box-Muller pair
        uint32_t w0, w1, w2, w3;
        philox4x32_10(p >> 1, (uint32_t)b, n, 0u, A.keys, w0, w1, w2, w3);
        const bool hi_half = (p & 1u) != 0u;
        box_muller_fast(A.mt, sL, uniform32(A.mt, hi_half ? w2 : w0), uniform32(A.mt, hi_half ? w3 : w1), A.A_q, z[0], z[1]);
      }
      double eps[2];
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        // S1; eps = the particle's RF gain of this turn (the epsilon of Eq. 5, T4)
        eps[i] = 0.0;
        if (NCAV > 0) {
#pragma unroll
          for (int c = 0; c < NCAV; ++c) {
            const double yv = __dadd_rn(__dmul_rn(A.cav_w[c], tau[i]), A.cav_ph[c]);
            double sv = sin_rf_fast(A.mt, yv);
            if (__builtin_expect(!(fabs(yv) < 65536.0), 0)) sv = sin_rf_slow(yv);
            del[i] = fma(A.cav_amp[c], sv, del[i]);
            eps[i] = fma(A.cav_amp[c], sv, eps[i]);
          }
        } else {
#pragma unroll 1
          for (int c = 0; c < A.n_cav; ++c) {
            const double yv = __dadd_rn(__dmul_rn(A.cav_w[c], tau[i]), A.cav_ph[c]);
            double sv = sin_rf_fast(A.mt, yv);
            if (__builtin_expect(!(fabs(yv) < 65536.0), 0)) sv = sin_rf_slow(yv);
            del[i] = fma(A.cav_amp[c], sv, del[i]);
            eps[i] = fma(A.cav_amp[c], sv, eps[i]);
          }
        }
        del[i] -= A.loss;
        if (RAD) del[i] = fma(del[i], A.one_minus_DE, z[i]);  // S2
        tau[i] = fma(A.drift, del[i], tau[i]);                // S3
      }
      // Eqs. (3), (4) with the turn's delta (T1) and Eq. (5) lines 2, 3 (T4, T5: one Philox block per particle, counter
      // (i, b, n, tag 2) -> (r_x, r_x', r_y, r_y')).  The sin / cos polynomials of a particle's four angles (two
      // betatron phases, two Box-Muller angles) are the same two polynomials: evaluated in lock step, LOCK particles
      // at a time, so that 8 LOCK independent DFMA chains are in flight.
      constexpr int LOCK = MBT_LOCK6;
#pragma unroll
      for (int i0 = 0; i0 < 2; i0 += LOCK) {
        constexpr int NA = (RAD ? 4 : 2) * LOCK;
        AngState ang[2 * LOCK];
        BmState bm[2 * LOCK];
        double f2[NA], ps[NA], pc[NA];
        const double dummy[1] = {0.0};
        double dummy_p[1];
#pragma unroll
        for (int l = 0; l < LOCK; ++l) {
          const int i = i0 + l;
          ang[2 * l] = turns_head(fma(A6.px.t_xi, del[i], A6.px.t_frac));
          ang[2 * l + 1] = turns_head(fma(A6.py.t_xi, del[i], A6.py.t_frac));
          f2[2 * l] = ang[2 * l].f2;
          f2[2 * l + 1] = ang[2 * l + 1].f2;
          if (RAD) {
            uint32_t w0, w1, w2, w3;
            philox4x32_10(2u * p + (uint32_t)i, (uint32_t)b, n, 2u, A.keys, w0, w1, w2, w3);
            bm[2 * l] = box_muller_head(A.mt, sL, uniform32(A.mt, w0), uniform32(A.mt, w1), 1.0);
            bm[2 * l + 1] = box_muller_head(A.mt, sL, uniform32(A.mt, w2), uniform32(A.mt, w3), 1.0);
            f2[2 * LOCK + 2 * l] = bm[2 * l].f2;
            f2[2 * LOCK + 2 * l + 1] = bm[2 * l + 1].f2;
          }
        }
        horner7_lockstep<0, NA>(A.mt, dummy, dummy_p, f2, ps, pc);
#pragma unroll
        for (int l = 0; l < LOCK; ++l) {
          const int i = i0 + l;
          betatron_tail(A.mt, A6.px, ang[2 * l], ps[2 * l], pc[2 * l], x[i], xp[i], del[i]);
          betatron_tail(A.mt, A6.py, ang[2 * l + 1], ps[2 * l + 1], pc[2 * l + 1], y[i], yp[i], del[i]);
          if (RAD) {
            double z0, z1, z2, z3;
            box_muller_tail(A.mt, bm[2 * l], ps[2 * LOCK + 2 * l], pc[2 * LOCK + 2 * l], z0, z1);
            box_muller_tail(A.mt, bm[2 * l + 1], ps[2 * LOCK + 2 * l + 1], pc[2 * LOCK + 2 * l + 1], z2, z3);
            const double num = 1.0 + del[i];
            const double adia = div_near_one(num, num + eps[i]);
            x[i] = fma(A6.px.exc_u, z0, x[i]);
            xp[i] = fma(xp[i], adia, A6.px.exc_up * z1);
            y[i] = fma(A6.py.exc_u, z2, y[i]);
            yp[i] = fma(yp[i], adia, A6.py.exc_up * z3);
          }
        }
      }
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        t[i] = __dmul_rn(__dsub_rn(tau[i], lo_new), A.invDelta);  // S4
        in[i] = live[i] && in_window(t[i], hi_nb);
      }
    }
    // S4: counts, and (MAP) the dipole sums of the turn's bins (T6).  Branch-free: everything that is not in the
    // window lands in the sink bin nb.
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const int j = in[i] ? __double2int_rd(t[i]) : nb;
      atomicAdd(&sH[j], 1u);
      if (MAP) {
        if (live[i]) {
          sxx = fma(x[i], x[i], sxx);
          syy = fma(y[i], y[i], syy);
        }
        const bool okx = ((uint32_t)__double2hiint(x[i]) & 0x7FFFFFFFu) < fx.xmax_hi;
        const bool oky = ((uint32_t)__double2hiint(y[i]) & 0x7FFFFFFFu) < fy.xmax_hi;
        const double mx = fma(okx && live[i] ? x[i] : 0.0, fx.inv_lsb, MBT_MAGIC);  // a padding slot deposits zero
        const double my = fma(oky && live[i] ? y[i] : 0.0, fy.inv_lsb, MBT_MAGIC);
        const uint32_t xl = (uint32_t)__double2loint(mx), xh = (uint32_t)(__double2hiint(mx) - 0x43380000);
        const uint32_t yl = (uint32_t)__double2loint(my), yh = (uint32_t)(__double2hiint(my) - 0x43380000);
        const uint32_t ox = atomicAdd(&sLo[j], xl), oy = atomicAdd(&sLo[(nb + 1) + j], yl);
        atomicAdd(&sHi[j], xh + ((ox + xl) < xl ? 1u : 0u));
        atomicAdd(&sHi[(nb + 1) + j], yh + ((oy + yl) < yl ? 1u : 0u));
        if (__builtin_expect(live[i] && !(okx && oky), 0)) {  // beyond X_max: fp64, straight to the global table
          if (!okx) atomicAdd(&A6.Sov[((size_t)b * 2) * (nb + 1) + j], x[i]);
          if (!oky) atomicAdd(&A6.Sov[((size_t)b * 2 + 1) * (nb + 1) + j], y[i]);
        }
      }
    }
    if (MAP) {
      *reinterpret_cast<double2 *>(A.tau + o) = make_double2(tau[0], tau[1]);
      *reinterpret_cast<double2 *>(A6.x + o) = make_double2(x[0], x[1]);
      *reinterpret_cast<double2 *>(A6.y + o) = make_double2(y[0], y[1]);
    }
    *reinterpret_cast<double2 *>(A.delta + o) = make_double2(del[0], del[1]);
    *reinterpret_cast<double2 *>(A6.xp + o) = make_double2(xp[0], xp[1]);
    *reinterpret_cast<double2 *>(A6.yp + o) = make_double2(yp[0], yp[1]);
  }

  // S7 and the scale sums: warp shuffles, then one atomic per CTA and bunch
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    st += __shfl_down_sync(0xffffffffu, st, o);
    sd += __shfl_down_sync(0xffffffffu, sd, o);
    stt += __shfl_down_sync(0xffffffffu, stt, o);
    sdd += __shfl_down_sync(0xffffffffu, sdd, o);
    sxx += __shfl_down_sync(0xffffffffu, sxx, o);
    syy += __shfl_down_sync(0xffffffffu, syy, o);
    nout += __shfl_down_sync(0xffffffffu, nout, o);
  }
  if ((tid & 31) == 0) {
    double *r = s_red[tid >> 5];
    r[0] = st; r[1] = sd; r[2] = stt; r[3] = sdd; r[4] = sxx; r[5] = syy;
    s_nout[tid >> 5] = nout;
  }
  __syncthreads();
  if (tid < 6) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < kPassThreads / 32; ++w) s += s_red[w][tid];
    if (tid < 4) atomicAdd(&A.mom_acc[(size_t)b * 4 + tid], s);
    else if (MAP) atomicAdd(&A6.acc2[(size_t)b * 2 + (tid - 4)], s);
  } else if (tid == 6) {
    uint32_t s = 0u;
#pragma unroll
    for (int w = 0; w < kPassThreads / 32; ++w) s += s_nout[w];
    if (s) atomicAdd(&A.nout_acc[b], (unsigned long long)s);
  }
  for (int j = tid; j < nb + 1; j += kPassThreads) {
    const uint32_t c = sH[j];
    if (c && j < nb) atomicAdd(&A.hist[(size_t)b * nb + j], c);
    if (MAP) {
#pragma unroll
      for (int a = 0; a < 2; ++a) {
        const unsigned long long v = ((unsigned long long)sHi[a * (nb + 1) + j] << 32) | sLo[a * (nb + 1) + j];
        if (v) atomicAdd(&A6.Sfix[((size_t)b * 2 + a) * (nb + 1) + j], v);
      }
    }
  }
  if (MAP) {
    if (tid == 0 && A.tile_turn) A.tile_turn[(size_t)b * gridDim.x + blockIdx.x] = n;
    if (A.count_done) {  // release this CTA's counts and sums and count it: the wake kernels' CTAs of the bunch wait for it
      __syncthreads();
      if (tid == 0) {
        __threadfence();
        atomicAdd(&A.bunch_done[b], 1u);
        if (A6.bunch_done_tr) atomicAdd(&A6.bunch_done_tr[b], 1u);
      }
    }
  }
}

struct TWakeArgs {
  int32_t M, nb, gather, fix_bits;
  uint32_t Np;
  const double *qm;     // [M]
  const double *wt;     // [nb] transverse table wt[k] = sum_r W_perp_r(k Delta), wt[0] = 0
  unsigned long long *Sfix;   // [M][2][nb+1] in: sums of this turn (entry nb: outside the window); out: zero
  double *Sov;                // [M][2][nb+1] likewise
  double *log_tr;             // [log_cap][M][4] mean x, mean y, rms x, rms y per turn, or nullptr
  int64_t log_cap;
  int32_t Krw;                // resistive-wall history depth in turns (0: off)
  double *ring_g;             // [Krw+2][M][2] source strengths Q_b ubar [C m], slot = turn % (Krw+2): k_rw of a turn reads
                              // Krw+1 slots; the spare one is what the next turn writes while trailing bunches still read
  const uint32_t *rw_ready;   // [M] (k_rw's flags) awaited before a ring_g slot is overwritten; used with use_flags only
  const uint32_t *turn_tr;    // the turn being closed (written by the pass; ctrl->turn is k_wake's to bump, beside us)
  FixScale *fix;              // [M][2] in: the scale the sums were deposited with; out: the next turn's
  double *acc2;               // [M][2] in: sum u^2 of this turn's mapped state; out: zero
  double *S_last;             // [M][2][nb] observable copy of the sums [m]
  double *K;                  // [M][2][nb] kick tables [V]
  WakeCell *cellX, *cellY;    // [M][nb+2] their gather cells (as WakeCell of mbt_kernels.cuh)
  uint32_t *tr_ready;         // [M] per-bunch sequencing: turn whose tables of bunch b are complete; the turn
  int32_t use_flags;          //     being closed is then tr_ready[b] + 1 (turn_tr may already belong to the next pass)
  uint32_t *bunch_done_tr;    // [M] pass CTAs of the bunch counted for the transverse side of k_wake6
};

// X_max = 2^E >= 64 sqrt(<u^2>) (E clamped; <u^2> = 0 or not finite: E = 0, every non-zero offset then takes the fp64 path)
__device__ __forceinline__ FixScale make_fix_scale(double mean_sq, int fix_bits) {
  int E = 0;
  if (mean_sq > 0.0 && mean_sq < 1.0e300) {
    int e2;
    frexp(mean_sq, &e2);             // mean_sq = m 2^e2, m in [1/2, 1)  ->  rms < 2^((e2 + 1) / 2)
    E = ((e2 + 1) >> 1) + 6;         // ceil(e2 / 2) + 6
    E = max(-400, min(400, E));
  }
  FixScale f;
  f.inv_lsb = scalbn(1.0, fix_bits - E);
  f.lsb = scalbn(1.0, E - fix_bits);
  f.xmax_hi = (uint32_t)__double2hiint(scalbn(1.0, E));
  f.pad = 0u;
  return f;
}

// k segments per output quad of the Toeplitz sums in k_wake_tr: as many as 256 threads allow, at most 8
__host__ __device__ inline int wake_tr_segments(int nb) {
  const int Q = (nb + 3) / 4;
  const int G = 256 / Q;
  return G < 1 ? 1 : (G > 8 ? 8 : G);
}
__host__ __device__ inline size_t wake_tr_smem_bytes(int nb) {
  return ((size_t)5 * nb + (nb + 8) + (size_t)wake_tr_segments(nb) * 2 * nb) * sizeof(double);
}

// Eq. (6b): strictly causal sum over the earlier bins, both planes; one CTA per bunch.  Also closes the fixed-point
// dipole sums of the turn and chooses the next turn's scale.
// s_w: wake_tr_smem_bytes(nb) of shared memory: [5][nb]: wt, q Sx, q Sy, Kx, Ky; then the padded table [nb+8] and the
// partial sums.  Called by every thread of a 256-thread CTA: by k_wake_tr, or by the y = 1 CTAs of k_wake6.
__device__ __forceinline__ void wake_tr_body(const TWakeArgs &A, const int b, double *s_w) {
  double *swp = s_w + 5 * A.nb;    // swp[3 + l] = wt[l]; zero for the lags -3..0 below and up to 4 beyond the table
  const int tid = threadIdx.x, nb = A.nb;
  double *sw = s_w, *sx = s_w + nb, *sy = s_w + 2 * nb, *kx = s_w + 3 * nb, *ky = s_w + 4 * nb;
  const uint32_t n_turn = A.use_flags ? __ldcg(&A.tr_ready[b]) + 1u : *A.turn_tr;
  const double qm = A.qm[b];
  FixScale fx, fy;  // the scale this turn's sums were deposited with: written by this bunch's CTA of the turn before (L2)
  fx.inv_lsb = __ldcg(&A.fix[2 * b].inv_lsb); fx.lsb = __ldcg(&A.fix[2 * b].lsb); fx.xmax_hi = 0u; fx.pad = 0u;
  fy.inv_lsb = __ldcg(&A.fix[2 * b + 1].inv_lsb); fy.lsb = __ldcg(&A.fix[2 * b + 1].lsb); fy.xmax_hi = 0u; fy.pad = 0u;
  const size_t ox = ((size_t)b * 2) * nb, oy = ox + nb;                  // S_last, K: [M][2][nb]
  const size_t fxo = ((size_t)b * 2) * (nb + 1), fyo = fxo + (nb + 1);   // Sfix, Sov: [M][2][nb+1]
  long long tix = 0, tiy = 0;   // integer totals over the bins and the sink: exact, so the centroid is reproducible
  double tox = 0.0, toy = 0.0;
  for (int j = tid; j < nb + 1; j += 256) {
    const long long ix = (long long)__ldcg(&A.Sfix[fxo + j]), iy = (long long)__ldcg(&A.Sfix[fyo + j]);  // accumulated by atomics: L2
    const double ovx = __ldcg(&A.Sov[fxo + j]), ovy = __ldcg(&A.Sov[fyo + j]);
    A.Sfix[fxo + j] = 0ull; A.Sfix[fyo + j] = 0ull;
    A.Sov[fxo + j] = 0.0; A.Sov[fyo + j] = 0.0;
    tix += ix; tiy += iy; tox += ovx; toy += ovy;
    if (j < nb) {
      const double vx = fma((double)ix, fx.lsb, ovx), vy = fma((double)iy, fy.lsb, ovy);
      A.S_last[ox + j] = vx; A.S_last[oy + j] = vy;
      sx[j] = qm * vx;
      sy[j] = qm * vy;
      sw[j] = A.wt[j];
      swp[3 + j] = j > 0 ? A.wt[j] : 0.0;
    }
  }
  if (tid < 3) swp[tid] = 0.0;
  if (tid < 5) swp[3 + nb + tid] = 0.0;
  // centroid of the bunch (all particles): per-turn log, and W3: source strength Q_b ubar = (Q_b / N_p) sum of offsets
  if (A.Krw > 0 || A.log_tr) {
    __shared__ long long s_ti[8][2];
    __shared__ double s_to[8][2];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      tix += __shfl_down_sync(0xffffffffu, tix, o); tiy += __shfl_down_sync(0xffffffffu, tiy, o);
      tox += __shfl_down_sync(0xffffffffu, tox, o); toy += __shfl_down_sync(0xffffffffu, toy, o);
    }
    if ((tid & 31) == 0) { s_ti[tid >> 5][0] = tix; s_ti[tid >> 5][1] = tiy; s_to[tid >> 5][0] = tox; s_to[tid >> 5][1] = toy; }
    // The slot of turn n last held turn n - Krw - 2, whose last readers are the k_rw CTAs of turn n - 2 (they sum the turns
    // n - 2 - Krw .. n - 2).  With the per-bunch flags nothing else orders a trailing bunch's k_rw CTA against this write
    // (a leading bunch runs ahead by design), so wait for every bunch's rw_ready >= n - 2: two turns of slack, true on
    // arrival in practice, and those CTAs belong to a launch four kernels back (resident or done: no deadlock).
    if (A.use_flags && A.Krw > 0)
      for (int bp = tid; bp < A.M; bp += 256) wait_turn(&A.rw_ready[bp], n_turn - 2u);
    __syncthreads();
    if (tid < 2) {
      long long ti = 0;
      double to = 0.0;
      for (int w = 0; w < 8; ++w) { ti += s_ti[w][tid]; to += s_to[w][tid]; }
      const double total = fma((double)ti, tid == 0 ? fx.lsb : fy.lsb, to);
      const uint32_t n = n_turn;
      if (A.Krw > 0) A.ring_g[((size_t)(n % (uint32_t)(A.Krw + 2)) * A.M + b) * 2 + tid] = qm * total;
      if (A.log_tr && n >= 1u && (int64_t)n <= A.log_cap) {
        const double iN = 1.0 / (double)A.Np, mean = total * iN;
        double *row = A.log_tr + ((size_t)(n - 1u) * A.M + b) * 4;
        row[tid] = mean;
        row[2 + tid] = sqrt(fmax(__ldcg(&A.acc2[2 * b + tid]) * iN - mean * mean, 0.0));  // acc2 is reset further down
      }
    }
  }
  __syncthreads();
  if (tid < 2) {
    A.fix[2 * b + tid] = make_fix_scale(__ldcg(&A.acc2[2 * b + tid]) / (double)A.Np, A.fix_bits);
    A.acc2[2 * b + tid] = 0.0;
  }
  // Toeplitz sums, register-blocked (the plain loop is shared-memory-bandwidth bound: 12 wavefronts per 8 MACs): a
  // thread owns four consecutive outputs j0..j0+3 and a segment of k; per k it loads one new table value into a
  // sliding window w[j0+i-k] and the two sources (a broadcast), 4 wavefronts per 8 MACs.  G segments per output
  // quad, partial sums added in segment order (reproducible).  Against one output per thread, same run, CUDA events,
  // k_wake + k_wake_tr: c3 31.8 -> 29.7 us, c4 55.1 -> 54.1 us, c5 (500 bins) 124 -> 111 us.
  {
    const int Q = (nb + 3) / 4, G = wake_tr_segments(nb), L = (nb + G - 1) / G;
    double *part = s_w + 5 * nb + (nb + 8);  // [G][2][nb]
    for (int item = tid; item < Q * G; item += 256) {  // one pass unless nb > 1024
      const int q = item % Q, g = item / Q;
      const int j0 = 4 * q, k_lo = g * L, k_end = min(min(k_lo + L, nb), j0 + 3);
      double ax[4] = {0.0, 0.0, 0.0, 0.0}, ay[4] = {0.0, 0.0, 0.0, 0.0};
      if (k_lo < k_end) {
        const double *wp = swp + (j0 - k_lo) + 3;  // wp[i] = w[j0 + i - k], zero for lags <= 0
        double w0 = wp[0], w1 = wp[1], w2 = wp[2], w3 = wp[3];
#pragma unroll 4
        for (int k = k_lo; k < k_end; ++k) {
          const double a = sx[k], c = sy[k];
          ax[0] = fma(w0, a, ax[0]); ay[0] = fma(w0, c, ay[0]);
          ax[1] = fma(w1, a, ax[1]); ay[1] = fma(w1, c, ay[1]);
          ax[2] = fma(w2, a, ax[2]); ay[2] = fma(w2, c, ay[2]);
          ax[3] = fma(w3, a, ax[3]); ay[3] = fma(w3, c, ay[3]);
          w3 = w2; w2 = w1; w1 = w0;
          wp -= 1;
          w0 = wp[0];
        }
      }
#pragma unroll
      for (int i = 0; i < 4; ++i)
        if (j0 + i < nb) {
          part[((size_t)g * 2) * nb + j0 + i] = ax[i];
          part[((size_t)g * 2 + 1) * nb + j0 + i] = ay[i];
        }
    }
    __syncthreads();
    for (int j = tid; j < nb; j += 256) {
      double ax = 0.0, ay = 0.0;
      for (int gg = 0; gg < G; ++gg) { ax += part[((size_t)gg * 2) * nb + j]; ay += part[((size_t)gg * 2 + 1) * nb + j]; }
      kx[j] = ax; ky[j] = ay;
      A.K[ox + j] = ax;
      A.K[oy + j] = ay;
    }
  }
  __syncthreads();
  for (int k = tid; k < nb + 2; k += 256) {
    WakeCell cx{0.0, 0.0}, cy{0.0, 0.0};
    if (A.gather == 1) {
      if (k <= nb) {
        const int lo = k > 0 ? k - 1 : 0, hi = k < nb ? k : nb - 1;
        cx.mid = 0.5 * (kx[lo] + kx[hi]); cx.dif = kx[hi] - kx[lo];
        cy.mid = 0.5 * (ky[lo] + ky[hi]); cy.dif = ky[hi] - ky[lo];
      }
    } else if (k < nb) {
      cx.mid = kx[k];
      cy.mid = ky[k];
    }
    A.cellX[(size_t)b * (nb + 2) + k] = cx;
    A.cellY[(size_t)b * (nb + 2) + k] = cy;
  }
  if (A.use_flags) {  // the bunch's tables, scale and source strength are written: publish them
    __syncthreads();
    if (tid == 0) {
      __threadfence();
      st_release_u32(&A.tr_ready[b], n_turn);
    }
  }
}

__global__ void __launch_bounds__(256) k_wake_tr(const __grid_constant__ TWakeArgs A) {
  extern __shared__ double s_wtr[];
  wake_tr_body(A, (int)blockIdx.x, s_wtr);
}

// Per-bunch sequencing of the 6-D turn: ONE wake kernel, grid (M, 2), launched as a programmatic dependent
// of the pass -- CTA (b, 0) builds the longitudinal wake of bunch b (wake_body), CTA (b, 1) its transverse kick tables
// (wake_tr_body) -- each as soon as the pass CTAs of ITS bunch are counted (two counters: each side resets its own).
// CTAs that become resident during the pass's last wave work on bunches that completed long before.
__global__ void __launch_bounds__(256, 3) k_wake6(const __grid_constant__ WakeArgs A, const __grid_constant__ TWakeArgs T) {
  extern __shared__ double smem_w6[];
  const int b = (int)blockIdx.x;
  uint32_t *cnt = blockIdx.y == 0 ? A.bunch_done : T.bunch_done_tr;
  if (threadIdx.x == 0) {
    while (ld_acquire_u32(&cnt[b]) < (uint32_t)A.tiles) {
    }
    cnt[b] = 0u;
  }
  __syncthreads();
  griddep_launch_dependents();  // k_rw or the next pass may come in: their CTAs wait for the flags of their own bunch
  if (blockIdx.y == 0) wake_body<false, true>(A, b, 0, smem_w6, A.smem_wake_bytes);
  else wake_tr_body(T, b, smem_w6);
}

// Long-range resistive-wall kick (readings W1..W5): one CTA per bunch b sums the sources of the last Krw turns (all
// bunches) and of this turn's bunches ahead, weight wrw[d] = (d T_rf)^-1/2 at the bucket distance
// d = (n - n') h + (s_b - s_b'); fixed summation order (reproducible).  Runs after k_wake_tr of the same turn, on the
// library's side stream beside k_wake.
struct RwArgs {
  int32_t M, Krw, h;
  const int32_t *bucket;  // [M]
  const double *ring_g;   // [Krw+2][M][2], slot = turn % (Krw+2)
  const double *wrw;      // [(Krw+1) h] weight at bucket distance d (entry 0 unused)
  double amp[2];
  double *rw;             // [M][2] out [V]
  const uint32_t *turn_tr;
  const uint32_t *tr_ready;  // [M] (k_wake6's transverse side)
  uint32_t *rw_ready;     // [M] per-bunch sequencing: turn whose kick of bunch b is complete (the turn summed is rw_ready[b] + 1)
  int32_t use_flags;
};
__global__ void __launch_bounds__(256) k_rw(const __grid_constant__ RwArgs A) {
  __shared__ double s_red[8][2];
  const int b = blockIdx.x, tid = threadIdx.x;
  griddep_launch_dependents();  // the next pass may come in: its CTAs wait for rw_ready
  // per-bunch sequencing: this turn's sources are those of the bunches AHEAD (W5); each is awaited through its tr_ready
  // flag below (CTAs of k_wake6, all resident or done before this kernel was let in).  The sources of the turns before
  // come from every bunch, also the trailing ones, whose k_wake6 CTA of turn n - 1 no launch boundary orders against
  // this CTA: they are awaited as tr_ready >= n - 1 (true on arrival in practice).
  const uint32_t n = A.use_flags ? __ldcg(&A.rw_ready[b]) + 1u : *A.turn_tr;
  const int sb = A.bucket[b];
  double sx = 0.0, sy = 0.0;
  // a thread keeps its source bunches bp (their bucket distance within a turn in a register) and walks the turns back;
  // the loads of one turn do not depend on the previous one's, so they overlap
  const int kmax = min(A.Krw, (int)min(n - 1u, (uint32_t)A.Krw));  // nothing before turn 1
  for (int bp = tid; bp < A.M; bp += 256) {
    const int ds = sb - A.bucket[bp];
    if (A.use_flags) wait_turn(&A.tr_ready[bp], ds > 0 ? n : n - 1u);
    const double2 *g = reinterpret_cast<const double2 *>(A.ring_g) + bp;
    uint32_t slot = n % (uint32_t)(A.Krw + 2);
#pragma unroll 4
    for (int k = 0; k <= kmax; ++k) {  // source: turn n - k, bunch bp, bucket distance d
      const int d = k * A.h + ds;
      const double w = d > 0 ? A.wrw[d] : 0.0;          // this turn (k = 0): only the bunches ahead
      const double2 gv = __ldcg(&g[(size_t)slot * A.M]);
      sx = fma(gv.x, w, sx);
      sy = fma(gv.y, w, sy);
      slot = slot == 0u ? (uint32_t)A.Krw + 1u : slot - 1u;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    sx += __shfl_down_sync(0xffffffffu, sx, o);
    sy += __shfl_down_sync(0xffffffffu, sy, o);
  }
  if ((tid & 31) == 0) { s_red[tid >> 5][0] = sx; s_red[tid >> 5][1] = sy; }
  __syncthreads();
  if (tid < 2) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += s_red[w][tid];
    A.rw[2 * b + tid] = A.amp[tid] * t;
  }
  if (A.use_flags) {
    __syncthreads();
    if (tid == 0) {
      __threadfence();
      st_release_u32(&A.rw_ready[b], n);
    }
  }
}

// per-bunch sequencing flags of the transverse wake kernels: "complete through `turn`"
__global__ void k_set_flags_tr(uint32_t *tr_ready, uint32_t *rw_ready, uint32_t *bunch_done_tr, int M, uint32_t turn) {
  for (int i = threadIdx.x; i < M; i += blockDim.x) { tr_ready[i] = turn; rw_ready[i] = turn; bunch_done_tr[i] = 0u; }
}

// scale of the fixed-point dipole sums from the state in memory (create, mbt_set_transverse): acc[M][8] of k_moments_tr
__global__ void k_fix_scale(int M, uint32_t Np, int fix_bits, const double *acc, FixScale *fix) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 2 * M) return;
  const int b = i >> 1, a = i & 1;
  fix[i] = make_fix_scale(acc[b * 8 + 4 + 2 * a] / (double)Np, fix_bits);
}

// sums for mbt_moments_transverse: out[M][8] += (sum x, x', y, y', sum x^2, x'^2, y^2, y'^2)
__device__ __forceinline__ double uniform32_plain(uint32_t x) { return ((double)x + 0.5) * 0x1p-32; }

struct TMomArgs {
  const double *x, *xp, *y, *yp;
  int64_t ld;
  uint32_t Np, tile;
};
__global__ void __launch_bounds__(256) k_moments_tr(const TMomArgs A, double *acc) {
  __shared__ double s_red[8][8];
  const int b = blockIdx.y, tid = threadIdx.x;
  const uint32_t i0 = blockIdx.x * A.tile, i1 = min(i0 + A.tile, A.Np);
  const size_t base = (size_t)b * A.ld;
  double s[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (uint32_t i = i0 + tid; i < i1; i += 256) {
    const double v[4] = {A.x[base + i], A.xp[base + i], A.y[base + i], A.yp[base + i]};
#pragma unroll
    for (int a = 0; a < 4; ++a) { s[a] += v[a]; s[4 + a] = fma(v[a], v[a], s[4 + a]); }
  }
#pragma unroll
  for (int a = 0; a < 8; ++a) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s[a] += __shfl_down_sync(0xffffffffu, s[a], o);
    if ((tid & 31) == 0) s_red[tid >> 5][a] = s[a];
  }
  __syncthreads();
  if (tid < 8) {
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < 8; ++w) t += s_red[w][tid];
    atomicAdd(&acc[(size_t)b * 8 + tid], t);
  }
}

__global__ void k_close_moments_tr(int M, uint32_t Np, const double *acc, double *out) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= M) return;
  const double iN = 1.0 / (double)Np;
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    const double m = acc[b * 8 + a] * iN;
    out[b * 8 + a] = m;
    out[b * 8 + 4 + a] = sqrt(fmax(acc[b * 8 + 4 + a] * iN - m * m, 0.0));
  }
}

// transverse initial distribution: Philox stream 3, counter (i, b, 0, 3), four normals (x, x', y, y')
__global__ void k_init_tr(double *x, double *xp, double *y, double *yp, int64_t ld, uint32_t Np, PhiloxKeys keys, double sx,
                          double sxp, double sy, double syp) {
  const int b = blockIdx.y;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < (uint32_t)ld; i += gridDim.x * blockDim.x) {
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    if (i < Np) {
      uint32_t w0, w1, w2, w3;
      philox4x32_10(i, (uint32_t)b, 0u, 3u, keys, w0, w1, w2, w3);
      box_muller_accurate(uniform32_plain(w0), uniform32_plain(w1), v[0], v[1]);
      box_muller_accurate(uniform32_plain(w2), uniform32_plain(w3), v[2], v[3]);
      v[0] *= sx; v[1] *= sxp; v[2] *= sy; v[3] *= syp;
    }
    const size_t q = (size_t)b * ld + i;
    x[q] = v[0]; xp[q] = v[1]; y[q] = v[2]; yp[q] = v[3];
  }
}

}  // namespace mbt
