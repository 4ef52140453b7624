// mbt_trans.cuh -- transverse planes (P:l.73-92 Eqs.(3)-(5), l.100-111 Eq.(6b); DESIGN.md
// readings T1..T8).  First correct CUDA path of this row: the transverse steps of a turn run in kernels of their own
// around the wake kernel, after the fused longitudinal pass (which is untouched):
//
//   k_pass        longitudinal: kick of turn n-1, map, binning of turn n            (mbt_kernels.cuh)
//   k_trans_map   Eqs. (3), (4) with the turn's delta, Eq. (5) lines 2-3, dipole deposit on the turn's window
//   k_wake        longitudinal wake of turn n                                       (mbt_kernels.cuh)
//   k_wake_tr     per bunch: K[j] = sum_{k<j} (Q_b/N_p) S[k] W_perp((j-k) Delta) for both planes
//   k_trans_kick  u' += K(tau)/E0 (gather as the longitudinal one); no transverse kick is ever pending
//
// Not fused and not tuned yet (library sincos / log, shared-memory fp64 atomics for the dipole sums): the bar of this
// stage is parity with the oracle.  Traffic: 80 B (map) + 56 B (kick) per particle-turn beside the pass's 32 B.
#pragma once
#include "mbt_kernels.cuh"

namespace mbt {

struct Plane {
  double two_pi_nu, xi, alpha, beta, gamma, eta, etap;
  double exc_u, exc_up;  // sigma_u sqrt(D_exc), sigma_up sqrt(D_exc)
};

struct TArgs {
  const double *tau, *delta;  // [M][ld] longitudinal store (read only here)
  double *x, *xp, *y, *yp;    // [M][ld]
  int64_t ld;
  uint32_t Np;
  int32_t M, nb;
  uint32_t tile;              // particles per CTA
  Plane px, py;
  int32_t rad;
  PhiloxKeys keys;
  // RF gain eps of Eq. (5): sum_c amp_c sin(w_c tau_before_drift + ph_c)
  int32_t n_cav;
  double cav_amp[kMaxCav], cav_w[kMaxCav], cav_ph[kMaxCav];
  double drift;
  // binning (as the pass)
  const double *lo_next;      // [M] window of this turn's binning (read by k_trans_map, before k_wake rotates it)
  const double *lo_hist;      // [M] the same window after k_wake (read by k_trans_kick)
  double invDelta, nb_d, invE0;
  int32_t gather;
  double *Sx, *Sy;            // [M][nb] dipole sums of the turn in flight (accumulated, consumed by k_wake_tr)
  const double *Kx, *Ky;      // [M][nb] kick tables [V]
  const Ctrl *ctrl;
};

// Eqs. (3), (4) for one plane (readings T2, T3), operation order as the oracle's
__device__ __forceinline__ void betatron_map(const Plane &p, double &u, double &up, double d) {
  const double psi = __dmul_rn(p.two_pi_nu, __dadd_rn(1.0, __dmul_rn(p.xi, d)));
  double sn, c;
  sincos(psi, &sn, &c);
  const double ub = u - p.eta * d, upb = up - p.etap * d;
  const double un = (c + p.alpha * sn) * ub + p.beta * sn * upb;
  const double upn = -p.gamma * sn * ub + (c - p.alpha * sn) * upb;
  u = p.eta * d + un;
  up = p.etap * d + upn;
}

__device__ __forceinline__ double uniform32_plain(uint32_t x) { return ((double)x + 0.5) * 0x1p-32; }

// after k_pass of turn n (tau, delta: mapped, not yet kicked by this turn's wake) and before k_wake of turn n
template <bool RAD>
__global__ void __launch_bounds__(256) k_trans_map(const __grid_constant__ TArgs A) {
  extern __shared__ double s_dip[];  // [2][nb]
  double *sSx = s_dip, *sSy = s_dip + A.nb;
  const int b = blockIdx.y, tid = threadIdx.x;
  for (int j = tid; j < 2 * A.nb; j += 256) s_dip[j] = 0.0;
  __syncthreads();
  const uint32_t n = A.ctrl->turn + 1u;  // k_wake has not bumped the counter yet: the turn in flight
  const double lo = A.lo_next[b];
  const uint32_t i0 = blockIdx.x * A.tile, i1 = min(i0 + A.tile, A.Np);
  const size_t base = (size_t)b * A.ld;
  for (uint32_t i = i0 + tid; i < i1; i += 256) {
    const double tau = A.tau[base + i], d = A.delta[base + i];
    double x = A.x[base + i], xp = A.xp[base + i], y = A.y[base + i], yp = A.yp[base + i];
    betatron_map(A.px, x, xp, d);
    betatron_map(A.py, y, yp, d);
    if (RAD) {
      // Eq. (5) lines 2, 3 (T4, T5): one Philox block per particle, counter (i, b, n, tag 2) -> (r_x, r_x', r_y, r_y')
      uint32_t w0, w1, w2, w3;
      philox4x32_10(i, (uint32_t)b, n, 2u, A.keys, w0, w1, w2, w3);
      double z0, z1, z2, z3;
      box_muller_accurate(uniform32_plain(w0), uniform32_plain(w1), z0, z1);
      box_muller_accurate(uniform32_plain(w2), uniform32_plain(w3), z2, z3);
      const double tau_old = fma(-A.drift, d, tau);  // tau before this turn's drift (to a rounding)
      double eps = 0.0;
      for (int c = 0; c < A.n_cav; ++c) eps += A.cav_amp[c] * sin(__dadd_rn(__dmul_rn(A.cav_w[c], tau_old), A.cav_ph[c]));
      const double adia = (1.0 + d) / (1.0 + d + eps);
      x += A.px.exc_u * z0;
      xp = xp * adia + A.px.exc_up * z1;
      y += A.py.exc_u * z2;
      yp = yp * adia + A.py.exc_up * z3;
    }
    A.x[base + i] = x; A.xp[base + i] = xp; A.y[base + i] = y; A.yp[base + i] = yp;
    // T6: dipole sums on the bins of this turn's histogram (the pass's S4 arithmetic)
    const double t = __dmul_rn(__dsub_rn(tau, lo), A.invDelta);
    if (t >= 0.0 && t < A.nb_d) {
      const int j = __double2int_rd(t);
      atomicAdd(&sSx[j], x);
      atomicAdd(&sSy[j], y);
    }
  }
  __syncthreads();
  for (int j = tid; j < A.nb; j += 256) {
    if (sSx[j] != 0.0) atomicAdd(&A.Sx[(size_t)b * A.nb + j], sSx[j]);
    if (sSy[j] != 0.0) atomicAdd(&A.Sy[(size_t)b * A.nb + j], sSy[j]);
  }
}

struct TWakeArgs {
  int32_t M, nb;
  const double *qm;     // [M]
  const double *wt;     // [nb] transverse table wt[k] = sum_r W_perp_r(k Delta), wt[0] = 0
  double *Sx, *Sy;      // [M][nb] in: sums of this turn; out: zero
  double *Sx_last, *Sy_last;  // [M][nb] observable copy
  double *Kx, *Ky;      // [M][nb] out
};

// Eq. (6b): strictly causal sum over the earlier bins; one CTA per bunch
__global__ void __launch_bounds__(256) k_wake_tr(const __grid_constant__ TWakeArgs A) {
  extern __shared__ double s_w[];  // [3][nb]: wt, q Sx, q Sy
  double *sw = s_w, *sx = s_w + A.nb, *sy = s_w + 2 * A.nb;
  const int b = blockIdx.x, tid = threadIdx.x, nb = A.nb;
  const double qm = A.qm[b];
  for (int j = tid; j < nb; j += 256) {
    const double vx = A.Sx[(size_t)b * nb + j], vy = A.Sy[(size_t)b * nb + j];
    A.Sx_last[(size_t)b * nb + j] = vx;
    A.Sy_last[(size_t)b * nb + j] = vy;
    A.Sx[(size_t)b * nb + j] = 0.0;
    A.Sy[(size_t)b * nb + j] = 0.0;
    sx[j] = qm * vx;
    sy[j] = qm * vy;
    sw[j] = A.wt[j];
  }
  __syncthreads();
  for (int j = tid; j < nb; j += 256) {
    double kx = 0.0, ky = 0.0;
    for (int k = 0; k < j; ++k) {
      kx = fma(sw[j - k], sx[k], kx);
      ky = fma(sw[j - k], sy[k], ky);
    }
    A.Kx[(size_t)b * nb + j] = kx;
    A.Ky[(size_t)b * nb + j] = ky;
  }
}

// after k_wake and k_wake_tr of turn n: u' += K(tau)/E0 for in-window particles (T7, T8)
__global__ void __launch_bounds__(256) k_trans_kick(const __grid_constant__ TArgs A) {
  extern __shared__ double s_k[];  // [2][nb]
  double *sKx = s_k, *sKy = s_k + A.nb;
  const int b = blockIdx.y, tid = threadIdx.x, nb = A.nb;
  for (int j = tid; j < nb; j += 256) { sKx[j] = A.Kx[(size_t)b * nb + j]; sKy[j] = A.Ky[(size_t)b * nb + j]; }
  __syncthreads();
  const double lo = A.lo_hist[b];
  const uint32_t i0 = blockIdx.x * A.tile, i1 = min(i0 + A.tile, A.Np);
  const size_t base = (size_t)b * A.ld;
  for (uint32_t i = i0 + tid; i < i1; i += 256) {
    const double t = __dmul_rn(__dsub_rn(A.tau[base + i], lo), A.invDelta);
    if (!(t >= 0.0 && t < A.nb_d)) continue;
    double vx, vy;
    if (A.gather == 0) {
      const int j = __double2int_rd(t);
      vx = sKx[j]; vy = sKy[j];
    } else {
      const double u = t - 0.5;
      if (u <= 0.0) { vx = sKx[0]; vy = sKy[0]; }
      else if (u >= (double)(nb - 1)) { vx = sKx[nb - 1]; vy = sKy[nb - 1]; }
      else {
        const int j0 = __double2int_rd(u);
        const double f = u - (double)j0;
        vx = sKx[j0] + f * (sKx[j0 + 1] - sKx[j0]);
        vy = sKy[j0] + f * (sKy[j0 + 1] - sKy[j0]);
      }
    }
    A.xp[base + i] += vx * A.invE0;
    A.yp[base + i] += vy * A.invE0;
  }
}

// sums for mbt_moments_transverse: out[M][8] += (sum x, x', y, y', sum x^2, x'^2, y^2, y'^2)
__global__ void __launch_bounds__(256) k_moments_tr(const __grid_constant__ TArgs A, double *acc) {
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
