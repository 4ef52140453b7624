// orc_tracker.cpp -- CPU ORACLE (test infrastructure, see orc.h).
//
// Plain single-threaded fp64 restatement of the per-turn longitudinal
// multi-bunch tracking method of arXiv:1809.00391, written step by step in the
// paper's order.  No blocking, fusion or reordering.  Build with
//     g++ -O2 -ffp-contract=off -std=c++17 -shared -fPIC
// (no FMA contraction: every product and sum below rounds separately).
//
// Turn n, for every bunch b and particle i:
//   1. RF kick + synchronous loss        P:l.65 Eq.(1), l.94 (harmonic-cavity list)
//   2. radiation damping + excitation    P:l.85 Eq.(5) line 1
//   3. drift with the UPDATED delta      P:l.67-69 Eq.(2) + the sentence before it (D1)
//   4. bin assignment + per-bin count    P:l.98, l.109-111
//   5. short-range wake on the bins      P:l.98 "excitation of this wake on each bin"
//   6. long-range resonator wake         P:l.229-237 (formula: reading D14)
//   7. wake kick                         P:l.102 Eq.(6a) (reading D9: delta -= V/E0)
//   8. per-bunch mean / rms              P:l.123-125
// and, with trans.enable (readings T1..T8, W1..W5):
//   3b. betatron map, excitation         P:l.73-92 Eqs.(3)-(5), after the longitudinal map (T1)
//   4b. per-bin dipole sums              P:l.104-111 (T6)
//   6b/7b. transverse wake and kick      P:l.100-107 Eq.(6b) (T7, T8)
//   9. long-range resistive-wall kick    P:l.117-119 (W1..W5), after the statistics of step 8
//
// PINS (tests/test_oracle_*.py, all run without a GPU):
//   philox4x32_10   Random123 known-answer vectors + cuRAND's host-callable Philox header
//   normal_pair     moments / KS test against scipy.stats.norm
//   resonator_wake  numerical inverse Fourier transform of the resonator impedance,
//                   loss factor of a binned Gaussian vs (1/pi) int Re Z exp(-w^2 s^2) dw
//   map (1,3)       small-amplitude synchrotron tune (FFT), Jacobian determinant 1
//   radiation (2)   centroid damping time, equilibrium energy spread
//   histogram (4)   numpy sort-and-count, sum + n_out = N_p, edge cases
//   SR wake (5)     numpy O(n^2) brute force, single occupied bin, energy bookkeeping
//   LR wake (6)     numpy brute-force pairwise sum, geometric-series closed form,
//                   lr_mode 1 (recurrence) against lr_mode 0 (definition)
//   whole loop      coupled-bunch growth rate vs the analytic uniform-fill formula, Eq.(7)
//   moments (8)     numpy mean / std
//   transverse      symplecticity, chromatic tune, dispersive fixed point, Courant-Snyder invariant; W_perp against
//                   its Lorentzian impedance; dipole sums vs numpy.bincount, Eq.(6b) written out; kick factor of a
//                   displaced Gaussian bunch from the impedance; coherent tune shift of the dipole line; adiabatic
//                   damping rate and equilibrium emittance (tests/test_oracle_transverse.py)
//   resistive wall  partial sums of k^-1/2 for a frozen offset, contiguous distance sum for a uniform fill, pairwise
//                   brute force, coupled-bunch growth / damping rates vs first-order theory (tests/test_oracle_rw.py)
//   history setters  orc_set_lr_history (rebuilds the per-turn aggregates ring_A) and orc_set_rw_history: checkpoint /
//                   resume into a fresh oracle is bit-identical to the uninterrupted run, both lr_modes, and is not
//                   when either setter is left out (tests/test_oracle_resume.py)
// No function of this file is "parity unpinned".
#include "orc.h"

#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

namespace {

typedef std::complex<double> cplx;
typedef long double ldbl;

thread_local std::string g_err = "";

int fail(int code, const std::string &msg) {
  g_err = msg;
  return code;
}

const ldbl PI_L = 3.141592653589793238462643383279502884L;
const double PI_D = 3.14159265358979323846;

// ---------------------------------------------------------------- Philox4x32-10
// Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11.
// Round: (hi0:lo0) = M0*c0, (hi1:lo1) = M1*c2;  c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0);
// the key is bumped by the Weyl constants AFTER each round's use.
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
    uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0;
    k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Reading D8: key = (seed mod 2^32, seed >> 32).  Initial-distribution stream (tag 1): the two
// uniforms use the top 52 bits of each 64-bit half, u = (k + 1/2) 2^-52, exactly representable and
// strictly inside (0,1); Box-Muller gives the pair (z_c, z_s).
void normal_pair(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                 double *u1o, double *u2o, double *zc, double *zs) {
  uint32_t ctr[4] = {c0, c1, c2, c3};
  uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
  uint32_t x[4];
  philox4x32_10(ctr, key, x);
  uint64_t w1 = ((uint64_t)x[1] << 32) | (uint64_t)x[0];
  uint64_t w2 = ((uint64_t)x[3] << 32) | (uint64_t)x[2];
  double u1 = ((double)(w1 >> 12) + 0.5) * 0x1p-52;
  double u2 = ((double)(w2 >> 12) + 0.5) * 0x1p-52;
  double r = std::sqrt(-2.0 * std::log(u1));
  double theta = 2.0 * PI_D * u2;
  *zc = r * std::cos(theta);
  *zs = r * std::sin(theta);
  if (u1o) *u1o = u1;
  if (u2o) *u2o = u2;
}

// Reading D8, excitation stream (tag 0): one Philox block serves FOUR consecutive particles of a bunch.  Each of
// its 32-bit words gives one uniform u = (x + 1/2) 2^-32 (exactly representable, strictly inside (0,1)); the
// words (x0, x1) are (u1, u2) of the Box-Muller pair (z[0], z[1]) of particles 4j, 4j+1 and (x2, x3) those of
// (z[2], z[3]) of particles 4j+2, 4j+3.
void normal_quad(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, double *uo, double *z) {
  uint32_t ctr[4] = {c0, c1, c2, c3};
  uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
  uint32_t x[4];
  philox4x32_10(ctr, key, x);
  for (int h = 0; h < 2; ++h) {
    double u1 = ((double)x[2 * h] + 0.5) * 0x1p-32;
    double u2 = ((double)x[2 * h + 1] + 0.5) * 0x1p-32;
    double r = std::sqrt(-2.0 * std::log(u1));
    double theta = 2.0 * PI_D * u2;
    z[2 * h] = r * std::cos(theta);
    z[2 * h + 1] = r * std::sin(theta);
    if (uo) { uo[2 * h] = u1; uo[2 * h + 1] = u2; }
  }
}

enum { TAG_EXCITATION = 0, TAG_INITIAL = 1, TAG_TRANSVERSE = 2, TAG_INITIAL_TRANSVERSE = 3 };

// ---------------------------------------------------------------- resonator
struct Resonator {
  double Rs, fr, Q;
  uint32_t flags;
  // derived (reading D10): w_r = 2 pi f_r, alpha = w_r/(2Q), wbar = sqrt(w_r^2 - alpha^2)
  ldbl alpha_l, wbar_l;
  double alpha, wbar;
  cplx C;  // 2 alpha Rs (1 + i alpha / wbar):  W(t>0) = Re[C exp(lambda t)]
};

void derive(Resonator &r) {
  ldbl wr = 2.0L * PI_L * (ldbl)r.fr;
  r.alpha_l = wr / (2.0L * (ldbl)r.Q);
  r.wbar_l = sqrtl(wr * wr - r.alpha_l * r.alpha_l);
  r.alpha = (double)r.alpha_l;
  r.wbar = (double)r.wbar_l;
  r.C = cplx(2.0 * r.alpha * r.Rs, 2.0 * r.alpha * r.Rs * (r.alpha / r.wbar));
}

// W(t) [V/C]: causal resonator wake, W(0) = alpha Rs = W(0+)/2 (beam-loading theorem), W(t<0) = 0.
double resonator_wake(const Resonator &r, double t) {
  if (t < 0.0) return 0.0;
  if (t == 0.0) return r.alpha * r.Rs;
  return 2.0 * r.alpha * r.Rs * std::exp(-r.alpha * t) *
         (std::cos(r.wbar * t) - (r.alpha / r.wbar) * std::sin(r.wbar * t));
}

// exp(lambda * dt), lambda = -alpha + i wbar, for dt up to K turns: the phase wbar*dt reaches
// 1e5..1e6 rad, so it is formed and reduced in extended precision, then rounded to fp64.
cplx exp_lambda(const Resonator &r, ldbl dt) {
  ldbl mag = expl(-r.alpha_l * dt);
  ldbl ph = r.wbar_l * dt;
  return cplx((double)(mag * cosl(ph)), (double)(mag * sinl(ph)));
}

}  // namespace

// ---------------------------------------------------------------- handle
struct orc_handle {
  // parameters
  orc_ring ring;
  std::vector<orc_cavity> cav;
  orc_radiation rad;
  int M = 0;
  int64_t Np = 0;
  std::vector<int32_t> bucket;
  std::vector<double> charge;
  double sigma_tau0 = 0, sigma_delta0 = 0;
  int nb = 0;
  double tau_lo = 0, tau_hi = 0;
  int gather = 1;
  int window_mode = 0;
  int32_t s_max = 0;                      // |shift| <= s_max keeps the window inside the bucket
  std::vector<int32_t> s_hist, s_next;    // [M] window shift in bins: of the current histogram / of the next binning
  std::vector<Resonator> res_lr;
  int K = 0;
  uint64_t seed = 0;
  int lr_mode = 0;
  int64_t log_cap = 0;
  // derived
  double omega_rf = 0, T_rf = 0, phi_s = 0, D_E = 0, A_q = 0, drift = 0, Delta = 0, invDelta = 0;
  std::vector<double> centre;  // c_j
  std::vector<double> w;       // SR table w_k = sum_r W_r(k Delta)
  bool have_sr = false;
  // state
  int64_t turn = 0;
  std::vector<double> tau, delta, tpos;
  std::vector<uint32_t> hist;
  std::vector<int64_t> n_out;
  std::vector<double> Vsr, Vlr, V;
  std::vector<cplx> ring_a;  // [(K+1)][M][R]: source phasors a[b][n'][r], slot n' % (K+1)
  std::vector<double> mom;   // [M][6]
  std::vector<double> log;   // [log_cap][M][6]
  // transverse planes (readings T1..T8); all empty when tr.enable == 0
  orc_transverse tr{};
  std::vector<Resonator> res_tr;
  std::vector<double> wt;                  // transverse table wt[k] = sum_r W_perp_r(k Delta), wt[0] = 0
  std::vector<double> x, xp, y, yp;        // [M][Np]
  std::vector<double> Sx, Sy, Kx, Ky;      // [M][nb] dipole sums [m] and kick tables [V]
  std::vector<double> mom_tr;              // [M][8]
  std::vector<double> log_tr;              // [log_cap][M][4] mean x, mean y, rms x, rms y per turn
  // long-range resistive wall (readings W1..W5)
  int Krw = 0;
  std::vector<double> ring_g;              // [(Krw+1)][M][2] source strengths Q_b ubar_{b,n'} [C m], slot n' % (Krw+1)
  std::vector<double> rw_kick;             // [M][2] kick of the last turn [V]
  double &g_at(int64_t n, int b, int a) { return ring_g[((size_t)(n % (Krw + 1)) * M + b) * 2 + a]; }
  // lr_mode 1 tables
  std::vector<cplx> g_step;  // [M-1][R] exp(lambda (s_{j+1}-s_j) T_rf)
  std::vector<cplx> g_hist;  // [K][R]   exp(lambda (k T0 - (s_{M-1}-s_0) T_rf)), k = 1..K
  std::vector<cplx> g_tail;  // [M][R]   exp(lambda (s_{M-1}-s_j) T_rf)
  std::vector<cplx> ring_A;  // [(K+1)][R] per-turn aggregates A_{n'}

  int R() const { return (int)res_lr.size(); }
  cplx &a_at(int64_t n, int b, int r) { return ring_a[((size_t)(n % (K + 1)) * M + b) * R() + r]; }
};

namespace {

ldbl dt_between(const orc_handle *h, int64_t dn, int ds) {
  ldbl T0 = (ldbl)h->ring.T0_s;
  return (ldbl)dn * T0 + (ldbl)ds * (T0 / (ldbl)h->ring.h);
}

// Reading T7 (the paper defers W_perp to its ref. [7], P:l.107): textbook transverse resonator wake,
// W_perp(t > 0) = (w_r^2 R / (Q wbar)) exp(-alpha t) sin(wbar t) [V/(C m)], R in Ohm/m, W_perp(t <= 0) = 0;
// its time integral is R / Q = |Z_perp(0)|.
double transverse_wake(const Resonator &r, double t) {
  if (!(t > 0.0)) return 0.0;
  double wr = 2.0 * PI_D * r.fr;
  return (wr * wr * r.Rs / (r.Q * r.wbar)) * std::exp(-r.alpha * t) * std::sin(r.wbar * t);
}

// Eqs. (3), (4) for one plane (readings T2, T3): Psi = 2 pi nu (1 + xi delta); the betatron part u - eta delta,
// u' - eta' delta is rotated by the Twiss matrix and the dispersive orbit is added back.
void betatron_map(const orc_plane &pl, double &u, double &up, double delta) {
  double psi = 2.0 * PI_D * pl.nu * (1.0 + pl.xi * delta);
  double c = std::cos(psi), sn = std::sin(psi);
  double gamma = (1.0 + pl.alpha * pl.alpha) / pl.beta_m;
  double ub = u - pl.eta_m * delta, upb = up - pl.etap * delta;
  double un = (c + pl.alpha * sn) * ub + pl.beta_m * sn * upb;
  double upn = -gamma * sn * ub + (c - pl.alpha * sn) * upb;
  u = pl.eta_m * delta + un;
  up = pl.etap * delta + upn;
}

// Reading D31: the window of bunch b starts at tau_lo + s Delta, s an integer number of bins
inline double window_lo(const orc_handle *h, int32_t s) {
  double off = (double)s * h->Delta;
  return h->tau_lo + off;
}
// centre of bin k of a window shifted by s bins
inline double bin_centre(const orc_handle *h, int32_t s, int k) { return window_lo(h, s) + ((double)k + 0.5) * h->Delta; }

// whole-bin step that brings the centroid of the counts back to the middle of the window:
// rint((sum_k (k + 1/2) c_k) / n_in - n_b / 2), half up, in exact integer arithmetic; 0 for an empty histogram
int32_t window_step(int nb, const uint32_t *c) {
  int64_t n_in = 0, m1 = 0;
  for (int k = 0; k < nb; ++k) { n_in += (int64_t)c[k]; m1 += (int64_t)k * (int64_t)c[k]; }
  if (n_in == 0) return 0;
  int64_t num = 2 * m1 + (2 - (int64_t)nb) * n_in, den = 2 * n_in;   // floor(num / den), den > 0
  int64_t q = num / den;
  if ((num % den != 0) && (num < 0)) q -= 1;
  return (int32_t)q;
}

// steps 1-3 for one particle; z is the unit normal of step 2
inline void map_one(const orc_handle *h, double &tau, double &delta, double z, double *eps_out = nullptr) {
  // 1. delta += sum_c (V_c/E0) sin(m_c w_rf tau + phi_c) - U0/E0   (terms left to right)
  const double E0 = h->ring.E0_eV;
  double eps = 0.0;  // relative energy gain in the RF cavities this turn (the epsilon of Eqs. (1), (5))
  for (size_t c = 0; c < h->cav.size(); ++c) {
    const orc_cavity &cv = h->cav[c];
    double term = (cv.V_volt / E0) * std::sin((double)cv.m * h->omega_rf * tau + cv.phase_rad);
    delta += term;
    eps += term;
  }
  if (eps_out) *eps_out = eps;
  delta -= h->ring.U0_eV / E0;
  // 2. delta = delta (1 - D_E) + sigma_delta sqrt(2 D_E) z
  if (h->rad.enable) delta = delta * (1.0 - h->D_E) + h->A_q * z;
  // 3. tau += alpha_c T0 delta  (the delta just updated, reading D1)
  tau += h->drift * delta;
}

void moments_of(const double *v, int64_t n, double &mean, double &rms) {
  double sm = 0; for (int64_t i = 0; i < n; ++i) sm += v[i];
  mean = sm / (double)n;
  double var = 0; for (int64_t i = 0; i < n; ++i) var += (v[i] - mean) * (v[i] - mean);
  rms = std::sqrt(var / (double)n);
}

void compute_moments(orc_handle *h) {
  if (h->tr.enable)
    for (int b = 0; b < h->M; ++b) {
      const double *c[4] = {&h->x[(size_t)b * h->Np], &h->xp[(size_t)b * h->Np], &h->y[(size_t)b * h->Np], &h->yp[(size_t)b * h->Np]};
      for (int a = 0; a < 4; ++a) moments_of(c[a], h->Np, h->mom_tr[(size_t)b * 8 + a], h->mom_tr[(size_t)b * 8 + 4 + a]);
    }
  // 8. population mean / rms over ALL particles of the bunch, two passes (reading D22)
  for (int b = 0; b < h->M; ++b) {
    const double *t = &h->tau[(size_t)b * h->Np];
    const double *d = &h->delta[(size_t)b * h->Np];
    double st = 0, sd = 0;
    for (int64_t i = 0; i < h->Np; ++i) { st += t[i]; sd += d[i]; }
    double mt = st / (double)h->Np, md = sd / (double)h->Np;
    double vt = 0, vd = 0;
    for (int64_t i = 0; i < h->Np; ++i) {
      vt += (t[i] - mt) * (t[i] - mt);
      vd += (d[i] - md) * (d[i] - md);
    }
    double *m = &h->mom[(size_t)b * 6];
    m[0] = (double)(h->Np - h->n_out[b]);
    m[1] = (double)h->n_out[b];
    m[2] = mt;
    m[3] = md;
    m[4] = std::sqrt(vt / (double)h->Np);
    m[5] = std::sqrt(vd / (double)h->Np);
  }
}

// step 4 for the current coordinates (also used after set_particles so that n_in / n_out and the
// histogram describe the uploaded state)
void bin_all(orc_handle *h) {
  std::fill(h->hist.begin(), h->hist.end(), 0u);
  std::fill(h->n_out.begin(), h->n_out.end(), (int64_t)0);
  std::fill(h->Sx.begin(), h->Sx.end(), 0.0);
  std::fill(h->Sy.begin(), h->Sy.end(), 0.0);
  for (int b = 0; b < h->M; ++b)
    for (int64_t i = 0; i < h->Np; ++i) {
      size_t p = (size_t)b * h->Np + i;
      // 4. t = (tau - tau_lo) * invDelta; in-window iff 0 <= t < n_b; j = floor(t)
      double t = (h->tau[p] - window_lo(h, h->s_hist[b])) * h->invDelta;
      h->tpos[p] = t;
      if (t >= 0.0 && t < (double)h->nb) {
        int j = (int)std::floor(t);
        h->hist[(size_t)b * h->nb + j] += 1u;
        if (h->tr.enable) {  // reading T6: q_k D_p(tau_k) of Eq. (6b) = (Q_b / N_p) * sum of the offsets in bin k
          h->Sx[(size_t)b * h->nb + j] += h->x[p];
          h->Sy[(size_t)b * h->nb + j] += h->y[p];
        }
      } else {
        h->n_out[b] += 1;
      }
    }
}

// steps 5 and 6 of turn n for the counts `hist` [M][nb] (on the windows s_hist): V_SR and V_LR on the bins.
// commit = true (the tracked turn): the source phasors of the counts enter the history ring (and, lr_mode 1, the
// per-turn aggregate); commit = false (orc_wake_from_counts): the handle is left untouched.
void build_wake(orc_handle *h, int64_t n, const uint32_t *hist, bool commit, double *Vsr, double *Vlr) {
  const int M = h->M, nb = h->nb, R = h->R(), K = h->K;
  const int64_t Np = h->Np;
  // 5: short-range wake, V_SR[b][j] = sum_{k<=j} w[j-k] q[b][k], q = (Q_b/N_p) hist
  std::vector<double> q((size_t)nb);
  for (int b = 0; b < M; ++b) {
    double qm = h->charge[b] / (double)Np;
    for (int k = 0; k < nb; ++k) q[k] = qm * (double)hist[(size_t)b * nb + k];
    double *Vs = &Vsr[(size_t)b * nb];
    if (h->have_sr)
      orc_sr_convolve(nb, h->w.data(), q.data(), Vs);
    else
      for (int j = 0; j < nb; ++j) Vs[j] = 0.0;
  }
  // 6: long-range resonator wake
  std::fill(Vlr, Vlr + (size_t)M * nb, 0.0);
  if (R > 0) {
    // source phasors a[b][n][r] = sum_k q[b][k] exp(-lambda_r c_k)
    std::vector<cplx> a_n((size_t)M * R);
    for (int b = 0; b < M; ++b) {
      double qm = h->charge[b] / (double)Np;
      for (int r = 0; r < R; ++r) {
        const Resonator &rs = h->res_lr[r];
        cplx lam(-rs.alpha, rs.wbar);
        cplx a(0.0, 0.0);
        for (int k = 0; k < nb; ++k) {
          double qk = qm * (double)hist[(size_t)b * nb + k];
          a += qk * std::exp(-lam * bin_centre(h, h->s_hist[b], k));
        }
        a_n[(size_t)b * R + r] = a;
        if (commit) h->a_at(n, b, r) = a;
      }
    }
    std::vector<cplx> P((size_t)M * R, cplx(0, 0));
    if (h->lr_mode == 0) {
      // THE definition: pairwise sum over H(b,n)
      for (int b = 0; b < M; ++b)
        for (int r = 0; r < R; ++r) {
          const Resonator &rs = h->res_lr[r];
          cplx acc(0, 0);
          int64_t first = (n - K > 1) ? (n - K) : 1;
          for (int64_t np = first; np <= n - 1; ++np)
            for (int bp = 0; bp < M; ++bp)
              acc += h->a_at(np, bp, r) * exp_lambda(rs, dt_between(h, n - np, h->bucket[b] - h->bucket[bp]));
          for (int bp = 0; bp < M; ++bp)
            if (h->bucket[bp] < h->bucket[b])
              acc += a_n[(size_t)bp * R + r] * exp_lambda(rs, dt_between(h, 0, h->bucket[b] - h->bucket[bp]));
          P[(size_t)b * R + r] = acc;
        }
    } else {
      // equivalent O(M+K) form; only decaying factors occur
      for (int r = 0; r < R; ++r) {
        cplx G(0, 0);
        for (int k = 1; k <= K && n - k >= 1; ++k)
          G += h->ring_A[(size_t)((n - k) % (K + 1)) * R + r] * h->g_hist[(size_t)(k - 1) * R + r];
        cplx Pj = G, own(0, 0);
        for (int j = 0; j < M; ++j) {
          P[(size_t)j * R + r] = Pj;
          own += a_n[(size_t)j * R + r] * h->g_tail[(size_t)j * R + r];
          if (j + 1 < M) Pj = (Pj + a_n[(size_t)j * R + r]) * h->g_step[(size_t)j * R + r];
        }
        if (commit) h->ring_A[(size_t)(n % (K + 1)) * R + r] = own;
      }
    }
    // V_LR[b][j] = sum_r Re[C_r exp(lambda_r c_j) P[b][r]]
    for (int b = 0; b < M; ++b)
      for (int j = 0; j < nb; ++j) {
        double v = 0.0;
        for (int r = 0; r < R; ++r) {
          const Resonator &rs = h->res_lr[r];
          cplx lam(-rs.alpha, rs.wbar);
          v += std::real(rs.C * std::exp(lam * bin_centre(h, h->s_hist[b], j)) * P[(size_t)b * R + r]);
        }
        Vlr[(size_t)b * nb + j] = v;
      }
  }
}

void one_turn(orc_handle *h) {
  const int M = h->M, nb = h->nb;
  const int64_t Np = h->Np;
  const int64_t n = h->turn + 1;
  // 1-3: single-particle map
  for (int b = 0; b < M; ++b)
  {
    double zq[4] = {0.0, 0.0, 0.0, 0.0};
    for (int64_t i = 0; i < Np; ++i) {
      size_t p = (size_t)b * Np + i;
      double z = 0.0;
      if (h->rad.enable) {
        // one block per four particles: counter (i >> 2, b, n, tag 0), particle i takes z[i & 3]
        if ((i & 3) == 0) normal_quad(h->seed, (uint32_t)(i >> 2), (uint32_t)b, (uint32_t)n, TAG_EXCITATION, nullptr, zq);
        z = zq[i & 3];
      }
      double eps = 0.0;
      map_one(h, h->tau[p], h->delta[p], z, &eps);
      if (h->tr.enable) {
        // reading T1: the transverse steps of a turn follow its longitudinal map and use the updated delta
        const double d = h->delta[p];
        betatron_map(h->tr.x, h->x[p], h->xp[p], d);   // Eqs. (3), (4)
        betatron_map(h->tr.y, h->y[p], h->yp[p], d);
        if (h->rad.enable) {
          // Eq. (5) lines 2, 3 (reading T4; the same for y): one Philox block per particle, counter (i, b, n, tag 2),
          // its four normals are (x, x', y, y')
          double zt[4];
          normal_quad(h->seed, (uint32_t)i, (uint32_t)b, (uint32_t)n, TAG_TRANSVERSE, nullptr, zt);
          const double adia = (1.0 + d) / (1.0 + d + eps);
          h->x[p] += h->tr.x.sigma_u_m * std::sqrt(h->tr.x.D_exc) * zt[0];
          h->xp[p] = h->xp[p] * adia + h->tr.x.sigma_up * std::sqrt(h->tr.x.D_exc) * zt[1];
          h->y[p] += h->tr.y.sigma_u_m * std::sqrt(h->tr.y.D_exc) * zt[2];
          h->yp[p] = h->yp[p] * adia + h->tr.y.sigma_up * std::sqrt(h->tr.y.D_exc) * zt[3];
        }
      }
    }
  }
  // 4: bins, on the window chosen after the previous turn (reading D31); then the window of the next turn
  h->s_hist = h->s_next;
  bin_all(h);
  if (h->window_mode == 1)
    for (int b = 0; b < M; ++b) {
      int64_t s = (int64_t)h->s_hist[b] + window_step(nb, &h->hist[(size_t)b * nb]);
      if (s > h->s_max) s = h->s_max;
      if (s < -(int64_t)h->s_max) s = -(int64_t)h->s_max;
      h->s_next[b] = (int32_t)s;
    }
  // 5, 6: wake potentials of this turn's counts (build_wake above); the source phasors enter the history ring
  build_wake(h, n, h->hist.data(), true, h->Vsr.data(), h->Vlr.data());
  for (size_t x = 0; x < h->V.size(); ++x) h->V[x] = h->Vsr[x] + h->Vlr[x];
  // 7: wake kick on in-window particles, delta -= v/E0 (reading D9)
  for (int b = 0; b < M; ++b) {
    const double *Vb = &h->V[(size_t)b * nb];
    for (int64_t i = 0; i < Np; ++i) {
      size_t p = (size_t)b * Np + i;
      double t = h->tpos[p];
      if (!(t >= 0.0 && t < (double)nb)) continue;
      double v;
      if (h->gather == 0) {
        v = Vb[(int)std::floor(t)];  // nearest grid point: the paper's "kick given to every particle in the bin"
      } else {
        double u = t - 0.5;  // linear between bin centres, held constant in the outer half bins (reading D12)
        if (u <= 0.0) v = Vb[0];
        else if (u >= (double)(nb - 1)) v = Vb[nb - 1];
        else {
          int j0 = (int)std::floor(u);
          double f = u - (double)j0;
          v = Vb[j0] + f * (Vb[j0 + 1] - Vb[j0]);
        }
      }
      h->delta[p] -= v / h->ring.E0_eV;
    }
  }
  // 6b/7b: transverse short-range wake and kick, Eq. (6b): K[j] = sum_{k<j} (Q_b/N_p) S[k] W_perp((j-k) Delta);
  // u' += K(tau)/E0 for in-window particles, gathered like the longitudinal wake (readings T7, T8)
  if (h->tr.enable) {
    for (int b = 0; b < M; ++b) {
      double qm = h->charge[b] / (double)Np;
      for (int j = 0; j < nb; ++j) {
        double kx = 0.0, ky = 0.0;
        for (int k = 0; k < j; ++k) {
          kx += h->wt[j - k] * (qm * h->Sx[(size_t)b * nb + k]);
          ky += h->wt[j - k] * (qm * h->Sy[(size_t)b * nb + k]);
        }
        h->Kx[(size_t)b * nb + j] = kx;
        h->Ky[(size_t)b * nb + j] = ky;
      }
      for (int64_t i = 0; i < Np; ++i) {
        size_t p = (size_t)b * Np + i;
        double t = h->tpos[p];
        if (!(t >= 0.0 && t < (double)nb)) continue;
        const double *T[2] = {&h->Kx[(size_t)b * nb], &h->Ky[(size_t)b * nb]};
        double v[2];
        for (int a = 0; a < 2; ++a) {
          if (h->gather == 0) v[a] = T[a][(int)std::floor(t)];
          else {
            double u = t - 0.5;
            if (u <= 0.0) v[a] = T[a][0];
            else if (u >= (double)(nb - 1)) v[a] = T[a][nb - 1];
            else { int j0 = (int)std::floor(u); double f = u - (double)j0; v[a] = T[a][j0] + f * (T[a][j0 + 1] - T[a][j0]); }
          }
        }
        h->xp[p] += v[0] / h->ring.E0_eV;
        h->yp[p] += v[1] / h->ring.E0_eV;
      }
    }
  }
  // 8: statistics
  compute_moments(h);
  // 9: long-range resistive-wall kick on the transverse planes (P:l.117-119; readings W1..W5), "launched only when wake
  // potential effects are calculated for all the bunches and the statistics have been updated": the sources are the
  // bunch centroids of the statistics just taken, this turn's for the bunches ahead and the last Krw turns' for all;
  // W_rw(t) = A / sqrt(t) (W2); every particle of the bunch gets the same kick, in the window or not (W4)
  if (h->tr.enable && h->Krw > 0) {
    for (int b = 0; b < M; ++b) {
      h->g_at(n, b, 0) = h->charge[b] * h->mom_tr[(size_t)b * 8 + 0];
      h->g_at(n, b, 1) = h->charge[b] * h->mom_tr[(size_t)b * 8 + 2];
    }
    const double amp[2] = {h->tr.rw_amp_x, h->tr.rw_amp_y};
    for (int b = 0; b < M; ++b) {
      double sum[2] = {0.0, 0.0};
      for (int64_t np = std::max<int64_t>(1, n - h->Krw); np <= n; ++np)
        for (int bp = 0; bp < M; ++bp) {
          if (np == n && h->bucket[bp] >= h->bucket[b]) continue;          // this turn: only the bunches ahead (W5)
          double dt = (double)dt_between(h, n - np, h->bucket[b] - h->bucket[bp]);
          double wgt = 1.0 / std::sqrt(dt);
          for (int a = 0; a < 2; ++a) sum[a] += h->g_at(np, bp, a) * wgt;
        }
      for (int a = 0; a < 2; ++a) h->rw_kick[(size_t)b * 2 + a] = amp[a] * sum[a];
      const double kx = h->rw_kick[(size_t)b * 2] / h->ring.E0_eV, ky = h->rw_kick[(size_t)b * 2 + 1] / h->ring.E0_eV;
      for (int64_t i = 0; i < Np; ++i) {
        h->xp[(size_t)b * Np + i] += kx;
        h->yp[(size_t)b * Np + i] += ky;
      }
    }
    compute_moments(h);  // the observable moments describe the state after the kick
  }
  h->turn = n;
  if (n - 1 < h->log_cap) std::memcpy(&h->log[(size_t)(n - 1) * M * 6], h->mom.data(), sizeof(double) * M * 6);
  if (h->tr.enable && n - 1 < h->log_cap)
    for (int b = 0; b < M; ++b)
      for (int a = 0; a < 4; ++a)   // mom_tr: mean x x' y y', rms x x' y y'  ->  mean x, mean y, rms x, rms y
        h->log_tr[((size_t)(n - 1) * M + b) * 4 + a] = h->mom_tr[(size_t)b * 8 + (a < 2 ? 2 * a : 4 + 2 * (a - 2))];
}

}  // namespace

extern "C" {

const char *orc_last_error(void) { return g_err.c_str(); }

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox4x32_10(ctr, key, out); }

void orc_normal_pair(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, double *u1, double *u2,
                     double *z_c, double *z_s) {
  normal_pair(seed, c0, c1, c2, c3, u1, u2, z_c, z_s);
}

void orc_normal_quad(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, double *u, double *z) {
  normal_quad(seed, c0, c1, c2, c3, u, z);
}

double orc_resonator_wake(double Rs, double fr, double Q, double t) {
  Resonator r{Rs, fr, Q, 0u, 0, 0, 0, 0, cplx()};
  derive(r);
  return resonator_wake(r, t);
}

// V[j] = sum_{k=0..j} w[j-k] q[k], k ascending -- the definition of the discrete causal convolution
void orc_sr_convolve(int32_t nb, const double *w, const double *q, double *V) {
  for (int j = 0; j < nb; ++j) {
    double acc = 0.0;
    for (int k = 0; k <= j; ++k) acc += w[j - k] * q[k];
    V[j] = acc;
  }
}

void orc_map_one(const orc_handle *h, double *tau, double *delta, double z) { map_one(h, *tau, *delta, z); }

int orc_create(const orc_params *p, orc_handle **out) {
  if (!p || !out) return fail(ORC_EINVAL, "null argument");
  *out = nullptr;
  const orc_ring &rg = p->ring;
  if (!(rg.E0_eV > 0) || !(rg.T0_s > 0) || rg.h < 1 || !std::isfinite(rg.alpha_c) || rg.alpha_c == 0.0 ||
      !std::isfinite(rg.U0_eV))
    return fail(ORC_EINVAL, "ring: need E0 > 0, T0 > 0, h >= 1, alpha_c != 0");
  if (p->n_cav < 1 || !p->cav) return fail(ORC_EINVAL, "need at least the main cavity");
  if (p->fill.n_bunches < 1 || !p->fill.bucket || !p->fill.charge_C || p->fill.n_per_bunch < 1 ||
      p->fill.n_per_bunch > 0xFFFFFFFFll)
    return fail(ORC_EINVAL, "fill: need n_bunches >= 1, 1 <= n_per_bunch < 2^32");
  for (int b = 0; b < p->fill.n_bunches; ++b) {
    if (p->fill.bucket[b] < 0 || p->fill.bucket[b] >= rg.h) return fail(ORC_EINVAL, "bucket out of [0,h)");
    if (b > 0 && p->fill.bucket[b] <= p->fill.bucket[b - 1]) return fail(ORC_EINVAL, "buckets not strictly increasing");
    if (!std::isfinite(p->fill.charge_C[b])) return fail(ORC_EINVAL, "charge not finite");
  }
  const orc_wake &wk = p->wake;
  if (wk.n_bins < 2) return fail(ORC_EINVAL, "n_bins < 2");
  if (!(wk.tau_hi_s > wk.tau_lo_s) || !((wk.tau_hi_s - wk.tau_lo_s) < rg.T0_s / rg.h))
    return fail(ORC_EINVAL, "window must satisfy 0 < tau_hi - tau_lo < T_rf");
  if (wk.gather_order != 0 && wk.gather_order != 1) return fail(ORC_EINVAL, "gather_order must be 0 or 1");
  if (wk.window_mode != 0 && wk.window_mode != 1) return fail(ORC_EINVAL, "window_mode must be 0 or 1");
  if (wk.n_res < 0 || (wk.n_res > 0 && !wk.res)) return fail(ORC_EINVAL, "resonator list");
  if (wk.n_table < 0 || (wk.n_table > 0 && !wk.sr_table)) return fail(ORC_EINVAL, "sr_table");
  if (p->rad.enable && (!(p->rad.damping_turns > 0) || !(p->rad.sigma_delta >= 0)))
    return fail(ORC_EINVAL, "radiation: need damping_turns > 0, sigma_delta >= 0");
  if (p->log_capacity_turns < 0) return fail(ORC_EINVAL, "log_capacity_turns < 0");

  orc_handle *h = new (std::nothrow) orc_handle();
  if (!h) return fail(ORC_ENOMEM, "out of memory");
  try {
    h->ring = rg;
    h->cav.assign(p->cav, p->cav + p->n_cav);
    h->rad = p->rad;
    h->M = p->fill.n_bunches;
    h->Np = p->fill.n_per_bunch;
    h->bucket.assign(p->fill.bucket, p->fill.bucket + h->M);
    h->charge.assign(p->fill.charge_C, p->fill.charge_C + h->M);
    h->sigma_tau0 = p->fill.sigma_tau0_s;
    h->sigma_delta0 = p->fill.sigma_delta0;
    h->nb = wk.n_bins;
    h->tau_lo = wk.tau_lo_s;
    h->tau_hi = wk.tau_hi_s;
    h->gather = wk.gather_order;
    h->window_mode = wk.window_mode;
    h->seed = p->seed;
    h->lr_mode = p->lr_mode;
    h->log_cap = p->log_capacity_turns;

    // derived constants
    h->omega_rf = 2.0 * PI_D * (double)rg.h / rg.T0_s;
    h->T_rf = rg.T0_s / (double)rg.h;
    h->D_E = p->rad.enable ? 2.0 / p->rad.damping_turns : 0.0;
    h->A_q = p->rad.enable ? p->rad.sigma_delta * std::sqrt(2.0 * h->D_E) : 0.0;
    h->drift = rg.alpha_c * rg.T0_s;
    h->Delta = (h->tau_hi - h->tau_lo) / (double)h->nb;
    h->invDelta = (double)h->nb / (h->tau_hi - h->tau_lo);
    h->centre.resize(h->nb);
    for (int j = 0; j < h->nb; ++j) h->centre[j] = h->tau_lo + ((double)j + 0.5) * h->Delta;

    // synchronous phase (reading D3): V1 sin(phi_s) = U0 - sum_h V_h sin(phi_h), on the stable side
    for (int c = 1; c < p->n_cav; ++c)
      if (std::isnan(h->cav[c].phase_rad)) { delete h; return fail(ORC_EINVAL, "only cavity 0 may leave its phase open"); }
    if (std::isnan(h->cav[0].phase_rad)) {
      double u_eff = rg.U0_eV;
      for (int c = 1; c < p->n_cav; ++c) u_eff -= h->cav[c].V_volt * std::sin(h->cav[c].phase_rad);
      double s = u_eff / h->cav[0].V_volt;
      if (!(std::fabs(s) <= 1.0)) { delete h; return fail(ORC_EINVAL, "U0 exceeds the RF voltage: no synchronous phase"); }
      h->cav[0].phase_rad = (rg.alpha_c > 0.0) ? PI_D - std::asin(s) : std::asin(s);
    }
    h->phi_s = h->cav[0].phase_rad;

    // wake sources
    h->w.assign(h->nb, 0.0);
    for (int r = 0; r < wk.n_res; ++r) {
      const orc_resonator &in = wk.res[r];
      if (!(in.Q > 0.5) || !(in.fr_Hz > 0) || !std::isfinite(in.Rs_ohm)) { delete h; return fail(ORC_EINVAL, "resonator: need Q > 1/2, fr > 0"); }
      Resonator rr{in.Rs_ohm, in.fr_Hz, in.Q, in.flags, 0, 0, 0, 0, cplx()};
      derive(rr);
      if (in.flags & ORC_RES_SR) {
        h->have_sr = true;
        for (int k = 0; k < h->nb; ++k) h->w[k] += resonator_wake(rr, (double)k * h->Delta);
      }
      if (in.flags & ORC_RES_LR) h->res_lr.push_back(rr);
    }
    if (wk.n_table > 0) {  // user-sampled wake at lag k*Delta, added to the resonator table
      h->have_sr = true;
      for (int k = 0; k < h->nb && k < wk.n_table; ++k) h->w[k] += wk.sr_table[k];
    }
    h->K = wk.history_turns;
    if (h->R() > 0 && h->K < 0) { delete h; return fail(ORC_EINVAL, "history_turns < 0"); }
    if (h->R() == 0) h->K = 0;

    // state
    size_t N = (size_t)h->M * (size_t)h->Np;
    h->tau.resize(N); h->delta.resize(N); h->tpos.resize(N);
    h->hist.assign((size_t)h->M * h->nb, 0u);
    h->n_out.assign(h->M, 0);
    h->s_hist.assign(h->M, 0);
    h->s_next.assign(h->M, 0);
    // the shifted window [tau_lo + s Delta, tau_hi + s Delta] stays inside the bucket [-T_rf/2, T_rf/2]
    {
      double room = std::fmin(0.5 * h->T_rf - h->tau_hi, h->tau_lo + 0.5 * h->T_rf);   // to the nearer bucket edge
      double smax = std::floor(room / h->Delta);
      h->s_max = (h->window_mode && smax > 0.0) ? (int32_t)std::fmin(smax, 1.0e6) : 0;
    }
    h->Vsr.assign((size_t)h->M * h->nb, 0.0);
    h->Vlr.assign((size_t)h->M * h->nb, 0.0);
    h->V.assign((size_t)h->M * h->nb, 0.0);
    h->ring_a.assign((size_t)(h->K + 1) * h->M * (h->R() ? h->R() : 1), cplx(0, 0));
    h->mom.assign((size_t)h->M * 6, 0.0);
    // transverse planes
    h->tr = p->trans;
    h->tr.res = nullptr;  // copied below
    if (h->tr.enable) {
      const orc_plane *pls[2] = {&h->tr.x, &h->tr.y};
      for (const orc_plane *pl : pls)
        if (!(pl->beta_m > 0) || !std::isfinite(pl->nu) || !std::isfinite(pl->alpha) || !(pl->D_exc >= 0) ||
            !(pl->sigma_u_m >= 0) || !(pl->sigma_up >= 0) || !(pl->sigma0_u_m >= 0) || !(pl->sigma0_up >= 0)) {
          delete h;
          return fail(ORC_EINVAL, "transverse plane: need beta > 0, D_exc >= 0, sigmas >= 0");
        }
      if (p->trans.n_res < 0 || (p->trans.n_res > 0 && !p->trans.res)) { delete h; return fail(ORC_EINVAL, "transverse resonator list"); }
      h->wt.assign(h->nb, 0.0);
      for (int r = 0; r < p->trans.n_res; ++r) {
        const orc_resonator &in = p->trans.res[r];
        if (!(in.Q > 0.5) || !(in.fr_Hz > 0) || !std::isfinite(in.Rs_ohm)) { delete h; return fail(ORC_EINVAL, "transverse resonator: need Q > 1/2, fr > 0"); }
        Resonator rr{in.Rs_ohm, in.fr_Hz, in.Q, in.flags, 0, 0, 0, 0, cplx()};
        derive(rr);
        h->res_tr.push_back(rr);
        for (int k = 0; k < h->nb; ++k) h->wt[k] += transverse_wake(rr, (double)k * h->Delta);
      }
      h->x.assign(N, 0.0); h->xp.assign(N, 0.0); h->y.assign(N, 0.0); h->yp.assign(N, 0.0);
      h->Sx.assign((size_t)h->M * h->nb, 0.0); h->Sy.assign((size_t)h->M * h->nb, 0.0);
      h->Kx.assign((size_t)h->M * h->nb, 0.0); h->Ky.assign((size_t)h->M * h->nb, 0.0);
      h->mom_tr.assign((size_t)h->M * 8, 0.0);
      if (p->trans.rw_turns < 0 || p->trans.rw_turns > 100000 || !std::isfinite(p->trans.rw_amp_x) || !std::isfinite(p->trans.rw_amp_y)) {
        delete h;
        return fail(ORC_EINVAL, "resistive wall: need 0 <= rw_turns <= 100000, finite amplitudes");
      }
      h->Krw = p->trans.rw_turns;
      h->ring_g.assign((size_t)(h->Krw + 1) * h->M * 2, 0.0);
      h->rw_kick.assign((size_t)h->M * 2, 0.0);
    }
    h->log.assign((size_t)h->log_cap * h->M * 6, 0.0);
    if (h->tr.enable) h->log_tr.assign((size_t)h->log_cap * h->M * 4, 0.0);
    if (h->R() > 0) {
      int R = h->R(), M = h->M, K = h->K;
      h->g_step.assign((size_t)M * R, cplx(0, 0));
      h->g_tail.assign((size_t)M * R, cplx(0, 0));
      h->g_hist.assign((size_t)(K ? K : 1) * R, cplx(0, 0));
      h->ring_A.assign((size_t)(K + 1) * R, cplx(0, 0));
      int span = h->bucket[M - 1] - h->bucket[0];
      for (int r = 0; r < R; ++r) {
        for (int j = 0; j + 1 < M; ++j)
          h->g_step[(size_t)j * R + r] = exp_lambda(h->res_lr[r], dt_between(h, 0, h->bucket[j + 1] - h->bucket[j]));
        for (int j = 0; j < M; ++j)
          h->g_tail[(size_t)j * R + r] = exp_lambda(h->res_lr[r], dt_between(h, 0, h->bucket[M - 1] - h->bucket[j]));
        for (int k = 1; k <= K; ++k) h->g_hist[(size_t)(k - 1) * R + r] = exp_lambda(h->res_lr[r], dt_between(h, k, -span));
      }
    }

    // initial distribution (reading D20): Philox stream 1, counter (i, b, 0, 1); tau = s_tau0 z_c, delta = s_delta0 z_s
    for (int b = 0; b < h->M; ++b)
      for (int64_t i = 0; i < h->Np; ++i) {
        double zc, zs;
        normal_pair(h->seed, (uint32_t)i, (uint32_t)b, 0u, TAG_INITIAL, nullptr, nullptr, &zc, &zs);
        h->tau[(size_t)b * h->Np + i] = h->sigma_tau0 * zc;
        h->delta[(size_t)b * h->Np + i] = h->sigma_delta0 * zs;
      }
    // transverse initial distribution: Philox stream 3, counter (i, b, 0, 3), four normals (x, x', y, y')
    if (h->tr.enable)
      for (int b = 0; b < h->M; ++b)
        for (int64_t i = 0; i < h->Np; ++i) {
          double z4[4];
          normal_quad(h->seed, (uint32_t)i, (uint32_t)b, 0u, TAG_INITIAL_TRANSVERSE, nullptr, z4);
          size_t q = (size_t)b * h->Np + i;
          h->x[q] = h->tr.x.sigma0_u_m * z4[0];
          h->xp[q] = h->tr.x.sigma0_up * z4[1];
          h->y[q] = h->tr.y.sigma0_u_m * z4[2];
          h->yp[q] = h->tr.y.sigma0_up * z4[3];
        }
    bin_all(h);
    compute_moments(h);
  } catch (const std::bad_alloc &) {
    delete h;
    return fail(ORC_ENOMEM, "out of memory");
  }
  *out = h;
  return 0;
}

int orc_track(orc_handle *h, int64_t n_turns) {
  if (!h || n_turns < 0) return fail(ORC_EINVAL, "bad argument");
  if (h->turn + n_turns > 0xFFFFFFFFll) return fail(ORC_EINVAL, "turn counter would exceed 2^32");
  for (int64_t t = 0; t < n_turns; ++t) one_turn(h);
  return 0;
}

int orc_moments(orc_handle *h, double *out) {
  if (!h || !out) return fail(ORC_EINVAL, "null argument");
  std::memcpy(out, h->mom.data(), sizeof(double) * h->mom.size());
  return 0;
}

int orc_destroy(orc_handle *h) {
  delete h;
  return 0;
}

int orc_get_particles(orc_handle *h, double *tau, double *delta) {
  if (!h || !tau || !delta) return fail(ORC_EINVAL, "null argument");
  std::memcpy(tau, h->tau.data(), sizeof(double) * h->tau.size());
  std::memcpy(delta, h->delta.data(), sizeof(double) * h->delta.size());
  return 0;
}

int orc_set_particles(orc_handle *h, const double *tau, const double *delta, int64_t turn) {
  if (!h || !tau || !delta || turn < 0) return fail(ORC_EINVAL, "bad argument");
  std::memcpy(h->tau.data(), tau, sizeof(double) * h->tau.size());
  std::memcpy(h->delta.data(), delta, sizeof(double) * h->delta.size());
  h->turn = turn;
  bin_all(h);
  compute_moments(h);
  return 0;
}

int orc_get_transverse(orc_handle *h, double *x, double *xp, double *y, double *yp) {
  if (!h || !h->tr.enable || !x || !xp || !y || !yp) return fail(ORC_EINVAL, "transverse planes not enabled / null argument");
  size_t bytes = sizeof(double) * h->x.size();
  std::memcpy(x, h->x.data(), bytes); std::memcpy(xp, h->xp.data(), bytes);
  std::memcpy(y, h->y.data(), bytes); std::memcpy(yp, h->yp.data(), bytes);
  return 0;
}

int orc_set_transverse(orc_handle *h, const double *x, const double *xp, const double *y, const double *yp) {
  if (!h || !h->tr.enable || !x || !xp || !y || !yp) return fail(ORC_EINVAL, "transverse planes not enabled / null argument");
  size_t bytes = sizeof(double) * h->x.size();
  std::memcpy(h->x.data(), x, bytes); std::memcpy(h->xp.data(), xp, bytes);
  std::memcpy(h->y.data(), y, bytes); std::memcpy(h->yp.data(), yp, bytes);
  bin_all(h);
  compute_moments(h);
  return 0;
}

int orc_get_dipole(orc_handle *h, double *Sx, double *Sy) {
  if (!h || !h->tr.enable) return fail(ORC_EINVAL, "transverse planes not enabled");
  if (Sx) std::memcpy(Sx, h->Sx.data(), sizeof(double) * h->Sx.size());
  if (Sy) std::memcpy(Sy, h->Sy.data(), sizeof(double) * h->Sy.size());
  return 0;
}

int orc_get_transverse_wake(orc_handle *h, double *Kx, double *Ky) {
  if (!h || !h->tr.enable) return fail(ORC_EINVAL, "transverse planes not enabled");
  if (Kx) std::memcpy(Kx, h->Kx.data(), sizeof(double) * h->Kx.size());
  if (Ky) std::memcpy(Ky, h->Ky.data(), sizeof(double) * h->Ky.size());
  return 0;
}

int orc_moments_transverse(orc_handle *h, double *out) {
  if (!h || !h->tr.enable || !out) return fail(ORC_EINVAL, "transverse planes not enabled / null argument");
  std::memcpy(out, h->mom_tr.data(), sizeof(double) * h->mom_tr.size());
  return 0;
}

int orc_get_transverse_log(orc_handle *h, int64_t first_turn, int64_t n, double *out) {
  if (!h || !h->tr.enable || !out || first_turn < 1 || n < 0) return fail(ORC_EINVAL, "bad argument");
  if (first_turn - 1 + n > h->log_cap || first_turn - 1 + n > h->turn) return fail(ORC_ESTATE, "turns not in the log");
  std::memcpy(out, &h->log_tr[(size_t)(first_turn - 1) * h->M * 4], sizeof(double) * (size_t)n * h->M * 4);
  return 0;
}

int orc_get_rw_kick(orc_handle *h, double *kx, double *ky) {
  if (!h || !h->tr.enable) return fail(ORC_EINVAL, "transverse planes not enabled");
  for (int b = 0; b < h->M; ++b) {
    if (kx) kx[b] = h->rw_kick[(size_t)b * 2];
    if (ky) ky[b] = h->rw_kick[(size_t)b * 2 + 1];
  }
  return 0;
}

// oldest first: row k holds turn (turn - Krw + 1 + k); turns < 1 are zero
int orc_get_rw_history(orc_handle *h, double *out) {
  if (!h || !h->tr.enable || !out) return fail(ORC_EINVAL, "transverse planes not enabled / null argument");
  for (int k = 0; k < h->Krw; ++k) {
    int64_t np = h->turn - h->Krw + 1 + k;
    for (int b = 0; b < h->M; ++b)
      for (int a = 0; a < 2; ++a) out[((size_t)k * h->M + b) * 2 + a] = np >= 1 ? h->g_at(np, b, a) : 0.0;
  }
  return 0;
}

int orc_set_rw_history(orc_handle *h, const double *in) {
  if (!h || !h->tr.enable || !in) return fail(ORC_EINVAL, "transverse planes not enabled / null argument");
  for (int k = 0; k < h->Krw; ++k) {
    int64_t np = h->turn - h->Krw + 1 + k;
    if (np < 1) continue;
    for (int b = 0; b < h->M; ++b)
      for (int a = 0; a < 2; ++a) h->g_at(np, b, a) = in[((size_t)k * h->M + b) * 2 + a];
  }
  return 0;
}

double orc_transverse_wake(double Rs, double fr, double Q, double t) {
  Resonator r{Rs, fr, Q, 0u, 0, 0, 0, 0, cplx()};
  derive(r);
  return transverse_wake(r, t);
}

void orc_betatron_map(const orc_plane *pl, double *u, double *up, double delta) { betatron_map(*pl, *u, *up, delta); }

int orc_get_window(orc_handle *h, int32_t *s_hist, int32_t *s_next) {
  if (!h) return fail(ORC_EINVAL, "null argument");
  if (s_hist) std::memcpy(s_hist, h->s_hist.data(), sizeof(int32_t) * h->M);
  if (s_next) std::memcpy(s_next, h->s_next.data(), sizeof(int32_t) * h->M);
  return 0;
}

int orc_set_window(orc_handle *h, const int32_t *s_hist, const int32_t *s_next) {
  if (!h || !s_hist || !s_next) return fail(ORC_EINVAL, "null argument");
  for (int b = 0; b < h->M; ++b)
    if (std::abs(s_hist[b]) > h->s_max || std::abs(s_next[b]) > h->s_max) return fail(ORC_EINVAL, "window shift beyond the bucket");
  std::memcpy(h->s_hist.data(), s_hist, sizeof(int32_t) * h->M);
  std::memcpy(h->s_next.data(), s_next, sizeof(int32_t) * h->M);
  bin_all(h);
  compute_moments(h);
  return 0;
}

int32_t orc_window_step(int32_t n_bins, const uint32_t *hist) { return window_step(n_bins, hist); }

int orc_get_histogram(orc_handle *h, uint32_t *out) {
  if (!h || !out) return fail(ORC_EINVAL, "null argument");
  std::memcpy(out, h->hist.data(), sizeof(uint32_t) * h->hist.size());
  return 0;
}

int orc_get_wake(orc_handle *h, double *total, double *sr, double *lr) {
  if (!h) return fail(ORC_EINVAL, "null argument");
  size_t bytes = sizeof(double) * h->V.size();
  if (total) std::memcpy(total, h->V.data(), bytes);
  if (sr) std::memcpy(sr, h->Vsr.data(), bytes);
  if (lr) std::memcpy(lr, h->Vlr.data(), bytes);
  return 0;
}

// Steps 5 and 6 of the turn just completed, evaluated for OTHER counts of that turn (hist[M][n_bins], on the current
// windows) with the history the handle holds for the turns before; nothing in the handle changes.  With the oracle's
// own counts it returns orc_get_wake()'s tables bit for bit (same code path, build_wake).  The parity tests use it when
// the CUDA path's counts differ from the oracle's by edge-adjacent particles (north_star (ii)): the wake is then
// compared on the CUDA path's own counts instead of being skipped.
int orc_wake_from_counts(orc_handle *h, const uint32_t *hist, double *total, double *sr, double *lr) {
  if (!h || !hist) return fail(ORC_EINVAL, "null argument");
  if (h->turn < 1) return fail(ORC_ESTATE, "no tracked turn");
  const size_t n = (size_t)h->M * h->nb;
  std::vector<double> vs(n), vl(n);
  build_wake(h, h->turn, hist, false, vs.data(), vl.data());
  for (size_t x = 0; x < n; ++x) {
    if (total) total[x] = vs[x] + vl[x];
    if (sr) sr[x] = vs[x];
    if (lr) lr[x] = vl[x];
  }
  return 0;
}

int orc_get_moment_log(orc_handle *h, int64_t first_turn, int64_t n, double *out) {
  if (!h || !out || first_turn < 1 || n < 0) return fail(ORC_EINVAL, "bad argument");
  if (first_turn - 1 + n > h->log_cap || first_turn - 1 + n > h->turn) return fail(ORC_ESTATE, "turns not in the log");
  std::memcpy(out, &h->log[(size_t)(first_turn - 1) * h->M * 6], sizeof(double) * (size_t)n * h->M * 6);
  return 0;
}

int orc_get_lr_history(orc_handle *h, double *out) {
  if (!h || !out) return fail(ORC_EINVAL, "null argument");
  int R = h->R(), M = h->M, K = h->K;
  for (int k = 0; k < K; ++k) {
    int64_t t = h->turn - K + 1 + k;
    for (int b = 0; b < M; ++b)
      for (int r = 0; r < R; ++r) {
        cplx a = (t >= 1) ? h->a_at(t, b, r) : cplx(0, 0);
        double *o = &out[(((size_t)k * M + b) * R + r) * 2];
        o[0] = a.real();
        o[1] = a.imag();
      }
  }
  return 0;
}

int orc_set_lr_history(orc_handle *h, const double *in) {
  if (!h || !in) return fail(ORC_EINVAL, "null argument");
  int R = h->R(), M = h->M, K = h->K;
  for (int k = 0; k < K; ++k) {
    int64_t t = h->turn - K + 1 + k;
    if (t < 1) continue;
    cplx A(0, 0);
    for (int r = 0; r < R; ++r) {
      cplx agg(0, 0);
      for (int b = 0; b < M; ++b) {
        const double *i2 = &in[(((size_t)k * M + b) * R + r) * 2];
        h->a_at(t, b, r) = cplx(i2[0], i2[1]);
        agg += h->a_at(t, b, r) * h->g_tail[(size_t)b * R + r];
      }
      h->ring_A[(size_t)(t % (K + 1)) * R + r] = agg;
    }
  }
  return 0;
}

int64_t orc_turn(const orc_handle *h) { return h ? h->turn : -1; }
double orc_phi_s(const orc_handle *h) { return h ? h->phi_s : NAN; }

}  // extern "C"
