/* orc.h -- C ABI of the CPU ORACLE of the longitudinal multi-bunch tracker.
 *
 * TEST INFRASTRUCTURE ONLY.  This is the plain, slow, single-threaded fp64
 * restatement of the per-turn method of arXiv:1809.00391 that the
 * CUDA library (include/mbt.h) is checked against.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.  It shares no code, header, table or helper with the CUDA path.
 *
 * All pointers are HOST pointers.  All arrays passed in are copied.
 * Every function returns 0 on success or a negative ORC_E* code; the text of
 * the last error is returned by orc_last_error().
 *
 * Passages followed (P:l.N = /root/reference/PAPER.md line N):
 *   P:l.63-71  Eqs.(1),(2)  energy kick and drift
 *   P:l.83-92  Eq.(5) line 1 radiation damping + quantum excitation
 *   P:l.94     list of additional harmonic cavities
 *   P:l.98-115 bins, wake on each bin, kick Eq.(6a)
 *   P:l.123-125 per-bunch mean / rms statistics
 *   P:l.229-237 HOM-driven coupled-bunch motion (long-range resonator wake)
 *   P:l.113     first / last occupied bin (read as: the bin window follows the bunch, reading D31)
 * plus the readings D1..D31 of DESIGN.md where the paper is silent.
 */
#ifndef ORC_H
#define ORC_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define ORC_EINVAL (-1)
#define ORC_ENOMEM (-2)
#define ORC_ESTATE (-3)

#define ORC_RES_SR 1u /* resonator enters the short-range table  */
#define ORC_RES_LR 2u /* resonator enters the long-range sum     */

typedef struct orc_handle orc_handle;

typedef struct { double E0_eV, T0_s, alpha_c, U0_eV; int32_t h; } orc_ring;
typedef struct { double V_volt; int32_t m; double phase_rad; } orc_cavity;
typedef struct { int32_t enable; double sigma_delta, damping_turns; } orc_radiation;
typedef struct {
  int32_t n_bunches; const int32_t *bucket; const double *charge_C;
  int64_t n_per_bunch; double sigma_tau0_s, sigma_delta0;
} orc_fill;
typedef struct { double Rs_ohm, fr_Hz, Q; uint32_t flags; } orc_resonator;
typedef struct {
  int32_t n_bins; double tau_lo_s, tau_hi_s; int32_t gather_order;
  int32_t n_res; const orc_resonator *res; int32_t history_turns;
  int32_t n_table; const double *sr_table;
  int32_t window_mode; /* 0: fixed window (reading D11); 1: window follows the bunch in whole bins (reading D31) */
} orc_wake;
/* ---- transverse planes (P:l.73-92 Eqs.(3)-(5), l.100-107 Eq.(6b); readings T1..T8) ----
 * One plane u in {x, y}: tune nu (Psi_0 = 2 pi nu), Twiss alpha, beta [m] (gamma = (1 + alpha^2) / beta),
 * chromaticity xi (Eq. 3: Psi = Psi_0 (1 + xi delta)), periodic dispersion eta [m], eta' (T2: the third column of the
 * matrix of Eq. 4 is read as the one of the periodic one-turn matrix, i.e. u - eta delta is what rotates),
 * Eq. 5: u += sigma_u sqrt(D_exc) r1, u' = u' (1 + delta) / (1 + delta + eps) + sigma_up sqrt(D_exc) r2,
 * initial distribution u = sigma0_u z, u' = sigma0_up z' (uncorrelated Gaussian, Philox tag 3). */
typedef struct { double nu, alpha, beta_m, xi, eta_m, etap, sigma_u_m, sigma_up, D_exc, sigma0_u_m, sigma0_up; } orc_plane;
/* transverse short-range wake: resonators with Rs in Ohm/m (flags ignored),
 * W_perp(t > 0) = (w_r^2 R / (Q wbar)) exp(-a t) sin(wbar t), W_perp(0) = 0 (T7); both planes use the same list */
/* long-range resistive-wall kick on the transverse planes (P:l.117-119; readings W1..W5): after
 * the wake kicks and the statistics of turn n, every particle of bunch b gets
 *   du' = (1/E0) sum_{(b',n') in H_rw(b,n)} Q_b' ubar_{b',n'} A_u / sqrt((n-n') T0 + (s_b - s_b') T_rf),
 * ubar the mean offset of ALL particles of bunch b' at the end of turn n', H_rw = the passages of the last rw_turns turns
 * (all bunches) and the earlier bunches of this turn; A_u = rw_amp_x, rw_amp_y [V s^(1/2) / (C m)]; rw_turns = 0: off */
typedef struct { int32_t enable; orc_plane x, y; int32_t n_res; const orc_resonator *res;
                 double rw_amp_x, rw_amp_y; int32_t rw_turns; } orc_transverse;

typedef struct {
  orc_ring ring; int32_t n_cav; const orc_cavity *cav; orc_radiation rad;
  orc_fill fill; orc_wake wake; uint64_t seed; int64_t log_capacity_turns;
  int32_t lr_mode; /* 0: pairwise sum (THE definition); 1: O(M+K) recurrence (long runs) */
  orc_transverse trans; /* enable = 0: longitudinal tracker only */
} orc_params;

int orc_create(const orc_params *p, orc_handle **out);
int orc_track(orc_handle *h, int64_t n_turns);
int orc_moments(orc_handle *h, double *out /* [M][6]: n_in n_out mean_tau mean_delta rms_tau rms_delta */);
int orc_destroy(orc_handle *h);
int orc_get_particles(orc_handle *h, double *tau, double *delta);
int orc_set_particles(orc_handle *h, const double *tau, const double *delta, int64_t turn);
int orc_get_histogram(orc_handle *h, uint32_t *out /* [M][n_bins] */);
int orc_get_wake(orc_handle *h, double *total, double *sr_only, double *lr_only /* each [M][n_bins] or NULL */);
/* steps 5, 6 of the turn just completed for OTHER counts hist[M][n_bins] of that turn (history of the turns before as
 * held by the handle; the handle is not changed); with the oracle's own counts: orc_get_wake()'s tables bit for bit */
int orc_wake_from_counts(orc_handle *h, const uint32_t *hist, double *total, double *sr_only, double *lr_only);
int orc_get_moment_log(orc_handle *h, int64_t first_turn, int64_t n, double *out /* [n][M][6] */);
/* source phasors a[b][n'][r] of the last K turns, oldest first: [K][M][R_lr][2] (re, im) */
int orc_get_lr_history(orc_handle *h, double *out);
int orc_set_lr_history(orc_handle *h, const double *in);
/* window shifts in bins (reading D31): s_hist[M] = window of the current histogram / wake, s_next[M] = window the
 * next turn will bin with; both 0 in window_mode 0 */
int orc_get_window(orc_handle *h, int32_t *s_hist, int32_t *s_next);
int orc_set_window(orc_handle *h, const int32_t *s_hist, const int32_t *s_next);
/* the whole-bin shift that re-centres a histogram: rint(centroid in bins - n_bins / 2), exact integer arithmetic */
int32_t orc_window_step(int32_t n_bins, const uint32_t *hist);
/* transverse state, each [M][N_p]; dipole sums S[b][k] = sum of u over the particles of bin k [m]; kick tables
 * K[b][j] = sum_{k<j} (Q_b/N_p) S[b][k] W_perp((j-k) Delta) [V]; moments out[M][8]: mean x x' y y', rms x x' y y' */
int orc_get_transverse(orc_handle *h, double *x, double *xp, double *y, double *yp);
int orc_set_transverse(orc_handle *h, const double *x, const double *xp, const double *y, const double *yp);
int orc_get_dipole(orc_handle *h, double *Sx, double *Sy);
int orc_get_transverse_wake(orc_handle *h, double *Kx, double *Ky);
int orc_moments_transverse(orc_handle *h, double *out);
double orc_transverse_wake(double Rs_ohm_per_m, double fr_Hz, double Q, double t_s);
/* resistive-wall kick of the last turn per bunch [V] (kx[M], ky[M]); source strengths Q_b ubar [C m] of the last
 * rw_turns turns, oldest first: [rw_turns][M][2] (x, y) */
/* per-turn log of the transverse statistics (P:l.123: "mean values and the RMS values ... of each bunch", turn by turn):
 * out[n][M][4] = mean x, mean y, rms x, rms y of the state at the end of turns first_turn .. first_turn+n-1 (the kicks
 * act on u' only, so these are the offsets after the turn's map and excitation); capacity = log_capacity_turns */
int orc_get_transverse_log(orc_handle *h, int64_t first_turn, int64_t n, double *out);
int orc_get_rw_kick(orc_handle *h, double *kx, double *ky);
int orc_get_rw_history(orc_handle *h, double *out);
int orc_set_rw_history(orc_handle *h, const double *in);
/* Eqs. (3), (4) for one particle of one plane (no excitation): u, u' in place */
void orc_betatron_map(const orc_plane *pl, double *u, double *up, double delta);
int64_t orc_turn(const orc_handle *h);
double orc_phi_s(const orc_handle *h);
const char *orc_last_error(void);

/* ---- unit-level entry points used by the pins (tests/) ------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* the two uniforms and the Box-Muller pair of one Philox call */
void orc_normal_pair(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                     double *u1, double *u2, double *z_c, double *z_s);
/* Excitation stream (reading D8): one Philox block -> four normals; u[4] (may be NULL) and z[4]:
 * (z[0], z[1]) = Box-Muller of the 32-bit uniforms of words (x0, x1), (z[2], z[3]) of (x2, x3). */
void orc_normal_quad(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, double *u, double *z);
double orc_resonator_wake(double Rs_ohm, double fr_Hz, double Q, double t_s);
void orc_sr_convolve(int32_t n_bins, const double *w, const double *q, double *V);
/* one application of the single-particle map (steps 1-3) without wake, z given */
void orc_map_one(const orc_handle *h, double *tau, double *delta, double z);

#ifdef __cplusplus
}
#endif
#endif
