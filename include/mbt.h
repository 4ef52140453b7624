/* mbt.h -- C ABI of the B200 (sm_100a) longitudinal multi-bunch macro-particle tracker.
 *
 * The library tracks M bunches of N_p macro-particles each through the per-turn
 * method of arXiv:1809.00391 (mbtrack / mbtrack-cuda).  Passages implemented
 * (P:l.N = PAPER.md line N; D# = reading listed in DESIGN.md):
 *
 *   S1  RF kick + synchronous loss       P:l.63-67 Eq.(1), l.94 (list of harmonic cavities)
 *   S2  radiation damping + excitation   P:l.83-92 Eq.(5) line 1     (Philox4x32-10, D8)
 *   S3  drift with the updated delta     P:l.67-71 Eq.(2)            (D1)
 *   S4  bin assignment + per-bin count   P:l.98, l.109-111           (D11)
 *   S5  short-range wake on the bins     P:l.98, l.107               (D10)
 *   S6  long-range resonator wake        P:l.229-237                 (D14)
 *   S0  wake kick  delta -= V(tau)/E0    P:l.102 Eq.(6a), l.115      (D9, D12)
 *   S7  per-bunch mean / rms             P:l.123-125                 (D22)
 * and, on a handle created with trans.enable:
 *   T   betatron map with chromaticity and dispersion   P:l.73-81 Eqs.(3), (4)     (T1-T3)
 *       transverse damping / excitation                 P:l.83-92 Eq.(5) lines 2-3 (T4, T5)
 *       per-bin dipole sums, transverse wake kick       P:l.100-111 Eq.(6b)        (T6-T8)
 *   W   long-range resistive-wall kick                  P:l.117-119                (W1-W5)
 *
 * Every step runs in CUDA kernels on the device; there is NO CPU fallback.  All
 * parameter structs are plain old data; every array passed to mbt_create is a
 * HOST pointer that is copied before the call returns (the caller keeps ownership).
 * Particle coordinates live on the device for the whole run (P:l.39) as two fp64
 * arrays tau[M][ld] and delta[M][ld], ld = mbt_particle_stride(N_p) (N_p rounded up
 * to a multiple of 4 so that every bunch starts on a 32-byte boundary).
 *
 * Every function returns 0 (MBT_OK) or a negative MBT_E* code; the text of the last
 * error of the calling thread is returned by mbt_last_error().  No exception and no
 * abort crosses this boundary.  Functions taking a handle are not thread-safe with
 * respect to the same handle.
 *
 * Observable state: mbt_track() may leave the wake kick of the last turn pending
 * (it is fused into the head of the next turn's pass); every getter and mbt_moments()
 * applies it first, so what the caller sees after mbt_track(h, n) is the state
 * "after turn n's kick", as in the sequential order of the paper (Fig. 2, P:l.47-51).
 */
#ifndef MBT_H
#define MBT_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define MBT_OK 0
#define MBT_EINVAL (-1) /* bad or inconsistent parameter                       */
#define MBT_ENOMEM (-2) /* host or device allocation failed                    */
#define MBT_ECUDA (-3)  /* a CUDA call failed; text in mbt_last_error()        */
#define MBT_ESTATE (-4) /* call not valid in the handle's current state        */

#define MBT_RES_SR 1u /* resonator enters the short-range (same bunch, same turn) table */
#define MBT_RES_LR 2u /* resonator enters the long-range (other bunches / turns) sum    */

#define MBT_MAX_CAVITIES 8   /* main + harmonic cavities (P:l.94)                 */
#define MBT_MAX_BINS 4096    /* bins per bunch                                    */
#define MBT_MAX_LR 8         /* long-range resonators                             */
#define MBT_MAX_BUNCHES 1024 /* filled buckets (the in-turn scan runs in one CTA) */

typedef struct mbt_handle mbt_handle; /* opaque, library-owned */

/* ring: reference energy [eV], revolution period [s], momentum compaction, energy loss per turn [eV],
 * harmonic number (P:l.63-71; Table 1 P:l.131-144 lists the same quantities) */
typedef struct { double E0_eV, T0_s, alpha_c, U0_eV; int32_t h; } mbt_ring;

/* one RF cavity: kick (V/E0) sin(m w_rf tau + phase).  cav[0] is the main cavity; if its phase is NaN the
 * library solves V_0 sin(phi_s) = U0 - sum_{c>0} V_c sin(phase_c) on the stable side (D3). */
typedef struct { double V_volt; int32_t m; double phase_rad; } mbt_cavity;

/* radiation (P:l.85 Eq.(5)): D_E = 2/damping_turns, noise amplitude sigma_delta sqrt(2 D_E) (D6) */
typedef struct { int32_t enable; double sigma_delta, damping_turns; } mbt_radiation;

/* fill pattern: bucket[] strictly increasing in [0,h); charge_C[b] bunch charge [C];
 * initial distribution: seeded Gaussian, tau = sigma_tau0 z_c, delta = sigma_delta0 z_s (D20) */
typedef struct {
  int32_t n_bunches; const int32_t *bucket; const double *charge_C;
  int64_t n_per_bunch; double sigma_tau0_s, sigma_delta0;
} mbt_fill;

/* resonator wake W(t>0) = 2 a Rs exp(-a t)[cos(wb t) - (a/wb) sin(wb t)], W(0) = a Rs, a = w_r/2Q (D10) */
typedef struct { double Rs_ohm, fr_Hz, Q; uint32_t flags; } mbt_resonator;

/* wake: n_bins half-open bins over [tau_lo, tau_hi) around every bucket centre (D11);
 * gather_order 1 = linear between bin centres (default), 0 = nearest grid point (P:l.98);
 * history_turns K: the long-range sum covers all bunches of turns n-K..n-1 and the earlier bunches of turn n;
 * sr_table (optional, n_table samples, V/C at lag k*Delta) is ADDED to the resonator table;
 * window_mode 0: the window is fixed (D11); 1: after each binning the window of a bunch moves by
 * rint(centroid of its counts in bins - n_bins/2) whole bins, clamped inside the bucket, and the kick of a turn uses
 * the window its wake was built on (D31; the paper's first / last occupied bin search, P:l.113, read as a window
 * that follows the bunch). */
typedef struct {
  int32_t n_bins; double tau_lo_s, tau_hi_s; int32_t gather_order;
  int32_t n_res; const mbt_resonator *res; int32_t history_turns;
  int32_t n_table; const double *sr_table;
  int32_t window_mode;
} mbt_wake;

/* ---- transverse planes (P:l.73-92 Eqs.(3)-(5), l.100-111 Eq.(6b); readings T1..T8)
 * One plane u in {x, y}: tune nu (Psi_0 = 2 pi nu), Twiss alpha, beta [m] (gamma = (1 + alpha^2) / beta), chromaticity
 * xi (Eq. 3), periodic dispersion eta [m], eta' (T2), Eq. (5): u += sigma_u sqrt(D_exc) r1,
 * u' = u' (1 + delta) / (1 + delta + eps) + sigma_up sqrt(D_exc) r2 (only with radiation enabled); initial
 * distribution u = sigma0_u z, u' = sigma0_up z'. */
typedef struct { double nu, alpha, beta_m, xi, eta_m, etap, sigma_u_m, sigma_up, D_exc, sigma0_u_m, sigma0_up; } mbt_plane;
/* transverse short-range wake of Eq. (6b): resonators with Rs in Ohm/m (flags ignored),
 * W_perp(t > 0) = (w_r^2 R / (Q wbar)) exp(-a t) sin(wbar t), W_perp(0) = 0 (T7); the same list for both planes.
 * enable = 0: longitudinal tracker only (none of the transverse entry points may then be called). */
/* Long-range resistive-wall kick on the transverse planes (P:l.117-119; DESIGN.md readings
 * W1..W5): after the wake kicks of turn n every particle of bunch b gets
 *   du' = (1/E0) sum_{(b',n')} Q_b' ubar_{b',n'} A_u / sqrt((n-n') T0 + (s_b - s_b') T_rf)
 * over the passages of the last rw_turns turns (all bunches) and the bunches ahead in this turn, ubar = the mean offset of
 * all particles of the bunch at the end of its turn; A_u = rw_amp_x, rw_amp_y [V s^(1/2) / (C m)]; rw_turns = 0: off. */
typedef struct { int32_t enable; mbt_plane x, y; int32_t n_res; const mbt_resonator *res;
                 double rw_amp_x, rw_amp_y; int32_t rw_turns; } mbt_transverse;

/* Kernel-selection knobs (measurement and test aid; they change how the path is launched, never what it computes).
 * Every member: 0 = the library's choice.  All-zero (what a zero-initialised mbt_params carries) is the production setting.
 *   tile_iters        iterations of 256 * pairs_per_thread particle pairs a pass CTA runs (> 0 fixes the tile size)
 *   pairs_per_thread  1 or 2 particle pairs advanced per thread and iteration of the longitudinal pass
 *   pdl               programmatic dependent launch: 1 off, 2 the pass only, 3 the pass and the wake kernel
 *   stages6           shared-memory stages of the 6-D pass (2..4)
 *   turn_mode         1: a turn is two launches (k_pass, k_wake); 2: one launch (the last pass CTA of a bunch builds that
 *                     bunch's wake, the last CTA of the grid closes the turn); 3: the chip-resident persistent kernel
 *                     (whole mbt_track in one cooperative launch; MBT_EINVAL if the particle store does not fit on chip)
 *   verbose           1: print the chosen launch shapes to stderr at create
 *   per_bunch_start   1: every pass CTA waits for the whole wake kernel before it (griddepcontrol.wait); 2 (= the library's
 *                     choice where one k_wake CTA serves a bunch): it waits for its own bunch's wake only, and the wake
 *                     kernel's CTA of a bunch for that bunch's pass CTAs only; 3: the former without the latter */
typedef struct {
  int32_t tile_iters, pairs_per_thread, pdl, stages6, turn_mode, verbose, per_bunch_start;
  int32_t reserved[1]; /* must be 0 */
} mbt_tuning;

/* Bunch sharding over several devices (the paper's own outlook, P:l.253: "splitting the bunches
 * among multiple GPUs").  Opt-in; the default path is one device (BASELINE north_star).  fill / bucket / charge_C describe
 * the WHOLE fill on every rank; the handle of `rank` owns the contiguous bunches mbt_shard_range() gives it (chunks of
 * ceil(n_bunches / world)): particles, counts, short-range wakes and moments of a bunch never leave its owner.  The only
 * coupling is the long-range sum: every turn each rank needs the source phasors a[b][r] of all bunches.  A turn is
 *     mbt_shard_turn_begin(h)   the pass and the first half of the wakes; this rank's rows of d_exchange are written
 *     all-gather of d_exchange  the CALLER's collective (e.g. torch.distributed.all_gather_into_tensor over NCCL, on
 *                               the handle's stream): equal chunks of ceil(n_bunches / world) * R_lr complex doubles, rank order
 *     mbt_shard_turn_end(h)     the phasor of every local bunch from the sources of ALL bunches ahead of it; turn closed
 * d_exchange: caller-owned DEVICE buffer of mbt_shard_exchange_doubles() doubles, 16-byte aligned (may be NULL without
 * long-range resonators).  Getters, setters and mbt_moments work on the rank's own bunches ([n_local][...]);
 * mbt_get / set_lr_history carry all n_bunches rows on every rank.  mbt_track returns MBT_ESTATE on a sharded handle. */
typedef struct { int32_t enable, rank, world; void *d_exchange; } mbt_shard;

typedef struct {
  mbt_ring ring;
  int32_t n_cav; const mbt_cavity *cav; /* HOST array, n_cav >= 1 */
  mbt_radiation rad;
  mbt_fill fill;
  mbt_wake wake;
  uint64_t seed;                /* Philox key (D8)                                                     */
  int64_t log_capacity_turns;   /* > 0: keep per-turn moments of turns 1..capacity on the device       */
  void *d_tau, *d_delta;        /* optional caller-owned DEVICE buffers (e.g. torch tensors), each
                                   n_bunches * mbt_particle_stride(n_per_bunch) doubles, 32-byte aligned,
                                   alive until mbt_destroy; both NULL -> the library allocates.  They are
                                   overwritten with the seeded initial distribution.                    */
  void *stream;                 /* cudaStream_t the library enqueues on (e.g. torch's current stream);
                                   NULL -> the library creates and owns a (blocking) stream             */
  int32_t device;               /* CUDA device ordinal; -1 -> the current device                        */
  mbt_transverse trans;         /* transverse planes; the library owns their four device arrays          */
  mbt_tuning tuning;            /* kernel-selection knobs; all zero = the library's choice               */
  mbt_shard shard;              /* bunch sharding over several devices; enable = 0: one device            */
} mbt_params;

/* Validates, allocates, builds the wake tables and draws the initial distribution on the device (P:l.37: the user chooses
 * the effects included -- radiation, harmonic cavities, short- and long-range wakes are each switched by a zero count or
 * flag; P:l.39: the particles then live on the GPU for the whole run; D20: seeded Gaussian start).
 * On failure *out is NULL. */
int mbt_create(const mbt_params *p, mbt_handle **out);

/* The per-turn loop of P:l.47-51 (Fig. 2) for n_turns turns: per turn S1 (P:l.63-67 Eq. 1, l.94), S2 (P:l.83-92 Eq. 5
 * line 1), S3 (P:l.67-71 Eq. 2), S4 (P:l.98, l.109-111), S5 (P:l.98, l.107), S6 (P:l.229-237), S0 (P:l.102 Eq. 6a, l.115),
 * S7 (P:l.123-125); with trans.enable also P:l.73-92 Eqs. (3)-(5), l.100-111 Eq. (6b), l.117-119.  Nothing returns to the
 * host inside the loop (the paper's host "controls the flow", P:l.39; here a CUDA graph, or one persistent kernel, does).
 * Enqueues on the handle's stream (asynchronous; the turn counter is cumulative and must stay below 2^32 because it is
 * a Philox counter word). */
int mbt_track(mbt_handle *h, int64_t n_turns);

/* P:l.123-125 ("statistical information of the bunches ... mean and standard deviation"), the longitudinal pair:
 * per-bunch statistics of the current state into HOST memory, out[M][6]:
 * n_in, n_out, mean_tau, mean_delta, rms_tau, rms_delta (population rms over all N_p particles, D22).
 * Synchronises the stream. */
int mbt_moments(mbt_handle *h, double *out);

/* Frees everything the library allocated (never the caller's d_tau / d_delta).  NULL is allowed. */
int mbt_destroy(mbt_handle *h);

/* ---- state access used by the parity tests (HOST pointers, packed [M][N_p]; each call synchronises) ---- */
/* the coordinates tau, delta of P:l.55-61 after the last tracked turn's wake kick (P:l.102 Eq. 6a) */
int mbt_get_particles(mbt_handle *h, double *tau, double *delta);
/* Upload coordinates and set the turn counter; the pending kick, the wake and the long-range history are
 * cleared (call mbt_set_lr_history AFTER this call when resuming in the middle of a run). */
int mbt_set_particles(mbt_handle *h, const double *tau, const double *delta, int64_t turn);
/* per-bin particle counts (P:l.109-111: "number of particles in each bin") of the current state, out[M][n_bins] */
int mbt_get_histogram(mbt_handle *h, uint32_t *out);
/* V(tau_j) of P:l.102-107 on the bin centres: the short-range convolution (P:l.98) and the long-range resonator sum
 * (P:l.229-237; D14) built by the last tracked turn [V]; each of total / sr_only / lr_only is
 * [M][n_bins] or NULL.  All zero before the first turn and after mbt_set_particles. */
int mbt_get_wake(mbt_handle *h, double *total, double *sr_only, double *lr_only);
/* P:l.123: the statistics "at every turn" -- kept on the device instead of copied to the host each turn: per-turn
 * statistics of turns first_turn .. first_turn+n-1 (1-based), out[n][M][6]; needs log_capacity_turns */
int mbt_get_moment_log(mbt_handle *h, int64_t first_turn, int64_t n, double *out);
/* the history the long-range sum of P:l.229-237 runs over (D14; the resonator analogue of P:l.117 "information about
 * previous bunches"): source phasors a[b][n'][r] of the last K turns, oldest first, [K][M][R_lr][2] (re, im) */
int mbt_get_lr_history(mbt_handle *h, double *out);
int mbt_set_lr_history(mbt_handle *h, const double *in);
/* P:l.113 (first / last occupied bin, read as a window that follows the bunch, D31): window shifts in bins, HOST arrays of M int32 (either may be NULL in the getter): s_hist = window of the
 * current histogram and wake, s_next = window the next turn bins with.  mbt_set_particles resets both to 0; when
 * resuming, call mbt_set_window after it (it re-bins the state; |shift| beyond the bucket -> MBT_EINVAL). */
int mbt_get_window(mbt_handle *h, int32_t *s_hist, int32_t *s_next);
int mbt_set_window(mbt_handle *h, const int32_t *s_hist, const int32_t *s_next);

/* ---- transverse planes (HOST pointers; packed [M][N_p] for coordinates, [M][n_bins] for the bin tables) ----
 * The transverse steps of a turn are fused into the 6-D pass (k_pass6: betatron map, excitation, dipole deposit, and the
 * transverse kicks of the turn before); k_wake_tr convolves the dipole sums (Eq. 6b), k_rw sums the resistive-wall
 * sources.  Like the longitudinal kick, the transverse kicks of the last tracked turn stay pending inside the library;
 * every getter applies them first, so what is observed is the state after the turn's kicks (as in the oracle).
 * All of these return MBT_EINVAL on a handle created without trans.enable.  mbt_set_transverse replaces the four
 * coordinates of every particle (the longitudinal state, the turn counter and the histories stay). */
int mbt_get_transverse(mbt_handle *h, double *x, double *xp, double *y, double *yp);
int mbt_set_transverse(mbt_handle *h, const double *x, const double *xp, const double *y, const double *yp);
/* dipole sums S[b][k] = sum of u over the particles of bin k [m] and kick tables
 * K[b][j] = sum_{k<j} (Q_b/N_p) S[b][k] W_perp((j-k) Delta) [V] of the last tracked turn (NULL entries are skipped) */
int mbt_get_dipole(mbt_handle *h, double *Sx, double *Sy);
int mbt_get_transverse_wake(mbt_handle *h, double *Kx, double *Ky);
/* per-turn log of the transverse statistics (P:l.123), kept on the device when log_capacity_turns > 0:
 * out[n][M][4] = mean x, mean y, rms x, rms y of the state at the end of turns first_turn .. first_turn+n-1 (from the
 * pass's own sums: no extra pass over the particles).  MBT_ESTATE if the turns are not in the log. */
int mbt_get_transverse_log(mbt_handle *h, int64_t first_turn, int64_t n, double *out);
/* resistive-wall kick of the last tracked turn per bunch [V] (kx[M], ky[M]; NULL entries are skipped); source strengths
 * Q_b ubar [C m] of the last rw_turns turns, oldest first: [rw_turns][M][2] (x, y) -- get / set as the long-range
 * history (set after mbt_set_particles, which fixes the turn the rows refer to) */
int mbt_get_rw_kick(mbt_handle *h, double *kx, double *ky);
int mbt_get_rw_history(mbt_handle *h, double *out);
int mbt_set_rw_history(mbt_handle *h, const double *in);
/* out[M][8]: mean x x' y y', rms x x' y y' (population), of the current state */
int mbt_moments_transverse(mbt_handle *h, double *out);

/* ---- statistics without any device allocation ----
 * P:l.123-125 (per-bunch mean and standard deviation of the coordinates), the same sums mbt_moments_transverse forms, as
 * a free-standing call on the CALLER's device arrays that never allocates.
 *
 * Who needs it.  The handle-based calls keep their partial sums in memory mbt_create took from cudaMalloc.  Two kinds of
 * caller cannot work that way: (1) a monitor that samples the beam on a second stream while mbt_track runs -- cudaMalloc
 * and cudaFree serialise against all work in flight on the device, so an allocating call would stall the very run it
 * watches; (2) a host that has given all of HBM to its own pool (a caching allocator, a run sized to the card), where a
 * cudaMalloc issued from inside a library may fail.  Here the partial sums live in a fixed array compiled into the library
 * (MBT_NOALLOC_MAX_BUNCHES * 8 doubles = 64 KiB, held by every GPU that loads libmbt.so until the process exits); the
 * call issues one memset and two kernel launches and calls neither cudaMalloc nor cudaFree nor any allocating routine.
 *
 * Arguments.  d_x, d_xp, d_y, d_yp: DEVICE arrays [n_bunches][ld] of doubles, the first n_per_bunch entries of each row
 * are summed (ld >= n_per_bunch; any four coordinate arrays will do, e.g. tau, delta twice).  d_out: DEVICE array
 * [n_bunches][8], written with mean x, x', y, y', then population rms x, x', y, y' -- the layout of
 * mbt_moments_transverse.  stream: the cudaStream_t to enqueue on (NULL = the default stream).  The call is
 * asynchronous: d_out is complete when the stream reaches that point.  All pointers belong to the device that is current
 * at the call; the caller keeps ownership of all of them.
 *
 * Limits and errors.  n_bunches > MBT_NOALLOC_MAX_BUNCHES, n_bunches < 1, n_per_bunch outside 1 .. 2^32-1, ld <
 * n_per_bunch or a NULL pointer: MBT_EINVAL, nothing enqueued, text in mbt_last_error().  CUDA failures: MBT_ECUDA.
 *
 * First call on a device.  It looks up where the fixed array sits on that device (once; later calls reuse the answer).
 * That look-up can make the CUDA runtime load the library's code onto the device, so make the first call per device
 * early, before beginning any stream capture.
 *
 * Sharing.  There is ONE array per device, shared by every call from every thread and stream, and it keeps the sums of
 * the last call.  Each call zeroes the rows it uses before accumulating, so calls that follow one another on one stream
 * are independent.  Calls that can overlap on the GPU (different streams without an ordering between them, or host
 * threads enqueueing on different streams) race on the array and give wrong statistics: order them, or keep to one stream. */
#define MBT_NOALLOC_MAX_BUNCHES 1024
int mbt_bunch_stats_noalloc(const double *d_x, const double *d_xp, const double *d_y, const double *d_yp,
                            int32_t n_bunches, int64_t n_per_bunch, int64_t ld, double *d_out, void *stream);

/* ---- introspection ---- */
int64_t mbt_turn(const mbt_handle *h);        /* completed turns, -1 on NULL                 */
double mbt_phi_s(const mbt_handle *h);        /* synchronous phase of cav[0] [rad]           */
int64_t mbt_particle_stride(int64_t n_per_bunch); /* ld of the device arrays                 */
/* The tiling a pass would get (host logic only, no device needed): a bunch of pairs_per_bunch particle pairs, CTAs that
 * advance `stride` pairs per iteration, M bunches, `slots` CTAs resident on the device at once.  Even tiles (the last
 * at least 3/4 of the others) and, among those, the count that minimises ceil(w)/w (1 + 1/iterations), w = tiles M /
 * slots; tile_iters > 0 fixes the iterations per tile instead (mbt_tuning.tile_iters).  Writes pairs per tile and tiles
 * per bunch; MBT_EINVAL on non-positive arguments. */
int mbt_plan_tiles(int64_t pairs_per_bunch, int64_t stride, int32_t M, int32_t slots, int32_t tile_iters,
                   uint32_t *tile_pairs, int32_t *tiles);
/* DEVICE pointers of the particle store (for zero-copy wrapping, e.g. torch.from_blob-like views); applies a pending kick
 * first.  The library cannot see writes through these pointers (or into caller-owned d_tau / d_delta): after changing
 * coordinates in place call mbt_invalidate(), else mbt_moments / mbt_get_histogram return the statistics of the state the
 * library last closed.  (In-place writes never touch the wake, the history or the turn counter.) */
int mbt_device_pointers(mbt_handle *h, void **d_tau, void **d_delta, int64_t *ld);
/* ---- bunch sharding (mbt_shard above); the first two are host-only ---- */
/* the bunches rank owns: first index and count (count may be 0 for the last ranks; mbt_create refuses such a rank) */
int mbt_shard_range(int32_t n_bunches, int32_t world, int32_t rank, int32_t *first, int32_t *count);
/* doubles in the exchange buffer: world * ceil(n_bunches / world) * n_lr * 2; -1 on bad arguments */
int64_t mbt_shard_exchange_doubles(int32_t n_bunches, int32_t world, int32_t n_lr);
int mbt_shard_turn_begin(mbt_handle *h);
int mbt_shard_turn_end(mbt_handle *h);
/* The particle store was modified behind the library's back: the next getter re-derives counts and moments from memory. */
int mbt_invalidate(mbt_handle *h);
/* kernels launched by this handle so far (bench.py's gpu_launches) */
int64_t mbt_launch_count(const mbt_handle *h);
/* kernel launches per tracked turn of this handle: 1 (one-launch turn), 2 (k_pass, k_wake), 3 / 4 with the transverse
 * planes (+ k_wake_tr, + k_rw); a sharded handle: 3, or 4 with long-range resonators (mbt_shard_turn_begin: pass, first half
 * of the wakes; mbt_shard_turn_end: scatter of the gathered sources, second half); 0 for the chip-resident turn loop (one
 * launch per mbt_track call); -1 on NULL */
int mbt_launches_per_turn(const mbt_handle *h);
/* Seconds of device time of the most recent mbt_track call, measured with CUDA events recorded on the handle's
 * stream around the enqueued turns; synchronises.  Negative on error. */
double mbt_last_track_seconds(mbt_handle *h);
/* Measurement aid: tracks n_turns (1..65536) turns with plain launches instead of graph replay and brackets
 * every kernel with CUDA events on the handle's stream; returns the summed device time [s] of the fused
 * particle pass and of the wake kernel.  The turns are real turns (state and turn counter advance).
 * Synchronises. */
int mbt_track_profiled(mbt_handle *h, int64_t n_turns, double *pass_seconds, double *wake_seconds);
/* Run one Philox4x32-10 block on the device (known-answer tests of the device generator). */
int mbt_philox_selftest(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* Device normals exactly as the excitation step draws them (reading D8: one Philox block serves four consecutive
 * particles): HOST arrays of n counters (c0,c1,c2,c3) in ctr[n][4]; out[n][4]: (out[0], out[1]) = Box-Muller pair of
 * the 32-bit uniforms of words (x0, x1), (out[2], out[3]) that of (x2, x3). */
int mbt_normal_selftest(uint64_t seed, int64_t n, const uint32_t *ctr, double *out);
const char *mbt_last_error(void); /* thread-local, never NULL */
const char *mbt_version(void);

#ifdef __cplusplus
}
#endif
#endif
