// mbt.cu -- host side of the C ABI declared in include/mbt.h: validation, table construction,
// device memory, per-turn sequencing (CUDA graph replay of {k_pass, k_wake}) and the getters.
// No step of the method runs on the host: the host only derives constants and tables at create time.
#include "../../include/mbt.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "mbt_kernels.cuh"
#include "mbt_trans.cuh"
#include "mbt_resident.cuh"

using namespace mbt;

namespace {

thread_local std::string g_err;

// mbt_tuning.turn_mode 0 (the library's choice) is always two launches per turn.  The one-launch turn (turn_mode 2) and the
// chip-resident turn loop (turn_mode 3) are complete and parity-tested, but measured slower on every BASELINE workload
// (DESIGN.md sections 7.5, 7.6; e.g. c4: 0.238 vs 0.218 ms per turn), so neither is ever picked automatically.

int fail(int code, const std::string &msg) {
  g_err = msg;
  return code;
}

#define CU(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      char buf_[512];                                                                              \
      snprintf(buf_, sizeof buf_, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
      return fail(e_ == cudaErrorMemoryAllocation ? MBT_ENOMEM : MBT_ECUDA, buf_);                 \
    }                                                                                              \
  } while (0)

typedef long double ldbl;
const ldbl PI_L = 3.141592653589793238462643383279502884L;
const double PI_D = 3.14159265358979323846;

struct Res {
  double Rs, fr, Q;
  ldbl alpha, wbar;  // alpha = w_r / 2Q, wbar = sqrt(w_r^2 - alpha^2)     (D10)
};

Res make_res(const mbt_resonator &in) {
  Res r{in.Rs_ohm, in.fr_Hz, in.Q, 0, 0};
  const ldbl wr = 2.0L * PI_L * (ldbl)in.fr_Hz;
  r.alpha = wr / (2.0L * (ldbl)in.Q);
  r.wbar = sqrtl(wr * wr - r.alpha * r.alpha);
  return r;
}

// W(t) [V/C], W(0) = alpha Rs, W(t<0) = 0
double res_wake(const Res &r, ldbl t) {
  if (t < 0) return 0.0;
  if (t == 0) return (double)(r.alpha * (ldbl)r.Rs);
  return (double)(2.0L * r.alpha * (ldbl)r.Rs * expl(-r.alpha * t) * (cosl(r.wbar * t) - (r.alpha / r.wbar) * sinl(r.wbar * t)));
}

// exp(sign * lambda * t), lambda = -alpha + i wbar, evaluated in extended precision (phases reach 1e6 rad)
cplx exp_lambda(const Res &r, ldbl t) {
  const ldbl mag = expl(-r.alpha * t), ph = r.wbar * t;
  return cplx{(double)(mag * cosl(ph)), (double)(mag * sinl(ph))};
}

// Device buffer.  Zero-filling and uploads are enqueued on the HANDLE's stream -- the stream every kernel and copy of the
// handle runs on -- so that they are ordered against them also when the caller's stream is a non-blocking one (the legacy
// default stream, which cudaMemset / cudaMemcpy use, is not ordered against such streams).  cudaMemcpyAsync from pageable
// host memory returns once the source has been staged, so the host vector may go out of scope after the call.
template <class T>
struct DevBuf {
  T *p = nullptr;
  size_t n = 0;
  cudaError_t alloc(size_t count, cudaStream_t st) {
    n = count;
    if (count == 0) count = 1;
    cudaError_t e = cudaMalloc((void **)&p, count * sizeof(T));
    if (e == cudaSuccess) e = cudaMemsetAsync(p, 0, count * sizeof(T), st);
    return e;
  }
  cudaError_t upload(const std::vector<T> &v, cudaStream_t st) {
    cudaError_t e = alloc(v.size(), st);
    if (e == cudaSuccess && !v.empty()) e = cudaMemcpyAsync(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st);
    return e;
  }
  void release() {
    if (p) cudaFree(p);
    p = nullptr;
  }
};

}  // namespace

struct mbt_handle {
  int device = 0;
  cudaStream_t stream = nullptr;
  bool own_stream = false;
  int Mg = 0, b0 = 0;        // bunches of the whole fill, global index of this handle's first one (Mg = M, b0 = 0 unless sharded)
  bool sharded = false;
  int shard_rank = 0, shard_world = 1, shard_chunk = 0;
  int shard_phase = 0;       // 0: between turns; 1: mbt_shard_turn_begin done, the exchange is the caller's move
  cplx *xbuf = nullptr;      // caller-owned exchange buffer [world * chunk][R]
  int M = 0, nb = 0, R = 0, K = 0, slots = 2;  // slots of the long-range rings: K + 1, at least 2
  int64_t Np = 0, ld = 0;
  bool own_particles = false;
  double *d_tau = nullptr, *d_delta = nullptr;
  double phi_s = 0.0;
  int64_t turn = 0;        // host mirror of ctrl.turn
  bool dirty = true;       // observable quantities (pending kick, moments, counts) need a flush
  bool pointers_out = false;  // mbt_device_pointers has handed the store out: in-place writes are possible from now on
  bool wake_valid = false; // a tracked turn has built a wake since create / set_particles
  int64_t launches = 0;
  int64_t log_cap = 0;
  int grid_pass = 0;
  size_t smem_pass = 0, smem_wake = 0;
  Args args;
  WakeArgs wargs;
  DevBuf<double> qm, w, Vsr, mom_acc, mom_last, mom_log, scratch_a, scratch_b, scratch_c;
  DevBuf<WakeCell> cellSR;
  DevBuf<CellF> cellF;
  DevBuf<cplx> Esrc, F, g_step, g_tail, g_hist, a_cur, ring_a, ring_A, P;
  DevBuf<uint32_t> hist, hist_last;
  DevBuf<unsigned long long> nout_acc;
  DevBuf<int32_t> s_hist, s_next;
  DevBuf<uint32_t> rd_cnt, wr_cnt;
  // transverse planes (mbt_trans.cuh); empty unless trans
  bool trans = false;
  Args6 args6;
  TWakeArgs twargs;
  TMomArgs tmargs;
  int grid_tr = 0, grid_pass6 = 0, fix_bits = kFixBitsMax;
  size_t smem_pass6 = 0;
  void (*fn_map6)(const Args6) = nullptr;    // k_pass6<true, ...>
  void (*fn_flush6)(const Args6) = nullptr;  // k_pass6<false, ...>
  DevBuf<double> tx, txp, ty, typ, wt, Sov, S_last, Ktab, acc2, mom_tr_acc, mom_tr;
  DevBuf<unsigned long long> Sfix;
  DevBuf<FixScale> fix;
  DevBuf<WakeCell> cellX, cellY;
  int Krw = 0;                 // resistive-wall history depth (0: off)
  RwArgs rwargs;
  DevBuf<double> ring_g, rw, wrw, log_tr;
  DevBuf<int32_t> d_bucket;
  DevBuf<uint32_t> turn_tr;
  cudaStream_t stream2 = nullptr;          // side stream: k_wake_tr and k_rw run beside k_wake (fork / join by events)
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  int wake_splits = 1;
  DevBuf<double> lo_hist, lo_next;
  DevBuf<cplx> shift_src, shift_wit;
  int window_mode = 0;
  int32_t s_max = 0;
  double tau_lo = 0.0, Delta = 0.0;
  DevBuf<Ctrl> ctrl;
  void (*fn_map)(const Args, const WakeArgs) = nullptr;    // k_pass<true, ...> chosen for this handle's effects
  void (*fn_flush)(const Args, const WakeArgs) = nullptr;  // k_pass<false, ...>
  // chip-resident turn loop (mbt_resident.cuh): one cooperative launch per mbt_track call
  bool resident = false;
  void (*fn_res)(const Args, const WakeArgs, const ResArgs) = nullptr;
  ResArgs rargs;
  WakeArgs wargs_res;
  size_t smem_res = 0;
  int grid_res = 0;
  DevBuf<uint32_t> res_bar;
  bool fused = false;  // a turn is ONE launch: the pass's last CTA of a bunch builds the bunch's wake (mbt_tuning.turn_mode 2)
  DevBuf<uint32_t> bunch_done;
  DevBuf<uint32_t> a_ready, bunch_ready, agg_ready, tile_turn, tr_ready, rw_ready;
  size_t smem_wake6 = 0;
  DevBuf<uint32_t> bunch_done_tr;
  bool pipe6 = false;  // 6-D turn as one chain of programmatic dependents with per-bunch flags
  DevBuf<cplx> gd;
  int npair = 1;
  int pdl = 1;  // bit 0: the pass, bit 1: k_wake launched as a programmatic dependent (longitudinal handles; mbt_tuning.pdl sets it).
                // Measured, us per turn, graph replay: pass only c1 10.8 -> 10.0, c3 16.6 -> 16.0, c4 223.9 -> 222.8; k_wake as
                // well helps c1 (9.1) but costs c2 and c3 (26.8, 19.3): its resident CTAs are in the way of the pass's tail
  DevBuf<LogTabEntry> logtab;
  // captured graphs of 1, 2, 4, ... 64 turns, built on demand: a run is replayed largest first.  Inside a graph the kernels
  // are chained as programmatic dependents; BETWEEN two graph launches the dependency is a full one (the wake kernel's
  // latency is exposed there), so few, long graphs: 300 turns are 4 x 64 + 32 + 8 + 4 (7 boundaries, where graphs of 16
  // and single turns made 30).
  static constexpr int kGraphLevels = 7;
  cudaGraphExec_t graphs[kGraphLevels] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  bool timed = false;
};

namespace {

// ---- the instantiations of the fused pass and their selection at create time
typedef void (*pass_fn)(const Args, const WakeArgs);

template <int NPAIR>
pass_fn select_map(bool rad, int gather, int n_cav) {
#define MBT_SEL_(R, G)                                                    \
  (n_cav == 1 ? (pass_fn)k_pass<true, R, G, 1, NPAIR>                      \
              : n_cav == 2 ? (pass_fn)k_pass<true, R, G, 2, NPAIR> : (pass_fn)k_pass<true, R, G, 0, NPAIR>)
  if (rad) return gather ? MBT_SEL_(true, 1) : MBT_SEL_(true, 0);
  return gather ? MBT_SEL_(false, 1) : MBT_SEL_(false, 0);
#undef MBT_SEL_
}
template <int NPAIR>
pass_fn select_flush(int gather) {
  return gather ? (pass_fn)k_pass<false, false, 1, 0, NPAIR> : (pass_fn)k_pass<false, false, 0, 0, NPAIR>;
}

// Tiles of a pass: pairs per CTA (a multiple of `stride`, the pairs a CTA advances per iteration) and tiles per bunch.
// Large workloads: the grid runs in waves of `slots` resident CTAs, and what a launch costs beyond its traffic is the
// last, partly filled wave and the per-CTA prologue (gather cells, barriers) and epilogue (count flush).  Measured at c4
// (k_pass: 7 ragged tiles of 16 iterations -> 4 even tiles of 25: 0.2063 -> 0.1958 ms; 3, 5, 6, 7 even tiles 0.199 ..
// 0.204; k_pass6: 13 ragged tiles of 16 -> 4 even tiles of 49: 0.864 -> 0.832 ms, 22 tiles of 9: 0.879).  So: even tiles
// (the last one at least 3/4 of the others) and among those the tile count that minimises
// ceil(w) / w (1 + 1 / iterations), w = tiles M / slots the number of waves, one iteration's worth of per-CTA work.
// The same rule serves the small workloads, where it settles just under one wave (c2, one bunch of 1e6: 391 CTAs of
// 5 iterations instead of 977 of 2: pass 23.7 -> 18.6 us).  tile_iters > 0 (mbt_tuning.tile_iters) fixes the iterations.
void choose_tiles(int64_t ppb, int64_t stride, int M, int slots, int tile_iters, bool verbose, uint32_t *tile_pairs, int *tiles) {
  const int64_t total = (ppb + stride - 1) / stride;  // iterations per bunch
  int64_t iters = tile_iters > 0 ? tile_iters : 0;
  if (iters == 0) {
    double best = 1.0e30;
    for (int64_t n = 1; n <= total; ++n) {
      const int64_t it = (total + n - 1) / n;
      const int64_t n_eff = (total + it - 1) / it, last = total - (n_eff - 1) * it;
      if (n_eff != n) continue;  // the same tiling as a smaller n
      if (n_eff > 1 && 4 * last < 3 * it) continue;
      const double w = (double)(n_eff * M) / (double)slots, cost = std::ceil(w) / w * (1.0 + 1.0 / (double)it);
      if (cost < best) { best = cost; iters = it; }
    }
  }
  if (iters == 0) {
    iters = 16;
    while (iters > 1 && (int64_t)M * ((ppb + iters * stride - 1) / (iters * stride)) < 2ll * slots) iters /= 2;
  }
  *tile_pairs = (uint32_t)(iters * stride);
  *tiles = (int)((ppb + iters * stride - 1) / (iters * stride));
  if (verbose)
    fprintf(stderr, "mbt: choose_tiles ppb %lld stride %lld M %d slots %d -> %lld iterations, %d tiles\n", (long long)ppb,
            (long long)stride, M, slots, (long long)iters, *tiles);
}

typedef void (*res_fn)(const Args, const WakeArgs, const ResArgs);
res_fn select_resident(bool rad, int gather, int n_cav) {
#define MBT_SEL_(R, G) (n_cav == 1 ? (res_fn)k_resident<R, G, 1> : n_cav == 2 ? (res_fn)k_resident<R, G, 2> : (res_fn)k_resident<R, G, 0>)
  if (rad) return gather ? MBT_SEL_(true, 1) : MBT_SEL_(true, 0);
  return gather ? MBT_SEL_(false, 1) : MBT_SEL_(false, 0);
#undef MBT_SEL_
}

typedef void (*pass6_fn)(const Args6);
pass6_fn select_map6(bool rad, int gather, int n_cav) {
#define MBT_SEL_(R, G)                                             \
  (n_cav == 1 ? (pass6_fn)k_pass6<true, R, G, 1>                    \
              : n_cav == 2 ? (pass6_fn)k_pass6<true, R, G, 2> : (pass6_fn)k_pass6<true, R, G, 0>)
  if (rad) return gather ? MBT_SEL_(true, 1) : MBT_SEL_(true, 0);
  return gather ? MBT_SEL_(false, 1) : MBT_SEL_(false, 0);
#undef MBT_SEL_
}
pass6_fn select_flush6(int gather) { return gather ? (pass6_fn)k_pass6<false, false, 1, 0> : (pass6_fn)k_pass6<false, false, 0, 0>; }

// launch as a programmatic dependent of the kernel before it on the stream (mbt_kernels.cuh, griddepcontrol)
template <typename... KArgs, typename... Vals>
cudaError_t launch_dependent(void (*fn)(KArgs...), dim3 grid, int threads, size_t smem, cudaStream_t st, const Vals &...a) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(threads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, fn, a...);
}

// the pass of a tracked turn: the longitudinal one, or the fused 6-D one of a handle with the transverse planes.
// Every enqueue_* returns the first launch error (a bad configuration shows up here, not at a later synchronise).
cudaError_t enqueue_pass(mbt_handle *h) {
  if (h->trans) {
    if (h->pipe6) return launch_dependent(h->fn_map6, dim3(h->grid_pass6, h->M), kPassThreads, h->smem_pass6, h->stream, h->args6);
    h->fn_map6<<<dim3(h->grid_pass6, h->M), kPassThreads, h->smem_pass6, h->stream>>>(h->args6);
    return cudaGetLastError();
  }
  if (h->pdl & 1)
    return launch_dependent(h->fn_map, dim3(h->grid_pass, h->M), kPassThreads, h->smem_pass, h->stream, h->args, h->wargs);
  h->fn_map<<<dim3(h->grid_pass, h->M), kPassThreads, h->smem_pass, h->stream>>>(h->args, h->wargs);
  return cudaGetLastError();
}
// the wake kernels of a turn: k_wake on the handle's stream; the transverse ones (independent of it: they read what the
// pass wrote, and the next pass waits for both) on the side stream.  Under stream capture this becomes a fork and a join
// in the graph.  In the one-launch turn there is nothing to enqueue: the pass has built the wakes.
cudaError_t enqueue_wakes(mbt_handle *h) {
  if (h->fused) return cudaSuccess;
  cudaError_t e = cudaSuccess;
#define MBT_E_(call) do { if (e == cudaSuccess) e = (call); } while (0)
  if (h->pipe6) {  // one stream, every kernel a programmatic dependent of the one before; per-bunch flags order the data
    MBT_E_(launch_dependent(k_wake6, dim3(h->M, 2), kWakeThreads, h->smem_wake6, h->stream, h->wargs, h->twargs));
    if (h->Krw > 0) MBT_E_(launch_dependent(k_rw, dim3(h->M), 256, (size_t)0, h->stream, h->rwargs));
    return e;
  }
  if (h->trans) {
    MBT_E_(cudaEventRecord(h->ev_fork, h->stream));
    MBT_E_(cudaStreamWaitEvent(h->stream2, h->ev_fork, 0));
    k_wake_tr<<<h->M, 256, wake_tr_smem_bytes(h->nb), h->stream2>>>(h->twargs);
    MBT_E_(cudaGetLastError());
    if (h->Krw > 0) {
      k_rw<<<h->M, 256, 0, h->stream2>>>(h->rwargs);
      MBT_E_(cudaGetLastError());
    }
    MBT_E_(cudaEventRecord(h->ev_join, h->stream2));
  }
  if ((h->pdl & 2) && !h->trans) {
    MBT_E_(launch_dependent(k_wake, dim3(h->M, h->wake_splits), kWakeThreads, h->smem_wake, h->stream, h->wargs));
  } else {
    k_wake<<<dim3(h->M, h->wake_splits), kWakeThreads, h->smem_wake, h->stream>>>(h->wargs);
    MBT_E_(cudaGetLastError());
  }
  if (h->trans) MBT_E_(cudaStreamWaitEvent(h->stream, h->ev_join, 0));
#undef MBT_E_
  return e;
}
// launches per tracked turn: 1 in the one-launch turn, else 2; 3 with the transverse planes; 4 with their resistive-wall kick;
// a sharded handle: pass, first half of the wakes, (with long-range resonators) the scatter of the gathered sources, second half
int launches_per_turn(const mbt_handle *h) {
  if (h->sharded) return h->R > 0 ? 4 : 3;
  return h->resident ? 0 : h->fused ? 1 : h->trans ? (h->pipe6 ? (h->Krw > 0 ? 3 : 2) : (h->Krw > 0 ? 4 : 3)) : 2;
}

cudaError_t enqueue_turn(mbt_handle *h) {
  cudaError_t e = enqueue_pass(h);
  return e == cudaSuccess ? enqueue_wakes(h) : e;
}

// scale of the fixed-point dipole sums from the transverse state in memory
int rescale_transverse(mbt_handle *h) {
  CU(cudaMemsetAsync(h->mom_tr_acc.p, 0, sizeof(double) * h->M * 8, h->stream));
  k_moments_tr<<<dim3(h->grid_tr, h->M), 256, 0, h->stream>>>(h->tmargs, h->mom_tr_acc.p);
  k_fix_scale<<<(2 * h->M + 127) / 128, 128, 0, h->stream>>>(h->M, (uint32_t)h->Np, h->fix_bits, h->mom_tr_acc.p, h->fix.p);
  h->launches += 2;
  CU(cudaGetLastError());
  return 0;
}

int build_graph(mbt_handle *h, int turns, cudaGraphExec_t *out) {
  cudaGraph_t g = nullptr;
  CU(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
  cudaError_t le = cudaSuccess;
  for (int t = 0; t < turns && le == cudaSuccess; ++t) le = enqueue_turn(h);
  cudaError_t ce = cudaStreamEndCapture(h->stream, &g);  // always end the capture, also after a failed launch
  if (le != cudaSuccess || ce != cudaSuccess) {
    if (g) cudaGraphDestroy(g);
    cudaGetLastError();
    return fail(MBT_ECUDA, std::string("capturing a turn failed: ") + cudaGetErrorString(le != cudaSuccess ? le : ce));
  }
  cudaError_t e = cudaGraphInstantiate(out, g, 0);
  cudaGraphDestroy(g);
  CU(e);
  return 0;
}

// apply the pending kick, close moments and counts of the current state
int flush(mbt_handle *h) {
  if (!h->dirty) return 0;
  CU(cudaSetDevice(h->device));
  WakeArgs wa = h->wargs;
  wa.mode = 1;
  wa.S = 1;
  wa.bunch_wait = 0;
  if (h->trans) h->fn_flush6<<<dim3(h->grid_pass6, h->M), kPassThreads, h->smem_pass6, h->stream>>>(h->args6);
  else h->fn_flush<<<dim3(h->grid_pass, h->M), kPassThreads, h->smem_pass, h->stream>>>(h->args, wa);
  CU(cudaGetLastError());
  k_wake<<<h->M, kWakeThreads, h->smem_wake, h->stream>>>(wa);
  CU(cudaGetLastError());
  k_clear_pending<<<1, 1, 0, h->stream>>>(h->ctrl.p);
  CU(cudaGetLastError());
  h->launches += 3;
  // a handle on caller-owned buffers stays dirty: the caller may write the coordinates in place at any time (mbt.h)
  h->dirty = !h->own_particles || h->pointers_out;
  return 0;
}

void destroy(mbt_handle *h) {
  if (!h) return;
  cudaSetDevice(h->device);
  if (h->stream) cudaStreamSynchronize(h->stream);
  for (cudaGraphExec_t g : h->graphs)
    if (g) cudaGraphExecDestroy(g);
  if (h->stream2) { cudaStreamSynchronize(h->stream2); cudaStreamDestroy(h->stream2); }
  if (h->ev_fork) cudaEventDestroy(h->ev_fork);
  if (h->ev_join) cudaEventDestroy(h->ev_join);
  if (h->ev0) cudaEventDestroy(h->ev0);
  if (h->ev1) cudaEventDestroy(h->ev1);
  if (h->own_particles) {
    if (h->d_tau) cudaFree(h->d_tau);
    if (h->d_delta) cudaFree(h->d_delta);
  }
  h->qm.release(); h->w.release(); h->Vsr.release(); h->mom_acc.release(); h->mom_last.release(); h->mom_log.release();
  h->scratch_a.release(); h->scratch_b.release(); h->scratch_c.release();
  h->cellSR.release(); h->cellF.release();
  h->rd_cnt.release(); h->wr_cnt.release(); h->bunch_done.release();
  h->a_ready.release(); h->bunch_ready.release(); h->agg_ready.release(); h->gd.release(); h->tile_turn.release(); h->res_bar.release(); h->tr_ready.release(); h->rw_ready.release(); h->bunch_done_tr.release();
  h->tx.release(); h->txp.release(); h->ty.release(); h->typ.release(); h->wt.release(); h->Sfix.release(); h->Sov.release();
  h->S_last.release(); h->Ktab.release(); h->acc2.release(); h->fix.release(); h->cellX.release(); h->cellY.release();
  h->mom_tr_acc.release(); h->mom_tr.release();
  h->ring_g.release(); h->rw.release(); h->wrw.release(); h->d_bucket.release(); h->log_tr.release(); h->turn_tr.release();
  h->s_hist.release(); h->s_next.release(); h->lo_hist.release(); h->lo_next.release();
  h->shift_src.release(); h->shift_wit.release();
  h->Esrc.release(); h->F.release(); h->g_step.release(); h->g_tail.release(); h->g_hist.release(); h->a_cur.release();
  h->ring_a.release(); h->ring_A.release(); h->P.release(); h->logtab.release();
  h->hist.release(); h->hist_last.release(); h->nout_acc.release(); h->ctrl.release();
  if (h->own_stream && h->stream) cudaStreamDestroy(h->stream);
  delete h;
}

}  // namespace

namespace {
int upload_window(mbt_handle *h, const int32_t *s_hist, const int32_t *s_next) {
  std::vector<double> lh(h->M), ln(h->M);
  for (int b = 0; b < h->M; ++b) {
    double off_h = (double)s_hist[b] * h->Delta, off_n = (double)s_next[b] * h->Delta;
    lh[b] = h->tau_lo + off_h;
    ln[b] = h->tau_lo + off_n;
    if (lh[b] == 0.0) lh[b] = -0.0;
    if (ln[b] == 0.0) ln[b] = -0.0;
  }
  CU(cudaMemcpyAsync(h->s_hist.p, s_hist, sizeof(int32_t) * h->M, cudaMemcpyHostToDevice, h->stream));
  CU(cudaMemcpyAsync(h->s_next.p, s_next, sizeof(int32_t) * h->M, cudaMemcpyHostToDevice, h->stream));
  CU(cudaMemcpyAsync(h->lo_hist.p, lh.data(), sizeof(double) * h->M, cudaMemcpyHostToDevice, h->stream));
  CU(cudaMemcpyAsync(h->lo_next.p, ln.data(), sizeof(double) * h->M, cudaMemcpyHostToDevice, h->stream));
  CU(cudaStreamSynchronize(h->stream));  // the host vectors go out of scope
  return 0;
}
}  // namespace

namespace {
// the chip-resident turn loop: one cooperative launch per (at most 2^20) turns
int track_resident(mbt_handle *h, int64_t n_turns) {
  CU(cudaEventRecord(h->ev0, h->stream));
  int64_t left = n_turns;
  while (left > 0) {
    const int64_t chunk = std::min<int64_t>(left, 1 << 20);
    CU(cudaMemsetAsync(h->res_bar.p, 0, 2 * sizeof(uint32_t), h->stream));
    ResArgs ra = h->rargs;
    ra.n_turns = (int32_t)chunk;
    void *args[3] = {(void *)&h->args, (void *)&h->wargs_res, (void *)&ra};
    CU(cudaLaunchCooperativeKernel((const void *)h->fn_res, dim3(h->grid_res), dim3(kPassThreads), args, h->smem_res, h->stream));
    left -= chunk;
    h->launches += 1;
  }
  k_sync_flags<<<1, 256, 0, h->stream>>>(h->ctrl.p, h->a_ready.p, h->Mg * (h->R ? h->R : 1), h->bunch_ready.p, h->M, h->agg_ready.p,
                                         h->tile_turn.p, (int)h->tile_turn.n);
  CU(cudaGetLastError());
  h->launches += 1;
  CU(cudaEventRecord(h->ev1, h->stream));
  h->timed = true;
  h->turn += n_turns;
  h->dirty = true;
  h->wake_valid = true;
  return 0;
}
}  // namespace

extern "C" {

const char *mbt_last_error(void) { return g_err.c_str(); }
const char *mbt_version(void) { return "mbt-b200 0.1 (sm_100a)"; }
int64_t mbt_particle_stride(int64_t n) { return n < 0 ? -1 : (n + 3) / 4 * 4; }
int mbt_plan_tiles(int64_t ppb, int64_t stride, int32_t M, int32_t slots, int32_t tile_iters, uint32_t *tile_pairs,
                   int32_t *tiles) {
  if (ppb < 1 || stride < 1 || M < 1 || slots < 1 || tile_iters < 0 || !tile_pairs || !tiles) return fail(MBT_EINVAL, "bad argument");
  int n = 0;
  choose_tiles(ppb, stride, M, slots, tile_iters, false, tile_pairs, &n);
  *tiles = n;
  return 0;
}
int64_t mbt_turn(const mbt_handle *h) { return h ? h->turn : -1; }
double mbt_phi_s(const mbt_handle *h) { return h ? h->phi_s : NAN; }
int64_t mbt_launch_count(const mbt_handle *h) { return h ? h->launches : -1; }
int mbt_launches_per_turn(const mbt_handle *h) { return h ? launches_per_turn(h) : -1; }

int mbt_create(const mbt_params *p, mbt_handle **out) {
  if (!p || !out) return fail(MBT_EINVAL, "null argument");
  *out = nullptr;
  const mbt_ring &rg = p->ring;
  if (!(rg.E0_eV > 0) || !(rg.T0_s > 0) || rg.h < 1 || !std::isfinite(rg.alpha_c) || rg.alpha_c == 0.0 ||
      !std::isfinite(rg.U0_eV))
    return fail(MBT_EINVAL, "ring: need E0 > 0, T0 > 0, h >= 1, alpha_c != 0");
  if (p->n_cav < 1 || p->n_cav > MBT_MAX_CAVITIES || !p->cav)
    return fail(MBT_EINVAL, "need 1..MBT_MAX_CAVITIES cavities, cav[0] the main one");
  const mbt_fill &fl = p->fill;
  if (fl.n_bunches < 1 || fl.n_bunches > MBT_MAX_BUNCHES || !fl.bucket || !fl.charge_C)
    return fail(MBT_EINVAL, "fill: need 1 <= n_bunches <= MBT_MAX_BUNCHES and bucket / charge arrays");
  if (fl.n_per_bunch < 1 || fl.n_per_bunch > 0x7FFFFFFEll) return fail(MBT_EINVAL, "fill: need 1 <= n_per_bunch < 2^31 - 1");
  for (int b = 0; b < fl.n_bunches; ++b) {
    if (fl.bucket[b] < 0 || fl.bucket[b] >= rg.h) return fail(MBT_EINVAL, "bucket out of [0,h)");
    if (b > 0 && fl.bucket[b] <= fl.bucket[b - 1]) return fail(MBT_EINVAL, "buckets not strictly increasing");
    if (!std::isfinite(fl.charge_C[b])) return fail(MBT_EINVAL, "charge not finite");
  }
  if (!(fl.sigma_tau0_s >= 0) || !(fl.sigma_delta0 >= 0)) return fail(MBT_EINVAL, "initial sigmas must be >= 0");
  const mbt_wake &wk = p->wake;
  if (wk.n_bins < 2 || wk.n_bins > MBT_MAX_BINS) return fail(MBT_EINVAL, "need 2 <= n_bins <= MBT_MAX_BINS");
  if (!(wk.tau_hi_s > wk.tau_lo_s) || !((wk.tau_hi_s - wk.tau_lo_s) < rg.T0_s / rg.h))
    return fail(MBT_EINVAL, "window must satisfy 0 < tau_hi - tau_lo < T_rf");
  if (wk.gather_order != 0 && wk.gather_order != 1) return fail(MBT_EINVAL, "gather_order must be 0 or 1");
  if (wk.window_mode != 0 && wk.window_mode != 1) return fail(MBT_EINVAL, "window_mode must be 0 or 1");
  if (wk.n_res < 0 || (wk.n_res > 0 && !wk.res)) return fail(MBT_EINVAL, "resonator list");
  if (wk.n_table < 0 || (wk.n_table > 0 && !wk.sr_table)) return fail(MBT_EINVAL, "sr_table");
  if (p->rad.enable && (!(p->rad.damping_turns > 0) || !(p->rad.sigma_delta >= 0)))
    return fail(MBT_EINVAL, "radiation: need damping_turns > 0, sigma_delta >= 0");
  if (p->log_capacity_turns < 0) return fail(MBT_EINVAL, "log_capacity_turns < 0");
  if ((p->d_tau == nullptr) != (p->d_delta == nullptr)) return fail(MBT_EINVAL, "give both d_tau and d_delta or neither");
  if (p->d_tau && (((uintptr_t)p->d_tau | (uintptr_t)p->d_delta) & 31u)) return fail(MBT_EINVAL, "d_tau / d_delta must be 32-byte aligned");
  for (int c = 1; c < p->n_cav; ++c)
    if (std::isnan(p->cav[c].phase_rad)) return fail(MBT_EINVAL, "only cav[0] may leave its phase open");
  const mbt_transverse &tr = p->trans;
  if (tr.enable) {
    const mbt_plane *pls[2] = {&tr.x, &tr.y};
    for (const mbt_plane *pl : pls)
      if (!(pl->beta_m > 0) || !std::isfinite(pl->nu) || !std::isfinite(pl->alpha) || !(pl->D_exc >= 0) ||
          !(pl->sigma_u_m >= 0) || !(pl->sigma_up >= 0) || !(pl->sigma0_u_m >= 0) || !(pl->sigma0_up >= 0))
        return fail(MBT_EINVAL, "transverse plane: need beta > 0, D_exc >= 0, sigmas >= 0");
    if (tr.n_res < 0 || (tr.n_res > 0 && !tr.res)) return fail(MBT_EINVAL, "transverse resonator list");
    if (tr.rw_turns < 0 || tr.rw_turns > 100000 || !std::isfinite(tr.rw_amp_x) || !std::isfinite(tr.rw_amp_y))
      return fail(MBT_EINVAL, "resistive wall: need 0 <= rw_turns <= 100000, finite amplitudes");
    for (int r = 0; r < tr.n_res; ++r)
      if (!(tr.res[r].Q > 0.5) || !(tr.res[r].fr_Hz > 0) || !std::isfinite(tr.res[r].Rs_ohm))
        return fail(MBT_EINVAL, "transverse resonator: need Q > 1/2, fr > 0");
  }
  const mbt_shard &sh = p->shard;
  if (sh.enable) {
    if (sh.world < 1 || sh.rank < 0 || sh.rank >= sh.world) return fail(MBT_EINVAL, "shard: need 0 <= rank < world");
    if (p->trans.enable) return fail(MBT_EINVAL, "shard: not available with the transverse planes");
    if (sh.world > fl.n_bunches) return fail(MBT_EINVAL, "shard: more ranks than bunches");
  }
  const mbt_tuning &tn = p->tuning;
  if (tn.tile_iters < 0 || tn.pairs_per_thread < 0 || tn.pairs_per_thread > 2 || tn.pdl < 0 || tn.pdl > 3 || tn.stages6 < 0 ||
      (tn.stages6 != 0 && (tn.stages6 < 2 || tn.stages6 > kMaxStages6)) || tn.turn_mode < 0 || tn.turn_mode > 3 ||
      tn.verbose < 0 || tn.per_bunch_start < 0 || tn.per_bunch_start > 3 || tn.reserved[0] != 0)
    return fail(MBT_EINVAL, "tuning: a member is out of range (see mbt_tuning in mbt.h; all zero = the library's choice)");
  int n_lr = 0;
  for (int r = 0; r < wk.n_res; ++r) {
    if (!(wk.res[r].Q > 0.5) || !(wk.res[r].fr_Hz > 0) || !std::isfinite(wk.res[r].Rs_ohm))
      return fail(MBT_EINVAL, "resonator: need Q > 1/2, fr > 0");
    if (wk.res[r].flags & MBT_RES_LR) ++n_lr;
  }
  if (n_lr > MBT_MAX_LR) return fail(MBT_EINVAL, "too many long-range resonators");
  if (n_lr > 0 && wk.history_turns < 0) return fail(MBT_EINVAL, "history_turns < 0");

  int dev = p->device;
  if (dev < 0) CU(cudaGetDevice(&dev));
  CU(cudaSetDevice(dev));
  cudaDeviceProp prop;
  CU(cudaGetDeviceProperties(&prop, dev));

  mbt_handle *h = new (std::nothrow) mbt_handle();
  if (!h) return fail(MBT_ENOMEM, "out of memory");
  h->device = dev;
  h->stream = (cudaStream_t)p->stream;
  if (!h->stream) {  // stream capture is not allowed on the legacy default stream: use an own (blocking) stream
    cudaError_t e_ = cudaStreamCreate(&h->stream);
    if (e_ != cudaSuccess) {
      h->stream = nullptr;
      destroy(h);
      return fail(MBT_ECUDA, std::string("cudaStreamCreate failed: ") + cudaGetErrorString(e_));
    }
    h->own_stream = true;
  }
  // bunch sharding (S:8(f) rank 4): this handle owns the contiguous bunches [b0, b0 + M) of the fill's Mg
  const int Mg = h->Mg = fl.n_bunches;
  {
    int first = 0, count = Mg;
    if (sh.enable) {
      h->sharded = true;
      h->shard_rank = sh.rank;
      h->shard_world = sh.world;
      h->shard_chunk = (Mg + sh.world - 1) / sh.world;
      first = sh.rank * h->shard_chunk;
      count = std::max(0, std::min(h->shard_chunk, Mg - first));
      if (count == 0) { destroy(h); return fail(MBT_EINVAL, "shard: this rank owns no bunch (use fewer ranks)"); }
    }
    h->b0 = first;
    h->M = count;
  }
  const int M = h->M, b0 = h->b0;
  const int32_t *bucket_g = fl.bucket;   // the whole fill (long-range sums run over it)
  const int nb = h->nb = wk.n_bins;
  const int R = h->R = n_lr;
  const int K = h->K = n_lr ? wk.history_turns : 0;
  h->Np = fl.n_per_bunch;
  h->ld = mbt_particle_stride(h->Np);
  h->log_cap = p->log_capacity_turns;

#define CUH(call)                                                                                  \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      char buf_[512];                                                                              \
      snprintf(buf_, sizeof buf_, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
      cudaGetLastError();                                                                          \
      destroy(h);                                                                                  \
      return fail(e_ == cudaErrorMemoryAllocation ? MBT_ENOMEM : MBT_ECUDA, buf_);                 \
    }                                                                                              \
  } while (0)

  // ---- derived constants (fp64, once)
  Args &A = h->args;
  memset(&A, 0, sizeof A);
  const double E0 = rg.E0_eV;
  const double omega_rf = 2.0 * PI_D * (double)rg.h / rg.T0_s;
  std::vector<mbt_cavity> cav(p->cav, p->cav + p->n_cav);
  if (std::isnan(cav[0].phase_rad)) {
    // synchronous phase (D3): V_0 sin(phi_s) = U0 - sum_{c>0} V_c sin(phi_c), alpha_c cos(phi_s) < 0
    double u_eff = rg.U0_eV;
    for (int c = 1; c < p->n_cav; ++c) u_eff -= cav[c].V_volt * std::sin(cav[c].phase_rad);
    const double s = u_eff / cav[0].V_volt;
    if (!(std::fabs(s) <= 1.0)) {
      destroy(h);
      return fail(MBT_EINVAL, "U0 exceeds the RF voltage: no synchronous phase");
    }
    cav[0].phase_rad = (rg.alpha_c > 0.0) ? PI_D - std::asin(s) : std::asin(s);
  }
  h->phi_s = cav[0].phase_rad;
  A.n_cav = p->n_cav;
  for (int c = 0; c < p->n_cav; ++c) {
    A.cav_amp[c] = cav[c].V_volt / E0;
    A.cav_w[c] = (double)cav[c].m * omega_rf;
    A.cav_ph[c] = cav[c].phase_rad;
  }
  A.loss = rg.U0_eV / E0;
  A.rad = p->rad.enable ? 1 : 0;
  const double D_E = p->rad.enable ? 2.0 / p->rad.damping_turns : 0.0;  // D6
  A.one_minus_DE = 1.0 - D_E;
  A.A_q = p->rad.enable ? p->rad.sigma_delta * std::sqrt(2.0 * D_E) : 0.0;
  A.keys = philox_expand_key((uint32_t)(p->seed & 0xFFFFFFFFull), (uint32_t)(p->seed >> 32));
  A.drift = rg.alpha_c * rg.T0_s;
  A.nb = nb;
  A.gather = wk.gather_order;
  A.invDelta = (double)nb / (wk.tau_hi_s - wk.tau_lo_s);
  A.nb_d = (double)nb;
  A.invE0 = 1.0 / E0;
  A.ld = h->ld;
  A.Np = (uint32_t)h->Np;
  A.ppb = (uint32_t)(h->ld / 2);
  A.M = M;
  A.total_pairs = (int64_t)M * (h->ld / 2);
  A.R = R;

  // ---- tables (extended precision on the host, rounded once to fp64)
  const double Delta = (wk.tau_hi_s - wk.tau_lo_s) / (double)nb;
  std::vector<double> centre(nb);
  for (int j = 0; j < nb; ++j) centre[j] = wk.tau_lo_s + ((double)j + 0.5) * Delta;
  std::vector<double> w(nb, 0.0);
  bool have_sr = false;
  std::vector<Res> lr;
  std::vector<cplx> Cr;
  for (int r = 0; r < wk.n_res; ++r) {
    const Res rr = make_res(wk.res[r]);
    if (wk.res[r].flags & MBT_RES_SR) {
      have_sr = true;
      for (int k = 0; k < nb; ++k) w[k] += res_wake(rr, (ldbl)((double)k * Delta));
    }
    if (wk.res[r].flags & MBT_RES_LR) {
      lr.push_back(rr);
      // C_r = 2 alpha Rs (1 + i alpha / wbar):  W(t > 0) = Re[C_r exp(lambda_r t)]
      const ldbl two_a_rs = 2.0L * rr.alpha * (ldbl)rr.Rs;
      Cr.push_back(cplx{(double)two_a_rs, (double)(two_a_rs * rr.alpha / rr.wbar)});
    }
  }
  if (wk.n_table > 0) {
    have_sr = true;
    for (int k = 0; k < nb && k < wk.n_table; ++k) w[k] += wk.sr_table[k];
  }
  std::vector<cplx> Esrc((size_t)R * nb), F((size_t)R * nb), g_step((size_t)Mg * (R ? R : 1)), g_tail((size_t)Mg * (R ? R : 1)),
      g_hist((size_t)(K ? K : 1) * (R ? R : 1));
  const ldbl T0 = (ldbl)rg.T0_s, Trf = T0 / (ldbl)rg.h;
  for (int r = 0; r < R; ++r) {
    for (int k = 0; k < nb; ++k) {
      // exp(-lambda c_k) and C_r exp(lambda c_k): |c_k| < T_rf / 2, a few radians of phase
      const ldbl c = (ldbl)centre[k];
      const ldbl mg = expl(lr[r].alpha * c), ph = -lr[r].wbar * c;
      Esrc[(size_t)r * nb + k] = cplx{(double)(mg * cosl(ph)), (double)(mg * sinl(ph))};
      const ldbl mg2 = expl(-lr[r].alpha * c), ph2 = lr[r].wbar * c;
      const ldbl ere = mg2 * cosl(ph2), eim = mg2 * sinl(ph2);
      F[(size_t)r * nb + k] = cplx{(double)((ldbl)Cr[r].re * ere - (ldbl)Cr[r].im * eim),
                                   (double)((ldbl)Cr[r].re * eim + (ldbl)Cr[r].im * ere)};
    }
    const int span = bucket_g[Mg - 1] - bucket_g[0];
    for (int j = 0; j < Mg; ++j) {
      if (j + 1 < Mg) g_step[(size_t)j * R + r] = exp_lambda(lr[r], (ldbl)(bucket_g[j + 1] - bucket_g[j]) * Trf);
      g_tail[(size_t)j * R + r] = exp_lambda(lr[r], (ldbl)(bucket_g[Mg - 1] - bucket_g[j]) * Trf);
    }
    for (int k = 1; k <= K; ++k) g_hist[(size_t)(k - 1) * R + r] = exp_lambda(lr[r], (ldbl)k * T0 - (ldbl)span * Trf);
  }
  std::vector<double> qm(M);
  for (int b = 0; b < M; ++b) qm[b] = fl.charge_C[b0 + b] / (double)h->Np;

  // ---- device memory
  const size_t N = (size_t)M * (size_t)h->ld;
  if (p->d_tau) {
    h->d_tau = (double *)p->d_tau;
    h->d_delta = (double *)p->d_delta;
  } else {
    h->own_particles = true;
    CUH(cudaMalloc((void **)&h->d_tau, N * sizeof(double)));
    CUH(cudaMalloc((void **)&h->d_delta, N * sizeof(double)));
  }
  CUH(h->qm.upload(qm, h->stream));
  if (have_sr) CUH(h->w.upload(w, h->stream));
  CUH(h->Esrc.upload(Esrc, h->stream));
  CUH(h->F.upload(F, h->stream));
  {  // gather cells of the constant tables F_r (same cell definition as k_wake applies to V_SR)
    std::vector<CellF> cf((size_t)(R ? R : 1) * (nb + 2), CellF{cplx{0, 0}, cplx{0, 0}});
    for (int r = 0; r < R; ++r)
      for (int k = 0; k < nb + 2; ++k) {
        CellF c{cplx{0, 0}, cplx{0, 0}};
        if (wk.gather_order == 1) {
          if (k <= nb) {
            const cplx lo = F[(size_t)r * nb + (k > 0 ? k - 1 : 0)], hi = F[(size_t)r * nb + (k < nb ? k : nb - 1)];
            c.mid = cplx{0.5 * (lo.re + hi.re), 0.5 * (lo.im + hi.im)};
            c.dif = cplx{hi.re - lo.re, hi.im - lo.im};
          }
        } else if (k < nb) {
          c.mid = F[(size_t)r * nb + k];
        }
        cf[(size_t)r * (nb + 2) + k] = c;
      }
    CUH(h->cellF.upload(cf, h->stream));
  }
  CUH(h->cellSR.alloc((size_t)M * (nb + 2), h->stream));
  // ---- bunch-following window (D31): shifts in whole bins, |s| <= s_max keeps the window inside the bucket
  h->window_mode = wk.window_mode;
  h->tau_lo = wk.tau_lo_s;
  h->Delta = Delta;
  {
    const double T_rf = rg.T0_s / (double)rg.h;
    const double room = std::fmin(0.5 * T_rf - wk.tau_hi_s, wk.tau_lo_s + 0.5 * T_rf);  // to the nearer bucket edge
    const double smax = std::floor(room / Delta);
    h->s_max = (wk.window_mode && smax > 0.0) ? (int32_t)std::fmin(smax, 1.0e6) : 0;
    std::vector<double> lo0(M, (wk.tau_lo_s == 0.0) ? -0.0 : wk.tau_lo_s);  // 0 stored as -0.0: see in_window()
    CUH(h->lo_hist.upload(lo0, h->stream));
    CUH(h->lo_next.upload(lo0, h->stream));
    CUH(h->s_hist.alloc(M, h->stream));
    CUH(h->s_next.alloc(M, h->stream));
    if (wk.window_mode && R > 0) {
      const int W = 2 * h->s_max + 1;
      std::vector<cplx> ss((size_t)R * W), sw((size_t)R * W);
      for (int r = 0; r < R; ++r)
        for (int i = 0; i < W; ++i) {
          const ldbl t = (ldbl)(i - h->s_max) * (ldbl)Delta;
          const ldbl mg = expl(lr[r].alpha * t), ph = lr[r].wbar * t;
          ss[(size_t)r * W + i] = cplx{(double)(mg * cosl(ph)), (double)(-mg * sinl(ph))};               // exp(-lambda t)
          sw[(size_t)r * W + i] = cplx{(double)(cosl(ph) / mg), (double)(sinl(ph) / mg)};                // exp(+lambda t)
        }
      CUH(h->shift_src.upload(ss, h->stream));
      CUH(h->shift_wit.upload(sw, h->stream));
    }
  }
  CUH(h->g_step.upload(g_step, h->stream));
  CUH(h->g_tail.upload(g_tail, h->stream));
  CUH(h->g_hist.upload(g_hist, h->stream));
  {  // exp(lambda_r d T_rf) over the bucket distance d (one-launch turn: the per-bunch phasor gather)
    std::vector<cplx> gd((size_t)(R ? R : 1) * rg.h, cplx{1.0, 0.0});
    for (int r = 0; r < R; ++r)
      for (int d = 0; d < rg.h; ++d) gd[(size_t)r * rg.h + d] = exp_lambda(lr[r], (ldbl)d * Trf);
    CUH(h->gd.upload(gd, h->stream));
    CUH(h->d_bucket.upload(std::vector<int32_t>(bucket_g, bucket_g + Mg), h->stream));
    CUH(h->a_ready.alloc((size_t)Mg * (R ? R : 1), h->stream));
    CUH(h->bunch_ready.alloc(M, h->stream));
    CUH(h->agg_ready.alloc(1, h->stream));
  }
  CUH(h->Vsr.alloc((size_t)M * nb, h->stream));
  CUH(h->a_cur.alloc((size_t)M * (R ? R : 1), h->stream));
  h->slots = K + 1 < 2 ? 2 : K + 1;
  CUH(h->ring_a.alloc((size_t)h->slots * Mg * (R ? R : 1), h->stream));
  CUH(h->ring_A.alloc((size_t)h->slots * (R ? R : 1), h->stream));
  CUH(h->P.alloc((size_t)M * (R ? R : 1), h->stream));
  CUH(h->hist.alloc((size_t)M * nb, h->stream));
  CUH(h->hist_last.alloc((size_t)M * nb, h->stream));
  CUH(h->mom_acc.alloc((size_t)M * 4, h->stream));
  CUH(h->nout_acc.alloc((size_t)M, h->stream));
  CUH(h->mom_last.alloc((size_t)M * 6, h->stream));
  if (h->log_cap > 0) CUH(h->mom_log.alloc((size_t)h->log_cap * M * 6, h->stream));
  CUH(h->ctrl.alloc(1, h->stream));
  CUH(h->logtab.upload(std::vector<LogTabEntry>(kLogTabHost, kLogTabHost + 128), h->stream));

  A.tau = h->d_tau;
  A.delta = h->d_delta;
  A.Vsr = h->Vsr.p;
  A.P = h->P.p;
  A.F = h->F.p;
  A.cellSR = h->cellSR.p;
  A.cellF = h->cellF.p;
  A.hist = h->hist.p;
  A.lo_hist = h->lo_hist.p;
  A.lo_next = h->lo_next.p;
  A.mom_acc = h->mom_acc.p;
  A.nout_acc = h->nout_acc.p;
  A.ctrl = h->ctrl.p;
  A.logtab = h->logtab.p;
  A.mt = make_math_tab();

  WakeArgs &Wa = h->wargs;
  memset(&Wa, 0, sizeof Wa);
  Wa.M = M; Wa.nb = nb; Wa.R = R; Wa.K = K; Wa.Np = (uint32_t)h->Np; Wa.mode = 0;
  {  // few bunches and many bins: deal the convolution of a bunch out over S CTAs (<= 2 waves of CTAs).  Sharing a bunch
     // costs three dependent elections (atomics, fences, a reload of V_SR): ~3 us, what one CTA needs for the whole
     // register-blocked convolution of ~500 bins -- so up to 512 bins a bunch has ONE CTA (which also gives it the per-bunch
     // phasor gather and the per-bunch start of the next pass); tuning.wake_splits overrides.
    const int pairs = (nb + 1) / 2;
    int S = nb <= 512 ? 1 : (pairs + 31) / 32;
    const int room = (2 * prop.multiProcessorCount + M - 1) / M;
    if (S > room) S = room;
    if (S > 64) S = 64;
    if (tn.reserved[0] > 0) S = std::min(tn.reserved[0], std::min(room, 64));  // measurement: forced number of splits
    if (S < 1 || sh.enable) S = 1;  // a sharded handle runs the per-bunch phasor gather: one CTA per bunch
    h->wake_splits = S;
  }
  CUH(h->rd_cnt.alloc(M, h->stream));
  CUH(h->wr_cnt.alloc(M, h->stream));
  Wa.S = h->wake_splits; Wa.rd_cnt = h->rd_cnt.p; Wa.wr_cnt = h->wr_cnt.p;
  Wa.qm = h->qm.p;
  Wa.w = have_sr ? h->w.p : nullptr;
  Wa.Esrc = h->Esrc.p; Wa.g_step = h->g_step.p; Wa.g_tail = h->g_tail.p; Wa.g_hist = h->g_hist.p;
  Wa.hist = h->hist.p; Wa.hist_last = h->hist_last.p; Wa.Vsr = h->Vsr.p;
  Wa.cellSR = h->cellSR.p; Wa.gather = wk.gather_order;
  Wa.window_mode = wk.window_mode; Wa.s_max = h->s_max; Wa.tau_lo = wk.tau_lo_s; Wa.Delta = Delta;
  Wa.s_hist = h->s_hist.p; Wa.s_next = h->s_next.p; Wa.lo_hist = h->lo_hist.p; Wa.lo_next = h->lo_next.p;
  Wa.shift_src = h->shift_src.p; Wa.shift_wit = h->shift_wit.p;
  Wa.a_cur = h->a_cur.p; Wa.ring_a = h->ring_a.p; Wa.ring_A = h->ring_A.p; Wa.P = h->P.p;
  Wa.mom_acc = h->mom_acc.p; Wa.nout_acc = h->nout_acc.p; Wa.mom_last = h->mom_last.p;
  Wa.mom_log = h->log_cap > 0 ? h->mom_log.p : nullptr;
  Wa.log_cap = h->log_cap;
  Wa.ctrl = h->ctrl.p;
  if (sh.enable && R > 0) {
    if (!sh.d_exchange || ((uintptr_t)sh.d_exchange & 15u)) { destroy(h); return fail(MBT_EINVAL, "shard: d_exchange must be a 16-byte aligned device buffer (mbt_shard_exchange_doubles)"); }
    h->xbuf = (cplx *)sh.d_exchange;
  }
  Wa.Mg = Mg; Wa.b0 = b0; Wa.part = 0; Wa.xbuf = h->xbuf;
  Wa.h = rg.h; Wa.slots = h->slots; Wa.bucket = h->d_bucket.p; Wa.gd = h->gd.p;
  Wa.a_ready = h->a_ready.p; Wa.bunch_ready = h->bunch_ready.p; Wa.agg_ready = h->agg_ready.p;

  // ---- launch shapes: one resident wave of CTAs, each owning a contiguous run of pairs
  // two pairs per thread (twice the independent arithmetic per warp, 2 CTAs/SM) pay off except for small
  // two-cavity workloads, where the four sine chains per thread cost more registers than they hide latency
  if (tn.pdl) h->pdl = tn.pdl == 1 ? 0 : tn.pdl == 2 ? 1 : 3;  // mbt_tuning.pdl: 1 off, 2 the pass, 3 the pass and k_wake
  h->npair = kDefaultNPair ? kDefaultNPair : ((p->n_cav == 1 || (int64_t)M * h->Np >= 10000000ll) ? 2 : 1);
  if (tn.pairs_per_thread) h->npair = tn.pairs_per_thread;
  const bool rad_on = p->rad.enable != 0;
  h->fn_map = h->npair == 2 ? select_map<2>(rad_on, wk.gather_order, p->n_cav) : select_map<1>(rad_on, wk.gather_order, p->n_cav);
  h->fn_flush = h->npair == 2 ? select_flush<2>(wk.gather_order) : select_flush<1>(wk.gather_order);
  h->smem_pass = pass_smem_bytes(nb, h->npair);
  // k_wake: the convolution's shared memory + the staged source factors (if <= 64 KB), or the scan's staged operands (if
  // the scan runs and they fit in 96 KB).  Kept small: every CTA of the launch should be resident at once.
  {
    size_t need = wake_smem_bytes(nb, Mg);
    const size_t stage_e = (size_t)R * nb * sizeof(cplx) + 16;
    if (R > 0 && stage_e <= 64u * 1024u) need += stage_e;
    // one CTA per bunch: the per-bunch phasor gather replaces the scan.  A bunch's CTA waits only for CTAs of a lower
    // index, which were dispatched before it: no deadlock whether or not all M CTAs are resident at once (they are up to
    // 3 x 148 bunches: __launch_bounds__(256, 3) and the carve-out below)
    CUH(cudaFuncSetAttribute(k_wake, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
    const bool gather = h->wake_splits == 1;
    if (!gather && scan_smem_bytes(M, R) <= 96u * 1024u) need = std::max(need, scan_smem_bytes(M, R));
    h->smem_wake = need;
    Wa.gather_P = gather ? 1 : 0;
  }
  Wa.smem_wake_bytes = (uint32_t)h->smem_wake;
  Wa.smem_pass_bytes = (uint32_t)h->smem_pass;
  CUH(cudaFuncSetAttribute((const void *)h->fn_map, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_pass));
  CUH(cudaFuncSetAttribute((const void *)h->fn_flush, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_pass));
  CUH(cudaFuncSetAttribute(k_wake, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_wake));
  // all CTAs of k_wake should be resident at once: with the default carve-out only two per SM were (the third of an SM
  // started when the first had finished: 15 us later)
  CUH(cudaFuncSetAttribute(k_wake, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
  // tiles (choose_tiles)
  {
    int occ = 0;
    CUH(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)h->fn_map, kPassThreads, h->smem_pass));
    if (occ < 1) occ = 1;
    choose_tiles(h->ld / 2, (int64_t)kPassThreads * h->npair, M, prop.multiProcessorCount * occ, tn.tile_iters, tn.verbose != 0,
                 &A.tile_pairs, &h->grid_pass);
  }

  // ---- one launch per turn (mbt_tuning.turn_mode): the last pass CTA of a bunch builds the bunch's wake in the (drained)
  // particle stages, the last CTA of the grid closes the turn.  Not with the transverse planes (their wake kernels run
  // beside k_wake on a side stream).
  CUH(h->bunch_done.alloc(M, h->stream));
  A.bunch_done = h->bunch_done.p;
  A.b0 = b0;
  CUH(h->tile_turn.alloc((size_t)M * h->grid_pass, h->stream));
  A.tile_turn = h->tile_turn.p;
  A.bunch_ready = h->bunch_ready.p;
  // a pass CTA starts on its own bunch's wake (one k_wake CTA per bunch publishes bunch_ready) instead of on the whole grid
  A.flag_wait = (!tr.enable && !sh.enable && h->wargs.gather_P && tn.per_bunch_start != 1) ? 1 : 0;
  h->fused = !tr.enable && !sh.enable && tn.turn_mode == 2;
  if (tn.turn_mode == 2 && tr.enable) {
    destroy(h);
    return fail(MBT_EINVAL, "tuning.turn_mode 2 (one launch per turn) is not available with the transverse planes");
  }
  if (h->fused && h->smem_pass < wake_smem_bytes(nb, Mg)) h->fused = false;  // cannot happen for nb <= MBT_MAX_BINS
  A.fused = h->fused ? 1 : 0;
  if (h->fused) A.flag_wait = 0;  // the one-launch turn waits for its predecessor grid (it wrote the particles)
  // ... and the wake kernel's CTA of a bunch starts on its own bunch's pass CTAs (launched as a programmatic dependent)
  if (A.flag_wait && tn.per_bunch_start != 3) {
    A.count_done = 1;
    h->wargs.bunch_wait = 1;
    h->wargs.tiles = h->grid_pass;
    h->wargs.bunch_done = h->bunch_done.p;
    if (!tn.pdl) h->pdl |= 2;
  }
  if (tn.verbose)
    fprintf(stderr, "mbt: %s, %d pair(s) per thread, grid %d x %d, %zu B shared memory per CTA, pdl %d\n",
            h->fused ? "one launch per turn" : "two launches per turn", h->npair, h->grid_pass, M, h->smem_pass, h->pdl);

  // ---- chip-resident turn loop (mbt_tuning.turn_mode 3 only): grid = M x G_b CTAs, all resident (cooperative launch),
  // each holding tile_pairs pairs of one bunch in shared memory
  if (!tr.enable && !sh.enable && tn.turn_mode == 3) {
    res_fn fn = select_resident(rad_on, wk.gather_order, p->n_cav);
    const int64_t ppb = h->ld / 2, stride = (int64_t)kPassThreads * 2;
    bool ok = false;
    for (int occ = 2; occ >= 1 && !ok; --occ) {
      int gb = (prop.multiProcessorCount * occ) / M;                        // CTAs per bunch
      gb = (int)std::min<int64_t>(gb, (ppb + stride - 1) / stride);         // at least one full iteration per CTA
      if (gb < 1) continue;
      uint32_t tile = (uint32_t)((ppb + gb - 1) / gb);
      tile += tile & 1u;
      const size_t wake_bytes = (h->smem_wake + 15) & ~(size_t)15;
      const size_t smem = resident_smem_bytes(tile, nb, wake_bytes);
      if (smem > (size_t)prop.sharedMemPerBlockOptin) continue;
      if (cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { cudaGetLastError(); continue; }
      int got = 0;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&got, (const void *)fn, kPassThreads, smem) != cudaSuccess) { cudaGetLastError(); continue; }
      if ((int64_t)got * prop.multiProcessorCount < (int64_t)gb * M) continue;
      int coop = 0;
      cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
      if (!coop) continue;
      ok = true;
      h->resident = true;
      h->fn_res = fn;
      h->grid_res = gb * M;
      h->smem_res = smem;
      memset(&h->rargs, 0, sizeof h->rargs);
      h->rargs.ctas_per_bunch = gb;
      h->rargs.tile_pairs = tile;
      h->rargs.wake_off = (uint32_t)(smem - wake_bytes - 16 + 15) & ~15u;
      h->rargs.wake_bytes = (uint32_t)wake_bytes;
      h->wargs_res = h->wargs;
      h->wargs_res.S = std::min(h->wake_splits, gb);
      h->wargs_res.bunch_wait = 0;
    }
    if (ok) {
      CUH(h->res_bar.alloc(2, h->stream));
      h->rargs.bar = h->res_bar.p;
    } else if (tn.turn_mode == 3) {
      destroy(h);
      return fail(MBT_EINVAL, "tuning.turn_mode 3: the particle store does not fit in the chip's shared memory (or no cooperative launch)");
    }
    if (tn.verbose && ok)
      fprintf(stderr, "mbt: chip-resident turn loop, %d CTAs per bunch, %u pairs per CTA, %zu B shared memory per CTA\n",
              h->rargs.ctas_per_bunch, h->rargs.tile_pairs, h->smem_res);
  } else if (tn.turn_mode == 3) {
    destroy(h);
    return fail(MBT_EINVAL, "tuning.turn_mode 3 (chip-resident) is not available with the transverse planes or bunch sharding");
  }

  // ---- initial distribution (D20) on the device
  {
    dim3 grid((unsigned)((h->ld + 255) / 256 < 1024 ? (h->ld + 255) / 256 : 1024), (unsigned)M);
    k_init<<<grid, 256, 0, h->stream>>>(h->d_tau, h->d_delta, h->ld, (uint32_t)h->Np, M, b0, A.keys, fl.sigma_tau0_s,
                                         fl.sigma_delta0);
    h->launches += 1;
    CUH(cudaGetLastError());
  }
  // ---- transverse planes (mbt_trans.cuh)
  if (tr.enable) {
    h->trans = true;
    std::vector<double> wt(nb, 0.0);
    for (int r = 0; r < tr.n_res; ++r) {
      const Res rr = make_res(tr.res[r]);
      const ldbl wr = 2.0L * PI_L * (ldbl)rr.fr;
      for (int k = 1; k < nb; ++k) {  // W_perp(t > 0) = (w_r^2 R / (Q wbar)) exp(-a t) sin(wbar t), W_perp(0) = 0 (T7)
        const ldbl t = (ldbl)((double)k * Delta);
        wt[k] += (double)((wr * wr * (ldbl)rr.Rs / ((ldbl)rr.Q * rr.wbar)) * expl(-rr.alpha * t) * sinl(rr.wbar * t));
      }
    }
    CUH(h->wt.upload(wt, h->stream));
    CUH(h->tx.alloc(N, h->stream)); CUH(h->txp.alloc(N, h->stream)); CUH(h->ty.alloc(N, h->stream)); CUH(h->typ.alloc(N, h->stream));
    CUH(h->Sfix.alloc((size_t)M * 2 * (nb + 1), h->stream)); CUH(h->Sov.alloc((size_t)M * 2 * (nb + 1), h->stream));
    // long-range resistive wall (W1..W5): source ring, kick per bunch, weights (d T_rf)^-1/2 by bucket distance d
    h->Krw = tr.rw_turns;
    CUH(h->ring_g.alloc((size_t)(h->Krw + 2) * M * 2, h->stream));  // Krw + 1 slots are read per turn, one spare (TWakeArgs)
    CUH(h->rw.alloc((size_t)M * 2, h->stream));
    {
      std::vector<double> wr((size_t)(h->Krw + 1) * rg.h, 0.0);
      for (size_t d = 1; d < wr.size(); ++d)
        wr[d] = (double)(1.0L / sqrtl((ldbl)d * ((ldbl)rg.T0_s / (ldbl)rg.h)));
      CUH(h->wrw.upload(wr, h->stream));
    }
    RwArgs &Rw = h->rwargs;
    memset(&Rw, 0, sizeof Rw);
    Rw.M = M; Rw.Krw = h->Krw; Rw.h = rg.h; Rw.bucket = h->d_bucket.p; Rw.ring_g = h->ring_g.p; Rw.wrw = h->wrw.p;
    CUH(h->turn_tr.alloc(1, h->stream));
    CUH(cudaStreamCreateWithFlags(&h->stream2, cudaStreamNonBlocking));
    CUH(cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming));
    CUH(cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming));
    Rw.amp[0] = tr.rw_amp_x; Rw.amp[1] = tr.rw_amp_y; Rw.rw = h->rw.p; Rw.turn_tr = h->turn_tr.p;
    CUH(h->S_last.alloc((size_t)M * 2 * nb, h->stream)); CUH(h->Ktab.alloc((size_t)M * 2 * nb, h->stream));
    CUH(h->cellX.alloc((size_t)M * (nb + 2), h->stream)); CUH(h->cellY.alloc((size_t)M * (nb + 2), h->stream));
    CUH(h->fix.alloc((size_t)M * 2, h->stream)); CUH(h->acc2.alloc((size_t)M * 2, h->stream));
    CUH(h->mom_tr_acc.alloc((size_t)M * 8, h->stream)); CUH(h->mom_tr.alloc((size_t)M * 8, h->stream));
    // bits of the fixed-point dipole sums: N_p 2^bits <= 2^62 (mbt_trans.cuh)
    h->fix_bits = kFixBitsMax;
    while (h->fix_bits > 20 && (double)h->Np * std::ldexp(1.0, h->fix_bits) > std::ldexp(1.0, 62)) h->fix_bits -= 1;
    Args6 &T = h->args6;
    memset(&T, 0, sizeof T);
    T.L = A;
    T.x = h->tx.p; T.xp = h->txp.p; T.y = h->ty.p; T.yp = h->typ.p;
    const mbt_plane *pls[2] = {&tr.x, &tr.y};
    Plane *dst[2] = {&T.px, &T.py};
    for (int a = 0; a < 2; ++a) {
      const mbt_plane &q = *pls[a];
      Plane &d = *dst[a];
      d.t_frac = q.nu - std::floor(q.nu);
      d.t_xi = q.nu * q.xi;
      d.alpha = q.alpha; d.beta = q.beta_m; d.gamma = (1.0 + q.alpha * q.alpha) / q.beta_m;
      d.eta = q.eta_m; d.etap = q.etap;
      d.exc_u = q.sigma_u_m * std::sqrt(q.D_exc);
      d.exc_up = q.sigma_up * std::sqrt(q.D_exc);
    }
    T.cellX = h->cellX.p; T.cellY = h->cellY.p;
    T.Sfix = h->Sfix.p; T.Sov = h->Sov.p; T.fix = h->fix.p; T.acc2 = h->acc2.p; T.rw = h->rw.p; T.turn_tr = h->turn_tr.p;
    h->fn_map6 = select_map6(rad_on, wk.gather_order, p->n_cav);
    h->fn_flush6 = select_flush6(wk.gather_order);
    if (pass6_smem_bytes(nb, 2) > (size_t)prop.sharedMemPerBlockOptin) {
      char buf[160];
      snprintf(buf, sizeof buf, "transverse planes: n_bins = %d needs %zu bytes of shared memory per CTA (limit %zu)", nb,
               pass6_smem_bytes(nb, 2), (size_t)prop.sharedMemPerBlockOptin);
      destroy(h);
      return fail(MBT_EINVAL, buf);
    }
    // two stages (48 KB) in flight per CTA: three measured the same to 1 % (c4 0.839 vs 0.834 ms, c5 2.41 vs 2.37), four
    // cost a CTA per SM
    T.stages = tn.stages6 ? tn.stages6 : 2;
    h->smem_pass6 = pass6_smem_bytes(nb, T.stages);
    CUH(cudaFuncSetAttribute((const void *)h->fn_map6, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_pass6));
    CUH(cudaFuncSetAttribute((const void *)h->fn_flush6, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_pass6));
    CUH(cudaFuncSetAttribute(k_wake_tr, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wake_tr_smem_bytes(nb)));
    {
      int occ = 0;
      CUH(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)h->fn_map6, kPassThreads, h->smem_pass6));
      if (occ < 1) occ = 1;
      choose_tiles(h->ld / 2, kPassThreads, M, prop.multiProcessorCount * occ, tn.tile_iters, tn.verbose != 0, &T.tile_pairs,
                   &h->grid_pass6);
    }
    // per-bunch sequencing of the 6-D turn (as the longitudinal one): one k_wake CTA per bunch, launches chained
    CUH(h->tr_ready.alloc(M, h->stream));
    CUH(h->rw_ready.alloc(M, h->stream));
    CUH(h->bunch_done_tr.alloc(M, h->stream));
    h->pipe6 = h->wargs.gather_P && tn.per_bunch_start != 1 && tn.pdl != 1;
    if (h->pipe6) {
      h->tile_turn.release();
      CUH(h->tile_turn.alloc((size_t)M * h->grid_pass6, h->stream));
      T.L.tile_turn = h->tile_turn.p;
      T.L.bunch_ready = h->bunch_ready.p;
      T.L.flag_wait = 1;
      T.L.count_done = 1;
      T.tr_ready = h->tr_ready.p;
      T.rw_ready = h->Krw > 0 ? h->rw_ready.p : nullptr;
      T.bunch_done_tr = h->bunch_done_tr.p;
      h->smem_wake6 = std::max(h->smem_wake, wake_tr_smem_bytes(nb));
      CUH(cudaFuncSetAttribute(k_wake6, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_wake6));
      CUH(cudaFuncSetAttribute(k_wake6, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
      h->wargs.bunch_wait = 1;
      h->wargs.tiles = h->grid_pass6;
      h->wargs.bunch_done = h->bunch_done.p;
    }
    TMomArgs &Tm = h->tmargs;
    Tm.x = h->tx.p; Tm.xp = h->txp.p; Tm.y = h->ty.p; Tm.yp = h->typ.p; Tm.ld = h->ld; Tm.Np = (uint32_t)h->Np; Tm.tile = 8192;
    h->grid_tr = (int)((h->Np + Tm.tile - 1) / Tm.tile);
    TWakeArgs &Tw = h->twargs;
    memset(&Tw, 0, sizeof Tw);
    Tw.M = M; Tw.nb = nb; Tw.gather = wk.gather_order; Tw.fix_bits = h->fix_bits; Tw.Np = (uint32_t)h->Np;
    Tw.qm = h->qm.p; Tw.wt = h->wt.p;
    Tw.Sfix = h->Sfix.p; Tw.Sov = h->Sov.p; Tw.fix = h->fix.p; Tw.acc2 = h->acc2.p;
    Tw.S_last = h->S_last.p; Tw.K = h->Ktab.p; Tw.cellX = h->cellX.p; Tw.cellY = h->cellY.p;
    Tw.Krw = h->Krw; Tw.ring_g = h->ring_g.p; Tw.turn_tr = h->turn_tr.p;
    if (h->log_cap > 0) CUH(h->log_tr.alloc((size_t)h->log_cap * M * 4, h->stream));
    Tw.log_tr = h->log_cap > 0 ? h->log_tr.p : nullptr;
    Tw.log_cap = h->log_cap;
    Tw.tr_ready = h->tr_ready.p; Tw.use_flags = h->pipe6 ? 1 : 0; Tw.bunch_done_tr = h->bunch_done_tr.p;
    Tw.rw_ready = h->rw_ready.p;
    h->rwargs.rw_ready = h->rw_ready.p; h->rwargs.tr_ready = h->tr_ready.p; h->rwargs.use_flags = h->pipe6 ? 1 : 0;
    dim3 grid((unsigned)((h->ld + 255) / 256 < 1024 ? (h->ld + 255) / 256 : 1024), (unsigned)M);
    k_init_tr<<<grid, 256, 0, h->stream>>>(h->tx.p, h->txp.p, h->ty.p, h->typ.p, h->ld, (uint32_t)h->Np, A.keys,
                                           tr.x.sigma0_u_m, tr.x.sigma0_up, tr.y.sigma0_u_m, tr.y.sigma0_up);
    if (int rc = rescale_transverse(h)) { destroy(h); return rc; }
    h->launches += 1;
    CUH(cudaGetLastError());
  }
  CUH(cudaEventCreate(&h->ev0));
  CUH(cudaEventCreate(&h->ev1));
  CUH(cudaStreamSynchronize(h->stream));
#undef CUH
  h->dirty = true;
  *out = h;
  return 0;
}

int mbt_track(mbt_handle *h, int64_t n_turns) {
  if (!h || n_turns < 0) return fail(MBT_EINVAL, "bad argument");
  if (h->turn + n_turns > 0xFFFFFFFFll) return fail(MBT_EINVAL, "turn counter would exceed 2^32");
  if (h->sharded) return fail(MBT_ESTATE, "a sharded handle advances by mbt_shard_turn_begin / (all-gather) / mbt_shard_turn_end");
  CU(cudaSetDevice(h->device));
  if (n_turns == 0) return 0;
  if (h->resident) return track_resident(h, n_turns);
  for (int lv = mbt_handle::kGraphLevels - 1; lv >= 0; --lv)  // build what this call needs before the timed region
    if (((n_turns >> lv) & 1) || (lv == mbt_handle::kGraphLevels - 1 && (n_turns >> lv)))
      if (!h->graphs[lv]) {
        int rc = build_graph(h, 1 << lv, &h->graphs[lv]);
        if (rc) return rc;
      }
  CU(cudaEventRecord(h->ev0, h->stream));
  int64_t left = n_turns;
  for (int lv = mbt_handle::kGraphLevels - 1; lv >= 0; --lv)
    while (left >= (1ll << lv)) {
      CU(cudaGraphLaunch(h->graphs[lv], h->stream));
      left -= 1ll << lv;
      if (lv < mbt_handle::kGraphLevels - 1) break;  // every smaller size at most once
    }
  CU(cudaEventRecord(h->ev1, h->stream));
  h->timed = true;
  h->launches += launches_per_turn(h) * n_turns;
  h->turn += n_turns;
  h->dirty = true;
  h->wake_valid = true;
  return 0;
}

int mbt_track_profiled(mbt_handle *h, int64_t n_turns, double *pass_seconds, double *wake_seconds) {
  if (!h || n_turns < 1 || n_turns > 65536 || !pass_seconds || !wake_seconds) return fail(MBT_EINVAL, "bad argument");
  if (h->turn + n_turns > 0xFFFFFFFFll) return fail(MBT_EINVAL, "turn counter would exceed 2^32");
  if (h->sharded) return fail(MBT_ESTATE, "not available on a sharded handle");
  CU(cudaSetDevice(h->device));
  if (h->resident) {  // one launch does everything: its device time is the "pass", there is no separate wake kernel
    if (int rc = track_resident(h, n_turns)) return rc;
    const double sec = mbt_last_track_seconds(h);
    if (sec < 0) return MBT_ECUDA;
    *pass_seconds = sec;
    *wake_seconds = 0.0;
    return 0;
  }
  struct Events {  // destroyed on every exit path
    std::vector<cudaEvent_t> v;
    ~Events() { for (cudaEvent_t e : v) if (e) cudaEventDestroy(e); }
  } evs;
  evs.v.assign((size_t)n_turns * 3, nullptr);
  std::vector<cudaEvent_t> &ev = evs.v;
  for (auto &e : ev) CU(cudaEventCreate(&e));
  CU(cudaEventRecord(h->ev0, h->stream));
  for (int64_t t = 0; t < n_turns; ++t) {
    CU(cudaEventRecord(ev[3 * t], h->stream));
    CU(enqueue_pass(h));
    CU(cudaEventRecord(ev[3 * t + 1], h->stream));
    CU(enqueue_wakes(h));
    CU(cudaEventRecord(ev[3 * t + 2], h->stream));
    h->launches += launches_per_turn(h);
    h->turn += 1;
    h->dirty = true;
    h->wake_valid = true;
  }
  CU(cudaEventRecord(h->ev1, h->stream));
  h->timed = true;
  CU(cudaStreamSynchronize(h->stream));
  double ps = 0.0, ws = 0.0;
  for (int64_t t = 0; t < n_turns; ++t) {
    float a = 0.f, b = 0.f;
    CU(cudaEventElapsedTime(&a, ev[3 * t], ev[3 * t + 1]));
    CU(cudaEventElapsedTime(&b, ev[3 * t + 1], ev[3 * t + 2]));
    ps += (double)a * 1e-3;
    ws += (double)b * 1e-3;
  }
  *pass_seconds = ps;
  *wake_seconds = ws;
  return 0;
}

double mbt_last_track_seconds(mbt_handle *h) {
  if (!h || !h->timed) { fail(MBT_ESTATE, "no tracked call to time"); return -1.0; }
  if (cudaEventSynchronize(h->ev1) != cudaSuccess) { fail(MBT_ECUDA, "event synchronize failed"); return -1.0; }
  float ms = 0.f;
  if (cudaEventElapsedTime(&ms, h->ev0, h->ev1) != cudaSuccess) { fail(MBT_ECUDA, "event elapsed failed"); return -1.0; }
  return (double)ms * 1e-3;
}

int mbt_moments(mbt_handle *h, double *out) {
  if (!h || !out) return fail(MBT_EINVAL, "null argument");
  int rc = flush(h);
  if (rc) return rc;
  CU(cudaMemcpyAsync(out, h->mom_last.p, sizeof(double) * h->M * 6, cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_destroy(mbt_handle *h) {
  destroy(h);
  return 0;
}

int mbt_device_pointers(mbt_handle *h, void **d_tau, void **d_delta, int64_t *ld) {
  if (!h) return fail(MBT_EINVAL, "null argument");
  int rc = flush(h);
  if (rc) return rc;
  if (d_tau) *d_tau = h->d_tau;
  if (d_delta) *d_delta = h->d_delta;
  if (ld) *ld = h->ld;
  h->pointers_out = true;  // in-place writes are possible from now on: every later getter re-derives counts and moments
  h->dirty = true;
  return 0;
}

int mbt_shard_range(int32_t n_bunches, int32_t world, int32_t rank, int32_t *first, int32_t *count) {
  if (n_bunches < 1 || world < 1 || rank < 0 || rank >= world || !first || !count) return fail(MBT_EINVAL, "bad argument");
  const int chunk = (n_bunches + world - 1) / world;
  *first = std::min(rank * chunk, n_bunches);
  *count = std::max(0, std::min(chunk, n_bunches - rank * chunk));
  return 0;
}

int64_t mbt_shard_exchange_doubles(int32_t n_bunches, int32_t world, int32_t n_lr) {
  if (n_bunches < 1 || world < 1 || n_lr < 0) return -1;
  const int64_t chunk = (n_bunches + world - 1) / world;
  return (int64_t)world * chunk * n_lr * 2;
}

int mbt_shard_turn_begin(mbt_handle *h) {
  if (!h) return fail(MBT_EINVAL, "null argument");
  if (!h->sharded) return fail(MBT_ESTATE, "not a sharded handle");
  if (h->shard_phase != 0) return fail(MBT_ESTATE, "mbt_shard_turn_end has not closed the turn before");
  if (h->turn + 1 > 0xFFFFFFFFll) return fail(MBT_EINVAL, "turn counter would exceed 2^32");
  CU(cudaSetDevice(h->device));
  // the pass over this rank's bunches, then the first half of their wakes: counts, S5, gather cells, moments, and the S6
  // sources into this rank's rows of the exchange buffer
  h->fn_map<<<dim3(h->grid_pass, h->M), kPassThreads, h->smem_pass, h->stream>>>(h->args, h->wargs);
  CU(cudaGetLastError());
  WakeArgs wa = h->wargs;
  wa.part = 1;
  k_wake<<<dim3(h->M, 1), kWakeThreads, h->smem_wake, h->stream>>>(wa);
  CU(cudaGetLastError());
  h->launches += 2;
  h->shard_phase = 1;
  h->dirty = true;
  return 0;
}

int mbt_shard_turn_end(mbt_handle *h) {
  if (!h) return fail(MBT_EINVAL, "null argument");
  if (!h->sharded) return fail(MBT_ESTATE, "not a sharded handle");
  if (h->shard_phase != 1) return fail(MBT_ESTATE, "mbt_shard_turn_begin first");
  CU(cudaSetDevice(h->device));
  // the exchange buffer now holds the sources of ALL bunches: into the history ring, flags raised; then the second half
  // of the wakes of this rank's bunches (phasor gather over all bunches ahead, on any rank) and the closing of the turn
  if (h->R > 0) {
    const int rows = h->Mg;
    k_shard_scatter<<<(rows * h->R + 255) / 256, 256, 0, h->stream>>>(h->xbuf, rows, h->R, h->Mg, h->slots, h->ctrl.p, h->ring_a.p,
                                                                      h->a_ready.p);
    CU(cudaGetLastError());
    h->launches += 1;
  }
  WakeArgs wa = h->wargs;
  wa.part = 2;
  k_wake<<<dim3(h->M, 1), kWakeThreads, h->smem_wake, h->stream>>>(wa);
  CU(cudaGetLastError());
  h->launches += 1;
  h->shard_phase = 0;
  h->turn += 1;
  h->dirty = true;
  h->wake_valid = true;
  return 0;
}

int mbt_invalidate(mbt_handle *h) {
  if (!h) return fail(MBT_EINVAL, "null argument");
  h->dirty = true;
  return 0;
}

int mbt_get_particles(mbt_handle *h, double *tau, double *delta) {
  if (!h || !tau || !delta) return fail(MBT_EINVAL, "null argument");
  int rc = flush(h);
  if (rc) return rc;
  const size_t n = (size_t)h->M * h->Np;
  if (h->ld == h->Np) {
    CU(cudaMemcpyAsync(tau, h->d_tau, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaMemcpyAsync(delta, h->d_delta, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  } else {
    if (h->scratch_a.n < n) { h->scratch_a.release(); CU(h->scratch_a.alloc(n, h->stream)); }
    dim3 grid((unsigned)((h->Np + 255) / 256 < 1024 ? (h->Np + 255) / 256 : 1024), (unsigned)h->M);
    k_pack<<<grid, 256, 0, h->stream>>>(h->d_tau, h->ld, (uint32_t)h->Np, h->scratch_a.p);
    CU(cudaMemcpyAsync(tau, h->scratch_a.p, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    k_pack<<<grid, 256, 0, h->stream>>>(h->d_delta, h->ld, (uint32_t)h->Np, h->scratch_a.p);
    CU(cudaMemcpyAsync(delta, h->scratch_a.p, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    h->launches += 2;
  }
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_set_particles(mbt_handle *h, const double *tau, const double *delta, int64_t turn) {
  if (!h || !tau || !delta || turn < 0 || turn > 0xFFFFFFFFll) return fail(MBT_EINVAL, "bad argument");
  CU(cudaSetDevice(h->device));
  if (h->trans) {  // a pending transverse kick belongs to x', y', which this call does not replace: apply it first
    int rc = flush(h);
    if (rc) return rc;
  }
  const size_t n = (size_t)h->M * h->Np;
  if (h->ld == h->Np) {
    CU(cudaMemcpyAsync(h->d_tau, tau, n * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(h->d_delta, delta, n * sizeof(double), cudaMemcpyHostToDevice, h->stream));
  } else {
    if (h->scratch_a.n < n) { h->scratch_a.release(); CU(h->scratch_a.alloc(n, h->stream)); }
    dim3 grid((unsigned)((h->ld + 255) / 256 < 1024 ? (h->ld + 255) / 256 : 1024), (unsigned)h->M);
    CU(cudaMemcpyAsync(h->scratch_a.p, tau, n * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    k_unpack<<<grid, 256, 0, h->stream>>>(h->scratch_a.p, h->ld, (uint32_t)h->Np, h->d_tau);
    CU(cudaMemcpyAsync(h->scratch_a.p, delta, n * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    k_unpack<<<grid, 256, 0, h->stream>>>(h->scratch_a.p, h->ld, (uint32_t)h->Np, h->d_delta);
    h->launches += 2;
  }
  {
    std::vector<int32_t> zero(h->M, 0);
    int rc = upload_window(h, zero.data(), zero.data());
    if (rc) return rc;
  }
  k_set_ctrl<<<1, 256, 0, h->stream>>>(h->ctrl.p, (uint32_t)turn, 0u, h->a_ready.p, h->Mg * (h->R ? h->R : 1), h->bunch_ready.p, h->M,
                                       h->agg_ready.p, h->bunch_done.p, h->tile_turn.p, (int)h->tile_turn.n);
  if (h->trans) k_set_flags_tr<<<1, 256, 0, h->stream>>>(h->tr_ready.p, h->rw_ready.p, h->bunch_done_tr.p, h->M, (uint32_t)turn);
  CU(cudaGetLastError());
  h->launches += 1;
  CU(cudaMemsetAsync(h->hist.p, 0, sizeof(uint32_t) * h->M * h->nb, h->stream));
  CU(cudaMemsetAsync(h->mom_acc.p, 0, sizeof(double) * h->M * 4, h->stream));
  CU(cudaMemsetAsync(h->nout_acc.p, 0, sizeof(unsigned long long) * h->M, h->stream));
  CU(cudaMemsetAsync(h->ring_a.p, 0, sizeof(cplx) * (h->ring_a.n ? h->ring_a.n : 1), h->stream));
  CU(cudaMemsetAsync(h->ring_A.p, 0, sizeof(cplx) * (h->ring_A.n ? h->ring_A.n : 1), h->stream));
  if (h->trans) CU(cudaMemsetAsync(h->ring_g.p, 0, sizeof(double) * (h->ring_g.n ? h->ring_g.n : 1), h->stream));
  CU(cudaStreamSynchronize(h->stream));
  h->turn = turn;
  h->dirty = true;
  h->wake_valid = false;
  return 0;
}

namespace {
int copy_out_packed(mbt_handle *h, const double *dev, double *host) {
  const size_t n = (size_t)h->M * h->Np;
  if (h->ld == h->Np) {
    CU(cudaMemcpyAsync(host, dev, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  } else {
    if (h->scratch_a.n < n) { h->scratch_a.release(); CU(h->scratch_a.alloc(n, h->stream)); }
    dim3 grid((unsigned)((h->Np + 255) / 256 < 1024 ? (h->Np + 255) / 256 : 1024), (unsigned)h->M);
    k_pack<<<grid, 256, 0, h->stream>>>(dev, h->ld, (uint32_t)h->Np, h->scratch_a.p);
    h->launches += 1;
    CU(cudaMemcpyAsync(host, h->scratch_a.p, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  }
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}
int copy_in_packed(mbt_handle *h, const double *host, double *dev) {
  const size_t n = (size_t)h->M * h->Np;
  if (h->ld == h->Np) {
    CU(cudaMemcpyAsync(dev, host, n * sizeof(double), cudaMemcpyHostToDevice, h->stream));
  } else {
    if (h->scratch_a.n < n) { h->scratch_a.release(); CU(h->scratch_a.alloc(n, h->stream)); }
    dim3 grid((unsigned)((h->ld + 255) / 256 < 1024 ? (h->ld + 255) / 256 : 1024), (unsigned)h->M);
    CU(cudaMemcpyAsync(h->scratch_a.p, host, n * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    k_unpack<<<grid, 256, 0, h->stream>>>(h->scratch_a.p, h->ld, (uint32_t)h->Np, dev);
    h->launches += 1;
  }
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}
}  // namespace

int mbt_get_transverse(mbt_handle *h, double *x, double *xp, double *y, double *yp) {
  if (!h || !h->trans || !x || !xp || !y || !yp) return fail(MBT_EINVAL, "transverse planes not enabled / null argument");
  CU(cudaSetDevice(h->device));
  int rc = flush(h);  // the transverse kick of the last turn may be pending, like the longitudinal one
  if (rc) return rc;
  if ((rc = copy_out_packed(h, h->tx.p, x)) || (rc = copy_out_packed(h, h->txp.p, xp)) ||
      (rc = copy_out_packed(h, h->ty.p, y)) || (rc = copy_out_packed(h, h->typ.p, yp)))
    return rc;
  return 0;
}

int mbt_set_transverse(mbt_handle *h, const double *x, const double *xp, const double *y, const double *yp) {
  if (!h || !h->trans || !x || !xp || !y || !yp) return fail(MBT_EINVAL, "transverse planes not enabled / null argument");
  CU(cudaSetDevice(h->device));
  int rc = flush(h);
  if (rc) return rc;
  if ((rc = copy_in_packed(h, x, h->tx.p)) || (rc = copy_in_packed(h, xp, h->txp.p)) ||
      (rc = copy_in_packed(h, y, h->ty.p)) || (rc = copy_in_packed(h, yp, h->typ.p)))
    return rc;
  if ((rc = rescale_transverse(h))) return rc;
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_get_dipole(mbt_handle *h, double *Sx, double *Sy) {
  if (!h || !h->trans) return fail(MBT_EINVAL, "transverse planes not enabled");
  CU(cudaSetDevice(h->device));
  const size_t row = sizeof(double) * (size_t)h->nb;  // device layout [M][2][nb]
  if (Sx) CU(cudaMemcpy2DAsync(Sx, row, h->S_last.p, 2 * row, row, h->M, cudaMemcpyDeviceToHost, h->stream));
  if (Sy) CU(cudaMemcpy2DAsync(Sy, row, h->S_last.p + h->nb, 2 * row, row, h->M, cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_get_transverse_wake(mbt_handle *h, double *Kx, double *Ky) {
  if (!h || !h->trans) return fail(MBT_EINVAL, "transverse planes not enabled");
  CU(cudaSetDevice(h->device));
  const size_t row = sizeof(double) * (size_t)h->nb;
  if (Kx) CU(cudaMemcpy2DAsync(Kx, row, h->Ktab.p, 2 * row, row, h->M, cudaMemcpyDeviceToHost, h->stream));
  if (Ky) CU(cudaMemcpy2DAsync(Ky, row, h->Ktab.p + h->nb, 2 * row, row, h->M, cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_get_transverse_log(mbt_handle *h, int64_t first_turn, int64_t n, double *out) {
  if (!h || !h->trans || !out || first_turn < 1 || n < 0) return fail(MBT_EINVAL, "bad argument");
  if (first_turn - 1 + n > h->log_cap || first_turn - 1 + n > h->turn) return fail(MBT_ESTATE, "turns not in the log");
  CU(cudaSetDevice(h->device));
  if (n == 0) return 0;
  CU(cudaMemcpyAsync(out, h->log_tr.p + (size_t)(first_turn - 1) * h->M * 4, sizeof(double) * (size_t)n * h->M * 4,
                     cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_get_rw_kick(mbt_handle *h, double *kx, double *ky) {
  if (!h || !h->trans) return fail(MBT_EINVAL, "transverse planes not enabled");
  CU(cudaSetDevice(h->device));
  std::vector<double> v((size_t)h->M * 2);
  CU(cudaMemcpyAsync(v.data(), h->rw.p, sizeof(double) * v.size(), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  for (int b = 0; b < h->M; ++b) {
    if (kx) kx[b] = v[(size_t)b * 2];
    if (ky) ky[b] = v[(size_t)b * 2 + 1];
  }
  return 0;
}

// rows oldest first: row k = turn (turn - Krw + 1 + k), zero for turns < 1; ring slot of turn n' = n' % (Krw + 2)
int mbt_get_rw_history(mbt_handle *h, double *out) {
  if (!h || !h->trans || !out) return fail(MBT_EINVAL, "transverse planes not enabled / null argument");
  CU(cudaSetDevice(h->device));
  const size_t row = (size_t)h->M * 2;
  std::vector<double> ring((size_t)(h->Krw + 2) * row);
  CU(cudaMemcpyAsync(ring.data(), h->ring_g.p, sizeof(double) * ring.size(), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  for (int k = 0; k < h->Krw; ++k) {
    const int64_t np = h->turn - h->Krw + 1 + k;
    for (size_t i = 0; i < row; ++i) out[(size_t)k * row + i] = np >= 1 ? ring[(size_t)(np % (h->Krw + 2)) * row + i] : 0.0;
  }
  return 0;
}

int mbt_set_rw_history(mbt_handle *h, const double *in) {
  if (!h || !h->trans || !in) return fail(MBT_EINVAL, "transverse planes not enabled / null argument");
  CU(cudaSetDevice(h->device));
  const size_t row = (size_t)h->M * 2;
  std::vector<double> ring((size_t)(h->Krw + 2) * row, 0.0);
  for (int k = 0; k < h->Krw; ++k) {
    const int64_t np = h->turn - h->Krw + 1 + k;
    if (np < 1) continue;
    for (size_t i = 0; i < row; ++i) ring[(size_t)(np % (h->Krw + 2)) * row + i] = in[(size_t)k * row + i];
  }
  CU(cudaMemcpyAsync(h->ring_g.p, ring.data(), sizeof(double) * ring.size(), cudaMemcpyHostToDevice, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_moments_transverse(mbt_handle *h, double *out) {
  if (!h || !h->trans || !out) return fail(MBT_EINVAL, "transverse planes not enabled / null argument");
  CU(cudaSetDevice(h->device));
  if (int rc = flush(h)) return rc;
  CU(cudaMemsetAsync(h->mom_tr_acc.p, 0, sizeof(double) * h->M * 8, h->stream));
  k_moments_tr<<<dim3(h->grid_tr, h->M), 256, 0, h->stream>>>(h->tmargs, h->mom_tr_acc.p);
  k_close_moments_tr<<<(h->M + 127) / 128, 128, 0, h->stream>>>(h->M, (uint32_t)h->Np, h->mom_tr_acc.p, h->mom_tr.p);
  h->launches += 2;
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(out, h->mom_tr.p, sizeof(double) * h->M * 8, cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_get_window(mbt_handle *h, int32_t *s_hist, int32_t *s_next) {
  if (!h) return fail(MBT_EINVAL, "null argument");
  CU(cudaSetDevice(h->device));
  if (s_hist) CU(cudaMemcpyAsync(s_hist, h->s_hist.p, sizeof(int32_t) * h->M, cudaMemcpyDeviceToHost, h->stream));
  if (s_next) CU(cudaMemcpyAsync(s_next, h->s_next.p, sizeof(int32_t) * h->M, cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_set_window(mbt_handle *h, const int32_t *s_hist, const int32_t *s_next) {
  if (!h || !s_hist || !s_next) return fail(MBT_EINVAL, "null argument");
  CU(cudaSetDevice(h->device));
  for (int b = 0; b < h->M; ++b)
    if (std::abs(s_hist[b]) > h->s_max || std::abs(s_next[b]) > h->s_max) return fail(MBT_EINVAL, "window shift beyond the bucket");
  int rc = upload_window(h, s_hist, s_next);
  if (rc) return rc;
  h->dirty = true;  // counts and n_in / n_out are re-derived on the new window by the next flush
  return 0;
}

int mbt_get_histogram(mbt_handle *h, uint32_t *out) {
  if (!h || !out) return fail(MBT_EINVAL, "null argument");
  int rc = flush(h);
  if (rc) return rc;
  CU(cudaMemcpyAsync(out, h->hist_last.p, sizeof(uint32_t) * h->M * h->nb, cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_get_wake(mbt_handle *h, double *total, double *sr, double *lr) {
  if (!h) return fail(MBT_EINVAL, "null argument");
  CU(cudaSetDevice(h->device));
  const size_t n = (size_t)h->M * h->nb;
  if (!h->wake_valid) {
    if (total) memset(total, 0, n * sizeof(double));
    if (sr) memset(sr, 0, n * sizeof(double));
    if (lr) memset(lr, 0, n * sizeof(double));
    return 0;
  }
  if (h->scratch_b.n < 3 * n) { h->scratch_b.release(); CU(h->scratch_b.alloc(3 * n, h->stream)); }
  double *dt = h->scratch_b.p, *ds = dt + n, *dl = ds + n;
  k_eval_wake<<<h->M, 256, 0, h->stream>>>(h->M, h->nb, h->R, h->Vsr.p, h->P.p, h->F.p, dt, ds, dl);
  h->launches += 1;
  if (total) CU(cudaMemcpyAsync(total, dt, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  if (sr) CU(cudaMemcpyAsync(sr, ds, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  if (lr) CU(cudaMemcpyAsync(lr, dl, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_get_moment_log(mbt_handle *h, int64_t first_turn, int64_t n, double *out) {
  if (!h || !out || first_turn < 1 || n < 0) return fail(MBT_EINVAL, "bad argument");
  if (first_turn - 1 + n > h->log_cap || first_turn - 1 + n > h->turn) return fail(MBT_ESTATE, "turns not in the log");
  int rc = flush(h);  // closes the moments of the last tracked turn
  if (rc) return rc;
  if (n == 0) return 0;
  CU(cudaMemcpyAsync(out, h->mom_log.p + (size_t)(first_turn - 1) * h->M * 6, sizeof(double) * (size_t)n * h->M * 6,
                     cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_get_lr_history(mbt_handle *h, double *out) {
  if (!h || !out) return fail(MBT_EINVAL, "null argument");
  CU(cudaSetDevice(h->device));
  const int M = h->Mg, R = h->R, K = h->K;  // rows of the whole fill (a sharded handle holds them all)
  if (R == 0 || K == 0) return 0;
  std::vector<cplx> ring((size_t)h->slots * M * R);
  CU(cudaMemcpyAsync(ring.data(), h->ring_a.p, ring.size() * sizeof(cplx), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  for (int k = 0; k < K; ++k) {
    const int64_t t = h->turn - K + 1 + k;
    for (int b = 0; b < M; ++b)
      for (int r = 0; r < R; ++r) {
        cplx a{0.0, 0.0};
        if (t >= 1) a = ring[((size_t)(t % h->slots) * M + b) * R + r];
        double *o = &out[(((size_t)k * M + b) * R + r) * 2];
        o[0] = a.re;
        o[1] = a.im;
      }
  }
  return 0;
}

int mbt_set_lr_history(mbt_handle *h, const double *in) {
  if (!h || !in) return fail(MBT_EINVAL, "null argument");
  CU(cudaSetDevice(h->device));
  const int M = h->Mg, R = h->R, K = h->K;  // rows of the whole fill (a sharded handle holds them all)
  if (R == 0 || K == 0) return 0;
  std::vector<cplx> ring((size_t)h->slots * M * R, cplx{0.0, 0.0});
  for (int k = 0; k < K; ++k) {
    const int64_t t = h->turn - K + 1 + k;
    if (t < 1) continue;
    for (int b = 0; b < M; ++b)
      for (int r = 0; r < R; ++r) {
        const double *i2 = &in[(((size_t)k * M + b) * R + r) * 2];
        ring[((size_t)(t % h->slots) * M + b) * R + r] = cplx{i2[0], i2[1]};
      }
  }
  CU(cudaMemcpyAsync(h->ring_a.p, ring.data(), ring.size() * sizeof(cplx), cudaMemcpyHostToDevice, h->stream));
  k_aggregate_history<<<h->slots, 32, 0, h->stream>>>(M, R, K, h->ring_a.p, h->g_tail.p, h->ring_A.p);
  h->launches += 1;
  CU(cudaGetLastError());
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

int mbt_philox_selftest(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  if (!ctr || !key || !out) return fail(MBT_EINVAL, "null argument");
  uint32_t *d = nullptr;
  CU(cudaMalloc((void **)&d, 4 * sizeof(uint32_t)));
  k_philox_selftest<<<1, 1>>>(ctr[0], ctr[1], ctr[2], ctr[3], philox_expand_key(key[0], key[1]), d);
  cudaError_t e = cudaMemcpy(out, d, 4 * sizeof(uint32_t), cudaMemcpyDeviceToHost);
  cudaFree(d);
  CU(e);
  return 0;
}

int mbt_normal_selftest(uint64_t seed, int64_t n, const uint32_t *ctr, double *out) {
  if (n < 0 || (n > 0 && (!ctr || !out))) return fail(MBT_EINVAL, "bad argument");
  if (n == 0) return 0;
  uint32_t *dc = nullptr;
  double *dz = nullptr;
  LogTabEntry *dl = nullptr;
  CU(cudaMalloc((void **)&dl, sizeof kLogTabHost));
  CU(cudaMemcpy(dl, kLogTabHost, sizeof kLogTabHost, cudaMemcpyHostToDevice));
  CU(cudaMalloc((void **)&dc, (size_t)n * 4 * sizeof(uint32_t)));
  cudaError_t e = cudaMalloc((void **)&dz, (size_t)n * 4 * sizeof(double));
  if (e != cudaSuccess) { cudaFree(dc); CU(e); }
  e = cudaMemcpy(dc, ctr, (size_t)n * 4 * sizeof(uint32_t), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    k_normal_selftest<<<148, 256>>>(n, dc, philox_expand_key((uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)), dl, make_math_tab(), dz);
    e = cudaMemcpy(out, dz, (size_t)n * 4 * sizeof(double), cudaMemcpyDeviceToHost);
  }
  cudaFree(dc);
  cudaFree(dz);
  cudaFree(dl);
  CU(e);
  return 0;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// mbt_bunch_stats_noalloc: the per-bunch statistics of P:l.123-125 for callers that must not allocate device memory.
//
// The handle-based statistics calls keep their per-bunch partial sums in a buffer mbt_create obtained with cudaMalloc.
// Some users of this library cannot afford that: a monitoring hook that runs beside a long mbt_track on a second stream
// (cudaMalloc and cudaFree serialise against everything in flight on the device, so an allocating call would stall the
// tracking stream it is meant to watch), and hosts that have handed all of HBM to a pool of their own (a framework's
// caching allocator, a run sized to the card) where a cudaMalloc from inside a library can simply fail.  For them the
// partial sums of this entry point live in the fixed array below, which is part of the library image: every GPU that
// loads libmbt.so carries its 64 KiB until the process exits, and nothing is allocated or freed at call time.
//
// g_stats_scratch is a __device__ symbol.  In host code its name is only the host-side shadow of that symbol, NOT a
// device address -- handing `g_stats_scratch` itself to a kernel would fault (or, on a system whose GPU can reach host
// memory, quietly sum into the wrong place).  The device address is asked for once per device with
// cudaGetSymbolAddress, with that device current, and that pointer is what the kernels get.
static __device__ __align__(256) double g_stats_scratch[MBT_NOALLOC_MAX_BUNCHES * 8];

namespace {
constexpr int kNoallocMaxDevices = 64;
double *g_stats_scratch_addr[kNoallocMaxDevices];  // device address of g_stats_scratch on device d; nullptr = not looked up
std::mutex g_stats_scratch_mutex;

// First call on a device: resolve the array's address there.  The look-up may make the CUDA runtime load this library's
// module onto the device, which is why the header asks for the first call to be made outside any stream capture.
int stats_scratch_on_current_device(double **out) {
  int dev = -1;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoallocMaxDevices) return fail(MBT_EINVAL, "mbt_bunch_stats_noalloc: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_stats_scratch_mutex);
  if (!g_stats_scratch_addr[dev]) {
    double *p = nullptr;
    CU(cudaGetSymbolAddress((void **)&p, g_stats_scratch));
    if (!p) return fail(MBT_ECUDA, "mbt_bunch_stats_noalloc: cudaGetSymbolAddress returned a null address");
    g_stats_scratch_addr[dev] = p;
  }
  *out = g_stats_scratch_addr[dev];
  return 0;
}
}  // namespace

extern "C" int mbt_bunch_stats_noalloc(const double *d_x, const double *d_xp, const double *d_y, const double *d_yp,
                                       int32_t n_bunches, int64_t n_per_bunch, int64_t ld, double *d_out, void *stream) {
  if (!d_x || !d_xp || !d_y || !d_yp || !d_out) return fail(MBT_EINVAL, "mbt_bunch_stats_noalloc: null argument");
  if (n_bunches < 1) return fail(MBT_EINVAL, "mbt_bunch_stats_noalloc: n_bunches must be at least 1");
  if (n_bunches > MBT_NOALLOC_MAX_BUNCHES) {
    char buf[192];
    snprintf(buf, sizeof buf, "mbt_bunch_stats_noalloc: %d bunches exceed the fixed scratch array (MBT_NOALLOC_MAX_BUNCHES = %d); "
             "split the call or use mbt_moments_transverse", (int)n_bunches, (int)MBT_NOALLOC_MAX_BUNCHES);
    return fail(MBT_EINVAL, buf);
  }
  if (n_per_bunch < 1 || n_per_bunch > 0xFFFFFFFFll) return fail(MBT_EINVAL, "mbt_bunch_stats_noalloc: n_per_bunch must be in 1 .. 2^32-1");
  if (ld < n_per_bunch) return fail(MBT_EINVAL, "mbt_bunch_stats_noalloc: ld is smaller than n_per_bunch");
  double *acc = nullptr;
  if (int rc = stats_scratch_on_current_device(&acc)) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  TMomArgs A;
  A.x = d_x; A.xp = d_xp; A.y = d_y; A.yp = d_yp; A.ld = ld; A.Np = (uint32_t)n_per_bunch; A.tile = 8192;
  const int grid_x = (int)((n_per_bunch + A.tile - 1) / A.tile);
  // The array still holds the sums of whoever called last (on this device, from any thread or stream): the rows this
  // call accumulates into must start from zero.  A memset of existing memory allocates nothing.
  CU(cudaMemsetAsync(acc, 0, sizeof(double) * (size_t)n_bunches * 8, st));
  k_moments_tr<<<dim3(grid_x, n_bunches), 256, 0, st>>>(A, acc);
  k_close_moments_tr<<<(n_bunches + 127) / 128, 128, 0, st>>>(n_bunches, (uint32_t)n_per_bunch, acc, d_out);
  CU(cudaGetLastError());
  return 0;
}
