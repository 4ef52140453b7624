#!/usr/bin/env python
"""bench.py -- throughput of the fused per-turn hot path (macro-particle-turns/s) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c4] [--transverse] [--impl mbt|reference]

A "step" is one tracked turn of the whole hot path over every macro-particle of the
workload.  The workload at N = 1 is BASELINE.json configs[3] ("c4": 363 bunches x 1e5 macro-particles, the
configuration the metric is quoted on), synthetic and seeded (paper_1809_00391_b200/workloads.py).  The particle
store (581 MB) is larger than the 126 MB L2, so no L2 flush is needed between steps.

N > 1: the path does not shard without a per-turn exchange that BASELINE north_star rules out ("no sharding, no
collectives"), so every rank tracks an independent replica of the workload (a parameter-scan replica; DESIGN.md
"Multi-GPU": replicas only) and `value` is the sum over ranks divided by the slowest rank's device time.

--transverse adds the transverse planes to the workload: 6-D state, 96 B per particle-turn,
the dominant kernel is then the fused 6-D pass k_pass6.  The default line is the longitudinal one BASELINE.json names.

--impl reference times the CPU oracle (oracle/, test infrastructure) on this host's cores, on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "macro-particle-turns/s"
BYTES_PER_PARTICLE_TURN = 32.0  # tau, delta read once and written once per turn, fp64
BYTES_PER_PARTICLE_TURN_6D = 96.0  # with the transverse planes: six fp64 coordinates


def _config(args, **over):
    from paper_1809_00391_b200 import workloads as W
    cfg = W.config(args.config, **over)
    if args.transverse:
        cfg["transverse"] = W.transverse_planes(rw_amp_x=2.0e9, rw_amp_y=1.0e9, rw_turns=args.rw_turns)
    return cfg


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(prefix="mbt_clocks_", suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "25"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
            t_end = time.time() + 5.0          # nvidia-smi needs a moment before its first line: wait for it, so that
            while time.time() < t_end and os.path.getsize(self.path) == 0:   # the samples fall inside the timed region
                time.sleep(0.02)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.1)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        try:
            with open(self.path) as f:
                for line in f:
                    c = [x.strip() for x in line.split(",")]
                    if len(c) < 9:
                        continue
                    try:
                        sm.append(float(c[1])); mx.append(float(c[2]))
                    except ValueError:
                        continue
                    try:
                        pw.append(float(c[3]))          # board power draw [W]
                    except ValueError:
                        pass
                    for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                        if v.lower().startswith("active"):
                            reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        if pw:
            pw.sort()
            out.update(power_w=pw[len(pw) // 2])        # median of the samples taken during the region
        return out


def _oracle_sample(args, budget_s, n_steps):
    """Bounded sample of the workload for the CPU oracle: same fill pattern, wake sources, bins and history;
    N_p reduced so that n_steps turns take about budget_s seconds (the oracle runs ~1e7 particle-turns/s/core)."""
    from paper_1809_00391_b200 import workloads as W
    full = W.config(args.config)
    m = len(full["fill"]["buckets"])
    np_full = full["fill"]["n_per_bunch"]
    per_step = budget_s / max(n_steps, 1) * (2.0e6 if args.transverse else 8.0e6)
    np_s = int(max(500, min(np_full, per_step / m)))
    return _config(args, n_per_bunch=np_s), np_s, m


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import orc
    cfg, np_s, m = _oracle_sample(args, 120.0, args.steps + args.warmup)
    o = orc.Oracle(cfg, lr_mode=1)
    o.track(args.warmup)
    t0 = time.perf_counter()
    o.track(args.steps)
    dt = time.perf_counter() - t0
    val = m * np_s * args.steps / dt
    sample = "%s fill/wake/bins, N_p=%d of %d per bunch, %d turns, lr_mode=1" % (args.config, np_s, W_np(args.config), args.steps)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "particle-turns/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_keys(args, 1),
        "cpu_baseline": {"value": val, "unit": "particle-turns/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "particle-turns/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def W_np(name):
    from paper_1809_00391_b200 import workloads as W
    return W.config(name)["fill"]["n_per_bunch"]


def _config_keys(args, world):
    """`config` of the JSON line: the same keys and values in both arms (they describe the workload, not the arm)."""
    from paper_1809_00391_b200 import workloads as W
    state = (BYTES_PER_PARTICLE_TURN_6D if args.transverse else BYTES_PER_PARTICLE_TURN) / 2 * W.n_particles(W.config(args.config))
    return {"workload": _workload_name(args), "parallelism": "replicas x%d" % world,
            "l2": "particle store larger than L2, no flush needed" if state > 126e6 else
                  "particle store fits L2 (latency-bound config, not an HBM roofline)"}


def _workload_name(args):
    from paper_1809_00391_b200 import workloads as W
    name = args.config
    c = W.config(name)
    f, w = c["fill"], c["wake"]
    s = "%s: %d bunches x %d macro-particles, %d bins, %d resonators (%d long-range, %d-turn history), fp64 SoA" % (
        name, len(f["buckets"]), f["n_per_bunch"], w["n_bins"], len(w["resonators"]),
        sum(1 for r in w["resonators"] if r["flags"] & 2), w["history_turns"])
    if args.transverse:
        s += " + transverse planes (6-D state, one transverse broadband resonator)"
        if args.rw_turns:
            s += " + long-range resistive-wall kick (%d-turn history)" % args.rw_turns
    return s


def run_sharded(args):
    """--sharded: the opt-in bunch-sharded path: the fill's bunches are split over the ranks, one
    all-gather of the source phasors per turn (NCCL; none at N = 1).  STRONG scaling: the workload is fixed.  Not the
    default line (BASELINE north_star fixes one GPU, no collectives); at N = 1 it measures what the host-driven turn
    (three or four plain launches per turn enqueued by the host, no graph) costs against mbt_track."""
    import torch
    import torch.distributed as dist
    from paper_1809_00391_b200 import build, sharded, workloads as W
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    cfg = _config(args)
    n_part = W.n_particles(cfg)
    K, Wm = args.steps, args.warmup
    trk = sharded.ShardedTracker(cfg, rank=rank, world=world, device=local)
    trk.track(Wm)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    l0 = trk.tracker.launch_count
    e0.record(trk.stream)
    trk.track(K)
    e1.record(trk.stream)
    launches = trk.tracker.launch_count - l0     # what the handle counted: 3 per turn, 4 with long-range resonators
    torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3
    if world > 1:
        t = torch.tensor([sec], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        sec = float(t.item())
    m = trk.tracker.moments()
    assert np_isfinite(m)
    if rank == 0:
        line = {"metric": METRIC, "value": n_part * K / sec, "unit": "particle-turns/s", "n_gpus": world, "steps": K, "warmup": Wm,
                "ms_per_step": sec / K * 1e3, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic", "config": dict(_config_keys(args, world), parallelism="bunch-sharded x%d" % world),
                "roofline": None, "gpu_launches": int(launches),
                "note": "opt-in sharded path: mbt_shard_turn_begin / all_gather_into_tensor / mbt_shard_turn_end per turn"}
        print(json.dumps(line))
    trk.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def np_isfinite(a):
    import numpy as np
    return bool(np.isfinite(a).all())


def run_mbt(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1809_00391_b200 import build, mbt, workloads as W

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    cfg = _config(args)
    n_part = W.n_particles(cfg)
    bytes_pt = BYTES_PER_PARTICLE_TURN_6D if args.transverse else BYTES_PER_PARTICLE_TURN
    K, Wm = args.steps, args.warmup

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    tuning = {k: v for k, v in (("turn_mode", args.turn_mode), ("tile_iters", args.tile_iters),
                                ("pairs_per_thread", args.pairs_per_thread), ("pdl", args.pdl), ("verbose", args.verbose), ("per_bunch_start", args.per_bunch_start)) if v}
    trk = mbt.Tracker(cfg, log_capacity_turns=0, device=local, tuning=tuning)
    trk.track(Wm)
    trk.moments()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = trk.launch_count
    barrier()
    trk.track(K)                       # device-timed inside the library with CUDA events on its stream
    barrier()
    sec = trk.last_track_seconds()
    launches = trk.launch_count - l0
    clocks = sampler.stop() if rank == 0 else None   # sampled during the timed region only
    if world > 1:
        t = torch.tensor([sec], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        sec = float(t.item())
    value = world * n_part * K / sec

    # per-kernel device time of the same K steps (event-bracketed plain launches), for the roofline.  The board's power
    # controller averages over a fraction of a second: a pause lets this second timed region start from the state the
    # first one started from (idle after the warm-up), instead of inheriting its heat.
    pause_s = float(os.environ.get("MBT_BENCH_PAUSE_S", "2.0"))
    time.sleep(pause_s)
    pass_s, wake_s = trk.track_profiled(min(K, 2000))
    kp = min(K, 2000)
    peak, peak_src = _peaks()
    achieved = bytes_pt * n_part / (pass_s / kp) / 1e9
    one_launch = trk.launches_per_turn == 1
    roofline = {"bound": "hbm", "kernel": "k_pass6<true>" if args.transverse else
                ("k_pass<true> (one launch per turn: pass + wake of the bunches it completes)" if one_launch else "k_pass<true>"),
                "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": None, "traffic_source": None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": bytes_pt * n_part,
                "pass_ms": pass_s / kp * 1e3, "wake_ms": wake_s / kp * 1e3,
                "pass_share_of_step": pass_s / (pass_s + wake_s),
                "whole_step_frac": bytes_pt * n_part / (sec / K) / 1e9 / peak,
                "timing": "CUDA events around each launch, %d turns of plain launches, started %.1f s after the graph-replayed "
                          "timed region (same idle start for both; the board is power-capped after ~0.1 s of load).  pass_ms is the kernel ALONE: "
                          "events between the launches serialise them, whereas in the graph-replayed step (ms_per_step) the wake kernel "
                          "runs beside the tail of its pass and the head of the next one (per-bunch flags, DESIGN.md 7.1) -- so the step "
                          "can be shorter than pass_ms + wake_ms, and even than pass_ms; whole_step_frac = algorithmic bytes / "
                          "ms_per_step / peak" % (kp, pause_s)}
    # DRAM bytes of one launch from the committed `ncu --set full` capture of this workload (profiles/traffic_<cfg>.txt)
    try:
        with open(os.path.join(ROOT, "profiles", "traffic_%s%s.txt" % (args.config, "t" if args.transverse else ""))) as f:
            for ln in f:
                if ln.startswith("dram_bytes_per_launch"):
                    roofline["traffic"] = float(ln.split()[1])
                    roofline["traffic_source"] = ("profiles/%s: dram__bytes_read.sum + dram__bytes_write.sum of one launch from the "
                                                  "committed `ncu --set full` capture named there (not measured in this run)" %
                                                  os.path.basename(f.name))
    except Exception:
        pass

    # the sustained state: the config's full number of turns (what a real run sees: after ~0.1 s of this load the board
    # sits at its power cap), bounded in wall time; then, without a pause, the per-kernel timing in that same state
    sustained = None
    if args.sustained:
        T = int(min(cfg["n_turns"], max(K, args.sustained_seconds / (sec / K))))
        samp2 = ClockSampler(local)
        if rank == 0:
            samp2.start()
        barrier()
        trk.track(T)
        barrier()
        sec_s = trk.last_track_seconds()
        kp2 = min(T, 1000)
        pass_s2, wake_s2 = trk.track_profiled(kp2)
        clocks2 = samp2.stop() if rank == 0 else None
        if world > 1:
            t = torch.tensor([sec_s], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            sec_s = float(t.item())
        sustained = {"steps": T, "value": world * n_part * T / sec_s, "ms_per_step": sec_s / T * 1e3,
                     "pass_ms": pass_s2 / kp2 * 1e3, "wake_ms": wake_s2 / kp2 * 1e3,
                     "frac": bytes_pt * n_part / (pass_s2 / kp2) / 1e9 / peak,
                     "whole_step_frac": bytes_pt * n_part / (sec_s / T) / 1e9 / peak, "clocks": clocks2,
                     # energy: median board power of rank 0's GPU over the region x the time of a turn / particles of a turn
                     "power_w_median": (clocks2 or {}).get("power_w"),
                     "joules_per_particle_turn": ((clocks2["power_w"] * (sec_s / T) / n_part)
                                                  if clocks2 and clocks2.get("power_w") else None),
                     "what": "mbt_track(%d) of the config's %d turns, graph replay, CUDA events; then %d event-bracketed turns "
                             "with no pause (pass_ms, frac: the dominant kernel in the power-capped state)" % (T, cfg["n_turns"], kp2)}
    trk.close()

    # end to end through the C ABI with HOST buffers: upload the particle state from pinned host memory, track K
    # turns with the per-turn statistics log, read the statistics back (what the paper's host loop does, P:l.123)
    e2e = None
    if True:
        ld = n_part // len(cfg["fill"]["buckets"])
        h_tau = torch.empty(n_part, dtype=torch.float64).pin_memory()
        h_delta = torch.empty(n_part, dtype=torch.float64).pin_memory()
        t2 = mbt.Tracker(cfg, log_capacity_turns=K, device=local, tuning=tuning)
        tau0, delta0 = t2.particles(h_tau.numpy().reshape(len(cfg["fill"]["buckets"]), ld),
                                    h_delta.numpy().reshape(len(cfg["fill"]["buckets"]), ld))
        out = np.empty((K, t2.M, 6))
        barrier()
        tr0 = t2.transverse_particles() if args.transverse else None
        barrier()
        t0 = time.perf_counter()
        t2.set_particles(tau0, delta0, 0)          # H2D of the whole state (pinned host memory)
        if tr0 is not None:
            t2.set_transverse(*tr0)                # ... and of the four transverse coordinates (pageable host memory)
        t2.track(K)
        out = t2.moment_log(1, K)                  # D2H of the per-turn statistics
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": world * n_part * K / dt, "unit": "particle-turns/s",
               "h2d_bytes_per_step": (48.0 if args.transverse else 16.0) * n_part / K, "d2h_bytes_per_step": float(out.nbytes) / K,
               "what": "mbt_set_particles (pinned host -> device) + mbt_track(K) + mbt_get_moment_log (device -> host), wall clock"}
        assert np.isfinite(out).all()
        t2.close()

    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        from oracle import orc
        turns = 2
        t0 = time.perf_counter()
        o = orc.Oracle(cfg, lr_mode=1)
        t_init = time.perf_counter() - t0
        t0 = time.perf_counter()
        o.track(turns)
        dt = time.perf_counter() - t0
        cpu = {"value": n_part * turns / dt, "unit": "particle-turns/s", "cores": 1, "kind": "oracle",
               "sample": "full %s state, %d turns, lr_mode=1 (init %.1f s not timed)" % (args.config, turns, t_init),
               "host_cores_available": os.cpu_count()}
        o.close()

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": "particle-turns/s", "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": sec / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": _config_keys(args, world),
            "roofline": roofline, "sustained": sustained, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
            "clocks": clocks, "tuning": tuning or "library's choice",
            "algorithmic_GBps_whole_step": bytes_pt * value / world / 1e9,
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", default="c4")
    ap.add_argument("--transverse", action="store_true")
    ap.add_argument("--rw-turns", type=int, default=0, help="with --transverse: resistive-wall history depth (0: off)")
    ap.add_argument("--impl", default="mbt", choices=["mbt", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sustained", dest="sustained", action="store_false", help="skip the full-length sustained run")
    ap.add_argument("--sustained-seconds", type=float, default=8.0, help="device-time bound of the sustained run")
    ap.add_argument("--turn-mode", type=int, default=0, help="mbt_tuning.turn_mode (0: the library's choice)")
    ap.add_argument("--tile-iters", type=int, default=0, help="mbt_tuning.tile_iters")
    ap.add_argument("--pairs-per-thread", type=int, default=0, help="mbt_tuning.pairs_per_thread")
    ap.add_argument("--pdl", type=int, default=0, help="mbt_tuning.pdl")
    ap.add_argument("--verbose", type=int, default=0)
    ap.add_argument("--per-bunch-start", type=int, default=0, help="mbt_tuning.per_bunch_start")
    ap.add_argument("--sharded", action="store_true", help="opt-in bunch-sharded path (strong scaling; see run_sharded)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    if args.sharded:
        return run_sharded(args)
    return run_mbt(args)


if __name__ == "__main__":
    sys.exit(main())
