"""Thin ctypes binding of the CUDA library (include/mbt.h): argument marshalling only.

Every step of the method runs in the library's CUDA kernels.  There is no CPU fallback: if
``csrc/libmbt.so`` is missing or cannot be loaded, importing a symbol from it raises.
The function names mirror the C ABI (``mbt_create`` -> ``Tracker(cfg)``, ``mbt_track`` -> ``.track(n)``, ...).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libmbt.so")

# every symbol include/mbt.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "mbt_create", "mbt_track", "mbt_moments", "mbt_destroy", "mbt_get_particles", "mbt_set_particles",
    "mbt_get_histogram", "mbt_get_wake", "mbt_get_moment_log", "mbt_get_lr_history", "mbt_set_lr_history", "mbt_get_window", "mbt_set_window",
    "mbt_turn", "mbt_phi_s", "mbt_particle_stride", "mbt_plan_tiles", "mbt_device_pointers", "mbt_invalidate", "mbt_shard_range", "mbt_shard_exchange_doubles", "mbt_shard_turn_begin", "mbt_shard_turn_end",
    "mbt_launch_count", "mbt_launches_per_turn",
    "mbt_get_transverse", "mbt_set_transverse", "mbt_get_dipole", "mbt_get_transverse_wake", "mbt_moments_transverse",
    "mbt_get_rw_kick", "mbt_get_rw_history", "mbt_set_rw_history", "mbt_get_transverse_log",
    "mbt_bunch_stats_noalloc",
    "mbt_last_track_seconds", "mbt_track_profiled", "mbt_philox_selftest", "mbt_normal_selftest", "mbt_last_error", "mbt_version",
]


class Ring(C.Structure):
    _fields_ = [("E0_eV", C.c_double), ("T0_s", C.c_double), ("alpha_c", C.c_double), ("U0_eV", C.c_double),
                ("h", C.c_int32)]


class Cavity(C.Structure):
    _fields_ = [("V_volt", C.c_double), ("m", C.c_int32), ("phase_rad", C.c_double)]


class Radiation(C.Structure):
    _fields_ = [("enable", C.c_int32), ("sigma_delta", C.c_double), ("damping_turns", C.c_double)]


class Fill(C.Structure):
    _fields_ = [("n_bunches", C.c_int32), ("bucket", C.POINTER(C.c_int32)), ("charge_C", C.POINTER(C.c_double)),
                ("n_per_bunch", C.c_int64), ("sigma_tau0_s", C.c_double), ("sigma_delta0", C.c_double)]


class Resonator(C.Structure):
    _fields_ = [("Rs_ohm", C.c_double), ("fr_Hz", C.c_double), ("Q", C.c_double), ("flags", C.c_uint32)]


class Wake(C.Structure):
    _fields_ = [("n_bins", C.c_int32), ("tau_lo_s", C.c_double), ("tau_hi_s", C.c_double),
                ("gather_order", C.c_int32), ("n_res", C.c_int32), ("res", C.POINTER(Resonator)),
                ("history_turns", C.c_int32), ("n_table", C.c_int32), ("sr_table", C.POINTER(C.c_double)),
                ("window_mode", C.c_int32)]


PLANE_FIELDS = ("nu", "alpha", "beta_m", "xi", "eta_m", "etap", "sigma_u_m", "sigma_up", "D_exc", "sigma0_u_m", "sigma0_up")


class Plane(C.Structure):
    _fields_ = [(k, C.c_double) for k in PLANE_FIELDS]


class Transverse(C.Structure):
    _fields_ = [("enable", C.c_int32), ("x", Plane), ("y", Plane), ("n_res", C.c_int32), ("res", C.POINTER(Resonator)),
                ("rw_amp_x", C.c_double), ("rw_amp_y", C.c_double), ("rw_turns", C.c_int32)]


TUNING_FIELDS = ("tile_iters", "pairs_per_thread", "pdl", "stages6", "turn_mode", "verbose", "per_bunch_start")


class Tuning(C.Structure):
    _fields_ = [(k, C.c_int32) for k in TUNING_FIELDS] + [("reserved", C.c_int32 * 1)]


class Shard(C.Structure):
    _fields_ = [("enable", C.c_int32), ("rank", C.c_int32), ("world", C.c_int32), ("d_exchange", C.c_void_p)]


class Params(C.Structure):
    _fields_ = [("ring", Ring), ("n_cav", C.c_int32), ("cav", C.POINTER(Cavity)), ("rad", Radiation),
                ("fill", Fill), ("wake", Wake), ("seed", C.c_uint64), ("log_capacity_turns", C.c_int64),
                ("d_tau", C.c_void_p), ("d_delta", C.c_void_p), ("stream", C.c_void_p), ("device", C.c_int32),
                ("trans", Transverse), ("tuning", Tuning), ("shard", Shard)]


class MbtError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("mbt error %d: %s" % (code, text))
        self.code = code


_lib = None


def lib():
    """Load csrc/libmbt.so (built by paper_1809_00391_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not found: run `python -m paper_1809_00391_b200.build` (no CPU fallback exists)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        H = C.c_void_p
        dp = C.POINTER(C.c_double)
        L.mbt_create.argtypes = [C.POINTER(Params), C.POINTER(H)]
        L.mbt_track.argtypes = [H, C.c_int64]
        L.mbt_moments.argtypes = [H, dp]
        L.mbt_destroy.argtypes = [H]
        L.mbt_get_particles.argtypes = [H, dp, dp]
        L.mbt_set_particles.argtypes = [H, dp, dp, C.c_int64]
        L.mbt_get_histogram.argtypes = [H, C.POINTER(C.c_uint32)]
        L.mbt_get_wake.argtypes = [H, dp, dp, dp]
        L.mbt_get_moment_log.argtypes = [H, C.c_int64, C.c_int64, dp]
        L.mbt_get_lr_history.argtypes = [H, dp]
        L.mbt_set_lr_history.argtypes = [H, dp]
        L.mbt_turn.argtypes = [H]
        L.mbt_turn.restype = C.c_int64
        L.mbt_phi_s.argtypes = [H]
        L.mbt_phi_s.restype = C.c_double
        L.mbt_particle_stride.argtypes = [C.c_int64]
        L.mbt_particle_stride.restype = C.c_int64
        L.mbt_plan_tiles.argtypes = [C.c_int64, C.c_int64, C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_uint32), C.POINTER(C.c_int32)]
        L.mbt_invalidate.argtypes = [H]
        L.mbt_shard_range.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.mbt_shard_exchange_doubles.argtypes = [C.c_int32, C.c_int32, C.c_int32]
        L.mbt_shard_exchange_doubles.restype = C.c_int64
        L.mbt_shard_turn_begin.argtypes = [H]
        L.mbt_shard_turn_end.argtypes = [H]
        L.mbt_launches_per_turn.argtypes = [H]
        L.mbt_device_pointers.argtypes = [H, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_int64)]
        L.mbt_launch_count.argtypes = [H]
        L.mbt_launch_count.restype = C.c_int64
        L.mbt_last_track_seconds.argtypes = [H]
        L.mbt_last_track_seconds.restype = C.c_double
        L.mbt_track_profiled.argtypes = [H, C.c_int64, dp, dp]
        L.mbt_get_window.argtypes = [H, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.mbt_set_window.argtypes = [H, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.mbt_get_transverse.argtypes = [H, dp, dp, dp, dp]
        L.mbt_set_transverse.argtypes = [H, dp, dp, dp, dp]
        L.mbt_get_dipole.argtypes = [H, dp, dp]
        L.mbt_get_transverse_wake.argtypes = [H, dp, dp]
        L.mbt_moments_transverse.argtypes = [H, dp]
        L.mbt_get_transverse_log.argtypes = [H, C.c_int64, C.c_int64, dp]
        L.mbt_get_rw_kick.argtypes = [H, dp, dp]
        L.mbt_get_rw_history.argtypes = [H, dp]
        L.mbt_set_rw_history.argtypes = [H, dp]
        L.mbt_philox_selftest.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.mbt_normal_selftest.argtypes = [C.c_uint64, C.c_int64, C.POINTER(C.c_uint32), dp]
        L.mbt_bunch_stats_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int64, C.c_int64,
                                              C.c_void_p, C.c_void_p]
        L.mbt_last_error.restype = C.c_char_p
        L.mbt_version.restype = C.c_char_p
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ck(rc):
    if rc != 0:
        raise MbtError(rc, lib().mbt_last_error().decode())


def particle_stride(n_per_bunch: int) -> int:
    return int(lib().mbt_particle_stride(int(n_per_bunch)))


def plan_tiles(pairs_per_bunch, stride, n_bunches, slots, tile_iters=0):
    """(pairs per tile, tiles per bunch) a pass would get (host logic, no device needed)."""
    tp, nt = C.c_uint32(), C.c_int32()
    _ck(lib().mbt_plan_tiles(int(pairs_per_bunch), int(stride), int(n_bunches), int(slots), int(tile_iters), C.byref(tp),
                             C.byref(nt)))
    return tp.value, nt.value


def shard_range(n_bunches, world, rank):
    """(first, count): the contiguous bunches `rank` of `world` owns (host logic, no device needed)."""
    a, b = C.c_int32(), C.c_int32()
    _ck(lib().mbt_shard_range(int(n_bunches), int(world), int(rank), C.byref(a), C.byref(b)))
    return a.value, b.value


def shard_exchange_doubles(n_bunches, world, n_lr):
    """Doubles in the exchange buffer of a sharded handle: world * ceil(n_bunches / world) * n_lr * 2."""
    return int(lib().mbt_shard_exchange_doubles(int(n_bunches), int(world), int(n_lr)))


NOALLOC_MAX_BUNCHES = 1024  # MBT_NOALLOC_MAX_BUNCHES of include/mbt.h


def bunch_stats_noalloc(d_x, d_xp, d_y, d_yp, n_bunches, n_per_bunch, ld, d_out, stream=0):
    """mbt_bunch_stats_noalloc: per-bunch mean / rms of four DEVICE arrays [n_bunches][ld] into the DEVICE array
    d_out[n_bunches][8], for callers that may not allocate device memory (a monitor beside a running mbt_track, a host
    whose own pool holds all of HBM): the partial sums live in a fixed 64 KiB array inside the library.  All pointer
    arguments are integer device addresses (e.g. ``tensor.data_ptr()``), `stream` a cudaStream_t as an integer.
    Asynchronous on `stream`; at most NOALLOC_MAX_BUNCHES bunches; calls overlapping on the GPU race (include/mbt.h)."""
    _ck(lib().mbt_bunch_stats_noalloc(C.c_void_p(d_x), C.c_void_p(d_xp), C.c_void_p(d_y), C.c_void_p(d_yp), int(n_bunches),
                                      int(n_per_bunch), int(ld), C.c_void_p(d_out), C.c_void_p(stream)))


def philox_selftest(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    _ck(lib().mbt_philox_selftest(c, k, o))
    return [int(x) for x in o]


def normal_selftest(seed, ctr):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    out = np.empty((ctr.shape[0], 4))
    _ck(lib().mbt_normal_selftest(int(seed), ctr.shape[0], ctr.ctypes.data_as(C.POINTER(C.c_uint32)), _dp(out)))
    return out


def make_params(cfg, log_capacity_turns=0, d_tau=None, d_delta=None, stream=None, device=-1, tuning=None, shard=None):
    """Workload dict (paper_1809_00391_b200.workloads) -> (mbt_params, keep-alive list).
    tuning: dict of mbt_tuning members (mbt.h), e.g. dict(turn_mode=1); omitted members are 0 = the library's choice."""
    f, w = cfg["fill"], cfg["wake"]
    m = len(f["buckets"])
    bucket = (C.c_int32 * m)(*f["buckets"])
    charge = (C.c_double * m)(*f["charge_C"])
    cav = (Cavity * len(cfg["cavities"]))(*[Cavity(c["V_volt"], c["m"], c["phase_rad"]) for c in cfg["cavities"]])
    nres = len(w["resonators"])
    res = (Resonator * max(nres, 1))(*[Resonator(r["Rs_ohm"], r["fr_Hz"], r["Q"], r["flags"]) for r in w["resonators"]])
    tbl = w.get("sr_table")
    tbl = None if tbl is None else np.ascontiguousarray(tbl, dtype=np.float64)
    p = Params()
    p.ring = Ring(**cfg["ring"])
    p.n_cav = len(cfg["cavities"])
    p.cav = cav
    p.rad = Radiation(**cfg["radiation"])
    p.fill = Fill(m, bucket, charge, int(f["n_per_bunch"]), f["sigma_tau0_s"], f["sigma_delta0"])
    p.wake = Wake(int(w["n_bins"]), w["tau_lo_s"], w["tau_hi_s"], int(w["gather_order"]), nres, res,
                  int(w["history_turns"]), 0 if tbl is None else len(tbl), None if tbl is None else _dp(tbl),
                  int(w.get("window_mode", 0)))
    p.seed = int(cfg["seed"])
    p.log_capacity_turns = int(log_capacity_turns)
    p.d_tau = d_tau
    p.d_delta = d_delta
    p.stream = stream
    p.device = int(device)
    for k, v in (tuning or {}).items():
        if k not in TUNING_FIELDS:
            raise KeyError(k)
        setattr(p.tuning, k, int(v))
    if shard:
        p.shard = Shard(1, int(shard["rank"]), int(shard["world"]), shard.get("d_exchange"))
    tr = cfg.get("transverse")
    tres = None
    if tr:
        tres = (Resonator * max(len(tr["resonators"]), 1))(
            *[Resonator(r["Rs_ohm"], r["fr_Hz"], r["Q"], r.get("flags", 1)) for r in tr["resonators"]])
        p.trans = Transverse(1, Plane(**{k: float(tr["x"][k]) for k in PLANE_FIELDS}),
                             Plane(**{k: float(tr["y"][k]) for k in PLANE_FIELDS}), len(tr["resonators"]), tres,
                             float(tr.get("rw_amp_x", 0.0)), float(tr.get("rw_amp_y", 0.0)), int(tr.get("rw_turns", 0)))
    return p, [bucket, charge, cav, res, tbl, tres]


class Tracker:
    """One mbt_handle.  `d_tau` / `d_delta` / `stream` are raw device pointers / cudaStream_t values (ints),
    e.g. ``tensor.data_ptr()`` and ``torch.cuda.current_stream().cuda_stream``."""

    def __init__(self, cfg, log_capacity_turns=0, d_tau=None, d_delta=None, stream=None, device=-1, tuning=None, shard=None):
        """shard: dict(rank=, world=, d_exchange=device pointer) makes this the handle of one rank of a bunch-sharded run
        (mbt_shard in mbt.h); self.M is then the number of bunches this rank owns, self.Mg that of the whole fill."""
        L = lib()
        f, w = cfg["fill"], cfg["wake"]
        self.Mg = len(f["buckets"])
        self.first_bunch, self.M = shard_range(self.Mg, shard["world"], shard["rank"]) if shard else (0, self.Mg)
        self.Np = int(f["n_per_bunch"])
        self.nb = int(w["n_bins"])
        self.R_lr = sum(1 for r in w["resonators"] if r["flags"] & 2)
        self.K = int(w["history_turns"]) if self.R_lr else 0
        self.K_rw = int((cfg.get("transverse") or {}).get("rw_turns", 0))
        p, self._keep = make_params(cfg, log_capacity_turns, d_tau, d_delta, stream, device, tuning, shard)
        self._h = C.c_void_p()
        self._L = L
        _ck(L.mbt_create(C.byref(p), C.byref(self._h)))

    def close(self):
        if getattr(self, "_h", None):
            self._L.mbt_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    @property
    def turn(self):
        return int(self._L.mbt_turn(self._h))

    @property
    def phi_s(self):
        return float(self._L.mbt_phi_s(self._h))

    @property
    def launches_per_turn(self):
        return int(self._L.mbt_launches_per_turn(self._h))

    @property
    def launch_count(self):
        return int(self._L.mbt_launch_count(self._h))

    def track(self, n):
        _ck(self._L.mbt_track(self._h, int(n)))

    def last_track_seconds(self):
        s = float(self._L.mbt_last_track_seconds(self._h))
        if s < 0:
            raise MbtError(-4, self._L.mbt_last_error().decode())
        return s

    def track_profiled(self, n):
        """(pass_seconds, wake_seconds): summed per-kernel device time of n event-bracketed turns."""
        a, b = C.c_double(), C.c_double()
        _ck(self._L.mbt_track_profiled(self._h, int(n), C.byref(a), C.byref(b)))
        return a.value, b.value

    def moments(self, out=None):
        if out is None:
            out = np.empty((self.M, 6))
        _ck(self._L.mbt_moments(self._h, _dp(out)))
        return out

    def particles(self, tau=None, delta=None):
        if tau is None:
            tau = np.empty((self.M, self.Np))
        if delta is None:
            delta = np.empty((self.M, self.Np))
        _ck(self._L.mbt_get_particles(self._h, _dp(tau), _dp(delta)))
        return tau, delta

    def set_particles(self, tau, delta, turn):
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        delta = np.ascontiguousarray(delta, dtype=np.float64)
        if tau.size != self.M * self.Np or delta.size != tau.size:
            raise ValueError("need M*Np coordinates")
        _ck(self._L.mbt_set_particles(self._h, _dp(tau), _dp(delta), int(turn)))

    def histogram(self):
        out = np.empty((self.M, self.nb), dtype=np.uint32)
        _ck(self._L.mbt_get_histogram(self._h, out.ctypes.data_as(C.POINTER(C.c_uint32))))
        return out

    def wake(self):
        tot = np.empty((self.M, self.nb))
        sr = np.empty_like(tot)
        lr = np.empty_like(tot)
        _ck(self._L.mbt_get_wake(self._h, _dp(tot), _dp(sr), _dp(lr)))
        return tot, sr, lr

    def moment_log(self, first_turn, n):
        out = np.empty((n, self.M, 6))
        _ck(self._L.mbt_get_moment_log(self._h, int(first_turn), int(n), _dp(out)))
        return out

    def shard_turn_begin(self):
        _ck(self._L.mbt_shard_turn_begin(self._h))

    def shard_turn_end(self):
        _ck(self._L.mbt_shard_turn_end(self._h))

    def lr_history(self):
        out = np.zeros((max(self.K, 0), self.Mg, max(self.R_lr, 0), 2))
        if out.size:
            _ck(self._L.mbt_get_lr_history(self._h, _dp(out)))
        return out

    def set_lr_history(self, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        if a.size:
            _ck(self._L.mbt_set_lr_history(self._h, _dp(a)))

    def window(self):
        """(s_hist[M], s_next[M]): window shifts in bins (reading D31)."""
        a = np.zeros(self.M, dtype=np.int32)
        b = np.zeros(self.M, dtype=np.int32)
        ip = C.POINTER(C.c_int32)
        _ck(self._L.mbt_get_window(self._h, a.ctypes.data_as(ip), b.ctypes.data_as(ip)))
        return a, b

    def set_window(self, s_hist, s_next):
        a = np.ascontiguousarray(s_hist, dtype=np.int32)
        b = np.ascontiguousarray(s_next, dtype=np.int32)
        ip = C.POINTER(C.c_int32)
        _ck(self._L.mbt_set_window(self._h, a.ctypes.data_as(ip), b.ctypes.data_as(ip)))

    def transverse_particles(self):
        """(x, x', y, y'), each [M][N_p]."""
        out = [np.empty((self.M, self.Np)) for _ in range(4)]
        _ck(self._L.mbt_get_transverse(self._h, *[_dp(a) for a in out]))
        return out

    def set_transverse(self, x, xp, y, yp):
        a = [np.ascontiguousarray(v, dtype=np.float64) for v in (x, xp, y, yp)]
        if any(v.size != self.M * self.Np for v in a):
            raise ValueError("need M*Np coordinates")
        _ck(self._L.mbt_set_transverse(self._h, *[_dp(v) for v in a]))

    def dipole(self):
        sx, sy = np.empty((self.M, self.nb)), np.empty((self.M, self.nb))
        _ck(self._L.mbt_get_dipole(self._h, _dp(sx), _dp(sy)))
        return sx, sy

    def transverse_wake(self):
        kx, ky = np.empty((self.M, self.nb)), np.empty((self.M, self.nb))
        _ck(self._L.mbt_get_transverse_wake(self._h, _dp(kx), _dp(ky)))
        return kx, ky

    def transverse_log(self, first_turn, n):
        """[n][M][4]: mean x, mean y, rms x, rms y at the end of each turn."""
        out = np.empty((n, self.M, 4))
        _ck(self._L.mbt_get_transverse_log(self._h, int(first_turn), int(n), _dp(out)))
        return out

    def rw_kick(self):
        """(kx[M], ky[M]): resistive-wall kick of the last tracked turn [V]."""
        kx, ky = np.zeros(self.M), np.zeros(self.M)
        _ck(self._L.mbt_get_rw_kick(self._h, _dp(kx), _dp(ky)))
        return kx, ky

    def rw_history(self):
        out = np.zeros((self.K_rw, self.M, 2))
        if out.size:
            _ck(self._L.mbt_get_rw_history(self._h, _dp(out)))
        return out

    def set_rw_history(self, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        if a.size:
            _ck(self._L.mbt_set_rw_history(self._h, _dp(a)))

    def moments_transverse(self):
        out = np.empty((self.M, 8))
        _ck(self._L.mbt_moments_transverse(self._h, _dp(out)))
        return out

    def invalidate(self):
        """The particle store was written in place (through device_pointers or caller-owned buffers)."""
        _ck(self._L.mbt_invalidate(self._h))

    def device_pointers(self):
        t, d, ld = C.c_void_p(), C.c_void_p(), C.c_int64()
        _ck(self._L.mbt_device_pointers(self._h, C.byref(t), C.byref(d), C.byref(ld)))
        return t.value, d.value, ld.value
