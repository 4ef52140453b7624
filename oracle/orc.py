"""ctypes loader for the CPU ORACLE (test infrastructure only, see oracle/orc.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It converts a workload dict
(paper_1809_00391_b200.workloads) into the oracle's own C structs; it shares no
code with the CUDA binding.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "orc_tracker.cpp")
_LIB = os.path.join(_HERE, "liborc.so")


def build(force: bool = False) -> str:
    """Compile the oracle: -O2, no FMA contraction, single translation unit."""
    hdr = os.path.join(_HERE, "orc.h")
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(hdr))):
        return _LIB
    cmd = ["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-Wall", "-o", _LIB + ".tmp", _SRC]
    subprocess.run(cmd, check=True, cwd=_HERE)
    os.replace(_LIB + ".tmp", _LIB)
    return _LIB


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


class Params(C.Structure):
    _fields_ = [("ring", Ring), ("n_cav", C.c_int32), ("cav", C.POINTER(Cavity)), ("rad", Radiation),
                ("fill", Fill), ("wake", Wake), ("seed", C.c_uint64), ("log_capacity_turns", C.c_int64),
                ("lr_mode", C.c_int32), ("trans", Transverse)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        H = C.c_void_p
        dp = C.POINTER(C.c_double)
        L.orc_create.argtypes = [C.POINTER(Params), C.POINTER(H)]
        L.orc_track.argtypes = [H, C.c_int64]
        L.orc_moments.argtypes = [H, dp]
        L.orc_destroy.argtypes = [H]
        L.orc_get_particles.argtypes = [H, dp, dp]
        L.orc_set_particles.argtypes = [H, dp, dp, C.c_int64]
        L.orc_get_histogram.argtypes = [H, C.POINTER(C.c_uint32)]
        L.orc_get_wake.argtypes = [H, dp, dp, dp]
        L.orc_wake_from_counts.argtypes = [H, C.POINTER(C.c_uint32), dp, dp, dp]
        L.orc_get_moment_log.argtypes = [H, C.c_int64, C.c_int64, dp]
        L.orc_get_lr_history.argtypes = [H, dp]
        L.orc_set_lr_history.argtypes = [H, dp]
        ip = C.POINTER(C.c_int32)
        L.orc_get_window.argtypes = [H, ip, ip]
        L.orc_set_window.argtypes = [H, ip, ip]
        L.orc_window_step.argtypes = [C.c_int32, C.POINTER(C.c_uint32)]
        L.orc_window_step.restype = C.c_int32
        L.orc_get_transverse.argtypes = [H, dp, dp, dp, dp]
        L.orc_set_transverse.argtypes = [H, dp, dp, dp, dp]
        L.orc_get_dipole.argtypes = [H, dp, dp]
        L.orc_get_transverse_wake.argtypes = [H, dp, dp]
        L.orc_moments_transverse.argtypes = [H, dp]
        L.orc_get_transverse_log.argtypes = [H, C.c_int64, C.c_int64, dp]
        L.orc_get_rw_kick.argtypes = [H, dp, dp]
        L.orc_get_rw_history.argtypes = [H, dp]
        L.orc_set_rw_history.argtypes = [H, dp]
        L.orc_transverse_wake.argtypes = [C.c_double] * 4
        L.orc_transverse_wake.restype = C.c_double
        L.orc_betatron_map.argtypes = [C.POINTER(Plane), dp, dp, C.c_double]
        L.orc_betatron_map.restype = None
        L.orc_turn.argtypes = [H]
        L.orc_turn.restype = C.c_int64
        L.orc_phi_s.argtypes = [H]
        L.orc_phi_s.restype = C.c_double
        L.orc_last_error.restype = C.c_char_p
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.orc_philox4x32_10.restype = None
        L.orc_normal_pair.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, dp, dp, dp, dp]
        L.orc_normal_pair.restype = None
        L.orc_normal_quad.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, dp, dp]
        L.orc_normal_quad.restype = None
        L.orc_resonator_wake.argtypes = [C.c_double] * 4
        L.orc_resonator_wake.restype = C.c_double
        L.orc_sr_convolve.argtypes = [C.c_int32, dp, dp, dp]
        L.orc_sr_convolve.restype = None
        L.orc_map_one.argtypes = [H, dp, dp, C.c_double]
        L.orc_map_one.restype = None
        _lib = L
    return _lib


class OrcError(RuntimeError):
    pass


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def transverse_wake(rs, fr, q, t):
    return float(lib().orc_transverse_wake(rs, fr, q, t))


def betatron_map(plane, u, up, delta):
    pl = Plane(**{k: float(plane[k]) for k in PLANE_FIELDS})
    a, b = C.c_double(u), C.c_double(up)
    lib().orc_betatron_map(C.byref(pl), C.byref(a), C.byref(b), float(delta))
    return a.value, b.value


def window_step(hist):
    h = np.ascontiguousarray(hist, dtype=np.uint32)
    return int(lib().orc_window_step(h.size, h.ctypes.data_as(C.POINTER(C.c_uint32))))


def normal_quad(seed, c0, c1, c2, c3):
    """Excitation stream: (u[4], z[4]) of one Philox block (reading D8)."""
    u = (C.c_double * 4)()
    z = (C.c_double * 4)()
    lib().orc_normal_quad(seed, c0, c1, c2, c3, u, z)
    return list(u), list(z)


def normal_pair(seed, c0, c1, c2, c3):
    v = [C.c_double() for _ in range(4)]
    lib().orc_normal_pair(seed, c0, c1, c2, c3, *[C.byref(x) for x in v])
    return tuple(x.value for x in v)  # u1, u2, z_c, z_s


def resonator_wake(rs, fr, q, t):
    return lib().orc_resonator_wake(rs, fr, q, t)


def sr_convolve(w, q):
    w = np.ascontiguousarray(w, dtype=np.float64)
    q = np.ascontiguousarray(q, dtype=np.float64)
    out = np.empty_like(q)
    lib().orc_sr_convolve(len(q), _dp(w), _dp(q), _dp(out))
    return out


class Oracle:
    """One oracle tracker instance built from a workload dict."""

    def __init__(self, cfg, log_capacity_turns=0, lr_mode=0):
        L = lib()
        f, w = cfg["fill"], cfg["wake"]
        self.M = len(f["buckets"])
        self.Np = int(f["n_per_bunch"])
        self.nb = int(w["n_bins"])
        self.R_lr = sum(1 for r in w["resonators"] if r["flags"] & 2)
        self.K = int(w["history_turns"]) if self.R_lr else 0
        self._bucket = (C.c_int32 * self.M)(*f["buckets"])
        self._charge = (C.c_double * self.M)(*f["charge_C"])
        self._cav = (Cavity * len(cfg["cavities"]))(*[Cavity(c["V_volt"], c["m"], c["phase_rad"]) for c in cfg["cavities"]])
        nres = len(w["resonators"])
        self._res = (Resonator * max(nres, 1))(*[Resonator(r["Rs_ohm"], r["fr_Hz"], r["Q"], r["flags"]) for r in w["resonators"]])
        tbl = w.get("sr_table")
        self._tbl = None if tbl is None else np.ascontiguousarray(tbl, dtype=np.float64)
        p = Params()
        p.ring = Ring(**cfg["ring"])
        p.n_cav = len(cfg["cavities"])
        p.cav = self._cav
        p.rad = Radiation(**cfg["radiation"])
        p.fill = Fill(self.M, self._bucket, self._charge, self.Np, f["sigma_tau0_s"], f["sigma_delta0"])
        p.wake = Wake(self.nb, w["tau_lo_s"], w["tau_hi_s"], w["gather_order"], nres, self._res, w["history_turns"],
                      0 if self._tbl is None else len(self._tbl),
                      None if self._tbl is None else _dp(self._tbl), int(w.get("window_mode", 0)))
        p.seed = cfg["seed"]
        p.log_capacity_turns = int(log_capacity_turns)
        p.lr_mode = int(lr_mode)
        tr = cfg.get("transverse")
        self.transverse = bool(tr)
        self.K_rw = 0
        if tr:
            self._tres = (Resonator * max(len(tr["resonators"]), 1))(
                *[Resonator(r["Rs_ohm"], r["fr_Hz"], r["Q"], r.get("flags", 1)) for r in tr["resonators"]])
            p.trans = Transverse(1, Plane(**{k: float(tr["x"][k]) for k in PLANE_FIELDS}),
                                 Plane(**{k: float(tr["y"][k]) for k in PLANE_FIELDS}), len(tr["resonators"]), self._tres,
                                 float(tr.get("rw_amp_x", 0.0)), float(tr.get("rw_amp_y", 0.0)), int(tr.get("rw_turns", 0)))
            self.K_rw = int(tr.get("rw_turns", 0))
        self._h = C.c_void_p()
        self._L = L
        self._ck(L.orc_create(C.byref(p), C.byref(self._h)))

    def _ck(self, rc):
        if rc != 0:
            raise OrcError("oracle error %d: %s" % (rc, self._L.orc_last_error().decode()))

    def close(self):
        if self._h:
            self._L.orc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def turn(self):
        return int(self._L.orc_turn(self._h))

    @property
    def phi_s(self):
        return float(self._L.orc_phi_s(self._h))

    def track(self, n):
        self._ck(self._L.orc_track(self._h, int(n)))

    def moments(self):
        out = np.empty((self.M, 6))
        self._ck(self._L.orc_moments(self._h, _dp(out)))
        return out

    def particles(self):
        tau = np.empty((self.M, self.Np))
        delta = np.empty((self.M, self.Np))
        self._ck(self._L.orc_get_particles(self._h, _dp(tau), _dp(delta)))
        return tau, delta

    def set_particles(self, tau, delta, turn):
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        delta = np.ascontiguousarray(delta, dtype=np.float64)
        assert tau.size == self.M * self.Np and delta.size == tau.size
        self._ck(self._L.orc_set_particles(self._h, _dp(tau), _dp(delta), int(turn)))

    def histogram(self):
        out = np.empty((self.M, self.nb), dtype=np.uint32)
        self._ck(self._L.orc_get_histogram(self._h, out.ctypes.data_as(C.POINTER(C.c_uint32))))
        return out

    def wake(self):
        tot = np.empty((self.M, self.nb))
        sr = np.empty_like(tot)
        lr = np.empty_like(tot)
        self._ck(self._L.orc_get_wake(self._h, _dp(tot), _dp(sr), _dp(lr)))
        return tot, sr, lr

    def wake_from_counts(self, hist):
        """(total, sr, lr) of the turn just completed for other counts of that turn (steps 5, 6; state unchanged)."""
        hist = np.ascontiguousarray(hist, dtype=np.uint32)
        assert hist.shape == (self.M, self.nb)
        tot = np.empty((self.M, self.nb))
        sr = np.empty_like(tot)
        lr = np.empty_like(tot)
        self._ck(self._L.orc_wake_from_counts(self._h, hist.ctypes.data_as(C.POINTER(C.c_uint32)), _dp(tot), _dp(sr), _dp(lr)))
        return tot, sr, lr

    def moment_log(self, first_turn, n):
        out = np.empty((n, self.M, 6))
        self._ck(self._L.orc_get_moment_log(self._h, int(first_turn), int(n), _dp(out)))
        return out

    def lr_history(self):
        out = np.zeros((max(self.K, 0), self.M, max(self.R_lr, 0), 2))
        if out.size:
            self._ck(self._L.orc_get_lr_history(self._h, _dp(out)))
        return out

    def set_lr_history(self, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        if a.size:
            self._ck(self._L.orc_set_lr_history(self._h, _dp(a)))

    def transverse_particles(self):
        """(x, x', y, y'), each [M][N_p]."""
        out = [np.empty((self.M, self.Np)) for _ in range(4)]
        self._ck(self._L.orc_get_transverse(self._h, *[_dp(a) for a in out]))
        return out

    def set_transverse(self, x, xp, y, yp):
        a = [np.ascontiguousarray(v, dtype=np.float64) for v in (x, xp, y, yp)]
        self._ck(self._L.orc_set_transverse(self._h, *[_dp(v) for v in a]))

    def dipole(self):
        sx, sy = np.empty((self.M, self.nb)), np.empty((self.M, self.nb))
        self._ck(self._L.orc_get_dipole(self._h, _dp(sx), _dp(sy)))
        return sx, sy

    def transverse_wake(self):
        kx, ky = np.empty((self.M, self.nb)), np.empty((self.M, self.nb))
        self._ck(self._L.orc_get_transverse_wake(self._h, _dp(kx), _dp(ky)))
        return kx, ky

    def transverse_log(self, first_turn, n):
        """[n][M][4]: mean x, mean y, rms x, rms y at the end of each turn."""
        out = np.empty((n, self.M, 4))
        self._ck(self._L.orc_get_transverse_log(self._h, int(first_turn), int(n), _dp(out)))
        return out

    def rw_kick(self):
        """(kx[M], ky[M]): resistive-wall kick of the last turn [V]."""
        kx, ky = np.zeros(self.M), np.zeros(self.M)
        self._ck(self._L.orc_get_rw_kick(self._h, _dp(kx), _dp(ky)))
        return kx, ky

    def rw_history(self):
        out = np.zeros((self.K_rw, self.M, 2))
        if out.size:
            self._ck(self._L.orc_get_rw_history(self._h, _dp(out)))
        return out

    def set_rw_history(self, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        if a.size:
            self._ck(self._L.orc_set_rw_history(self._h, _dp(a)))

    def moments_transverse(self):
        out = np.empty((self.M, 8))
        self._ck(self._L.orc_moments_transverse(self._h, _dp(out)))
        return out

    def window(self):
        """(s_hist[M], s_next[M]): window shifts in bins (reading D31)."""
        a = np.zeros(self.M, dtype=np.int32)
        b = np.zeros(self.M, dtype=np.int32)
        ip = C.POINTER(C.c_int32)
        self._ck(self._L.orc_get_window(self._h, a.ctypes.data_as(ip), b.ctypes.data_as(ip)))
        return a, b

    def set_window(self, s_hist, s_next):
        a = np.ascontiguousarray(s_hist, dtype=np.int32)
        b = np.ascontiguousarray(s_next, dtype=np.int32)
        ip = C.POINTER(C.c_int32)
        self._ck(self._L.orc_set_window(self._h, a.ctypes.data_as(ip), b.ctypes.data_as(ip)))

    def map_one(self, tau, delta, z=0.0):
        t = C.c_double(tau)
        d = C.c_double(delta)
        self._L.orc_map_one(self._h, C.byref(t), C.byref(d), float(z))
        return t.value, d.value
