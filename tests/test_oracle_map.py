"""Pins for the oracle's single-particle map, radiation step and statistics (no GPU).

(a) small-amplitude synchrotron tune vs Q_s = sqrt(h alpha_c V |cos phi_s| / (2 pi E0))   [BASELINE north_star (a)]
(b) centroid damping time vs the configured damping time                                   [north_star (b)]
(c) equilibrium rms energy spread vs the configured sigma_delta                            [north_star (c)]
plus: synchronous phase / fixed point, Jacobian determinant, no secular growth without radiation
(the energy spread stays flat over 50 000 turns), moments vs numpy.
"""
import math

import numpy as np
import pytest
from scipy.signal import hilbert

from paper_1809_00391_b200 import workloads as W


def _bare(n_per_bunch, radiation, seed=1, **rad):
    cfg = W.config("c1", n_per_bunch=n_per_bunch, radiation=radiation, seed=seed)
    cfg["wake"]["resonators"] = []          # no collective effects
    cfg["radiation"].update(rad)
    return cfg


def _qs_formula(cfg, phi_s):
    r = cfg["ring"]
    return math.sqrt(r["h"] * r["alpha_c"] * cfg["cavities"][0]["V_volt"] * abs(math.cos(phi_s)) / (2 * math.pi * r["E0_eV"]))


def test_synchronous_phase_and_fixed_point(orc):
    o = orc.Oracle(_bare(1, 0))
    # V1 sin(phi_s) = U0 on the stable side for alpha_c > 0 (D3): pi - asin(0.6/1.4)
    assert o.phi_s == pytest.approx(math.pi - math.asin(3.0 / 7.0), abs=1e-15)
    assert o.phi_s == pytest.approx(2.698682, abs=1e-6)
    # the synchronous particle does not move: RF gain cancels the radiation loss (Eq. 1)
    o.set_particles([0.0], [0.0], 0)
    o.track(1000)
    tau, delta = o.particles()
    assert abs(tau[0, 0]) < 1e-22 and abs(delta[0, 0]) < 1e-15
    # alpha_c < 0 (the paper's dc12c lattice, Table 1) puts phi_s on the other side
    cfg = _bare(1, 0)
    cfg["ring"]["alpha_c"] = -1.356e-4
    assert orc.Oracle(cfg).phi_s == pytest.approx(math.asin(3.0 / 7.0), abs=1e-15)


def test_pin_a_small_amplitude_synchrotron_tune(orc):
    n = 1 << 16
    cfg = _bare(1, 0)
    o = orc.Oracle(cfg, log_capacity_turns=n)
    o.set_particles([1.0e-12], [0.0], 0)
    o.track(n)
    x = o.moment_log(1, n)[:, 0, 2]
    x = (x - x.mean()) * np.hanning(n)
    s = np.abs(np.fft.rfft(x))
    k = int(np.argmax(s[1:])) + 1
    a, b, c = np.log(s[k - 1]), np.log(s[k]), np.log(s[k + 1])
    q_meas = (k + 0.5 * (a - c) / (a - 2 * b + c)) / n
    q_form = _qs_formula(cfg, o.phi_s)
    assert q_form == pytest.approx(2.0149168e-3, rel=1e-6)       # SURVEY.md 8(c) pin (a)
    assert q_meas == pytest.approx(q_form, rel=5e-3)             # north_star: formula, 0.5 %
    # exact tune of the linearised kick-drift map: cos(2 pi Q) = 1 + k d / 2
    r = cfg["ring"]
    kk = cfg["cavities"][0]["V_volt"] * (2 * math.pi * r["h"] / r["T0_s"]) * math.cos(o.phi_s) / r["E0_eV"]
    q_lin = math.acos(1.0 + kk * r["alpha_c"] * r["T0_s"] / 2.0) / (2 * math.pi)
    assert q_meas == pytest.approx(q_lin, rel=1e-4)              # FFT peak interpolation is good to ~0.01 bin
    # sharper estimate, independent of the FFT: upward zero crossings of tau(n), linearly interpolated
    y = o.moment_log(1, n)[:, 0, 2]
    up = np.nonzero((y[:-1] < 0) & (y[1:] >= 0))[0]
    tz = up + y[up] / (y[up] - y[up + 1])
    q_zero = (len(tz) - 1) / (tz[-1] - tz[0])
    assert q_zero == pytest.approx(q_lin, rel=2e-6)


def test_drift_uses_updated_delta_jacobian_is_symplectic(orc):
    o = orc.Oracle(_bare(1, 0))
    od = orc.Oracle(_bare(1, 1, sigma_delta=0.0, damping_turns=1.0e4))
    for tau0, del0 in [(0.0, 0.0), (7e-12, -2e-3), (-30e-12, 1e-3)]:
        for orc_i, det_want in [(o, 1.0), (od, 1.0 - 2.0e-4)]:
            ht, hd = 1e-13, 1e-6
            tp, dp = orc_i.map_one(tau0 + ht, del0)
            tm, dm = orc_i.map_one(tau0 - ht, del0)
            tP, dP = orc_i.map_one(tau0, del0 + hd)
            tM, dM = orc_i.map_one(tau0, del0 - hd)
            j11, j21 = (tp - tm) / (2 * ht), (dp - dm) / (2 * ht)
            j12, j22 = (tP - tM) / (2 * hd), (dP - dM) / (2 * hd)
            assert j11 * j22 - j12 * j21 == pytest.approx(det_want, abs=2e-6)
            # kick-then-drift: d tau'/d delta = alpha_c T0 d delta'/d delta (Eq. 2 with the new delta, D1)
            assert j12 == pytest.approx(1e-4 * 9.68e-7 * j22, rel=1e-6)


def test_no_secular_growth_without_radiation(orc):
    """PAPER.md l.146-154 (Fig. 3a): without SR the energy spread stays flat over 50 000 turns.
    The explicit-Euler reading of Eq.(2) would grow every amplitude by e^6 (D1)."""
    cfg = _bare(500, 0)
    o = orc.Oracle(cfg)
    r = cfg["ring"]
    w = 2 * math.pi * r["h"] / r["T0_s"]
    d = r["alpha_c"] * r["T0_s"]
    v = cfg["cavities"][0]["V_volt"] / r["E0_eV"]

    def mean_h():
        tau, delta = o.particles()
        pot = v * (np.cos(w * tau + o.phi_s) / w + tau * math.sin(o.phi_s) - math.cos(o.phi_s) / w)
        return float(np.mean(0.5 * d * delta**2 + pot))

    ws = 2 * math.pi * _qs_formula(cfg, o.phi_s) / r["T0_s"]

    def emittance():
        # linear-motion invariant of the (mismatched, breathing) bunch: rms_delta^2 + (w_s rms_tau / alpha_c)^2
        m = o.moments()[0]
        return m[5] ** 2 + (ws * m[4] / r["alpha_c"]) ** 2

    h0 = mean_h()
    e0 = emittance()
    o.track(50_000)
    h1 = mean_h()
    assert h0 > 0
    assert abs(h1 - h0) / h0 < 2e-3
    assert emittance() == pytest.approx(e0, rel=2e-2)             # breathing only, no e^12 in the squares
    assert 0.8e-3 < o.moments()[0, 5] < 1.4e-3                    # between the two breathing extremes (D20)


def test_pin_b_centroid_damping_time(orc):
    n = 30_000
    n_damp = 1.0e4
    o = orc.Oracle(_bare(1, 1, sigma_delta=0.0, damping_turns=n_damp), log_capacity_turns=n)
    o.set_particles([2.0e-12], [0.0], 0)
    o.track(n)
    x = o.moment_log(1, n)[:, 0, 2]
    env = np.abs(hilbert(x))
    sl = slice(2000, n - 2000)
    slope = np.polyfit(np.arange(n)[sl], np.log(env[sl]), 1)[0]
    assert -1.0 / slope == pytest.approx(n_damp, rel=1e-2)                    # north_star (b)
    assert slope == pytest.approx(0.5 * math.log(1.0 - 2.0 / n_damp), rel=2e-3)  # det of one-turn map = 1 - D_E


def test_pin_c_equilibrium_energy_spread(orc):
    """Protocol of PAPER.md l.158 ('equilibrium' = average over the last turns), with a short damping
    time so that the run stays in the CPU budget: 10 damping times, average over the last half."""
    sig = 1.0e-3
    cfg = _bare(10_000, 1, sigma_delta=sig, damping_turns=1000.0)
    cfg["fill"]["sigma_delta0"] = 0.2e-3       # start far from equilibrium
    cfg["fill"]["sigma_tau0_s"] = 2.0e-12
    n = 10_000
    o = orc.Oracle(cfg, log_capacity_turns=n)
    o.track(n)
    log = o.moment_log(1, n)
    rms = math.sqrt(np.mean(log[n // 2:, 0, 5] ** 2))
    assert rms == pytest.approx(sig, rel=1e-2)                                 # north_star (c)
    assert log[0, 0, 5] < 0.3e-3                                               # it really started elsewhere
    # matched bunch length sigma_tau = alpha_c sigma_delta / omega_s
    r = cfg["ring"]
    ws = 2 * math.pi * _qs_formula(cfg, o.phi_s) / r["T0_s"]
    rms_tau = math.sqrt(np.mean(log[n // 2:, 0, 4] ** 2))
    assert rms_tau == pytest.approx(r["alpha_c"] * sig / ws, rel=2e-2)


def test_excitation_stream_layout(orc):
    """Particle i of bunch b at turn n uses Philox counter (i>>2, b, n, 0) (reading D8: one block serves four consecutive
    particles): words (x0, x1) make the Box-Muller pair of particles 4j, 4j+1, (x2, x3) that of 4j+2, 4j+3; the even particle
    of a pair takes z_c, the odd one z_s."""
    cfg = _bare(5, 1)
    cfg["fill"]["buckets"] = [0, 7]
    cfg["fill"]["charge_C"] = [1e-9, 1e-9]
    o = orc.Oracle(cfg)
    tau0, del0 = o.particles()
    o.track(1)
    tau1, del1 = o.particles()
    o2 = orc.Oracle(cfg)
    for b in range(2):
        for i in range(5):
            _, z = orc.normal_quad(cfg["seed"], i >> 2, b, 1, 0)   # one block per four particles (D8)
            t, d = o2.map_one(tau0[b, i], del0[b, i], z[i & 3])
            assert t == tau1[b, i] and d == del1[b, i]
    # initial distribution: counter (i, b, 0, 1), tau = sigma_tau0 z_c, delta = sigma_delta0 z_s
    _, _, zc, zs = orc.normal_pair(cfg["seed"], 3, 1, 0, 1)
    assert tau0[1, 3] == 10e-12 * zc and del0[1, 3] == 1e-3 * zs


def test_moments_against_numpy(orc):
    cfg = W.tiny(m=3, n_per_bunch=1001)
    o = orc.Oracle(cfg)
    o.track(3)
    tau, delta = o.particles()
    m = o.moments()
    assert np.allclose(m[:, 2], tau.mean(axis=1), rtol=1e-13, atol=0)
    assert np.allclose(m[:, 3], delta.mean(axis=1), rtol=1e-12, atol=1e-20)
    assert np.allclose(m[:, 4], tau.std(axis=1), rtol=1e-13)
    assert np.allclose(m[:, 5], delta.std(axis=1), rtol=1e-13)
    assert np.all(m[:, 0] + m[:, 1] == 1001)
    log_o = orc.Oracle(cfg, log_capacity_turns=3)
    log_o.track(3)
    assert np.array_equal(log_o.moment_log(3, 1)[0], m)
