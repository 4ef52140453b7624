"""Pins of the oracle's long-range resistive-wall kick on the transverse planes (P:l.117-119;
DESIGN.md readings W1..W5): brute-force pairwise sum from the recorded centroids, closed forms for a frozen offset
(single bunch: partial sums of k^-1/2; uniform fill: one contiguous sum over bucket distances), the kick reaching
every particle, switches."""
import math

import numpy as np
import pytest

from paper_1809_00391_b200 import workloads as W

ZETA_HALF = -1.4603545088095868   # Riemann zeta(1/2)


def _sum_inv_sqrt(n):
    """sum_{k=1..n} k^-1/2 by Euler-Maclaurin (n >= 64: error < 1e-12); small n written out."""
    if n < 64:
        return sum(1.0 / math.sqrt(k) for k in range(1, n + 1))
    return 2 * math.sqrt(n) + ZETA_HALF + 0.5 / math.sqrt(n) - 1.0 / (24 * n**1.5) + 1.0 / (384 * n**3.5)


def _cfg(m=1, n_per_bunch=50, buckets=None, rw_turns=3, amp=(2.0e9, -0.7e9), frozen=True, **kw):
    cfg = W.tiny(m=m, n_per_bunch=n_per_bunch, n_bins=16, n_lr=0, radiation=0, buckets=buckets, **kw)
    cfg["wake"]["resonators"] = []
    tr = W.transverse_planes(xi_x=0.0, xi_y=0.0, eta_x=0.0)
    tr["resonators"] = []
    if frozen:                                   # integer tunes: the one-turn map is the identity, offsets stay put
        tr["x"]["nu"], tr["y"]["nu"] = 18.0, 5.0
    tr["rw_amp_x"], tr["rw_amp_y"], tr["rw_turns"] = amp[0], amp[1], rw_turns
    cfg["transverse"] = tr
    return cfg


def test_sum_helper():
    for n in (1, 5, 64, 100, 1000):
        assert abs(_sum_inv_sqrt(n) - sum(1.0 / math.sqrt(k) for k in range(1, n + 1))) < 1e-9


def test_single_bunch_frozen_offset_partial_sums(orc):
    """One bunch held at x0, y0: kick of turn n = Q u0 A sum_{k=1..min(K, n-1)} (k T0)^-1/2, constant from turn K+1 on;
    x' grows by kick / E0 per turn for every particle."""
    K = 20
    cfg = _cfg(m=1, n_per_bunch=40, rw_turns=K)
    o = orc.Oracle(cfg)
    n_p = 40
    x0, y0 = 2.0e-3, -5.0e-4
    o.set_transverse(np.full((1, n_p), x0), np.zeros((1, n_p)), np.full((1, n_p), y0), np.zeros((1, n_p)))
    q, e0, t0 = cfg["fill"]["charge_C"][0], cfg["ring"]["E0_eV"], cfg["ring"]["T0_s"]
    ax, ay = cfg["transverse"]["rw_amp_x"], cfg["transverse"]["rw_amp_y"]
    xp_prev = np.zeros(n_p)
    for n in range(1, K + 6):
        o.track(1)
        kx, ky = o.rw_kick()
        s = _sum_inv_sqrt(min(K, n - 1)) / math.sqrt(t0)
        x, xp, y, yp = o.transverse_particles()
        # the offsets drift by beta sin(2 pi nu) x' ~ 1e-15 x' per turn at an integer tune: use the actual centroid
        assert abs(kx[0] - q * x0 * ax * s) <= 1e-9 * abs(q * x0 * ax * s) + 1e-30
        assert abs(ky[0] - q * y0 * ay * s) <= 1e-9 * abs(q * y0 * ay * s) + 1e-30
        assert np.allclose(xp[0] - xp_prev, kx[0] / e0, rtol=1e-9, atol=1e-16)    # (gamma sin(2 pi nu) x0 ~ 1e-18 per turn)
        xp_prev = xp[0].copy()
    assert kx[0] != 0.0


def test_uniform_fill_contiguous_distance_sum(orc):
    """Every bucket filled, every bunch at the same offset and charge: the sources of bunch b at turn n > K sit at the
    bucket distances d = 1 .. K h + s_b without a gap (the bunches ahead in this turn, then K full turns), so
    kick_b = Q u0 A / sqrt(T_rf) sum_{d=1..K h + s_b} d^-1/2."""
    h, K, n_p = 484, 2, 2
    cfg = _cfg(m=h, n_per_bunch=n_p, buckets=list(range(h)), rw_turns=K)
    cfg["fill"]["charge_C"] = [1.0e-9] * h
    o = orc.Oracle(cfg)
    x0 = 1.0e-3
    o.set_transverse(np.full((h, n_p), x0), np.zeros((h, n_p)), np.full((h, n_p), -x0), np.zeros((h, n_p)))
    o.track(K + 1)
    kx, ky = o.rw_kick()
    t_rf = cfg["ring"]["T0_s"] / h
    ax, ay = cfg["transverse"]["rw_amp_x"], cfg["transverse"]["rw_amp_y"]
    for b in (0, 1, 7, 200, 483):
        want = 1.0e-9 * x0 / math.sqrt(t_rf) * _sum_inv_sqrt(K * h + b)
        assert abs(kx[b] - ax * want) < 1e-8 * abs(ax * want)
        assert abs(ky[b] + ay * want) < 1e-8 * abs(ay * want)


def test_pairwise_bruteforce_from_recorded_centroids(orc):
    """Irregular fill, unequal charges, moving offsets (real tunes): the kick of every turn against the pairwise sum
    written out in numpy from the centroids recorded turn by turn; same-turn sources are the bunches AHEAD only."""
    K, n_p, turns = 3, 64, 9
    cfg = _cfg(m=5, n_per_bunch=n_p, rw_turns=K, frozen=False)
    o = orc.Oracle(cfg)
    x, xp, y, yp = o.transverse_particles()
    off = np.array([[1e-3], [-2e-3], [5e-4], [0.0], [3e-3]])
    o.set_transverse(x + off, xp, y - 0.5 * off, yp)
    bk, qb = cfg["fill"]["buckets"], np.array(cfg["fill"]["charge_C"])
    t0, hh = np.longdouble(cfg["ring"]["T0_s"]), cfg["ring"]["h"]
    amp = (cfg["transverse"]["rw_amp_x"], cfg["transverse"]["rw_amp_y"])
    g = {}
    for n in range(1, turns + 1):
        o.track(1)
        m = o.moments_transverse()
        g[n] = np.stack([qb * m[:, 0], qb * m[:, 2]], axis=1)          # the kick acts on u' only: u is the turn's final one
        kx, ky = o.rw_kick()
        for b in range(5):
            want = np.zeros(2)
            for n2 in range(max(1, n - K), n + 1):
                for b2 in range(5):
                    if n2 == n and bk[b2] >= bk[b]:
                        continue
                    dt = float((n - n2) * t0 + (bk[b] - bk[b2]) * (t0 / hh))
                    want += g[n2][b2] / math.sqrt(dt)
            got = np.array([kx[b], ky[b]])
            assert np.all(np.abs(got - np.array(amp) * want) <= 1e-12 * np.abs(np.array(amp) * want).max() + 1e-300)
    hist = o.rw_history()
    assert hist.shape == (K, 5, 2) and np.allclose(hist[-1], g[turns], rtol=0, atol=0)
    assert np.array_equal(hist[0], g[turns - K + 1])


def test_kick_reaches_every_particle_and_switches(orc):
    """Same state, with and without the resistive wall: x' differs by kick / E0 for EVERY particle of the bunch, also
    those outside the bin window (W4); x, y, tau, delta untouched; rw_turns = 0 or zero amplitudes switch it off."""
    cfg = _cfg(m=3, n_per_bunch=200, rw_turns=2, frozen=False)
    cfg0 = _cfg(m=3, n_per_bunch=200, rw_turns=0, frozen=False)
    o, o0 = orc.Oracle(cfg), orc.Oracle(cfg0)
    tau, delta = o.particles()
    tau = tau.copy()
    tau[:, :5] = 80e-12                                              # outside the +-50 ps window
    x, xp, y, yp = o.transverse_particles()
    for oo in (o, o0):
        oo.set_particles(tau, delta, 0)
        oo.set_transverse(x + 1e-3, xp, y + 2e-3, yp)
    o.track(1); o0.track(1)                                          # turn 1: first bunch has no source yet
    o.track(1); o0.track(1)
    assert o.moments()[0, 1] >= 5
    kx, ky = o.rw_kick()
    a, a0 = o.transverse_particles(), o0.transverse_particles()
    assert np.array_equal(o.particles()[0], o0.particles()[0])
    assert np.any(kx != 0) and np.any(ky != 0) and not np.any(o0.rw_kick()[0])
    # two turns: the first turn's kick has rotated into x; compare a single turn from a common state instead
    s = [v.copy() for v in a0]
    o.set_transverse(*s); o0.set_transverse(*s)
    o.set_particles(*o0.particles(), 2); o0.set_particles(*o0.particles(), 2)
    o.track(1); o0.track(1)
    kx, ky = o.rw_kick()
    a, a0 = o.transverse_particles(), o0.transverse_particles()
    e0 = cfg["ring"]["E0_eV"]
    assert np.array_equal(a[0], a0[0]) and np.array_equal(a[2], a0[2])
    assert np.allclose(a[1] - a0[1], (kx / e0)[:, None], rtol=1e-9, atol=1e-25)
    assert np.allclose(a[3] - a0[3], (ky / e0)[:, None], rtol=1e-9, atol=1e-25)
    zero = _cfg(m=3, n_per_bunch=20, rw_turns=4, amp=(0.0, 0.0), frozen=False)
    oz = orc.Oracle(zero)
    oz.track(3)
    assert not np.any(oz.rw_kick()[0]) and not np.any(oz.rw_kick()[1])
    bad = _cfg(rw_turns=-1)
    with pytest.raises(Exception):
        orc.Oracle(bad)


def _rw_mode_sum(nu, m_prime, n_bunches, k_turns, t0):
    """Z_m' = sum_j exp(i 2 pi j (nu - m') / M) / sqrt(j T0 / M) over the sources of an equally spaced train of M point
    bunches, j = 1 .. K M + b counted in bunch spacings (averaged over the witness b: the K-turn cut is b-dependent)."""
    z = 0.0
    for b in range(n_bunches):
        j = np.arange(1, k_turns * n_bunches + b + 1)
        z += np.sum(np.exp(2j * np.pi * j * (nu - m_prime) / n_bunches) / np.sqrt(j * t0 / n_bunches))
    return z / n_bunches


def test_resistive_wall_coupled_bunch_growth_rate(orc):
    """Whole loop against linear theory: M = 22 equally spaced rigid bunches (one macro-particle each), betatron tune
    18.2.  In turn-sampled coordinates a = x / sqrt(beta) + i sqrt(beta) x' the eigen-patterns of the train are
    a_b ~ exp(i 2 pi (m' - nu) b / M), and to first order in the wake a turn multiplies mode m' by
    exp(-i mu) (1 + i kappa beta Z_m' / 2), kappa = Q A / E0: growth rate -kappa beta Im Z_m' / 2 per turn, fastest for
    m' = ceil(nu) = 19 (the classic resistive-wall mode), damped for m' = 17 (m' = 18 sits 0.2 below the tune, where
    the 30-turn cut of the history still moves its slowly converging sum by 10 %: not used).  Fitted, 5 %."""
    M, K, turns = 22, 30, 1200
    h = 484
    cfg = _cfg(m=M, n_per_bunch=1, buckets=list(range(0, h, h // M)), rw_turns=K, frozen=False, amp=(0.0, 0.0))
    cfg["fill"]["charge_C"] = [1.0e-9] * M
    tr = cfg["transverse"]
    nu, beta = tr["x"]["nu"], tr["x"]["beta_m"]
    q, e0, t0 = 1.0e-9, cfg["ring"]["E0_eV"], cfg["ring"]["T0_s"]
    z19, z18 = _rw_mode_sum(nu, 19, M, K, t0), _rw_mode_sum(nu, 17, M, K, t0)
    assert z19.imag < 0 < z18.imag
    amp = 2.0e-3 / (-q * beta * z19.imag / (2 * e0))               # growth 2e-3 per turn for m' = 19
    tr["rw_amp_x"] = amp
    want19, want18 = -q * amp / e0 * beta * z19.imag / 2, -q * amp / e0 * beta * z18.imag / 2
    o = orc.Oracle(cfg)
    b = np.arange(M)
    a0 = 1.0e-4 * (np.exp(2j * np.pi * (19 - nu) * b / M) + np.exp(2j * np.pi * (17 - nu) * b / M))
    zero = np.zeros((M, 1))
    o.set_transverse((math.sqrt(beta) * a0.real)[:, None], (a0.imag / math.sqrt(beta))[:, None], zero, zero)
    amp19, amp18 = np.empty(turns), np.empty(turns)
    for n in range(turns):
        o.track(1)
        x, xp, _, _ = o.transverse_particles()
        a = x[:, 0] / math.sqrt(beta) + 1j * math.sqrt(beta) * xp[:, 0]
        amp19[n] = abs(np.sum(a * np.exp(-2j * np.pi * (19 - nu) * b / M)))
        amp18[n] = abs(np.sum(a * np.exp(-2j * np.pi * (17 - nu) * b / M)))
    t = np.arange(turns)
    g19 = np.polyfit(t[100:], np.log(amp19[100:]), 1)[0]
    g18 = np.polyfit(t[100:600], np.log(amp18[100:600]), 1)[0]
    assert abs(want19 - 2.0e-3) < 1e-12
    assert abs(g19 / want19 - 1) < 0.05, (g19, want19)
    assert want18 < 0 and abs(g18 / want18 - 1) < 0.05, (g18, want18)
