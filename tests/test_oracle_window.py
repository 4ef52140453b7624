"""Pins of the bunch-following bin window (reading D31; SURVEY.md 8(f) rank 3, P:l.113), oracle only."""
import math
from fractions import Fraction

import numpy as np
import pytest

from paper_1809_00391_b200 import workloads as W


@pytest.fixture(scope="module")
def orc():
    from oracle import orc as o
    o.build()
    return o


def test_window_step_is_the_rounded_centroid_offset(orc):
    # step = rint(sum_k (k + 1/2) c_k / n_in - n_b / 2), half up, exact; 0 for an empty histogram
    rng = np.random.default_rng(3)
    for nb in (2, 3, 8, 301):
        for _ in range(50):
            c = rng.integers(0, 50, nb) * (rng.random(nb) < 0.3)
            got = orc.window_step(c)
            if c.sum() == 0:
                assert got == 0
                continue
            x = Fraction(int(((np.arange(nb) * 2 + 1) * c).sum()), int(2 * c.sum())) - Fraction(nb, 2)
            assert got == math.floor(x + Fraction(1, 2))
    assert orc.window_step([0, 0, 0, 0]) == 0
    assert orc.window_step([0, 0, 0, 7]) == 2 and orc.window_step([7, 0, 0, 0]) == -1   # 1.5 -> 2, -1.5 -> -1 (half up)


def _displaced(cfg, orc, shift_s):
    o = orc.Oracle(cfg)
    tau, delta = o.particles()
    o.set_particles(tau + shift_s, delta, 0)
    return o


def test_window_follows_a_displaced_bunch_and_stops_the_losses(orc):
    """A bunch sitting 30 ps off the bucket centre in a +-50 ps window (sigma 10 ps): the fixed window (D11) keeps
    ~2.3 % of it outside; the following window re-centres itself in whole bins after the first binning."""
    out = {}
    for mode in (0, 1):
        cfg = W.tiny(m=2, n_per_bunch=20000, n_bins=50, n_lr=1, radiation=0)
        cfg["wake"]["window_mode"] = mode
        for r in cfg["wake"]["resonators"]:
            r["Rs_ohm"] *= 1e-6                          # negligible wake: the comparison is about the window
        o = _displaced(cfg, orc, 30e-12)
        o.track(3)
        out[mode] = (o.moments(), o.window(), o.histogram())
    m0, w0, _ = out[0]
    m1, w1, h1 = out[1]
    assert np.all(w0[0] == 0) and np.all(w0[1] == 0)
    assert np.all(m0[:, 1] > 0.015 * 20000)              # Phi(-2) = 2.3 % beyond +50 ps
    delta = 100e-12 / 50
    assert np.all(np.abs(w1[0] - 30e-12 / delta) <= 1)   # shift = 15 bins +- 1
    assert np.all(m1[:, 1] < 10)                         # |x| > 5 sigma: 6e-7 per particle
    k = np.arange(50) + 0.5
    centroid = (h1 * k).sum(axis=1) / h1.sum(axis=1)
    assert np.all(np.abs(centroid - 25.0) <= 1.0)        # re-centred to within a bin (the bunch moves a little per turn)
    assert np.all(m1[:, 0] + m1[:, 1] == 20000)


def test_shifted_window_is_a_translation_of_the_grid(orc):
    """Same particles; window shifted by s whole bins vs particles shifted by -s bins in a fixed window: the same
    histogram (particles are placed on bin centres, away from the edges) and the same short-range wake."""
    nb, npb = 32, 500
    cfg = W.tiny(m=1, n_per_bunch=npb, n_bins=nb, n_lr=0, radiation=0)
    cfg["wake"]["window_mode"] = 1
    d = 100e-12 / nb
    rng = np.random.default_rng(5)
    k = rng.integers(6, 20, npb)
    tau = (-50e-12 + (k + 0.5) * d)[None, :]
    a = orc.Oracle(cfg)
    a.set_particles(tau, np.zeros_like(tau), 0)
    b = orc.Oracle(cfg)
    b.set_particles(tau, np.zeros_like(tau), 0)
    b.set_window([-5], [-5])
    ha, hb = a.histogram()[0], b.histogram()[0]
    assert ha.sum() == npb and hb.sum() == npb
    assert np.array_equal(hb[5:], ha[:-5]) and not hb[:5].any()


def _lr_brute_force_windows(orc, cfg, hists, shifts, n, lr_res):
    """Physical definition with every bin centre at its own window: c = tau_lo + (s + k + 1/2) Delta."""
    f, w = cfg["fill"], cfg["wake"]
    m, nb, k_hist = len(f["buckets"]), w["n_bins"], w["history_turns"]
    t0, h = cfg["ring"]["T0_s"], cfg["ring"]["h"]
    d = (w["tau_hi_s"] - w["tau_lo_s"]) / nb
    out = np.zeros((m, nb))
    for b in range(m):
        cj = w["tau_lo_s"] + (shifts[n][b] + np.arange(nb) + 0.5) * d
        for n2 in range(max(1, n - k_hist), n + 1):
            for b2 in range(m):
                if n2 == n and not f["buckets"][b2] < f["buckets"][b]:
                    continue
                ck = w["tau_lo_s"] + (shifts[n2][b2] + np.arange(nb) + 0.5) * d
                dt = (n - n2) * t0 + (f["buckets"][b] - f["buckets"][b2]) * (t0 / h)
                q = f["charge_C"][b2] / f["n_per_bunch"] * hists[n2][b2].astype(np.float64)
                for r in lr_res:
                    for j in range(nb):
                        for k in range(nb):
                            if q[k] != 0.0:
                                out[b, j] += q[k] * orc.resonator_wake(r["Rs_ohm"], r["fr_Hz"], r["Q"], cj[j] - ck[k] + dt)
    return out


@pytest.mark.parametrize("lr_mode", [0, 1])
def test_lr_wake_with_moving_windows_against_pairwise_brute_force(orc, lr_mode):
    """The long-range sum keeps using true bin-centre times when every bunch's window moves from turn to turn."""
    cfg = W.tiny(m=4, n_per_bunch=41, n_bins=8, k_hist=3, n_lr=2, radiation=0)
    cfg["wake"]["window_mode"] = 1
    o = orc.Oracle(cfg, lr_mode=lr_mode)
    tau, delta = o.particles()
    off = np.array([[12e-12], [-20e-12], [0.0], [33e-12]])
    o.set_particles(tau * 0.4 + off, delta, 0)            # narrow bunches, each at its own offset
    lr_res = [r for r in cfg["wake"]["resonators"] if r["flags"] & W.FLAG_LR]
    hists, shifts = {}, {}
    seen = set()
    for n in range(1, 7):
        o.track(1)
        hists[n] = o.histogram()
        shifts[n] = o.window()[0].copy()
        seen.update(int(s) for s in shifts[n])
        want = _lr_brute_force_windows(orc, cfg, hists, shifts, n, lr_res)
        vlr = o.wake()[2]
        assert np.allclose(vlr, want, rtol=0, atol=1e-10 * np.abs(want).max())
    assert len(seen) >= 3                                  # the windows did move, differently per bunch
