"""Pins for the oracle's binning, short-range and long-range wake (no GPU).

(d) histogram counts sum to N, equal an independent numpy sort-and-count               [BASELINE north_star (d)]
(e) convolution and long-range sums against O(N^2) brute force on tiny inputs          [north_star (e)]
plus: the resonator wake function against the Fourier transform of the resonator impedance,
the loss factor of a binned Gaussian against the frequency-domain integral, W(0) = W(0+)/2,
geometric-series closed form of the long-range sum, recurrence (lr_mode 1) against the definition.
"""
import math

import numpy as np
import pytest
from scipy import integrate

from paper_1809_00391_b200 import workloads as W


def _re_z(rs, fr, q, w):
    wr = 2 * math.pi * fr
    return rs / (1.0 + q * q * (wr / w - w / wr) ** 2)


def _abs_z(rs, fr, q, w):
    wr = 2 * math.pi * fr
    return rs / math.sqrt(1.0 + q * q * (wr / w - w / wr) ** 2)


# ------------------------------------------------------------------ wake function
@pytest.mark.parametrize("rs,fr,q", [(5e3, 10e9, 1.0), (2e4, 3e9, 4.0), (1e6, 1.2e9, 30.0)])
def test_resonator_wake_is_fourier_transform_of_impedance(orc, rs, fr, q):
    """int_0^inf W(t) exp(-i w t) dt = Z(w) = Rs / (1 + i Q (w_r/w - w/w_r)): real part and modulus."""
    wr = 2 * math.pi * fr
    alpha = wr / (2 * q)
    t_end = 45.0 / alpha                        # exp(-45) ~ 3e-20
    f = lambda t: orc.resonator_wake(rs, fr, q, t)
    for w in [0.5 * wr, 0.93 * wr, wr, 1.4 * wr]:
        n_osc = int(t_end * max(w, wr) / (2 * math.pi)) + 1
        pts = np.linspace(0, t_end, 4 * n_osc + 1)
        re = sum(integrate.quad(lambda t: f(t) * math.cos(w * t), a, b, epsabs=0, epsrel=1e-11)[0]
                 for a, b in zip(pts[:-1], pts[1:]))
        im = sum(integrate.quad(lambda t: f(t) * math.sin(w * t), a, b, epsabs=0, epsrel=1e-11)[0]
                 for a, b in zip(pts[:-1], pts[1:]))
        assert re == pytest.approx(_re_z(rs, fr, q, w), rel=1e-7, abs=1e-9 * rs)
        assert math.hypot(re, im) == pytest.approx(_abs_z(rs, fr, q, w), rel=1e-7)


def test_resonator_wake_special_values(orc):
    rs, fr, q = 5e3, 10e9, 1.0
    wr = 2 * math.pi * fr
    assert orc.resonator_wake(rs, fr, q, -1e-15) == 0.0                          # causal
    # beam-loading theorem: W(0) = W(0+)/2, W(0+) = w_r Rs / Q
    assert orc.resonator_wake(rs, fr, q, 1e-22) == pytest.approx(wr * rs / q, rel=1e-9)
    assert orc.resonator_wake(rs, fr, q, 0.0) == pytest.approx(0.5 * wr * rs / q, rel=1e-15)
    # Z(0) = 0: the wake integrates to zero
    alpha = wr / (2 * q)
    tot = integrate.quad(lambda t: orc.resonator_wake(rs, fr, q, t), 0, 60 / alpha, epsabs=0, epsrel=1e-12, limit=400)[0]
    assert abs(tot) < 1e-9 * rs


def test_loss_factor_of_binned_gaussian_matches_frequency_domain(orc):
    """k = (1/pi) int_0^inf Re Z(w) exp(-w^2 s^2) dw  vs  sum_jk p_j p_k W(c_j - c_k)  (SURVEY 8(c) pin, D10)."""
    rs, fr, q, sig = 5e3, 10e9, 1.0, 10e-12
    k_freq = integrate.quad(lambda w: _re_z(rs, fr, q, w) * math.exp(-(w * sig) ** 2), 1e3, 40 / sig,
                            epsabs=0, epsrel=1e-10, limit=500)[0] / math.pi
    assert k_freq == pytest.approx(6.3905e13, rel=2e-4)                          # SURVEY.md 8(c) value
    for nb, tol in [(200, 4e-4), (1000, 3e-5)]:
        edges = np.linspace(-5 * sig, 5 * sig, nb + 1)
        from scipy.stats import norm
        p = np.diff(norm.cdf(edges / sig))
        p /= p.sum()
        dt = edges[1] - edges[0]
        w = np.array([orc.resonator_wake(rs, fr, q, k * dt) for k in range(nb)])
        v = orc.sr_convolve(w, p)
        assert float(np.dot(p, v)) == pytest.approx(k_freq, rel=tol)


# ------------------------------------------------------------------ histogram (d)
def test_pin_d_histogram_against_numpy_sort_and_count(orc):
    cfg = W.tiny(m=4, n_per_bunch=5003, n_bins=37)
    cfg["fill"]["sigma_tau0_s"] = 30e-12        # a good fraction outside the +-50 ps window
    o = orc.Oracle(cfg)
    for _ in range(3):
        tau, _ = o.particles()
        h = o.histogram()
        m = o.moments()
        lo, hi, nb = cfg["wake"]["tau_lo_s"], cfg["wake"]["tau_hi_s"], cfg["wake"]["n_bins"]
        edges = lo + (hi - lo) * np.arange(nb + 1) / nb
        for b in range(o.M):
            ts = np.sort(tau[b])
            cum = np.searchsorted(ts, edges, side="left")                       # particles strictly below each edge
            want = np.diff(cum)
            assert np.array_equal(h[b], want.astype(np.uint32))
            assert int(h[b].sum()) + int(m[b, 1]) == o.Np
            assert int(m[b, 0]) == int(h[b].sum())
        assert m[:, 1].sum() > 100                                               # the out-of-window policy is exercised
        o.track(1)


def test_histogram_edges(orc):
    cfg = W.tiny(m=1, n_per_bunch=8, n_bins=8)
    o = orc.Oracle(cfg)
    lo, hi, nb = cfg["wake"]["tau_lo_s"], cfg["wake"]["tau_hi_s"], 8
    d = (hi - lo) / nb
    centres = lo + (np.arange(nb) + 0.5) * d
    o.set_particles(centres, np.zeros(8), 0)
    assert np.array_equal(o.histogram()[0], np.ones(8, dtype=np.uint32))        # centre c_j lands in bin j
    tau = np.array([lo, np.nextafter(lo, -1), hi, np.nextafter(hi, -1), math.nan, math.inf, -math.inf, 0.0])
    o.set_particles(tau, np.zeros(8), 0)
    h = o.histogram()[0]
    assert h[0] == 1 and h[7] == 1 and h[4] == 1 and h.sum() == 3                # half-open [lo, hi), NaN/inf out
    assert o.moments()[0, 1] == 5


# ------------------------------------------------------------------ short-range wake (e)
def test_pin_e_sr_convolution_brute_force(orc):
    rng = np.random.default_rng(5)
    for nb in [1, 2, 7, 64, 301]:
        w = rng.standard_normal(nb)
        q = rng.random(nb)
        v = orc.sr_convolve(w, q)
        assert np.allclose(v, np.convolve(w, q)[:nb], rtol=1e-12, atol=1e-13)    # library routine
        tz = np.array([[w[j - k] if j >= k else 0.0 for k in range(nb)] for j in range(nb)])
        assert np.allclose(v, tz @ q, rtol=1e-12, atol=1e-13)                    # lower-triangular Toeplitz
    # single occupied bin k: V[j] = q w[j-k] for j >= k, zero before it (causality)
    nb, k = 50, 17
    w = rng.standard_normal(nb)
    q = np.zeros(nb)
    q[k] = 2.5
    v = orc.sr_convolve(w, q)
    assert np.all(v[:k] == 0.0) and np.array_equal(v[k:], 2.5 * w[: nb - k])


def test_sr_wake_in_tracker_matches_definition_and_recurrence(orc):
    cfg = W.config("c1", n_per_bunch=3000)
    o = orc.Oracle(cfg)
    o.track(2)
    h = o.histogram()[0].astype(np.float64)
    _, vsr, vlr = o.wake()
    assert np.all(vlr == 0.0)
    nb = o.nb
    lo, hi = cfg["wake"]["tau_lo_s"], cfg["wake"]["tau_hi_s"]
    d = (hi - lo) / nb
    r = cfg["wake"]["resonators"][0]
    qk = cfg["fill"]["charge_C"][0] / o.Np * h
    # definition: V_j = sum_k q_k W(c_j - c_k)
    want = np.array([sum(qk[k] * orc.resonator_wake(r["Rs_ohm"], r["fr_Hz"], r["Q"], (j - k) * d) for k in range(j + 1))
                     for j in range(nb)])
    assert np.allclose(vsr[0], want, rtol=1e-12, atol=1e-12 * np.abs(want).max())
    # O(n) complex recurrence for a pure resonator: P <- (P + q_j) e^{lambda d}; V_j = Re[C P_j] + alpha R q_j
    wr = 2 * math.pi * r["fr_Hz"]
    al = wr / (2 * r["Q"])
    wb = math.sqrt(wr * wr - al * al)
    lam = complex(-al, wb)
    cc = 2 * al * r["Rs_ohm"] * complex(1.0, al / wb)
    p = 0j
    rec = np.empty(nb)
    for j in range(nb):
        rec[j] = (cc * p).real + al * r["Rs_ohm"] * qk[j]
        p = (p + qk[j]) * np.exp(lam * d)
    assert np.allclose(vsr[0], rec, rtol=1e-11, atol=1e-11 * np.abs(want).max())


def test_wake_kick_energy_bookkeeping_ngp_and_linear(orc):
    """NGP gather: sum_i (-E0 ddelta_i) = sum_j hist_j V_j (the beam loses what the wake takes).  Linear gather:
    each particle gets the interpolated value between bin centres, edge values held (D12)."""
    for gather in (0, 1):
        cfg = W.tiny(m=2, n_per_bunch=2001, n_bins=25, gather=gather, radiation=0)
        cfg["fill"]["sigma_tau0_s"] = 25e-12
        a = orc.Oracle(cfg)
        a.track(1)
        tau1, delta1 = a.particles()
        v, _, _ = a.wake()
        h = a.histogram()
        # the same turn without any wake source gives the pre-kick delta (tau is untouched by the kick)
        cfg0 = W.tiny(m=2, n_per_bunch=2001, n_bins=25, gather=gather, radiation=0)
        cfg0["fill"]["sigma_tau0_s"] = 25e-12
        cfg0["wake"]["resonators"] = []
        b = orc.Oracle(cfg0)
        b.track(1)
        tau0, delta0 = b.particles()
        assert np.array_equal(tau0, tau1)
        e0 = cfg["ring"]["E0_eV"]
        kick_v = -(delta1 - delta0) * e0
        lo, hi, nb = cfg["wake"]["tau_lo_s"], cfg["wake"]["tau_hi_s"], 25
        t = (tau1 - lo) * (nb / (hi - lo))
        inside = (t >= 0) & (t < nb)
        assert np.all(kick_v[~inside] == 0.0) and (~inside).sum() > 0            # no kick outside the window
        for bb in range(2):
            if gather == 0:
                assert kick_v[bb].sum() == pytest.approx(float(np.dot(h[bb], v[bb])), rel=1e-9)
                j = np.floor(t[bb][inside[bb]]).astype(int)
                assert np.allclose(kick_v[bb][inside[bb]], v[bb][j], rtol=1e-9, atol=1e-12 * np.abs(v).max())
            else:
                centres = np.arange(nb) + 0.5
                want = np.interp(t[bb][inside[bb]], centres, v[bb])              # np.interp holds the edge values
                assert np.allclose(kick_v[bb][inside[bb]], want, rtol=1e-9, atol=1e-9 * np.abs(v).max())


# ------------------------------------------------------------------ long-range wake (e)
def _lr_brute_force(orc, cfg, hists, n, sr_lr_resonators):
    """Physical definition, no phasors: V_LR[b][j] = sum over every earlier passage (b', n') in the K-turn
    window and every bin k of q_{b',n'}[k] * W_r(c_j - c_k + (n-n') T0 + (s_b - s_b') T_rf)."""
    f, w = cfg["fill"], cfg["wake"]
    m, nb, k_hist = len(f["buckets"]), w["n_bins"], w["history_turns"]
    t0, h = cfg["ring"]["T0_s"], cfg["ring"]["h"]
    d = (w["tau_hi_s"] - w["tau_lo_s"]) / nb
    c = w["tau_lo_s"] + (np.arange(nb) + 0.5) * d
    out = np.zeros((m, nb))
    for b in range(m):
        for n2 in range(max(1, n - k_hist), n + 1):
            for b2 in range(m):
                if n2 == n and not f["buckets"][b2] < f["buckets"][b]:
                    continue
                dt = (n - n2) * t0 + (f["buckets"][b] - f["buckets"][b2]) * (t0 / h)
                q = f["charge_C"][b2] / f["n_per_bunch"] * hists[n2][b2].astype(np.float64)
                for r in sr_lr_resonators:
                    for j in range(nb):
                        for k in range(nb):
                            if q[k] != 0.0:
                                out[b, j] += q[k] * orc.resonator_wake(r["Rs_ohm"], r["fr_Hz"], r["Q"], c[j] - c[k] + dt)
    return out


@pytest.mark.parametrize("lr_mode", [0, 1])
def test_pin_e_lr_wake_against_pairwise_brute_force(orc, lr_mode):
    cfg = W.tiny(m=5, n_per_bunch=37, n_bins=8, k_hist=3, n_lr=2)
    o = orc.Oracle(cfg, lr_mode=lr_mode)
    lr_res = [r for r in cfg["wake"]["resonators"] if r["flags"] & W.FLAG_LR]
    hists = {}
    for n in range(1, 8):
        o.track(1)
        hists[n] = o.histogram()
        _, _, vlr = o.wake()
        want = _lr_brute_force(orc, cfg, hists, n, lr_res)
        scale = np.abs(want).max()
        if n == 1:
            assert np.all(vlr[0] == 0.0)                  # nothing precedes the first bunch of the first turn
        assert scale > 0
        assert np.allclose(vlr, want, rtol=0, atol=1e-10 * scale)


@pytest.mark.parametrize("lr_mode", [0, 1])
def test_wake_from_counts_own_counts_bit_equal_other_counts_brute_force(orc, lr_mode):
    """orc_wake_from_counts (steps 5, 6 for other counts of the turn just completed): with the oracle's own counts it
    is orc_get_wake bit for bit and leaves the state alone; with counts moved between bins it equals the written-out
    short-range sum and the physical pairwise long-range sum (no phasors) of those counts."""
    cfg = W.tiny(m=5, n_per_bunch=37, n_bins=8, k_hist=3, n_lr=2)
    o = orc.Oracle(cfg, lr_mode=lr_mode)
    lr_res = [r for r in cfg["wake"]["resonators"] if r["flags"] & W.FLAG_LR]
    sr_res = [r for r in cfg["wake"]["resonators"] if r["flags"] & W.FLAG_SR]
    wk = cfg["wake"]
    nb = wk["n_bins"]
    d = (wk["tau_hi_s"] - wk["tau_lo_s"]) / nb
    w = np.array([sum(orc.resonator_wake(r["Rs_ohm"], r["fr_Hz"], r["Q"], k * d) for r in sr_res) for k in range(nb)])
    hists = {}
    for n in range(1, 7):
        o.track(1)
        hists[n] = o.histogram()
        before = [x.copy() for x in o.wake()] + [o.lr_history().copy()]
        same = o.wake_from_counts(hists[n])
        for a, b in zip(same, before[:3]):
            assert np.array_equal(a, b)
        # move one particle of every bunch to the neighbouring bin (what an edge-adjacent particle does)
        other = hists[n].copy()
        for b in range(other.shape[0]):
            k = int(np.argmax(other[b]))
            other[b, k] -= 1
            other[b, (k + 1) % nb] += 1
        tot, sr, lr = o.wake_from_counts(other)
        q = np.array(cfg["fill"]["charge_C"])[:, None] / cfg["fill"]["n_per_bunch"] * other
        want_sr = np.array([[sum(w[j - k] * q[b, k] for k in range(j + 1)) for j in range(nb)] for b in range(len(q))])
        assert np.allclose(sr, want_sr, rtol=1e-13, atol=0)
        want_lr = _lr_brute_force(orc, cfg, {**hists, n: other}, n, lr_res)
        assert np.allclose(lr, want_lr, rtol=0, atol=1e-10 * np.abs(want_lr).max())
        assert np.array_equal(tot, sr + lr)
        assert not np.array_equal(lr[1:], before[2][1:]) and not np.array_equal(sr, before[1])
        after = [x.copy() for x in o.wake()] + [o.lr_history().copy()]
        for a, b in zip(after, before):
            assert np.array_equal(a, b)                       # the handle is unchanged


def test_lr_recurrence_equals_definition_long_history(orc):
    cfg = W.tiny(m=5, n_per_bunch=101, n_bins=16, k_hist=6, n_lr=3, harmonic=True)
    a = orc.Oracle(cfg, lr_mode=0)
    b = orc.Oracle(cfg, lr_mode=1)
    for n in range(15):
        a.track(1)
        b.track(1)
        va, vb = a.wake()[2], b.wake()[2]
        assert np.allclose(va, vb, rtol=0, atol=1e-11 * np.abs(va).max())
    ta, da = a.particles()
    tb, db = b.particles()
    assert np.allclose(ta, tb, rtol=1e-12, atol=1e-25) and np.allclose(da, db, rtol=1e-11, atol=1e-18)


def test_lr_uniform_fill_geometric_series(orc):
    """Uniform fill, equal charges, every particle in the centre bin: bunch j of turn n sees
    q Re[C sum_{m=1}^{L} g^m], g = exp(lambda T0/M), L = min(K, n-1) M + j."""
    m, k_hist, nb, npb = 4, 3, 9, 10
    cfg = W.tiny(m=m, n_per_bunch=npb, n_bins=nb, k_hist=k_hist, n_lr=1, radiation=0,
                 buckets=[0, 121, 242, 363])
    q = 1.0e-15                                           # tiny charge: nobody leaves the centre bin
    cfg["fill"]["charge_C"] = [q] * m
    cfg["wake"]["resonators"] = [r for r in cfg["wake"]["resonators"] if r["flags"] & W.FLAG_LR]
    for r in cfg["wake"]["resonators"]:
        r["flags"] = W.FLAG_LR
    o = orc.Oracle(cfg)
    o.set_particles(np.zeros((m, npb)), np.zeros((m, npb)), 0)
    r = cfg["wake"]["resonators"][0]
    wr = 2 * math.pi * r["fr_Hz"]
    al = wr / (2 * r["Q"])
    wb = math.sqrt(wr * wr - al * al)
    cc = 2 * al * r["Rs_ohm"] * complex(1.0, al / wb)
    t0 = cfg["ring"]["T0_s"]
    for n in range(1, 7):
        o.track(1)
        h = o.histogram()
        assert np.all(h[:, nb // 2] == npb)
        vlr = o.wake()[2]
        for j in range(m):
            ll = min(k_hist, n - 1) * m + j
            # sum_{m=1..L} Re[C exp(lambda m T0/M)] term by term with the phase reduced in extended precision
            s = 0.0
            for mm in range(1, ll + 1):
                dt = np.longdouble(mm) * np.longdouble(t0) / m
                ph = float((np.longdouble(wb) * dt) % (2 * np.pi * np.longdouble(1)))
                s += (cc * math.exp(-al * float(dt)) * complex(math.cos(ph), math.sin(ph))).real
            assert vlr[j, nb // 2] == pytest.approx(q * s, rel=1e-8, abs=1e-9 * q * abs(cc))


def test_user_sampled_table_resistive_inductive_power_law(orc):
    """a user-sampled short-range table (here R + L + a t^-3/2 power law) is added to the
    resonator table and convolved like it.  Pins: with the table alone, V is the textbook grid form
    R I_j + L (I_j - I_{j-1}) / Delta + power-law sum, written out with numpy; with a resonator as well, the sum."""
    cfg = W.tiny(m=2, n_per_bunch=3000, n_bins=32, n_lr=0)
    wk = cfg["wake"]
    nb = wk["n_bins"]
    delta = (wk["tau_hi_s"] - wk["tau_lo_s"]) / nb
    R, L, A = 700.0, 3.0e-9, 2.0e-4
    tbl = W.sampled_wake_table(nb, delta, r_ohm=R, l_henry=L, rw_amp=A)
    both = W.tiny(m=2, n_per_bunch=3000, n_bins=32, n_lr=0)
    both["wake"]["sr_table"] = tbl
    only = W.tiny(m=2, n_per_bunch=3000, n_bins=32, n_lr=0)
    only["wake"]["sr_table"] = tbl
    only["wake"]["resonators"] = []
    o_res, o_both, o_only = orc.Oracle(cfg), orc.Oracle(both), orc.Oracle(only)
    for o in (o_res, o_both, o_only):
        o.track(1)
    h = o_only.histogram().astype(np.float64)
    v_only = o_only.wake()[1]
    for b in range(2):
        q = h[b] * only["fill"]["charge_C"][b] / only["fill"]["n_per_bunch"]
        cur = q / delta                                            # bin current [A]
        want = R * cur + L * (cur - np.concatenate([[0.0], cur[:-1]])) / delta
        for j in range(nb):
            for k in range(j):
                want[j] += A * ((j - k) * delta) ** -1.5 * q[k]
        assert np.allclose(v_only[b], want, rtol=1e-12, atol=1e-12 * np.abs(want).max())
    # identical particles in all three (the wake kick comes after the binning of turn 1): superposition
    assert np.array_equal(o_res.histogram(), o_both.histogram())
    v_sum = o_res.wake()[1] + v_only
    assert np.allclose(o_both.wake()[1], v_sum, rtol=1e-12, atol=1e-12 * np.abs(v_sum).max())
