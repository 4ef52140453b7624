"""Pin (f) for the oracle's whole loop: a single narrow-band resonator on an upper synchrotron sideband of a
uniformly filled ring drives coupled-bunch mode mu at the analytic rate (BASELINE north_star (f), 10 %).

Analytic rate (the uniform-fill formula of which PAPER.md l.233 Eq.(7) is the two-term truncation):
    1/tau_mu = alpha_c I0 / (2 (E0/e) T0 w_s) * sum_p w_p Re Z(w_p) exp(-(w_p sigma_tau)^2),
    w_p = (p M + mu) w0 + w_s,  I0 = M q / T0.
The resonator sits at f_r = (p M + mu) f0 + f_s, so mode mu grows and mode M - mu (which sees the resonator on
its lower sideband) is damped at the same rate: both signs are checked, which fixes the sign conventions of the
map (D3), of the wake kick (D9) and of the time ordering in the long-range sum (D14).
"""
import math

import numpy as np
import pytest
from scipy.signal import hilbert

from paper_1809_00391_b200 import workloads as W


def test_pin_f_coupled_bunch_growth_rate_uniform_fill(orc):
    m_b, mu, p = 11, 6, 105
    q_b, rs, qual = 2.0e-9, 1.0e6, 1.0e4
    cfg = W.config("c1", n_per_bunch=200, radiation=0)
    r = cfg["ring"]
    t0 = r["T0_s"]
    f0 = 1.0 / t0
    cfg["fill"]["buckets"] = [k * (r["h"] // m_b) for k in range(m_b)]
    cfg["fill"]["charge_C"] = [q_b] * m_b
    phi_s = math.pi - math.asin(r["U0_eV"] / cfg["cavities"][0]["V_volt"])
    q_s = math.sqrt(r["h"] * r["alpha_c"] * cfg["cavities"][0]["V_volt"] * abs(math.cos(phi_s)) / (2 * math.pi * r["E0_eV"]))
    f_s = q_s * f0
    f_r = (p * m_b + mu) * f0 + f_s
    # validity of the formula: resonator much wider than f_s, history covers the decay
    assert f_r / qual > 10 * f_s
    k_hist = 25
    assert math.exp(-(2 * math.pi * f_r / (2 * qual)) * k_hist * t0) < 1e-3
    cfg["wake"]["resonators"] = [dict(Rs_ohm=rs, fr_Hz=f_r, Q=qual, flags=W.FLAG_LR)]
    cfg["wake"]["history_turns"] = k_hist
    cfg["wake"]["n_bins"] = 100
    cfg["wake"]["gather_order"] = 1

    n = 6000
    o = orc.Oracle(cfg, log_capacity_turns=n, lr_mode=1)
    tau, delta = o.particles()
    tau += 1.0e-12 * np.cos(2 * np.pi * mu * np.arange(m_b) / m_b)[:, None]   # equal mix of modes mu and M - mu
    o.set_particles(tau, delta, 0)
    o.track(n)
    log = o.moment_log(1, n)
    assert log[-1, :, 1].sum() == 0                                              # nobody left the window
    cent = log[:, :, 2] - log[:, :, 2].mean(axis=0)
    # analytic signal in time separates exp(-i w_s n) from exp(+i w_s n), then DFT over the bunch index
    amp = np.abs(np.fft.fft(hilbert(cent, axis=0), axis=1))
    sl = slice(500, n - 500)
    turns = np.arange(n)

    def fitted(mode):
        return float(np.polyfit(turns[sl], np.log(amp[sl, mode]), 1)[0])

    sig_tau = float(np.mean(log[:, :, 4]))
    w0, ws, wr = 2 * math.pi * f0, 2 * math.pi * f_s, 2 * math.pi * f_r

    def analytic(mode):
        s = 0.0
        for pp in range(-400, 401):
            wp = (pp * m_b + mode) * w0 + ws
            re_z = rs / (1.0 + qual * qual * (wr / wp - wp / wr) ** 2)
            s += wp * re_z * math.exp(-(wp * sig_tau) ** 2)
        i0 = m_b * q_b / t0
        return r["alpha_c"] * i0 / (2.0 * r["E0_eV"] * t0 * ws) * s * t0            # per turn

    g_up, g_dn = analytic(mu), analytic(m_b - mu)
    assert g_up > 2e-4 and g_dn < -2e-4
    assert g_up < 0.05 * 2 * math.pi * q_s                                       # growth << synchrotron frequency
    assert fitted(mu) == pytest.approx(g_up, rel=0.10)                           # north_star (f)
    assert fitted(m_b - mu) == pytest.approx(g_dn, rel=0.10)
    assert fitted(mu) == pytest.approx(g_up, rel=0.03)                           # what the oracle actually reaches
    # all other modes neither grow nor decay at anything like this rate
    for mode in range(m_b):
        if mode not in (mu, m_b - mu):
            assert abs(fitted(mode)) < 0.2 * g_up
