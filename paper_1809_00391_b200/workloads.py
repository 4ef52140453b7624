"""Seeded synthetic workloads (inputs only) shared by the CUDA path and the CPU oracle.

This module holds NONE of the method's arithmetic: it only writes down the
parameter sets of BASELINE.json `configs[0..4]` (called c1..c5 here, SURVEY.md
section 8 table) plus a few tiny brute-force cases, as plain Python dicts. Each
side (paper_1809_00391_b200.mbt for the CUDA library, oracle/orc.py for the CPU
oracle) converts the dict into its own C structs with its own code.

Readings that fill the gaps of BASELINE.json (all listed in DESIGN.md):
  * common ring (c1): E0 = 2.4 GeV, h = 484, f_rf = 500 MHz -> T0 = h / f_rf,
    V1 = 1.4 MV, U0 = 0.6 MeV, alpha_c = +1e-4, sigma_delta = 1e-3,
    damping time 1e4 turns; initial Gaussian sigma_tau0 = 10 ps, sigma_delta0 = 1e-3;
  * harmonic cavity (c2, c5): ideal m = 3, V = 0.45 MV, phase 0 (alpha_c > 0);
  * windows: +-50 ps (c1, c3, c4), +-250 ps (c2, c5);
  * c3 buckets round(k*484/3) = {0, 161, 323};
  * c4 charges ~ N(1 nC, 2 %) from numpy's default_rng(4) (input generation,
    not part of the tracked method);
  * c5: 1 nC per bunch, BB as c1, HOMs (1.2 GHz, 1e4, 1 MOhm),
    (2.1 GHz, 1e3, 0.1 MOhm), (1.6 GHz, 3e4, 1 MOhm);
  * seed = config number; gather: c1 NGP (BASELINE "200 NGP bins"), others linear.

Resonator flags: bit0 = contributes to the short-range (same bunch, same turn)
table, bit1 = contributes to the long-range (other bunches / earlier turns) sum.
"""
from __future__ import annotations

import copy
import math

import numpy as np

FLAG_SR = 1
FLAG_LR = 2

_F_RF = 500.0e6
_H = 484


def _ring():
    return dict(E0_eV=2.4e9, T0_s=_H / _F_RF, alpha_c=1.0e-4, U0_eV=0.6e6, h=_H)


def _main_cavity():
    # phase NaN -> each side solves the synchronous phase itself (reading D3)
    return dict(V_volt=1.4e6, m=1, phase_rad=math.nan)


def _harmonic_cavity():
    return dict(V_volt=0.45e6, m=3, phase_rad=0.0)


def _bb(rs=5.0e3):
    return dict(Rs_ohm=rs, fr_Hz=10.0e9, Q=1.0, flags=FLAG_SR)


def _hom(rs, fr, q):
    return dict(Rs_ohm=rs, fr_Hz=fr, Q=q, flags=FLAG_SR | FLAG_LR)


def _base(seed, buckets, charges, n_per_bunch, n_bins, half_window, gather, res, hist_turns, cav, n_turns):
    return dict(
        ring=_ring(),
        cavities=cav,
        radiation=dict(enable=1, sigma_delta=1.0e-3, damping_turns=1.0e4),
        seed=int(seed),
        fill=dict(
            buckets=[int(b) for b in buckets],
            charge_C=[float(q) for q in charges],
            n_per_bunch=int(n_per_bunch),
            sigma_tau0_s=10.0e-12,
            sigma_delta0=1.0e-3,
        ),
        wake=dict(
            n_bins=int(n_bins),
            tau_lo_s=-float(half_window),
            tau_hi_s=float(half_window),
            gather_order=int(gather),
            resonators=res,
            history_turns=int(hist_turns),
            sr_table=None,
        ),
        n_turns=int(n_turns),
    )


def c1():
    return _base(1, [0], [1.0e-9], 10_000, 200, 50e-12, 0, [_bb(5e3)], 0, [_main_cavity()], 1000)


def c2():
    return _base(2, [0], [5.0e-9], 1_000_000, 1000, 250e-12, 1, [_bb(20e3)], 0,
                 [_main_cavity(), _harmonic_cavity()], 10_000)


def c3():
    buckets = [int(round(k * _H / 3.0)) for k in range(3)]
    return _base(3, buckets, [1.0e-9] * 3, 100_000, 500, 50e-12, 1,
                 [_bb(5e3), _hom(1.0e6, 1.2e9, 1.0e4)], 10, [_main_cavity()], 20_000)


def c4():
    m = 363
    rng = np.random.default_rng(4)
    charges = 1.0e-9 * (1.0 + 0.02 * rng.standard_normal(m))
    return _base(4, range(m), charges, 100_000, 300, 50e-12, 1,
                 [_bb(5e3), _hom(1.0e6, 1.2e9, 1.0e4), _hom(0.5e6, 2.1e9, 5.0e3)], 20,
                 [_main_cavity()], 10_000)


def c5():
    m = 484
    return _base(5, range(m), [1.0e-9] * m, 200_000, 500, 250e-12, 1,
                 [_bb(5e3), _hom(1.0e6, 1.2e9, 1.0e4), _hom(0.1e6, 2.1e9, 1.0e3), _hom(1.0e6, 1.6e9, 3.0e4)],
                 50, [_main_cavity(), _harmonic_cavity()], 5_000)


CONFIGS = dict(c1=c1, c2=c2, c3=c3, c4=c4, c5=c5)


def config(name: str, **overrides):
    """Return a deep copy of config `name` with optional overrides.

    Recognised overrides: n_per_bunch, n_turns, seed, n_bunches (keep the first
    n buckets/charges), radiation (0/1), gather_order, history_turns, n_bins.
    """
    cfg = copy.deepcopy(CONFIGS[name]())
    for k, v in overrides.items():
        if v is None:
            continue
        if k == "n_per_bunch":
            cfg["fill"]["n_per_bunch"] = int(v)
        elif k == "n_turns":
            cfg["n_turns"] = int(v)
        elif k == "seed":
            cfg["seed"] = int(v)
        elif k == "n_bunches":
            cfg["fill"]["buckets"] = cfg["fill"]["buckets"][: int(v)]
            cfg["fill"]["charge_C"] = cfg["fill"]["charge_C"][: int(v)]
        elif k == "radiation":
            cfg["radiation"]["enable"] = int(v)
        elif k == "gather_order":
            cfg["wake"]["gather_order"] = int(v)
        elif k == "history_turns":
            cfg["wake"]["history_turns"] = int(v)
        elif k == "n_bins":
            cfg["wake"]["n_bins"] = int(v)
        else:
            raise KeyError(k)
    return cfg


def tiny(m=5, n_per_bunch=37, n_bins=8, k_hist=3, seed=11, buckets=None, n_lr=2, gather=1, harmonic=False,
         radiation=1):
    """Small irregular-fill case for brute-force cross-checks (ragged sizes on purpose)."""
    if buckets is None:
        buckets = [0, 3, 4, 100, 483][:m]
    rng = np.random.default_rng(seed)
    charges = 1.0e-9 * (1.0 + 0.3 * rng.random(len(buckets)))
    res = [_bb(5e3)]
    homs = [_hom(1.0e6, 1.2e9, 1.0e4), _hom(0.5e6, 2.1e9, 5.0e3), _hom(1.0e6, 1.6e9, 3.0e4)]
    res += homs[:n_lr]
    cav = [_main_cavity()] + ([_harmonic_cavity()] if harmonic else [])
    cfg = _base(seed, buckets, charges, n_per_bunch, n_bins, 50e-12, gather, res, k_hist, cav, 9)
    cfg["radiation"]["enable"] = int(radiation)
    return cfg


def transverse_planes(nu_x=18.2, nu_y=5.3, beta_x=8.0, beta_y=4.0, alpha_x=0.0, alpha_y=0.0, xi_x=1.0, xi_y=1.0,
                      eta_x=0.1, etap_x=0.0, emit_x=3.0e-10, emit_y=3.0e-12, u0_over_e0=2.5e-4, rs_ohm_per_m=1.0e6,
                      fr_hz=5.0e9, q=1.0, rw_amp_x=0.0, rw_amp_y=0.0, rw_turns=0):
    """Synthetic transverse-plane parameters (inputs only) for cfg["transverse"].
    sigma_u = sqrt(emit beta), sigma_up = sqrt(emit gamma); D_exc = (U0/E0) / (beta gamma), the value for which
    the excitation of Eq. (5) balances its adiabatic damping at the emittance `emit` (reading T4); the
    initial distribution is the equilibrium one (uncorrelated, alpha = 0 by default); one broadband transverse
    resonator for both planes.  rw_*: long-range resistive-wall kick (readings W1..W5), W_rw(t) = rw_amp / sqrt(t)
    [V/(C m)] with a synthetic amplitude, history of rw_turns turns (0: off)."""
    def plane(nu, a, b, xi, eta, etap, emit):
        g = (1.0 + a * a) / b
        return dict(nu=nu, alpha=a, beta_m=b, xi=xi, eta_m=eta, etap=etap, sigma_u_m=math.sqrt(emit * b),
                    sigma_up=math.sqrt(emit * g), D_exc=u0_over_e0 / (b * g), sigma0_u_m=math.sqrt(emit * b),
                    sigma0_up=math.sqrt(emit * g))
    return dict(x=plane(nu_x, alpha_x, beta_x, xi_x, eta_x, etap_x, emit_x),
                y=plane(nu_y, alpha_y, beta_y, xi_y, 0.0, 0.0, emit_y),
                resonators=[dict(Rs_ohm=rs_ohm_per_m, fr_Hz=fr_hz, Q=q, flags=FLAG_SR)],
                rw_amp_x=float(rw_amp_x), rw_amp_y=float(rw_amp_y), rw_turns=int(rw_turns))


def sampled_wake_table(n_bins, delta_s, r_ohm=0.0, l_henry=0.0, rw_amp=0.0):
    """User-sampled short-range wake w[k] at lag k*Delta [V/C] for `wake["sr_table"]` (the
    wake sources the paper lists beside resonators, P:l.98 "resistive-wall effects ... purely resistive and inductive
    components", whose formulas are only in its ref. [7]).  Input generation, not the method: the tracker just
    convolves whatever table it is given.  Textbook grid forms:
      * pure resistance R:  V = R I, I_j = q_j / Delta        ->  w[0] += R / Delta
      * pure inductance L:  V = L dI/dt (backward difference) ->  w[0] += L / Delta^2, w[1] -= L / Delta^2
      * resistive-wall-like power law, amplitude synthetic:   ->  w[k] += rw_amp * (k Delta)^(-3/2), k >= 1
    """
    w = np.zeros(int(n_bins))
    w[0] += r_ohm / delta_s + l_henry / delta_s**2
    if n_bins > 1:
        w[1] -= l_henry / delta_s**2
        k = np.arange(1, int(n_bins))
        w[1:] += rw_amp * (k * delta_s) ** -1.5
    return w


def n_particles(cfg) -> int:
    return len(cfg["fill"]["buckets"]) * cfg["fill"]["n_per_bunch"]
