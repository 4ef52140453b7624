"""Comparison helpers for the GPU-vs-oracle parity tests (tolerances of BASELINE.json north_star (i)-(iii),
made precise by DESIGN.md reading D23)."""
import json
import os

import numpy as np

TOL_PARTICLE = 1e-12   # north_star (i): single-turn coordinates, relative (scale: max(|x|, sigma_x of the bunch))
TOL_WAKE = 1e-10       # north_star (iii): wake potentials, relative to max_j |V[b][j]|
TOL_EDGE = 1e-12       # north_star (ii): particles this close (in bin units) to a bin edge may change bin


def particle_errors(x_gpu, x_cpu):
    """max over particles of |x_gpu - x_cpu| / max(|x_cpu|, sigma_x(bunch)), per D23; arrays [M][Np]."""
    x_gpu = np.asarray(x_gpu)
    x_cpu = np.asarray(x_cpu)
    sig = x_cpu.std(axis=1, keepdims=True)
    sig = np.where(sig > 0, sig, np.abs(x_cpu).max(axis=1, keepdims=True))
    scale = np.maximum(np.abs(x_cpu), sig)
    scale = np.where(scale > 0, scale, 1.0)
    return float(np.max(np.abs(x_gpu - x_cpu) / scale))


def wake_error(v_gpu, v_cpu):
    """max over bunches and bins of |dV| / max_j |V_cpu[b][j]| (D23); all-zero rows must match exactly."""
    v_gpu = np.asarray(v_gpu)
    v_cpu = np.asarray(v_cpu)
    scale = np.abs(v_cpu).max(axis=1, keepdims=True)
    zero = scale[:, 0] == 0
    if zero.any():
        assert np.all(v_gpu[zero] == 0.0)
    scale = np.where(scale > 0, scale, 1.0)
    return float(np.max(np.abs(v_gpu - v_cpu) / scale))


def histogram_mismatch(h_gpu, h_cpu, tau_cpu, cfg, shifts=None):
    """Counts must be bit-exact, except for particles within TOL_EDGE (bin units) of a bin edge.

    Returns (n_mismatching_bins, n_edge_particles).  Raises if the mismatch cannot be explained by
    edge-adjacent particles of the oracle's tau."""
    h_gpu = np.asarray(h_gpu, dtype=np.int64)
    h_cpu = np.asarray(h_cpu, dtype=np.int64)
    diff = h_gpu - h_cpu
    bad = int(np.count_nonzero(diff))
    w = cfg["wake"]
    nb = w["n_bins"]
    inv = nb / (w["tau_hi_s"] - w["tau_lo_s"])
    lo = w["tau_lo_s"]
    if shifts is not None:
        lo = lo + np.asarray(shifts, dtype=np.float64)[:, None] * ((w["tau_hi_s"] - w["tau_lo_s"]) / nb)
    t = (np.asarray(tau_cpu) - lo) * inv
    edge = np.abs(t - np.rint(t)) < TOL_EDGE * np.maximum(1.0, np.abs(t))
    n_edge = int(np.count_nonzero(edge))
    if bad:
        # every unit of count that moved must belong to an edge-adjacent particle
        assert np.abs(diff).sum() <= 2 * n_edge, "histogram differs by more than the edge-adjacent particles allow"
    return bad, n_edge


def assert_counts_consistent(m_gpu, m_cpu, hist_gpu, n_per_bunch, bad, n_edge):
    """n_in / n_out (integers): always equal to the GPU's own counts and to N_p in sum; equal to the oracle's when the
    histograms agree, else different from them by no more than the edge-adjacent particles (only one sitting on a
    window end changes n_in at all)."""
    n_in_g = np.asarray(hist_gpu, dtype=np.int64).sum(axis=1)
    assert np.array_equal(m_gpu[:, 0], n_in_g.astype(np.float64)), "n_in is not the sum of the counts"
    assert np.all(m_gpu[:, 0] + m_gpu[:, 1] == float(n_per_bunch)), "n_in + n_out != N_p"
    if bad == 0:
        assert np.array_equal(m_cpu[:, :2], m_gpu[:, :2])
    else:
        assert np.abs(m_gpu[:, 0] - m_cpu[:, 0]).sum() <= n_edge and np.abs(m_gpu[:, 1] - m_cpu[:, 1]).sum() <= n_edge


def resume_on_gpu(o, trk, cfg=None):
    """Upload the oracle's current state (particles, turn, long-range history) into the GPU tracker."""
    tau, delta = o.particles()
    trk.set_particles(tau, delta, o.turn)
    if cfg is not None and cfg["wake"].get("window_mode", 0):
        trk.set_window(*o.window())                 # after set_particles (which resets the shifts)
    trk.set_lr_history(o.lr_history())
    return tau, delta


def assert_single_turn_parity(o, trk, cfg, turns=1, tol_particle=TOL_PARTICLE, tol_wake=TOL_WAKE, after_resume=None):
    """Both sides advance `turns` turns from the oracle's current state; everything observable is compared."""
    resume_on_gpu(o, trk, cfg)
    if after_resume is not None:
        after_resume(trk)
    o.track(turns)
    trk.track(turns)
    tau_c, delta_c = o.particles()
    tau_g, delta_g = trk.particles()
    e_tau = particle_errors(tau_g, tau_c)
    e_delta = particle_errors(delta_g, delta_c)
    assert e_tau <= tol_particle, "tau differs by %.3e (relative, D23)" % e_tau
    assert e_delta <= tol_particle, "delta differs by %.3e (relative, D23)" % e_delta
    sh_c, sn_c = o.window()
    sh_g, sn_g = trk.window()
    assert np.array_equal(sh_c, sh_g) and np.array_equal(sn_c, sn_g), "window shifts differ (D31)"
    hist_g = trk.histogram()
    bad, n_edge = histogram_mismatch(hist_g, o.histogram(), tau_c, cfg, shifts=sh_c)
    # north_star (iii): the wake is ALWAYS compared.  If the counts differ by edge-adjacent particles, the expected wake
    # is the oracle's steps 5-6 of the same turn evaluated on the GPU's counts (orc_wake_from_counts: same statements,
    # same history), so S5 / S6 are checked on that branch too.
    tot_c, sr_c, lr_c = o.wake() if bad == 0 else o.wake_from_counts(hist_g)
    tot_g, sr_g, lr_g = trk.wake()
    e_w = max(wake_error(tot_g, tot_c), wake_error(sr_g, sr_c), wake_error(lr_g, lr_c))
    assert e_w <= tol_wake, "wake differs by %.3e (relative, D23)" % e_w
    m_c, m_g = o.moments(), trk.moments()
    assert_counts_consistent(m_g, m_c, hist_g, o.Np, bad, n_edge)
    # means: absolute error against the rms of the same coordinate; rms: relative
    assert np.all(np.abs(m_g[:, 2] - m_c[:, 2]) <= 1e-11 * np.maximum(m_c[:, 4], np.abs(m_c[:, 2])) + 1e-300)
    assert np.all(np.abs(m_g[:, 3] - m_c[:, 3]) <= 1e-11 * np.maximum(m_c[:, 5], np.abs(m_c[:, 3])) + 1e-300)
    for k in (4, 5):
        ref = np.maximum(m_c[:, k], np.abs(m_c[:, k - 2]))
        assert np.all(np.abs(m_g[:, k] - m_c[:, k]) <= 1e-8 * ref + 1e-300), (m_g[:, k], m_c[:, k])
    return dict(e_tau=e_tau, e_delta=e_delta, e_wake=e_w, hist_bad_bins=bad, edge_particles=n_edge)


def report(name, numbers):
    """Append one record of measured parity numbers (errors, mismatching bins, edge-adjacent particle counts) to
    gpurun_out/parity_report.jsonl at the repo root; the tracked table in DESIGN.md section 8 is copied from it."""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = os.path.join(root, "gpurun_out")
    try:
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_report.jsonl"), "a") as f:
            f.write(json.dumps({"case": name, **numbers}, default=float) + "\n")
    except OSError:
        pass
    print(name, numbers)
