"""CPU-only unit tests of the parity harness itself (tests/parity.py): the branch that runs when the GPU's counts differ
from the oracle's by particles sitting on a bin edge (BASELINE north_star (ii): such particles "may change bin" and are
to be counted and reported).  On the GPU that branch has never fired -- every full-size run so far had zero mismatching
bins -- so its Python logic (histogram_mismatch's "<= 2 n_edge" rule, assert_counts_consistent's else-arm, the
wake_from_counts arm of assert_single_turn_parity, the per-bunch `shifts` broadcast) is pinned here with a stand-in for the
GPU side: a second oracle whose reported counts are edited after the turn.

  * a particle steered onto a bin edge (to an ulp: the oracle's own one-particle map, orc_map_one, is inverted by secant)
    is booked in the neighbouring bin by the stand-in: the comparison must PASS, reporting 2 mismatching bins and at least
    one edge-adjacent particle, with the wake compared against the oracle's steps 5-6 on the stand-in's counts;
  * the same with the stand-in's wake left as built from the UNEDITED counts must FAIL (so the branch does compare wakes);
  * a particle that is nowhere near an edge booked in the wrong bin must FAIL;
  * the same three with window_mode = 1 and displaced bunches, i.e. with non-zero per-bunch window shifts."""
import numpy as np
import pytest

from paper_1809_00391_b200 import workloads as W
from parity import TOL_EDGE, assert_counts_consistent, assert_single_turn_parity, histogram_mismatch


class EditedCounts:
    """Stands in for mbt.Tracker in assert_single_turn_parity: an oracle of its own, whose counts are edited by `edit`
    (hist -> hist) after tracking; the wake it reports is the oracle's steps 5-6 on the edited counts (what a device that
    had binned that way would have built), unless stale_wake."""

    def __init__(self, orc, cfg, edit, stale_wake=False):
        self.g = orc.Oracle(cfg, lr_mode=0)
        self.edit, self.stale_wake = edit, stale_wake

    def set_particles(self, tau, delta, turn): self.g.set_particles(tau, delta, turn)
    def set_window(self, a, b): self.g.set_window(a, b)
    def set_lr_history(self, a): self.g.set_lr_history(a)
    def track(self, n): self.g.track(n)
    def particles(self): return self.g.particles()
    def window(self): return self.g.window()
    def histogram(self): return self.edit(self.g.histogram().copy())
    def wake(self): return self.g.wake() if self.stale_wake else self.g.wake_from_counts(self.histogram())
    def moments(self): return self.g.moments()


def _steer_onto_edge(o, cfg, b, i, j_edge, shift=0):
    """Change particle (b, i) of the oracle's state so that after ONE turn its tau is the lower edge of bin j_edge of bunch
    b's window (moved by `shift` bins), to rounding.  Radiation is off in these configurations, so the turn's map of one
    particle is orc_map_one with z = 0; tau_0 = 0 makes the RF kick cancel the synchronous loss, and delta_0 is found by
    secant on the oracle's own map."""
    w = cfg["wake"]
    width = (w["tau_hi_s"] - w["tau_lo_s"]) / w["n_bins"]
    target = w["tau_lo_s"] + (j_edge + shift) * width
    f = lambda d: o.map_one(0.0, d)[0] - target
    d0, d1 = 0.0, 1e-4
    for _ in range(60):
        f0, f1 = f(d0), f(d1)
        if f1 == f0:
            break
        d0, d1 = d1, d1 - f1 * (d1 - d0) / (f1 - f0)
    assert abs(f(d1)) <= 4 * np.spacing(abs(target))
    tau, delta = o.particles()
    tau[b, i], delta[b, i] = 0.0, d1
    o.set_particles(tau, delta, o.turn)            # resets the window: the caller re-installs the one it wants
    return target


def _move(b, j_from, j_to):
    def edit(h):
        assert h[b, j_from] > 0
        h[b, j_from] -= 1
        h[b, j_to] += 1
        return h
    return edit


def _setup(orc, window_mode):
    cfg = W.tiny(m=4, n_per_bunch=203, n_bins=16, k_hist=3, n_lr=2, radiation=0)
    cfg["wake"]["window_mode"] = window_mode
    o = orc.Oracle(cfg, lr_mode=0)
    if window_mode:
        tau, delta = o.particles()
        o.set_particles(tau * 0.5 + np.array([[12e-12], [-20e-12], [0.0], [30e-12]]), delta, 0)
    o.track(5)
    return cfg, o


@pytest.mark.parametrize("window_mode", [0, 1])
def test_edge_adjacent_particle_in_the_neighbouring_bin_is_accepted_and_reported(orc, window_mode):
    cfg, o = _setup(orc, window_mode)
    b, i, j = 2, 17, 9
    s_next = int(o.window()[1][b])             # the window turn 6 bins bunch b with
    if window_mode:
        assert len(set(int(s) for s in o.window()[1])) >= 3      # the shifts really differ from bunch to bunch
    sh, sn = o.window()
    _steer_onto_edge(o, cfg, b, i, j, shift=s_next)
    if window_mode:
        o.set_window(sh, sn)
    # which side of the edge does the oracle book it on?  (advance a copy)
    probe = orc.Oracle(cfg, lr_mode=0)
    probe.set_particles(*o.particles(), o.turn)
    if window_mode:
        probe.set_window(sh, sn)
    probe.set_lr_history(o.lr_history())
    probe.track(1)
    t1 = probe.particles()[0][b, i]
    w = cfg["wake"]
    inv = w["n_bins"] / (w["tau_hi_s"] - w["tau_lo_s"])
    pos = (t1 - w["tau_lo_s"]) * inv - int(probe.window()[0][b])
    assert abs(pos - j) < TOL_EDGE * j, pos
    j_orc = j if pos >= j else j - 1
    j_other = j - 1 if j_orc == j else j
    r = assert_single_turn_parity(o, EditedCounts(orc, cfg, _move(b, j_orc, j_other)), cfg)
    assert r["hist_bad_bins"] == 2 and r["edge_particles"] >= 1
    assert r["e_tau"] == 0.0 and r["e_wake"] == 0.0     # both sides ran the same statements on the same counts


@pytest.mark.parametrize("window_mode", [0, 1])
def test_edge_branch_still_compares_the_wake(orc, window_mode):
    cfg, o = _setup(orc, window_mode)
    b, i, j = 1, 5, 7
    sh, sn = o.window()
    _steer_onto_edge(o, cfg, b, i, j, shift=int(sn[b]))
    if window_mode:
        o.set_window(sh, sn)
    ok = False
    for j_from, j_to in ((j, j - 1), (j - 1, j)):       # whichever side the oracle booked it on, one of the two applies
        o2 = orc.Oracle(cfg, lr_mode=0)
        o2.set_particles(*o.particles(), o.turn)
        if window_mode:
            o2.set_window(sh, sn)
        o2.set_lr_history(o.lr_history())
        try:
            with pytest.raises(AssertionError, match="wake differs"):
                assert_single_turn_parity(o2, EditedCounts(orc, cfg, _move(b, j_from, j_to), stale_wake=True), cfg)
            ok = True
        except AssertionError as e:                      # the edit's own precondition (empty source bin) on the wrong side
            if "wake differs" in str(e):
                raise
    assert ok


@pytest.mark.parametrize("window_mode", [0, 1])
def test_particle_away_from_any_edge_in_the_wrong_bin_is_refused(orc, window_mode):
    cfg, o = _setup(orc, window_mode)
    h = o.histogram()
    b = 0
    j = int(np.argmax(h[b]))                             # a well-filled bin: its particles are not on an edge
    with pytest.raises(AssertionError, match="edge-adjacent"):
        assert_single_turn_parity(o, EditedCounts(orc, cfg, _move(b, j, j + 1)), cfg)


def test_histogram_mismatch_counts_units_not_bins(orc):
    """The rule is on moved COUNTS: two units moved with a single edge-adjacent particle is one too many."""
    cfg = W.tiny(m=2, n_per_bunch=50, n_bins=8, radiation=0)
    w = cfg["wake"]
    width = (w["tau_hi_s"] - w["tau_lo_s"]) / 8
    tau = np.full((2, 50), w["tau_lo_s"] + 2.5 * width)
    tau[1, 3] = w["tau_lo_s"] + 5 * width               # exactly on the edge between bins 4 and 5
    h = np.zeros((2, 8), dtype=np.uint32)
    h[0, 2] = 50; h[1, 2] = 49; h[1, 5] = 1
    g = h.copy(); g[1, 5] -= 1; g[1, 4] += 1
    assert histogram_mismatch(g, h, tau, cfg) == (2, 1)
    assert histogram_mismatch(h, h, tau, cfg) == (0, 1)
    g2 = g.copy(); g2[0, 2] -= 1; g2[0, 3] += 1          # a second unit moved, by a particle in mid-bin
    with pytest.raises(AssertionError):
        histogram_mismatch(g2, h, tau, cfg)
    # shifts: the same tau seen through windows moved by whole bins keeps the same edge set, per bunch
    assert histogram_mismatch(g, h, tau, cfg, shifts=np.array([3, -2])) == (2, 1)
    # assert_counts_consistent's else-arm: n_in may differ by at most the edge-adjacent particles
    m_c = np.array([[50.0, 0.0], [50.0, 0.0]])
    m_g = np.array([[50.0, 0.0], [49.0, 1.0]])
    hg = h.copy(); hg[1, 5] -= 1                          # the edge particle fell out of the window on the device
    assert_counts_consistent(m_g, m_c, hg, 50, bad=1, n_edge=1)
    with pytest.raises(AssertionError):
        assert_counts_consistent(m_g, m_c, hg, 50, bad=1, n_edge=0)
    with pytest.raises(AssertionError):
        assert_counts_consistent(m_g, m_c, hg, 50, bad=0, n_edge=1)
