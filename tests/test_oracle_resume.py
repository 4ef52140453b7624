"""Pins of the oracle's history setters, orc_set_lr_history and orc_set_rw_history (oracle/orc_tracker.cpp), which rebuild
state the turn loop otherwise builds itself: the ring of source phasors a[b][n'][r] with its per-turn aggregates ring_A (the
lr_mode = 1 form of the long-range sum, P:l.229-237, reading D14) and the ring of resistive-wall source strengths
(P:l.117-119, readings W1-W5).

The pin is a property no formula retyped here could satisfy by accident: checkpoint and resume.  An oracle is tracked past
the depth of both histories and its state read out through the getters; a FRESH oracle is given that state through
set_particles, set_window, set_lr_history, set_transverse and set_rw_history; both then track on.  Every observable of the
resumed run -- coordinates, counts, wakes, both histories, windows, moments -- must equal the uninterrupted run's bit for bit,
for the pairwise sum (lr_mode 0) and for the aggregate form (lr_mode 1).  A setter that dropped a row, put it in the wrong
slot, mixed up bunch and resonator, or rebuilt an aggregate with a wrong tail factor changes the first wake after the
resume (the histories enter it with weights of order one) and fails the comparison."""
import numpy as np
import pytest

from paper_1809_00391_b200 import workloads as W


def _cfg(window_mode, rw_turns):
    cfg = W.tiny(n_per_bunch=203, n_bins=16, k_hist=3)
    cfg["wake"]["window_mode"] = window_mode
    cfg["transverse"] = W.transverse_planes(rw_amp_x=2.0e9, rw_amp_y=1.0e9, rw_turns=rw_turns)
    return cfg


def _observables(o):
    out = {"tau": o.particles()[0], "delta": o.particles()[1], "hist": o.histogram(), "lr_history": o.lr_history(),
           "rw_history": o.rw_history(), "moments": o.moments(), "moments_tr": o.moments_transverse()}
    for k, v in zip(("V", "Vsr", "Vlr"), o.wake()):
        out[k] = v
    for k, v in zip(("x", "xp", "y", "yp"), o.transverse_particles()):
        out[k] = v
    for k, v in zip(("Kx", "Ky"), o.transverse_wake()):
        out[k] = v
    for k, v in zip(("rw_x", "rw_y"), o.rw_kick()):
        out[k] = v
    for k, v in zip(("s_hist", "s_next"), o.window()):
        out[k] = v
    return out


@pytest.mark.parametrize("lr_mode", [0, 1])
@pytest.mark.parametrize("window_mode,rw_turns,n_ckpt", [(0, 2, 5), (1, 2, 7), (0, 4, 2), (1, 1, 4)])
def test_resume_through_the_history_setters_is_bit_identical(orc, lr_mode, window_mode, rw_turns, n_ckpt):
    cfg = _cfg(window_mode, rw_turns)
    a = orc.Oracle(cfg, lr_mode=lr_mode)
    a.track(n_ckpt)                       # (0, 4, 2): a checkpoint BEFORE the histories are full (rows of turns < 1 are zero)
    tau, delta = a.particles()
    s_hist, s_next = a.window()
    lr, rw, tr = a.lr_history(), a.rw_history(), a.transverse_particles()
    assert np.abs(lr).max() > 0 and np.abs(rw).max() > 0            # the histories matter in what follows
    b = orc.Oracle(cfg, lr_mode=lr_mode)
    b.set_particles(tau, delta, n_ckpt)
    b.set_window(s_hist, s_next)
    b.set_lr_history(lr)
    b.set_transverse(*tr)
    b.set_rw_history(rw)
    assert b.turn == n_ckpt
    assert np.array_equal(b.lr_history(), lr) and np.array_equal(b.rw_history(), rw)   # get(set(x)) = x
    for step in (1, 3):                   # one turn, then on past the point where the set rows have all been consumed
        a.track(step); b.track(step)
        oa, ob = _observables(a), _observables(b)
        for k in oa:
            assert np.array_equal(oa[k], ob[k]), (k, step, np.abs(np.asarray(oa[k], float) - np.asarray(ob[k], float)).max())


def test_resume_without_the_histories_differs(orc):
    """The control: the same resume with the two setters left out is NOT the uninterrupted run (so the test above is
    sensitive to them), and leaving out either one alone is caught as well."""
    cfg = _cfg(0, 2)
    a = orc.Oracle(cfg, lr_mode=1)
    a.track(5)
    tau, delta = a.particles()
    lr, rw, tr = a.lr_history(), a.rw_history(), a.transverse_particles()
    a.track(1)
    for skip in ("lr", "rw"):
        b = orc.Oracle(cfg, lr_mode=1)
        b.set_particles(tau, delta, 5)
        if skip != "lr":
            b.set_lr_history(lr)
        b.set_transverse(*tr)
        if skip != "rw":
            b.set_rw_history(rw)
        b.track(1)
        if skip == "lr":
            assert not np.array_equal(a.wake()[2], b.wake()[2]) and not np.array_equal(a.particles()[1], b.particles()[1])
        else:
            assert not np.array_equal(a.rw_kick()[0], b.rw_kick()[0]) and not np.array_equal(a.transverse_particles()[1], b.transverse_particles()[1])
