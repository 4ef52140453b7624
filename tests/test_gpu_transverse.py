"""GPU-vs-oracle parity of the transverse planes through the C ABI (P:l.73-92 Eqs.(3)-(5),
l.100-111 Eq.(6b); readings T1..T8).  Same protocol as test_gpu_parity.py: the oracle's state is uploaded,
both sides advance one turn, everything observable is compared:
  coordinates (x, x', y, y') within 1e-12 relative (scale D23), dipole sums and kick tables within 1e-10 of the
  row maximum (the wake tolerance of north_star (iii)), moments 1e-8."""
import numpy as np
import pytest

from paper_1809_00391_b200 import workloads as W
from parity import TOL_PARTICLE, TOL_WAKE, assert_single_turn_parity, particle_errors, wake_error

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mbt():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device")
    from paper_1809_00391_b200 import build, mbt as _mbt
    build.build()
    _mbt.lib()
    return _mbt


def _cfg(tr=None, **kw):
    cfg = W.tiny(**kw)
    cfg["transverse"] = W.transverse_planes(**(tr or {}))
    return cfg


def assert_transverse_turn_parity(o, t, cfg, turns=1, tol=TOL_PARTICLE):
    """Upload the oracle's 6-D state, advance both sides, compare the transverse observables; the longitudinal ones
    go through assert_single_turn_parity (which does the tracking)."""
    t.set_transverse(*o.transverse_particles())
    hist_rw = o.rw_history()

    def more(trk):                               # after mbt_set_particles has fixed the turn the rows refer to
        trk.set_rw_history(hist_rw)
    r = assert_single_turn_parity(o, t, cfg, turns=turns, after_resume=more)
    if o.K_rw:
        for nm, g, c in zip(("rw_x", "rw_y"), t.rw_kick(), o.rw_kick()):
            scale = np.abs(c).max()
            r["e_" + nm] = float(np.abs(g - c).max() / scale) if scale > 0 else float(np.abs(g).max())
            assert r["e_" + nm] <= TOL_WAKE, "%s differs by %.3e" % (nm, r["e_" + nm])
        assert np.allclose(t.rw_history(), o.rw_history(), rtol=1e-10, atol=1e-12 * np.abs(o.rw_history()).max())
    names = ("x", "xp", "y", "yp")
    for nm, g, c in zip(names, t.transverse_particles(), o.transverse_particles()):
        e = particle_errors(g, c)
        assert e <= tol, "%s differs by %.3e (relative, D23)" % (nm, e)
        r["e_" + nm] = e
    if r["hist_bad_bins"] == 0:
        for nm, g, c in zip(("Sx", "Sy"), t.dipole(), o.dipole()):
            r["e_" + nm] = wake_error(g, c)
            assert r["e_" + nm] <= TOL_WAKE, "%s differs by %.3e" % (nm, r["e_" + nm])
        for nm, g, c in zip(("Kx", "Ky"), t.transverse_wake(), o.transverse_wake()):
            r["e_" + nm] = wake_error(g, c)
            assert r["e_" + nm] <= TOL_WAKE, "%s differs by %.3e" % (nm, r["e_" + nm])
    m_c, m_g = o.moments_transverse(), t.moments_transverse()
    for k in range(4):
        ref = np.maximum(m_c[:, 4 + k], np.abs(m_c[:, k]))
        assert np.all(np.abs(m_g[:, k] - m_c[:, k]) <= 1e-10 * ref + 1e-300), (k, m_g[:, k], m_c[:, k])
        assert np.all(np.abs(m_g[:, 4 + k] - m_c[:, 4 + k]) <= 1e-8 * ref + 1e-300), (k, m_g[:, 4 + k], m_c[:, 4 + k])
    return r


def test_transverse_initial_distribution(mbt, orc):
    for kw in (dict(n_per_bunch=37), dict(n_per_bunch=8193, m=3), dict(n_per_bunch=1, m=2)):
        cfg = _cfg(**kw)
        o = orc.Oracle(cfg)
        with mbt.Tracker(cfg) as t:
            for g, c in zip(t.transverse_particles(), o.transverse_particles()):
                assert particle_errors(g, c) <= TOL_PARTICLE
            tau_g, delta_g = t.particles()
            tau_c, delta_c = o.particles()
            assert particle_errors(tau_g, tau_c) <= TOL_PARTICLE and particle_errors(delta_g, delta_c) <= TOL_PARTICLE
            m_c, m_g = o.moments_transverse(), t.moments_transverse()
            assert np.allclose(m_g[:, 4:], m_c[:, 4:], rtol=1e-8)


VARIANTS = {
    "default": dict(n_per_bunch=513, n_bins=16),
    "no_radiation": dict(n_per_bunch=400, n_bins=16, radiation=0),
    "ngp": dict(n_per_bunch=257, n_bins=16, gather=0),
    "harmonic": dict(n_per_bunch=301, n_bins=32, harmonic=True),
    "no_long_wake": dict(n_per_bunch=1000, n_bins=16, n_lr=0),
    "one_particle": dict(n_per_bunch=1, m=2),
    "ragged_tiles": dict(n_per_bunch=8193 + 5, m=2, n_bins=64),
    "many_bins": dict(n_per_bunch=4000, m=2, n_bins=1023),
    "twiss": dict(n_per_bunch=999, n_bins=16, tr=dict(alpha_x=-0.7, alpha_y=1.3, etap_x=-0.015, xi_x=2.5, xi_y=-1.0)),
    "two_resonators": dict(n_per_bunch=777, n_bins=32),
}


@pytest.mark.parametrize("name", sorted(VARIANTS))
def test_transverse_single_turn_parity(mbt, orc, name):
    kw = dict(VARIANTS[name])
    cfg = _cfg(**kw)
    if name == "two_resonators":
        cfg["transverse"]["resonators"].append(dict(Rs_ohm=-3.0e5, fr_Hz=1.1e10, Q=4.0, flags=1))
    o = orc.Oracle(cfg)
    o.track(3)
    with mbt.Tracker(cfg) as t:
        for _ in range(3):
            r = assert_transverse_turn_parity(o, t, cfg)
        print(name, r)


RW_VARIANTS = {
    "five_bunches": dict(m=5, n_per_bunch=513, n_bins=16, rw=dict(rw_turns=3)),
    "one_bunch_deep": dict(m=1, n_per_bunch=300, n_bins=16, rw=dict(rw_turns=40)),
    "no_radiation_ngp": dict(m=4, n_per_bunch=257, n_bins=16, radiation=0, gather=0, rw=dict(rw_turns=2)),
    "x_only": dict(m=3, n_per_bunch=999, n_bins=32, rw=dict(rw_turns=5, rw_amp_y=0.0)),
    "ragged_tiles": dict(m=2, n_per_bunch=8193 + 7, n_bins=64, rw=dict(rw_turns=1)),
}


@pytest.mark.parametrize("name", sorted(RW_VARIANTS))
def test_resistive_wall_single_turn_parity(mbt, orc, name):
    """Long-range resistive-wall kick (readings W1..W5): the kick per bunch, the source history and, through x' and y',
    its application to every particle; bunches displaced so that the centroids are not noise, a few particles parked
    outside the bin window (they are kicked too, W4)."""
    kw = dict(RW_VARIANTS[name])
    rw = dict(rw_amp_x=2.0e9, rw_amp_y=-0.7e9)
    rw.update(kw.pop("rw"))
    cfg = _cfg(**kw)
    cfg["transverse"].update(rw)
    o = orc.Oracle(cfg)
    m, n_p = len(cfg["fill"]["buckets"]), cfg["fill"]["n_per_bunch"]
    tau, delta = o.particles()
    tau = tau.copy()
    tau[:, : min(3, n_p // 4)] = 90e-12
    o.set_particles(tau, delta, 0)
    x, xp, y, yp = o.transverse_particles()
    off = (1.0e-3 * (1 + np.arange(m)) * (-1.0) ** np.arange(m))[:, None]
    o.set_transverse(x + off, xp, y - 0.3 * off, yp)
    o.track(3)
    with mbt.Tracker(cfg) as t:
        for _ in range(4):
            r = assert_transverse_turn_parity(o, t, cfg)
        assert np.abs(t.rw_kick()[0]).max() > 0
        print(name, r)


def test_resistive_wall_on_the_c4_fill_and_without_resync(mbt, orc):
    """363 bunches, 20-turn resistive-wall history (7260 sources per bunch and turn), then eight turns on its own."""
    cfg = W.config("c4", n_per_bunch=256)
    cfg["transverse"] = W.transverse_planes()
    cfg["transverse"].update(rw_amp_x=2.0e9, rw_amp_y=1.0e9, rw_turns=20)
    o = orc.Oracle(cfg, lr_mode=0)
    x, xp, y, yp = o.transverse_particles()
    off = 1.0e-3 * np.sin(2 * np.pi * 5 * np.arange(363) / 363)[:, None]
    o.set_transverse(x + off, xp, y + 0.5 * off, yp)
    o.track(2)
    with mbt.Tracker(cfg) as t:
        r = assert_transverse_turn_parity(o, t, cfg)
        print(r)
        o.track(8)
        t.track(8)
        for g, c in zip(t.transverse_particles(), o.transverse_particles()):
            assert particle_errors(g, c) <= 1e-10
        for g, c in zip(t.rw_kick(), o.rw_kick()):
            assert np.abs(g - c).max() <= 1e-9 * np.abs(c).max()


def test_transverse_with_bunch_following_window(mbt, orc):
    cfg = _cfg(m=3, n_per_bunch=3001, n_bins=32)
    cfg["wake"]["window_mode"] = 1
    o = orc.Oracle(cfg)
    tau, delta = o.particles()
    o.set_particles(tau * 0.5 + np.array([[15e-12], [-22e-12], [0.0]]), delta, 0)
    o.track(2)
    with mbt.Tracker(cfg) as t:
        for _ in range(4):
            assert_transverse_turn_parity(o, t, cfg)
        assert len(set(int(s) for s in t.window()[0])) >= 2


def test_transverse_several_turns_without_resync(mbt, orc):
    """Ten turns from the common initial distribution, no re-synchronisation: the betatron phase advances by
    ~2 pi nu per turn, so rounding differences rotate but do not grow; histograms stay identical on this seed."""
    cfg = _cfg(m=3, n_per_bunch=5000, n_bins=32)
    o = orc.Oracle(cfg)
    with mbt.Tracker(cfg) as t:
        o.track(10)
        t.track(10)
        assert t.turn == 10
        for g, c in zip(t.transverse_particles(), o.transverse_particles()):
            assert particle_errors(g, c) <= 1e-10
        if np.array_equal(t.histogram(), o.histogram()):
            for g, c in zip(t.transverse_wake(), o.transverse_wake()):
                assert wake_error(g, c) <= 1e-9
        m_c, m_g = o.moments_transverse(), t.moments_transverse()
        assert np.allclose(m_g[:, 4:], m_c[:, 4:], rtol=1e-8)


@pytest.mark.parametrize("name,over", [("c3", dict(n_per_bunch=30_000)), ("c4", dict(n_per_bunch=1_500))])
def test_transverse_on_baseline_fills(mbt, orc, name, over):
    """The transverse planes on the fill patterns of BASELINE configs c3 / c4 (reduced N_p): several CTAs per bunch,
    363 bunches, long-range history in the longitudinal plane."""
    cfg = W.config(name, **over)
    cfg["transverse"] = W.transverse_planes()
    o = orc.Oracle(cfg, lr_mode=0)
    o.track(2)
    with mbt.Tracker(cfg) as t:
        r = assert_transverse_turn_parity(o, t, cfg)
        print(name, r)


def test_resistive_wall_growth_rate_long_run(mbt, orc):
    """Long run (north_star (iii): fitted growth rates within 5 %): the resistive-wall coupled-bunch instability of 22
    equally spaced bunches (the configuration pinned against linear theory in tests/test_oracle_rw.py, here with 64
    macro-particles per bunch), 1200 turns in one mbt_track call, growth of mode 19 fitted from the per-turn centroid log
    on both sides."""
    import math
    M, K, turns, n_p = 22, 30, 1200, 64
    cfg = W.tiny(m=M, n_per_bunch=n_p, n_bins=16, n_lr=0, radiation=0, buckets=list(range(0, 484, 22)))
    cfg["wake"]["resonators"] = []
    cfg["fill"]["charge_C"] = [1.0e-9] * M
    tr = W.transverse_planes(xi_x=0.0, xi_y=0.0, eta_x=0.0, rw_amp_x=3.0e10, rw_amp_y=0.0, rw_turns=K)
    tr["resonators"] = []
    cfg["transverse"] = tr
    nu, beta = tr["x"]["nu"], tr["x"]["beta_m"]
    b = np.arange(M)
    a0 = 1.0e-3 * np.exp(2j * np.pi * (19 - nu) * b / M)
    rates = []
    o = orc.Oracle(cfg, log_capacity_turns=turns)
    with mbt.Tracker(cfg, log_capacity_turns=turns) as t:
        x, xp, y, yp = o.transverse_particles()
        start = (x + (math.sqrt(beta) * a0.real)[:, None], xp + (a0.imag / math.sqrt(beta))[:, None], y, yp)
        for side in (o, t):
            side.set_transverse(*start)
            side.track(turns)
            cx = side.transverse_log(1, turns)[:, :, 0]                       # [turns][M] centroids
            amp = np.abs(cx @ np.exp(-2j * np.pi * (19 - nu) * b / M))
            n = np.arange(turns)
            rates.append(np.polyfit(n[300:], np.log(amp[300:]), 1)[0])
    assert rates[0] > 5e-4                                                     # it does grow
    assert abs(rates[1] / rates[0] - 1) < 0.05, rates


@pytest.mark.parametrize("rw_turns,m,npb", [(1, 5, 64), (2, 5, 33), (1, 40, 16), (3, 7, 64)])
def test_resistive_wall_ring_under_per_bunch_sequencing(mbt, rw_turns, m, npb):
    """The source ring of the resistive-wall kick (ring_g) under the per-bunch flags of DESIGN.md 7.1: a leading bunch may
    start its next turn while the k_rw CTA of a trailing bunch still sums this one, so the slot the next turn writes must
    not be one this turn reads (the ring has rw_turns + 2 slots and the writer waits for the readers of two turns back).
    Tiny bunches, short histories and hundreds of turns are where kernels of consecutive turns overlap most; the run
    must equal, bit for bit, the same library with grid-wide waits (per_bunch_start = 1)."""
    turns = 400
    buckets = sorted(set(int(b) for b in np.linspace(0, 482, m)))
    cfg = _cfg(tr=dict(rw_amp_x=2.0e9, rw_amp_y=1.0e9, rw_turns=rw_turns), m=len(buckets), buckets=buckets, n_per_bunch=npb,
               n_bins=8)
    with mbt.Tracker(cfg, log_capacity_turns=turns, tuning=dict(per_bunch_start=2)) as ta, \
            mbt.Tracker(cfg, log_capacity_turns=turns, tuning=dict(per_bunch_start=1)) as tb:
        for n in (turns // 3, 1, turns - turns // 3 - 1):
            ta.track(n); tb.track(n)
        for a, b in zip(ta.transverse_particles(), tb.transverse_particles()):
            assert np.array_equal(a, b)
        assert np.array_equal(ta.rw_history(), tb.rw_history())
        for a, b in zip(ta.rw_kick(), tb.rw_kick()):
            assert np.array_equal(a, b)
        la, lb = ta.transverse_log(1, turns), tb.transverse_log(1, turns)
        assert np.array_equal(la[..., :2], lb[..., :2])                  # centroids: from the exact integer totals
        assert np.allclose(la[..., 2:], lb[..., 2:], rtol=1e-9, atol=0)  # rms: sums of squares added by fp64 atomics


def test_transverse_log_matches_oracle(mbt, orc):
    """Per-turn log of mean / rms x, y (P:l.123) from the pass's own sums, twelve turns without re-synchronisation; one
    bunch displaced by 20 sigma (mean >> rms: the single-pass variance must survive the cancellation)."""
    cfg = _cfg(m=3, n_per_bunch=9001, n_bins=32)
    cfg["transverse"].update(rw_amp_x=2.0e9, rw_amp_y=-0.7e9, rw_turns=2)
    o = orc.Oracle(cfg, log_capacity_turns=12)
    with mbt.Tracker(cfg, log_capacity_turns=12) as t:
        x, xp, y, yp = o.transverse_particles()
        off = np.array([[1.0e-3], [0.0], [-2.0e-4]])
        o.set_transverse(x + off, xp, y - off, yp)
        t.set_transverse(x + off, xp, y - off, yp)
        o.track(12)
        t.track(12)
        lc, lg = o.transverse_log(1, 12), t.transverse_log(1, 12)
        sig = lc[:, :, 2:]
        assert np.all(np.abs(lg[:, :, :2] - lc[:, :, :2]) <= 1e-9 * np.maximum(sig, np.abs(lc[:, :, :2])))
        assert np.all(np.abs(lg[:, :, 2:] - lc[:, :, 2:]) <= 1e-7 * sig)
        with pytest.raises(mbt.MbtError):
            t.transverse_log(5, 9)


def test_transverse_kick_changes_the_angles(mbt, orc):
    """Not a no-op: with the transverse resonator removed the angles of the same turn differ by K(tau)/E0."""
    cfg = _cfg(m=1, n_per_bunch=4096, n_bins=32, radiation=0)
    cfg0 = _cfg(m=1, n_per_bunch=4096, n_bins=32, radiation=0)
    cfg0["transverse"]["resonators"] = []
    with mbt.Tracker(cfg) as t, mbt.Tracker(cfg0) as t0:
        x, xp, y, yp = t.transverse_particles()
        t.set_transverse(x + 1e-3, xp, y - 5e-4, yp)          # a dipole offset so that the sums are not noise
        t0.set_transverse(x + 1e-3, xp, y - 5e-4, yp)
        t.track(1)
        t0.track(1)
        kx, ky = t.transverse_wake()
        assert np.abs(kx).max() > 0 and np.abs(ky).max() > 0
        assert not t0.transverse_wake()[0].any()
        d = t.transverse_particles()[1] - t0.transverse_particles()[1]
        assert np.abs(d).max() > 0
        assert np.abs(d).max() <= np.abs(kx).max() / cfg["ring"]["E0_eV"] * (1 + 1e-12)
        assert np.array_equal(t.transverse_particles()[0], t0.transverse_particles()[0])   # the kick acts on u' only


def test_transverse_full_size_c4(mbt, orc):
    """The workload `bench.py --transverse --rw-turns 20` times (363 x 1e5 particles, 6-D, resistive wall), in its launch
    configuration: initial distribution and one tracked turn element by element against the oracle, then properties
    that hold at any size."""
    cfg = W.config("c4")
    cfg["transverse"] = W.transverse_planes(rw_amp_x=2.0e9, rw_amp_y=1.0e9, rw_turns=20)
    o = orc.Oracle(cfg, lr_mode=1)
    with mbt.Tracker(cfg) as t:
        for g, c in zip(t.transverse_particles(), o.transverse_particles()):
            assert particle_errors(g, c) <= TOL_PARTICLE
        del g, c
        o.track(1); t.track(1)
        errs = {}
        for nm, g, c in zip(("x", "xp", "y", "yp"), t.transverse_particles(), o.transverse_particles()):
            errs[nm] = particle_errors(g, c)
        del g, c
        tau_c, delta_c = o.particles()
        tau_g, delta_g = t.particles()
        errs["tau"], errs["delta"] = particle_errors(tau_g, tau_c), particle_errors(delta_g, delta_c)
        print(errs)
        assert max(errs.values()) <= TOL_PARTICLE, errs
        if np.array_equal(t.histogram(), o.histogram()):
            for g, c in zip(t.dipole() + t.transverse_wake(), o.dipole() + o.transverse_wake()):
                assert wake_error(g, c) <= TOL_WAKE
        for g, c in zip(t.rw_kick(), o.rw_kick()):
            assert np.abs(g - c).max() <= TOL_WAKE * np.abs(c).max()
        # the dipole sums are fixed-point integers: a second handle reproduces them bit for bit
        sx1, sy1 = t.dipole()
    with mbt.Tracker(cfg) as t2:
        t2.track(1)
        sx2, sy2 = t2.dipole()
        assert np.array_equal(sx1, sx2) and np.array_equal(sy1, sy2)
        m = t2.moments()
        assert np.all(t2.histogram().sum(axis=1) == m[:, 0]) and np.all(m[:, 0] + m[:, 1] == cfg["fill"]["n_per_bunch"])


def test_many_particles_per_bunch_fewer_fixed_point_bits(mbt, orc):
    """N_p > 2^18 per bunch: the fixed-point dipole sums give up bits so that N_p 2^bits stays below 2^62 (here 43,
    and 41 for the million-particle bunch of c2); sums, kicks and coordinates keep their tolerances."""
    cfg = _cfg(m=1, n_per_bunch=300_001, n_bins=64)
    o = orc.Oracle(cfg)
    x, xp, y, yp = o.transverse_particles()
    o.set_transverse(x + 2.0e-4, xp, y - 1.0e-5, yp)
    o.track(1)
    with mbt.Tracker(cfg) as t:
        r = assert_transverse_turn_parity(o, t, cfg)
        print(r)
    cfg = W.config("c2")
    cfg["transverse"] = W.transverse_planes()
    o = orc.Oracle(cfg)
    o.track(1)
    with mbt.Tracker(cfg) as t:
        r = assert_transverse_turn_parity(o, t, cfg)
        print(r)


def test_three_cavities_and_lost_particles(mbt, orc):
    """The generic cavity loop (more than two cavities) of both passes, and particles far off the bucket (the
    large-argument branch of the RF sine, |phase| >= 2^16 rad) in the 6-D pass; NaN offsets stay NaN and do not crash."""
    for transverse in (False, True):
        cfg = _cfg(m=2, n_per_bunch=1025, n_bins=32, harmonic=True) if transverse else W.tiny(m=2, n_per_bunch=1025, n_bins=32, harmonic=True)
        cfg["cavities"].append(dict(V_volt=0.12e6, m=4, phase_rad=0.7))
        o = orc.Oracle(cfg)
        tau, delta = o.particles()
        tau = tau.copy()
        tau[:, ::5] += 1.0e-4          # 3e5 rad of RF phase
        tau[:, 1::7] -= 3.0e-6
        o.set_particles(tau, delta, 0)
        o.track(2)
        with mbt.Tracker(cfg) as t:
            for _ in range(2):
                if transverse:
                    assert_transverse_turn_parity(o, t, cfg)
                else:
                    assert_single_turn_parity(o, t, cfg)
    cfg = _cfg(m=2, n_per_bunch=300, n_bins=16)
    o = orc.Oracle(cfg)
    x, xp, y, yp = [a.copy() for a in o.transverse_particles()]
    x[0, 3] = np.nan
    with mbt.Tracker(cfg) as t:
        t.set_transverse(x, xp, y, yp)
        o.set_transverse(x, xp, y, yp)
        t.track(2); o.track(2)
        g, c = t.transverse_particles(), o.transverse_particles()
        for a, b in zip(g, c):
            # the NaN poisons the x dipole sum of its bin, hence the x' kick of every particle behind it -- the same
            # particles on both sides; bunch 1 and the y plane never see it
            assert np.array_equal(np.isfinite(a), np.isfinite(b))
            ok = np.isfinite(b)
            assert np.allclose(a[ok], b[ok], rtol=1e-9, atol=1e-30)
        assert np.isfinite(g[2]).all() and np.isfinite(g[3]).all() and np.isfinite(g[0][1]).all()
        assert not np.isfinite(g[1][0]).all()
        assert np.array_equal(t.histogram(), o.histogram())


def test_transverse_on_a_caller_owned_stream(mbt, orc):
    """The caller's stream (a torch stream) with the library's side stream forked off it: 40 turns through the
    graph-replayed path (unrolled graph + single-turn graphs), twice, against the oracle; two handles on two streams at
    the same time do not disturb each other."""
    import torch
    cfg = _cfg(m=3, n_per_bunch=2500, n_bins=32)
    cfg["transverse"].update(rw_amp_x=2.0e9, rw_amp_y=1.0e9, rw_turns=3)
    o = orc.Oracle(cfg, log_capacity_turns=80)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    with mbt.Tracker(cfg, log_capacity_turns=80, stream=s1.cuda_stream) as a, \
            mbt.Tracker(cfg, log_capacity_turns=80, stream=s2.cuda_stream) as b:
        for _ in range(2):
            a.track(40); b.track(40)
            o.track(40)
        lc = o.transverse_log(1, 80)
        for t in (a, b):
            lg = t.transverse_log(1, 80)
            assert np.all(np.abs(lg[:, :, :2] - lc[:, :, :2]) <= 1e-8 * lc[:, :, 2:])
            for g, c in zip(t.transverse_particles(), o.transverse_particles()):
                assert particle_errors(g, c) <= 1e-9
        assert np.array_equal(a.dipole()[0], b.dipole()[0])        # fixed-point sums: identical bit for bit
        for u, v in zip(a.transverse_particles(), b.transverse_particles()):
            assert np.array_equal(u, v)


def test_set_particles_keeps_a_pending_transverse_kick(mbt):
    """mbt_set_particles replaces tau and delta only: the transverse kick still pending from the last tracked turn must
    reach x', y' first (it is not the caller's to lose)."""
    cfg = _cfg(m=2, n_per_bunch=3000, n_bins=32)
    cfg["transverse"].update(rw_amp_x=2.0e9, rw_amp_y=1.0e9, rw_turns=2)
    with mbt.Tracker(cfg) as a, mbt.Tracker(cfg) as b:
        for t in (a, b):
            x, xp, y, yp = t.transverse_particles()
            t.set_transverse(x + 1e-3, xp, y - 1e-3, yp)
            t.track(2)
        tau, delta = a.particles()                 # flushes the pending kicks of `a`
        ra = a.transverse_particles()
        b.set_particles(tau, delta, 2)             # no getter in between
        rb = b.transverse_particles()
        for u, v in zip(ra, rb):
            assert np.array_equal(u, v)


def test_transverse_edge_cases(mbt, orc):
    """Degenerate inputs of the 6-D pass: everybody outside the bin window (no dipole sums, no wake kick, the
    resistive-wall kick still reaches every particle); offsets far beyond the fixed-point range X_max = 64 rms (the
    fp64 overflow path of the dipole sums) and a bunch sitting exactly on the axis (<u^2> = 0)."""
    # (1) all particles outside the window
    cfg = _cfg(m=3, n_per_bunch=500, n_bins=16)
    cfg["transverse"].update(rw_amp_x=2.0e9, rw_amp_y=1.0e9, rw_turns=2)
    o = orc.Oracle(cfg)
    tau, delta = o.particles()
    o.set_particles(tau + 120e-12, delta * 0.0, 0)
    x, xp, y, yp = o.transverse_particles()
    o.set_transverse(x + 1e-3, xp, y - 1e-3, yp)
    o.track(2)
    with mbt.Tracker(cfg) as t:
        for _ in range(2):
            r = assert_transverse_turn_parity(o, t, cfg)
        assert np.all(t.moments()[:, 0] == 0) and not t.dipole()[0].any() and not t.transverse_wake()[0].any()
        assert np.abs(t.rw_kick()[0]).max() > 0
    # (2) outliers beyond X_max and an on-axis bunch
    cfg = _cfg(m=3, n_per_bunch=2049, n_bins=32)
    o = orc.Oracle(cfg)
    x, xp, y, yp = [a.copy() for a in o.transverse_particles()]
    x[0, ::97] = 0.5                               # 1e4 sigma_x: far outside 64 rms of the rest ... but they raise the rms
    x[0, 5] = 40.0                                 # ... and this one is beyond 64 rms whatever the others do
    y[0, 7] = -3.0
    x[1, :] = 0.0; xp[1, :] = 0.0; y[1, :] = 0.0; yp[1, :] = 0.0
    o.set_transverse(x, xp, y, yp)
    o.track(1)
    with mbt.Tracker(cfg) as t:
        for _ in range(3):
            r = assert_transverse_turn_parity(o, t, cfg)
        sx, sy = t.dipole()
        assert np.abs(sx[0]).max() > 1.0 and np.abs(sy[0]).max() > 0.5    # the outliers are in the sums
    # (3) too many bins for the 6-D pass's shared memory: a clean error, not a launch failure
    big = _cfg(m=1, n_per_bunch=64, n_bins=4000)
    with pytest.raises(mbt.MbtError) as e:
        mbt.Tracker(big)
    assert e.value.code == -1 and "shared memory" in str(e.value)


def test_transverse_entry_points_refuse_a_longitudinal_handle(mbt):
    cfg = W.tiny()
    with mbt.Tracker(cfg) as t:
        with pytest.raises(mbt.MbtError) as e:
            t.transverse_particles()
        assert e.value.code == -1
        with pytest.raises(mbt.MbtError):
            t.moments_transverse()
        with pytest.raises(mbt.MbtError):
            t.dipole()
        with pytest.raises(mbt.MbtError):
            t.rw_kick()
        with pytest.raises(mbt.MbtError):
            t.transverse_log(1, 0)
    bad = _cfg()
    bad["transverse"]["rw_turns"] = -2
    with pytest.raises(mbt.MbtError):
        mbt.Tracker(bad)
    bad = _cfg()
    bad["transverse"]["x"]["beta_m"] = 0.0
    with pytest.raises(mbt.MbtError):
        mbt.Tracker(bad)
