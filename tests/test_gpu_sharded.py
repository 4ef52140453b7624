"""Bunch sharding on ONE GPU: the handles of all ranks live on the same device and the all-gather
is replaced by device-to-device copies between their exchange buffers, phase by phase (no kernel waits for another
launch).  The kernels and host code are exactly those a multi-GPU run uses (mbt_shard_turn_begin / _end); only the
collective is emulated.  The sharded run is compared with the oracle like the single-device one."""
import numpy as np
import pytest

from paper_1809_00391_b200 import workloads as W
from parity import TOL_PARTICLE, histogram_mismatch, particle_errors, wake_error

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


class Ranks:
    """All ranks of a sharded run on one device."""

    def __init__(self, mbt, cfg, world, log_capacity_turns=0):
        import torch
        from paper_1809_00391_b200 import sharded
        self.torch, self.world = torch, world
        m = len(cfg["fill"]["buckets"])
        n_lr = sum(1 for r in cfg["wake"]["resonators"] if r["flags"] & 2)
        self.rows, self.per_rank, total = sharded.exchange_layout(m, world, n_lr)
        self.n_lr = n_lr
        self.x = [torch.zeros(max(total, 2), dtype=torch.float64, device="cuda") for _ in range(world)]
        self.t = [mbt.Tracker(cfg, log_capacity_turns=log_capacity_turns,
                              shard=dict(rank=r, world=world, d_exchange=self.x[r].data_ptr() if n_lr else None))
                  for r in range(world)]

    def track(self, n):
        for _ in range(n):
            for t in self.t:
                t.shard_turn_begin()
            self.torch.cuda.synchronize()
            for dst in range(self.world):                       # the all-gather, as copies
                for src in range(self.world):
                    if src != dst:
                        sl = slice(src * self.per_rank, (src + 1) * self.per_rank)
                        self.x[dst][sl].copy_(self.x[src][sl])
            self.torch.cuda.synchronize()
            for t in self.t:
                t.shard_turn_end()

    def gather(self, what):
        return np.concatenate([getattr(t, what)() for t in self.t], axis=0)

    def particles(self):
        parts = [t.particles() for t in self.t]
        return np.concatenate([p[0] for p in parts]), np.concatenate([p[1] for p in parts])

    def wake(self):
        ws = [t.wake() for t in self.t]
        return [np.concatenate([w[k] for w in ws]) for k in range(3)]

    def resume(self, o, window=False):
        tau, delta = o.particles()
        for t in self.t:
            sl = slice(t.first_bunch, t.first_bunch + t.M)
            t.set_particles(tau[sl], delta[sl], o.turn)
            if window:                                           # after set_particles, which resets the shifts; own bunches only
                s_hist, s_next = o.window()
                t.set_window(s_hist[sl], s_next[sl])
            t.set_lr_history(o.lr_history())                     # every rank holds the whole history
        return tau, delta

    def close(self):
        for t in self.t:
            t.close()


@pytest.mark.parametrize("world", [1, 2, 3])
@pytest.mark.parametrize("kw", [dict(n_per_bunch=1001), dict(n_per_bunch=300, n_lr=3, k_hist=2, harmonic=True), dict(n_per_bunch=64, n_lr=0)])
def test_sharded_single_turns_match_oracle(mbt, orc, world, kw):
    cfg = W.tiny(**kw)                                           # 5 bunches in buckets 0, 3, 4, 100, 483
    o = orc.Oracle(cfg, lr_mode=0)
    o.track(4)
    R = Ranks(mbt, cfg, world)
    try:
        assert [t.M for t in R.t] == [mbt.shard_range(5, world, r)[1] for r in range(world)]
        for _ in range(3):
            R.resume(o)
            o.track(1)
            R.track(1)
            tau_c, delta_c = o.particles()
            tau_g, delta_g = R.particles()
            assert particle_errors(tau_g, tau_c) <= TOL_PARTICLE and particle_errors(delta_g, delta_c) <= TOL_PARTICLE
            bad, _ = histogram_mismatch(R.gather("histogram"), o.histogram(), tau_c, cfg)
            assert bad == 0
            for g, c in zip(R.wake(), o.wake()):
                assert wake_error(g, c) <= 1e-10
            m_g, m_c = R.gather("moments"), o.moments()
            assert np.array_equal(m_g[:, :2], m_c[:, :2]) and np.allclose(m_g[:, 2:], m_c[:, 2:], rtol=1e-8, atol=1e-22)
            hist_c = o.lr_history()
            for t in R.t:                                        # the whole history on every rank
                assert t.lr_history().shape == hist_c.shape
                if hist_c.size:
                    assert np.allclose(t.lr_history(), hist_c, rtol=0, atol=1e-10 * np.abs(hist_c).max())
    finally:
        R.close()


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_with_bunch_following_window(mbt, orc, world):
    """mbt_shard with window_mode = 1 (reading D31): every bunch displaced differently, so the per-bunch window shifts
    differ across the ranks' bunches.  The shift of a bunch's window multiplies its long-range SOURCE phasor (indexed by the
    rank's LOCAL bunch) and the phasor it WITNESSES, which is summed over ring rows and ready-flags indexed by the GLOBAL
    bunch -- the local / global mix this test walks through.  Single turns from the oracle's state incl. its windows, then
    turns without re-synchronisation; launches_per_turn of a sharded handle is 4 with long-range resonators."""
    cfg = W.tiny(m=5, n_per_bunch=1501, n_bins=32, k_hist=3, n_lr=2)
    cfg["wake"]["window_mode"] = 1
    o = orc.Oracle(cfg, lr_mode=0)
    tau0, delta0 = o.particles()
    off = np.array([[12e-12], [-20e-12], [0.0], [30e-12], [-8e-12]])
    o.set_particles(tau0 * 0.5 + off, delta0, 0)
    o.track(4)
    R = Ranks(mbt, cfg, world)
    try:
        assert all(t.launches_per_turn == 4 for t in R.t)
        for _ in range(3):
            R.resume(o, window=True)
            o.track(1)
            R.track(1)
            tau_c, delta_c = o.particles()
            tau_g, delta_g = R.particles()
            assert particle_errors(tau_g, tau_c) <= TOL_PARTICLE and particle_errors(delta_g, delta_c) <= TOL_PARTICLE
            sh_c, sn_c = o.window()
            sh_g = np.concatenate([t.window()[0] for t in R.t]); sn_g = np.concatenate([t.window()[1] for t in R.t])
            assert np.array_equal(sh_c, sh_g) and np.array_equal(sn_c, sn_g)
            bad, _ = histogram_mismatch(R.gather("histogram"), o.histogram(), tau_c, cfg, shifts=sh_c)
            assert bad == 0
            for g, c in zip(R.wake(), o.wake()):
                assert wake_error(g, c) <= 1e-10
        assert len(set(int(s) for s in o.window()[0])) >= 3      # the windows really sit in different places
        # own runs from the same displaced start, no re-synchronisation
        o2 = orc.Oracle(cfg, lr_mode=0)
        o2.set_particles(tau0 * 0.5 + off, delta0, 0)
        for t in R.t:
            sl = slice(t.first_bunch, t.first_bunch + t.M)
            t.set_particles((tau0 * 0.5 + off)[sl], delta0[sl], 0)
        o2.track(8)
        R.track(8)
        assert np.array_equal(np.concatenate([t.window()[0] for t in R.t]), o2.window()[0])
        assert np.array_equal(R.gather("histogram"), o2.histogram())
        assert particle_errors(R.particles()[1], o2.particles()[1]) <= 1e-10
        assert wake_error(R.wake()[0], o2.wake()[0]) <= 1e-9
    finally:
        R.close()


def test_sharded_run_without_resync_and_against_single_device(mbt, orc):
    """Nine turns from each side's own initial distribution (the Philox counters carry the GLOBAL bunch index): the sharded
    run against the oracle, and against the single-device library run on the c4 fill pattern (363 bunches over 4 ranks:
    chunks of 91, the last rank 90)."""
    cfg = W.tiny(n_per_bunch=777, n_bins=32)
    o = orc.Oracle(cfg, lr_mode=0)
    R = Ranks(mbt, cfg, 2)
    try:
        o.track(9)
        R.track(9)
        assert particle_errors(R.particles()[1], o.particles()[1]) <= 1e-10
        assert np.array_equal(R.gather("histogram"), o.histogram())
        assert wake_error(R.wake()[0], o.wake()[0]) <= 1e-9
        assert all(t.turn == 9 for t in R.t)
        with pytest.raises(mbt.MbtError):
            R.t[0].track(1)                                      # mbt_track is not how a sharded handle advances
    finally:
        R.close()
    cfg = W.config("c4", n_per_bunch=1500)
    R = Ranks(mbt, cfg, 4)
    try:
        with mbt.Tracker(cfg) as t:
            t.track(25)                                          # past the 20-turn history
            R.track(25)
            tau_s, delta_s = t.particles()
            tau_g, delta_g = R.particles()
            assert particle_errors(tau_g, tau_s) <= 1e-10 and particle_errors(delta_g, delta_s) <= 1e-10
            assert np.array_equal(R.gather("histogram"), t.histogram())
            assert wake_error(R.wake()[2], t.wake()[2]) <= 1e-10
    finally:
        R.close()
