"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol include/mbt.h
declares; the binding's struct layout matches the header (compiled probe); workloads are well-formed."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

from paper_1809_00391_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1809_00391_b200 import build
    return build.build()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "mbt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mbt_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(libpath):
    from paper_1809_00391_b200 import mbt
    lib = ctypes.CDLL(libpath)
    declared = _declared_symbols()
    assert len(declared) >= 20
    for s in declared:
        assert hasattr(lib, s), s
    assert sorted(mbt.SYMBOLS) == declared      # the binding covers exactly the header
    out = subprocess.run(["nm", "-D", "--defined-only", libpath], capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r" T (mbt_[a-z_0-9]+)", out))
    assert set(declared) <= exported


def test_host_only_entry_points(libpath):
    """Calls that touch no GPU: stride, version, error text, NULL handling."""
    from paper_1809_00391_b200 import mbt
    L = mbt.lib()
    assert mbt.particle_stride(37) == 40 and mbt.particle_stride(100000) == 100000 and mbt.particle_stride(1) == 4
    assert b"sm_100a" in L.mbt_version()
    assert L.mbt_turn(None) == -1
    assert L.mbt_destroy(None) == 0
    assert L.mbt_create(None, None) == -1
    assert b"null" in L.mbt_last_error()
    assert L.mbt_track(None, 1) == -1


def test_struct_layout_matches_header(tmp_path):
    """sizeof/offsetof of every struct as the C compiler sees the header vs the ctypes mirror."""
    from paper_1809_00391_b200 import mbt
    probe = tmp_path / "probe.c"
    probe.write_text('''
#include <stdio.h>
#include <stddef.h>
#include "mbt.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n", sizeof(mbt_ring), sizeof(mbt_cavity), sizeof(mbt_radiation), sizeof(mbt_fill),
         sizeof(mbt_resonator), sizeof(mbt_wake), sizeof(mbt_params), sizeof(mbt_tuning), sizeof(mbt_transverse), sizeof(mbt_plane));
  printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n", offsetof(mbt_params, cav), offsetof(mbt_params, rad), offsetof(mbt_params, fill),
         offsetof(mbt_params, wake), offsetof(mbt_params, seed), offsetof(mbt_params, d_tau), offsetof(mbt_params, stream),
         offsetof(mbt_params, device), offsetof(mbt_params, trans), offsetof(mbt_params, tuning),
         offsetof(mbt_tuning, pairs_per_thread), offsetof(mbt_tuning, turn_mode), offsetof(mbt_tuning, reserved));
  return 0;
}''')
    exe = tmp_path / "probe"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(probe)], check=True)
    a, b = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.strip().splitlines()
    sizes = [int(x) for x in a.split()]
    offs = [int(x) for x in b.split()]
    assert sizes == [ctypes.sizeof(c) for c in (mbt.Ring, mbt.Cavity, mbt.Radiation, mbt.Fill, mbt.Resonator, mbt.Wake, mbt.Params,
                                                mbt.Tuning, mbt.Transverse, mbt.Plane)]
    P, T = mbt.Params, mbt.Tuning
    assert offs == [P.cav.offset, P.rad.offset, P.fill.offset, P.wake.offset, P.seed.offset, P.d_tau.offset,
                    P.stream.offset, P.device.offset, P.trans.offset, P.tuning.offset,
                    T.pairs_per_thread.offset, T.turn_mode.offset, T.reserved.offset]


def test_make_params_marshalling():
    from paper_1809_00391_b200 import mbt
    cfg = W.config("c4", n_per_bunch=10)
    p, keep = mbt.make_params(cfg, log_capacity_turns=7)
    assert p.fill.n_bunches == 363 and p.fill.bucket[362] == 362 and p.fill.n_per_bunch == 10
    assert p.wake.n_res == 3 and p.wake.res[2].fr_Hz == 2.1e9 and p.wake.res[0].flags == 1
    assert p.wake.history_turns == 20 and p.log_capacity_turns == 7 and p.seed == 4
    assert np.isnan(p.cav[0].phase_rad)
    assert all(getattr(p.tuning, k) == 0 for k in mbt.TUNING_FIELDS) and list(p.tuning.reserved) == [0]
    p, keep = mbt.make_params(cfg, tuning=dict(turn_mode=1, tile_iters=3))
    assert p.tuning.turn_mode == 1 and p.tuning.tile_iters == 3 and p.tuning.pdl == 0
    with pytest.raises(KeyError):
        mbt.make_params(cfg, tuning=dict(no_such_knob=1))


def test_create_refuses_nonzero_reserved_tuning_word(libpath):
    """mbt.h: mbt_tuning.reserved "must be 0" -- any other value is MBT_EINVAL at validation, before a device is touched."""
    from paper_1809_00391_b200 import mbt
    L = mbt.lib()
    for bad in (1, -1):
        p, keep = mbt.make_params(W.config("c1"))
        p.tuning.reserved[0] = bad
        h = ctypes.c_void_p()
        assert L.mbt_create(ctypes.byref(p), ctypes.byref(h)) == -1 and not h.value
        assert b"tuning" in L.mbt_last_error()


def test_workloads_match_baseline_configs():
    shapes = {"c1": (1, 10_000, 200, 0, 1000), "c2": (1, 1_000_000, 1000, 0, 10_000), "c3": (3, 100_000, 500, 10, 20_000),
              "c4": (363, 100_000, 300, 20, 10_000), "c5": (484, 200_000, 500, 50, 5_000)}
    for name, (m, npb, nb, k, turns) in shapes.items():
        c = W.config(name)
        assert len(c["fill"]["buckets"]) == m and c["fill"]["n_per_bunch"] == npb
        assert c["wake"]["n_bins"] == nb and c["wake"]["history_turns"] == k and c["n_turns"] == turns
    c4 = W.config("c4")
    q = np.array(c4["fill"]["charge_C"])
    assert c4["fill"]["buckets"] == list(range(363)) and abs(q.mean() / 1e-9 - 1) < 5e-3 and 0.01 < q.std() / 1e-9 < 0.03
    assert W.config("c3")["fill"]["buckets"] == [0, 161, 323]
    assert len(W.config("c5")["cavities"]) == 2 and len(W.config("c5")["wake"]["resonators"]) == 4
    # seeded: two calls give identical inputs
    assert W.config("c4") == W.config("c4")


def test_pass_tiling_host_logic():
    """mbt_plan_tiles (no device needed): the tilings of the BASELINE workloads on a B200 (148 SMs x 2 or 3 resident CTAs)
    and the properties every tiling has: it covers the bunch, tiles are whole iterations, the last tile is at least
    3/4 of the others."""
    from paper_1809_00391_b200 import build, mbt
    build.build()
    assert mbt.plan_tiles(50_000, 512, 363, 296) == (25 * 512, 4)          # c4, k_pass two pairs per thread: 4.9 waves
    assert mbt.plan_tiles(100_000, 512, 484, 296) == (66 * 512, 3)         # c5
    assert mbt.plan_tiles(50_000, 256, 363, 296) == (49 * 256, 4)          # c4, k_pass6
    assert mbt.plan_tiles(500_000, 256, 1, 444) == (5 * 256, 391)          # c2: just under one wave
    assert mbt.plan_tiles(5_000, 512, 1, 296) == (512, 10)                 # c1: one iteration per CTA
    import random
    rng = random.Random(3)
    for _ in range(300):
        ppb = rng.randint(1, 400_000)
        stride = rng.choice([256, 512])
        m = rng.choice([1, 2, 3, 22, 121, 363, 484, 1000])
        slots = rng.choice([148, 296, 444])
        tp, nt = mbt.plan_tiles(ppb, stride, m, slots)
        assert tp % stride == 0 and tp > 0 and nt >= 1
        assert nt * tp >= ppb > (nt - 1) * tp                                # covers the bunch, no empty tile
        it = tp // stride
        last = -(-(ppb - (nt - 1) * tp) // stride)
        assert nt == 1 or 4 * last >= 3 * it
    assert mbt.plan_tiles(50_000, 512, 363, 296, tile_iters=16) == (16 * 512, 7)   # mbt_tuning.tile_iters
    with pytest.raises(mbt.MbtError):
        mbt.plan_tiles(0, 512, 1, 296)
