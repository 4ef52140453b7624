"""mbt_bunch_stats_noalloc against mbt_moments_transverse (GPU).

mbt_bunch_stats_noalloc is the statistics call for users who may not allocate device memory when they ask for the
statistics: a monitor sampling the beam on a second stream while mbt_track runs (cudaMalloc / cudaFree serialise against
everything in flight on the device, so an allocating call would stall the run it watches), or a host whose own memory
pool already holds all of HBM (a cudaMalloc from inside the library may then fail).  Its partial sums sit in one fixed
64 KiB array compiled into libmbt.so instead of in a buffer from cudaMalloc; every call on a device shares that array, and
the array keeps whatever the previous call left in it.

So the thing to check is not only that the numbers agree with the existing, handle-based path (mbt_moments_transverse,
which sums the same four coordinate arrays into memory mbt_create allocated), but that they still agree on a SECOND
call, made right after the first on a different beam state: left-over sums of call one must not leak into call two.
Both paths add their partial sums with floating-point atomics in whatever order the CTAs arrive, so they agree to rounding,
not bit for bit; the bars are the ones test_gpu_transverse.py holds mbt_moments_transverse to (means 1e-10, rms 1e-8, of
max(rms, |mean|)).

This file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here
must not hide the parity tests.  It makes no assumption about what ran before it -- the library looks up the array's
device address on the first call in the process, wherever that call comes from -- so it passes alone in a fresh process
and at the end of the whole suite alike."""
import numpy as np
import pytest

from paper_1809_00391_b200 import workloads as W

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


def _device_rows(torch, a, ld):
    """Host array [M][N_p] -> device tensor [M][ld] (ld >= N_p; the padding is filled with a value that would wreck the
    sums if the kernel read past N_p)."""
    m, n = a.shape
    d = torch.full((m, ld), 1.0e30, dtype=torch.float64, device="cuda")
    d[:, :n] = torch.from_numpy(np.ascontiguousarray(a)).to("cuda")
    return d


def _stats_noalloc(mbt, torch, coords, ld):
    """Upload four [M][N_p] host arrays and run the no-allocation entry point on torch's current stream."""
    m, n = coords[0].shape
    dev = [_device_rows(torch, c, ld) for c in coords]
    out = torch.full((m, 8), float("nan"), dtype=torch.float64, device="cuda")
    mbt.bunch_stats_noalloc(*(d.data_ptr() for d in dev), m, n, ld, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    return out.cpu().numpy()           # .cpu() waits for the stream: the call itself is asynchronous


def _assert_same_statistics(got, ref):
    for k in range(4):
        scale = np.maximum(ref[:, 4 + k], np.abs(ref[:, k]))
        assert np.all(np.abs(got[:, k] - ref[:, k]) <= 1e-10 * scale + 1e-300), ("mean", k, got[:, k], ref[:, k])
        assert np.all(np.abs(got[:, 4 + k] - ref[:, 4 + k]) <= 1e-8 * scale + 1e-300), ("rms", k, got[:, 4 + k], ref[:, 4 + k])


def test_noalloc_statistics_match_handle_path_on_two_calls_in_a_row(mbt):
    import torch
    torch.cuda.set_device(0)
    # 5 bunches of 20 001 particles: three 8192-particle tiles per bunch with a ragged last one, rows padded to ld
    cfg = W.tiny(n_per_bunch=20001, n_bins=32)
    cfg["transverse"] = W.transverse_planes()
    n = 20001
    ld = mbt.particle_stride(n) + 8
    with mbt.Tracker(cfg) as t:
        t.track(3)
        ref_a, state_a = t.moments_transverse(), t.transverse_particles()
        t.track(2)
        ref_b, state_b = t.moments_transverse(), t.transverse_particles()
    assert not np.array_equal(ref_a, ref_b)                     # the two calls really see different beams
    got_a = _stats_noalloc(mbt, torch, state_a, ld)             # first call: also the one that looks up the array
    got_b = _stats_noalloc(mbt, torch, state_b, ld)             # second call: the array still holds call one's sums
    _assert_same_statistics(got_a, ref_a)
    _assert_same_statistics(got_b, ref_b)
    # a third call on fewer bunches than before must not be disturbed by the rows it does not use
    got_c = _stats_noalloc(mbt, torch, [c[:2] for c in state_a], n)
    _assert_same_statistics(got_c, ref_a[:2])


def test_noalloc_rejects_what_the_fixed_array_cannot_hold(mbt):
    import torch
    torch.cuda.set_device(0)
    x = torch.zeros(8, dtype=torch.float64, device="cuda")
    out = torch.zeros(8, dtype=torch.float64, device="cuda")
    p, o = x.data_ptr(), out.data_ptr()
    with pytest.raises(mbt.MbtError) as e:
        mbt.bunch_stats_noalloc(p, p, p, p, mbt.NOALLOC_MAX_BUNCHES + 1, 1, 1, o)
    assert e.value.code == -1 and "MBT_NOALLOC_MAX_BUNCHES" in str(e.value)
    for bad in (dict(m=0, n=1, ld=1), dict(m=1, n=0, ld=1), dict(m=1, n=8, ld=4), dict(m=1, n=2 ** 32, ld=2 ** 32)):
        with pytest.raises(mbt.MbtError) as e:
            mbt.bunch_stats_noalloc(p, p, p, p, bad["m"], bad["n"], bad["ld"], o)
        assert e.value.code == -1
    with pytest.raises(mbt.MbtError):
        mbt.bunch_stats_noalloc(p, p, 0, p, 1, 8, 8, o)
    torch.cuda.synchronize()
    assert float(out.abs().sum()) == 0.0                        # nothing was enqueued by the refused calls
