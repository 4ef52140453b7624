"""Pins for the oracle's own Philox4x32-10 and its uniform -> normal transform (reading D8)."""
import os
import shutil
import subprocess

import numpy as np
import pytest
from scipy import stats

HERE = os.path.dirname(os.path.abspath(__file__))


def _kat():
    rows = []
    with open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(x, 16) for x in line.split()]
            rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_philox_known_answer_vectors(orc):
    rows = _kat()
    assert len(rows) == 3
    for ctr, key, want in rows:
        assert orc.philox(ctr, key) == want


def test_philox_against_cuda_toolkit_host_implementation(orc, tmp_path):
    """Independent implementation: the CUDA toolkit's curand_philox4x32_x.h compiled for the HOST."""
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    exe = str(tmp_path / "cph")
    subprocess.run([nvcc, "-Wno-deprecated-gpu-targets", "-o", exe, os.path.join(HERE, "aux", "curand_philox_host.cu")],
                   check=True, capture_output=True)
    out = subprocess.run([exe, "200"], check=True, capture_output=True, text=True).stdout.strip().splitlines()
    assert len(out) == 200
    for line in out:
        lhs, rhs = line.split("->")
        v = [int(x, 16) for x in lhs.split()]
        want = [int(x, 16) for x in rhs.split()]
        assert orc.philox(v[0:4], v[4:6]) == want


def test_uniforms_are_top_52_bits_plus_half(orc):
    # u = (k + 1/2) 2^-52 with k the top 52 bits of (x1:x0) resp. (x3:x2): exact in fp64, strictly in (0,1)
    for seed, c in [(1, (0, 0, 1, 0)), (0xDEADBEEF12345678, (7, 3, 99, 1)), (2**64 - 1, (2**32 - 1,) * 4)]:
        x = orc.philox(list(c), [seed & 0xFFFFFFFF, seed >> 32])
        u1, u2, zc, zs = orc.normal_pair(seed, *c)
        k1 = ((x[1] << 32) | x[0]) >> 12
        k2 = ((x[3] << 32) | x[2]) >> 12
        from fractions import Fraction
        assert Fraction(u1) == Fraction(2 * k1 + 1, 2**53)
        assert Fraction(u2) == Fraction(2 * k2 + 1, 2**53)
        assert 0.0 < u1 < 1.0 and 0.0 < u2 < 1.0
        # Box-Muller pair, evaluated here with mpmath-free high-precision-by-construction numpy longdouble
        r = np.sqrt(-2.0 * np.log(np.longdouble(u1)))
        th = 2.0 * np.pi * np.longdouble(u2)
        assert abs(float(r * np.cos(th)) - zc) < 1e-14
        assert abs(float(r * np.sin(th)) - zs) < 1e-14


def test_excitation_uniforms_are_32_bit_words_plus_half(orc):
    # excitation stream (reading D8): u_k = (x_k + 1/2) 2^-32 for each word of the block, exact in fp64, in (0,1);
    # (z0, z1) is the Box-Muller pair of (u0, u1), (z2, z3) that of (u2, u3)
    from fractions import Fraction
    for seed, c in [(1, (0, 0, 1, 0)), (0xDEADBEEF12345678, (7, 3, 99, 0)), (2**64 - 1, (2**32 - 1,) * 4)]:
        x = orc.philox(list(c), [seed & 0xFFFFFFFF, seed >> 32])
        u, z = orc.normal_quad(seed, *c)
        for k in range(4):
            assert Fraction(u[k]) == Fraction(2 * x[k] + 1, 2**33)
            assert 0.0 < u[k] < 1.0
        for h in range(2):
            r = np.sqrt(-2.0 * np.log(np.longdouble(u[2 * h])))
            th = 2.0 * np.pi * np.longdouble(u[2 * h + 1])
            assert abs(float(r * np.cos(th)) - z[2 * h]) < 1e-14
            assert abs(float(r * np.sin(th)) - z[2 * h + 1]) < 1e-14


def test_normals_are_standard_normal(orc):
    n = 100_000
    for draw in ("quad", "pair"):
        if draw == "quad":   # excitation stream: four normals per block
            z = np.array([orc.normal_quad(12345, i, 2, 7, 0)[1] for i in range(n // 2)]).ravel()
        else:                # initial-distribution stream: two normals per block
            z = np.array([orc.normal_pair(12345, i, 2, 0, 1)[2:] for i in range(n)]).ravel()
        m = z.size
        assert abs(z.mean()) < 4.0 / np.sqrt(m)
        assert abs(z.var() - 1.0) < 4.0 * np.sqrt(2.0 / m)
        assert abs(stats.kurtosis(z)) < 4.0 * np.sqrt(24.0 / m)
        assert abs(stats.skew(z)) < 4.0 * np.sqrt(6.0 / m)
        assert stats.kstest(z, "norm").pvalue > 1e-3
        # the members of a block are uncorrelated
        assert abs(np.corrcoef(z[0::2], z[1::2])[0, 1]) < 4.0 / np.sqrt(m / 2)
        if draw == "quad":
            assert abs(np.corrcoef(z[0::4], z[2::4])[0, 1]) < 4.0 / np.sqrt(m / 4)
            assert abs(np.corrcoef(z[1::4], z[3::4])[0, 1]) < 4.0 / np.sqrt(m / 4)


def test_streams_differ_by_tag_turn_bunch(orc):
    for draw in (orc.normal_pair, orc.normal_quad):
        base = draw(1, 5, 0, 1, 0)
        assert draw(1, 5, 0, 1, 1) != base   # tag
        assert draw(1, 5, 0, 2, 0) != base   # turn
        assert draw(1, 5, 1, 1, 0) != base   # bunch
        assert draw(2, 5, 0, 1, 0) != base   # seed
        assert draw(1 << 32, 5, 0, 1, 0) != draw(0, 5, 0, 1, 0)  # high key word is used
