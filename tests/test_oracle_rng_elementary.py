"""Pins for the oracle's random stream and fp32 elementary functions.

Nothing here compares the oracle with itself: Philox against published known answers and the
cuRAND header constants; the fixed-operation fp32 log / sincos against libm in fp64 over ALL 2^24
inputs the tracer can ever feed them."""
import os
import re

import numpy as np
import pytest

import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(GOLD, "philox4x32_10_kat.txt")) if l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert O.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])


def test_philox_constants_match_curand_header():
    path = "/usr/local/cuda/include/curand_philox4x32_x.h"
    if not os.path.exists(path):
        pytest.skip("CUDA toolkit header not present")
    txt = open(path).read()
    want = {"PHILOX_W32_0": 0x9E3779B9, "PHILOX_W32_1": 0xBB67AE85,
            "PHILOX_M4x32_0": 0xD2511F53, "PHILOX_M4x32_1": 0xCD9E8D57}
    for name, val in want.items():
        m = re.search(r"#define\s+%s\s+\(?(0x[0-9A-Fa-f]+)" % name, txt)
        assert m and int(m.group(1), 16) == val


def test_philox_counter_sensitivity():
    # each counter / key word must matter (a dropped word would collide)
    base = O.philox4x32_10((1, 2, 3, 4), (5, 6))
    seen = {base}
    for i in range(4):
        c = [1, 2, 3, 4]
        c[i] += 1
        seen.add(O.philox4x32_10(c, (5, 6)))
    seen.add(O.philox4x32_10((1, 2, 3, 4), (6, 6)))
    seen.add(O.philox4x32_10((1, 2, 3, 4), (5, 7)))
    assert len(seen) == 7


def _ulp_err(approx32, exact64):
    exact32 = exact64.astype(np.float32)
    ulp = np.spacing(np.abs(exact32)).astype(np.float64)
    ulp[ulp == 0] = np.finfo(np.float32).tiny
    return np.abs(approx32.astype(np.float64) - exact64) / ulp


def test_fp32_log_exhaustive():
    """-ln(w) for every w = k 2^-24, k = 1..2^24 (all values 1-u0 can take): <= 2 ulp of libm fp64."""
    k = np.arange(1, (1 << 24) + 1, dtype=np.float64)
    w = (k / (1 << 24)).astype(np.float32)
    got = O.neg_log_f32(w)
    ref = -np.log(w.astype(np.float64))
    assert got[-1] == 0.0 and np.all(got >= 0)
    nz = ref > 0
    err = _ulp_err(got[nz], ref[nz])
    assert err.max() <= 2.0, err.max()
    # monotone non-increasing in w (a free-path sampler must preserve order of the uniforms)
    assert np.all(np.diff(got.astype(np.float64)) <= 0)
    # mean of -ln(1-u) over the lattice = 1 - O(2^-24 * 24)
    assert abs(got.astype(np.float64).mean() - 1.0) < 1e-5


def test_fp32_sincos_exhaustive():
    k = np.arange(0, 1 << 24, dtype=np.float64)
    u = (k / (1 << 24)).astype(np.float32)
    s, c = O.sincos_2pi_f32(u)
    ang = 2.0 * np.pi * u.astype(np.float64)
    assert np.abs(s.astype(np.float64) - np.sin(ang)).max() < 1.5e-7
    assert np.abs(c.astype(np.float64) - np.cos(ang)).max() < 1.5e-7
    n2 = s.astype(np.float64) ** 2 + c.astype(np.float64) ** 2
    assert np.abs(n2 - 1).max() < 4e-7
    # exact values at the quarter turns
    q = [0, 1 << 22, 1 << 23, 3 << 22]
    assert list(s[q]) == [0.0, 1.0, 0.0, -1.0] and list(c[q]) == [1.0, 0.0, -1.0, 0.0]
