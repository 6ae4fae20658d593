"""Pins P1/P2 of the oracle's random streams: Philox4x32-10 words against the
published known answers and against ATen's own engine; uniforms exact dyadic rationals built from
the documented bit layout; Box-Muller normals against the normal law (moments + Kolmogorov-Smirnov)."""
import os
import subprocess
import sys

import numpy as np
import pytest
from scipy import stats

from oracle import api as O

HERE = os.path.dirname(os.path.abspath(__file__))


def _kat_rows():
    rows = []
    with open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(x, 16) for x in line.split()]
            rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_philox_known_answers():
    rows = _kat_rows()
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert O.philox4x32_10(ctr, key) == out


@pytest.fixture(scope="module")
def aten_bin(tmp_path_factory):
    import torch
    inc = os.path.join(os.path.dirname(torch.__file__), "include")
    if not os.path.exists(os.path.join(inc, "ATen", "core", "PhiloxRNGEngine.h")):
        pytest.skip("ATen Philox header not present")
    exe = str(tmp_path_factory.mktemp("aten") / "aten_philox_pin")
    subprocess.run(["g++", "-O1", "-std=c++17", "-I" + inc, os.path.join(HERE, "aten_philox_pin.cpp"), "-o", exe],
                   check=True)
    return exe


def test_philox_matches_aten_engine(aten_bin):
    """A library routine (at::Philox4_32) evaluated on random counters/keys and on the sampler's own
    counter layout must give the oracle's words."""
    g = np.random.default_rng(123)
    cases = [tuple(int(x) for x in g.integers(0, 2 ** 32, 6)) for _ in range(40)]
    args = []
    for c0, c1, c2, c3, k0, k1 in cases:
        args += [str(k0 | (k1 << 32)), str(c2 | (c3 << 32)), str(c0 | (c1 << 32))]
    out = subprocess.run([aten_bin] + args, check=True, capture_output=True, text=True).stdout.split("\n")
    for (c0, c1, c2, c3, k0, k1), line in zip(cases, out):
        assert O.philox4x32_10([c0, c1, c2, c3], [k0, k1]) == [int(x, 16) for x in line.split()]


def test_stream_counter_layout(aten_bin):
    """key = seed words; counter = (obj lo, kind<<24 | obj bits 32..55, t, d)."""
    cases = [(0, 0, 0, 1, 0), (7, 1, 0, 5, 2), (0xDEADBEEFCAFE, 0, 299_999, 10_000, 1),
             (3, 0, (1 << 40) + 17, 2 ** 32 - 1, 3)]
    args = []
    for seed, kind, obj, t, d in cases:
        c0, c1 = obj & 0xFFFFFFFF, (kind << 24) | ((obj >> 32) & 0xFFFFFF)
        args += [str(seed), str(t | (d << 32)), str(c0 | (c1 << 32))]
    out = subprocess.run([aten_bin] + args, check=True, capture_output=True, text=True).stdout.split("\n")
    for (seed, kind, obj, t, d), line in zip(cases, out):
        assert O.stream_words(seed, kind, obj, t, d) == [int(x, 16) for x in line.split()]


def test_uniform_f64_is_the_documented_dyadic_rational():
    for obj in (0, 1, 12345, 299_999):
        for t in (1, 2, 1000):
            w = O.stream_words(9, O.KIND_PLATE, obj, t, 0)
            k = ((w[0] >> 6) << 26) | (w[1] >> 6)            # 52 bits
            u = O.uniform_f64(9, O.KIND_PLATE, obj, t, 0)
            assert 0.0 < u < 1.0
            # exact: (k + 1/2) 2^-52 has 53 significant bits
            assert u == (2 * k + 1) / float(2 ** 53)
            assert float(u).hex() == ((2 * k + 1) / float(2 ** 53)).hex()


def test_uniform_extremes_never_hit_0_or_1():
    # the smallest / largest representable outputs of the mapping are strictly inside (0,1)
    lo, hi = (0 + 0.5) * 2.0 ** -52, ((2 ** 52 - 1) + 0.5) * 2.0 ** -52
    assert lo > 0.0 and hi < 1.0 and np.log(hi) < 0.0
    lo32 = np.float32(0.5) * np.float32(2.0 ** -23)
    hi32 = (np.float32(2 ** 23 - 1) + np.float32(0.5)) * np.float32(2.0 ** -23)
    assert lo32 > 0 and hi32 < 1


def test_normals_f64_follow_the_normal_law():
    n_obj = 60_000
    z = np.array([O.normals_f64(5, O.KIND_PLATE, i, 3, 2) for i in range(n_obj)])   # (n_obj, 2)
    for col in (z[:, 0], z[:, 1], z.reshape(-1)):
        assert abs(col.mean()) < 4.0 / np.sqrt(col.size)
        assert abs(col.var() - 1.0) < 4.0 * np.sqrt(2.0 / col.size)
        assert stats.kstest(col, "norm").pvalue > 1e-3
    # the two members of a Box-Muller pair are uncorrelated; radius^2 is chi^2_2
    assert abs(np.corrcoef(z[:, 0], z[:, 1])[0, 1]) < 4.0 / np.sqrt(n_obj)
    assert stats.kstest((z ** 2).sum(1), "chi2", args=(2,)).pvalue > 1e-3
    # skewness / excess kurtosis
    assert abs(stats.skew(z.reshape(-1))) < 0.03 and abs(stats.kurtosis(z.reshape(-1))) < 0.06


def test_normals_are_a_function_of_the_documented_words():
    """z0 = sqrt(-2 ln u1) cos(2 pi u2) with u1 from (w0,w1), u2 from (w2,w3) of draw d=1 -- evaluated with
    mpmath at 40 digits, so a swapped word, a sin/cos swap or a missing factor fails."""
    import mpmath as mp
    mp.mp.dps = 40
    for obj, t in ((0, 1), (17, 9), (299_999, 10_000)):
        w = O.stream_words(2, O.KIND_THETA, obj, t, 1)
        u1 = mp.mpf(2 * (((w[0] >> 6) << 26) | (w[1] >> 6)) + 1) / mp.mpf(2) ** 53
        u2 = mp.mpf(2 * (((w[2] >> 6) << 26) | (w[3] >> 6)) + 1) / mp.mpf(2) ** 53
        r = mp.sqrt(-2 * mp.log(u1))
        z = O.normals_f64(2, O.KIND_THETA, obj, t, 2)
        assert abs(z[0] - float(r * mp.cos(2 * mp.pi * u2))) < 1e-14 * max(1.0, abs(z[0]))
        assert abs(z[1] - float(r * mp.sin(2 * mp.pi * u2))) < 1e-14 * max(1.0, abs(z[1]))
    # draws beyond the first pair come from d = 2, 3, ...
    z5 = O.normals_f64(2, O.KIND_THETA, 0, 4, 5)
    w = O.stream_words(2, O.KIND_THETA, 0, 4, 3)
    u1 = mp.mpf(2 * (((w[0] >> 6) << 26) | (w[1] >> 6)) + 1) / mp.mpf(2) ** 53
    u2 = mp.mpf(2 * (((w[2] >> 6) << 26) | (w[3] >> 6)) + 1) / mp.mpf(2) ** 53
    assert abs(z5[4] - float(mp.sqrt(-2 * mp.log(u1)) * mp.cos(2 * mp.pi * u2))) < 1e-14


def _u52(wa, wb):
    import mpmath as mp
    return mp.mpf(2 * (((wa >> 6) << 26) | (wb >> 6)) + 1) / mp.mpf(2) ** 53


def test_plate_draws_f64_are_the_documented_function_of_the_pair_words():
    """objects draw in pairs m = i >> 1.  p = 1: ONE call per pair (draw 0 of pair m), every word a
    32-bit uniform (w + 1/2) 2^-32: w0 -> u1, w1 -> u2, cos branch for the even object, sin branch for the odd one,
    accept uniform from w2 / w3.  p >= 2: 52-bit accept uniform from draw 0 of pair m, words (w0,w1) for the even object
    and (w2,w3) for the odd one; normals per object, draws 1.. of object i.  Evaluated with mpmath."""
    import mpmath as mp
    mp.mp.dps = 40
    for i, t in ((0, 1), (1, 1), (17, 9), (299_998, 10_000), (299_999, 10_000), (2 ** 33 + 5, 3)):
        m, h = i >> 1, i & 1
        a = O.stream_words(9, O.KIND_PLATE, m, t, 0)
        z, u = O.plate_draws_f64(9, i, t, 1)
        u32 = lambda w: mp.mpf(2 * w + 1) / mp.mpf(2) ** 33
        assert u == float(u32(a[3] if h else a[2])) and 2.0 ** -33 <= u <= 1 - 2.0 ** -33
        u1, u2 = u32(a[0]), u32(a[1])
        r = mp.sqrt(-2 * mp.log(u1))
        want = r * (mp.sin(2 * mp.pi * u2) if h else mp.cos(2 * mp.pi * u2))
        assert abs(z[0] - float(want)) < 1e-14 * max(1.0, abs(z[0]))
        # p = 2: uniform as above, normals are the per-object Box-Muller pair
        z2, u_2 = O.plate_draws_f64(9, i, t, 2)
        assert u_2 == float(_u52(a[2], a[3]) if h else _u52(a[0], a[1]))
        assert np.array_equal(z2, O.normals_f64(9, O.KIND_PLATE, i, t, 2))


def test_plate_draws_follow_their_laws_and_pairs_are_independent():
    n = 60_000
    d = [O.plate_draws_f64(13, i, 5, 1) for i in range(n)]
    z = np.array([x[0][0] for x in d]); u = np.array([x[1] for x in d])
    assert abs(z.mean()) < 4 / np.sqrt(n) and abs(z.var() - 1) < 4 * np.sqrt(2 / n)
    assert stats.kstest(z, "norm").pvalue > 1e-3 and stats.kstest(u, "uniform").pvalue > 1e-3
    assert 0 < u.min() and u.max() < 1
    ze, zo, ue, uo = z[0::2], z[1::2], u[0::2], u[1::2]
    assert abs(np.corrcoef(ze, zo)[0, 1]) < 4 / np.sqrt(n / 2)
    assert abs(np.corrcoef(ue, uo)[0, 1]) < 4 / np.sqrt(n / 2)
    assert abs(np.corrcoef(ze, ue)[0, 1]) < 4 / np.sqrt(n / 2)
    # joint law of a pair: radius^2 ~ chi^2_2 and the angle uniform (full independence of the two normals)
    assert stats.kstest(ze ** 2 + zo ** 2, "chi2", args=(2,)).pvalue > 1e-3
    assert stats.kstest((np.arctan2(zo, ze) / (2 * np.pi)) % 1.0, "uniform").pvalue > 1e-3
    # consecutive iterations of one object are independent draws
    zt = np.array([O.plate_draws_f64(13, 7, t, 1)[0][0] for t in range(1, 20001)])
    assert abs(np.corrcoef(zt[:-1], zt[1:])[0, 1]) < 4 / np.sqrt(zt.size)
    assert stats.kstest(zt, "norm").pvalue > 1e-3


def test_plate_draws_f32():
    n = 40_000
    zs, us = np.empty(n, np.float32), np.empty(n, np.float32)
    for i in range(n):
        z, u = O.plate_draws_f32(11, i, 7, 1)
        zs[i] = z[0]; us[i] = u
    for i in (10, 11):
        w = O.stream_words(11, O.KIND_PLATE, i >> 1, 7, 0)
        assert us[i] == np.float32(((w[3 if i & 1 else 2] >> 9) + 0.5) * 2.0 ** -23)
        u1 = ((w[0] >> 9) + 0.5) * 2.0 ** -23
        u2 = ((w[1] >> 9) + 0.5) * 2.0 ** -23
        trig = np.sin if i & 1 else np.cos
        assert abs(float(zs[i]) - np.sqrt(-2 * np.log(u1)) * trig(2 * np.pi * u2)) < 1e-5
    assert 0 < us.min() and us.max() < 1
    assert stats.kstest(us.astype(np.float64), "uniform").pvalue > 1e-3
    assert stats.kstest(zs.astype(np.float64), "norm").pvalue > 1e-3
    assert abs(np.corrcoef(zs[0::2], zs[1::2])[0, 1]) < 4.0 / np.sqrt(n / 2)
    assert abs(np.corrcoef(us[0::2], us[1::2])[0, 1]) < 4.0 / np.sqrt(n / 2)
    # p = 2 keeps the per-object layout
    z2, u2_ = O.plate_draws_f32(11, 5, 7, 2)
    z0, z1, u = O.draws_f32(11, O.KIND_PLATE, 5, 7)
    assert z2[0] == z0 and z2[1] == z1 and u2_ == u


def test_draws_f32():
    n = 40_000
    zs, us = np.empty((n, 2), np.float32), np.empty(n, np.float32)
    for i in range(n):
        z0, z1, u = O.draws_f32(11, O.KIND_PLATE, i, 7)
        zs[i] = (z0, z1)
        us[i] = u
    w = O.stream_words(11, O.KIND_PLATE, 5, 7, 0)
    assert us[5] == np.float32(((w[2] >> 9) + 0.5) * 2.0 ** -23)
    u1 = ((w[0] >> 9) + 0.5) * 2.0 ** -23
    u2 = ((w[1] >> 9) + 0.5) * 2.0 ** -23
    assert abs(float(zs[5, 0]) - np.sqrt(-2 * np.log(u1)) * np.cos(2 * np.pi * u2)) < 1e-5
    assert abs(float(zs[5, 1]) - np.sqrt(-2 * np.log(u1)) * np.sin(2 * np.pi * u2)) < 1e-5
    assert 0 < us.min() and us.max() < 1
    assert stats.kstest(us.astype(np.float64), "uniform").pvalue > 1e-3
    assert stats.kstest(zs.reshape(-1).astype(np.float64), "norm").pvalue > 1e-3
    assert abs(np.corrcoef(zs[:, 0], us)[0, 1]) < 4.0 / np.sqrt(n)
