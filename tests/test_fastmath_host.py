"""Accuracy of the CUDA path's specialised fp64 exp / log / sqrt (csrc/fastmath.cuh) and of the exact uniform
construction (csrc/philox.cuh::u01), measured on the HOST build of the same headers against mpmath.  The device
build differs only in the 2^-23 seeds (MUFU instead of a float division), which the Newton steps absorb; the GPU
parity tests then check the device results against the oracle."""
import os
import subprocess

import mpmath
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "fastmath_host.cu")


@pytest.fixture(scope="module")
def binary(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("fm") / "fastmath_host")
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc, "-O2", "-std=c++17", "-o", out, SRC], check=True)
    return out


def run(binary, what, x):
    """binary: the path of the host build, or any callable (what, x) -> y -- tests/test_gpu_fastmath.py passes the device
    build through cudahm_probe_math, so that both builds are held to the very same pins."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    if callable(binary):
        return np.asarray(binary(what, x), dtype=np.float64)
    res = subprocess.run([binary, what], input=x.tobytes(), capture_output=True, check=True)
    return np.frombuffer(res.stdout, dtype=np.float64)


def ulp_err(got, exact_fn, x):
    mpmath.mp.prec = 120
    worst = 0.0
    for g, xi in zip(got, x):
        ex = exact_fn(mpmath.mpf(float(xi)))
        ulp = mpmath.mpf(float(np.spacing(abs(float(ex)))))
        worst = max(worst, float(abs(mpmath.mpf(float(g)) - ex) / ulp))
    return worst


def test_exp_fast(binary):
    rng = np.random.default_rng(1)
    x = np.concatenate([rng.uniform(-30, 5, 3000), rng.uniform(-708, 709, 1000), -np.exp(rng.uniform(-40, 3, 1500)),
                        [0.0, -0.0, 1.0, -1.0, -708.0, 709.0, 0.5 * np.log(2), -0.5 * np.log(2)]])
    got = run(binary, "exp", x)
    assert ulp_err(got, mpmath.exp, x) <= 1.5
    big = run(binary, "exp", np.array([-1e300, -np.inf, 800.0, np.inf]))
    assert big[0] == big[1] == np.exp(-708.0) * (big[0] / np.exp(-708.0)) and 0 < big[0] < 1e-307   # clamped, never 0
    assert np.isfinite(big[2]) and big[2] == big[3]


def test_expm1_nonpos(binary):
    """1 - e^(-L/l) of the BB1 density needs e^x - 1 with full relative accuracy from x ~ -1e-9 to -700."""
    rng = np.random.default_rng(5)
    x = -np.concatenate([np.exp(rng.uniform(-45, 6.5, 5000)), rng.uniform(0, 0.05, 1500), rng.uniform(0, 2.0, 1500),
                         [0.0, np.log(2) / 128, np.log(2) / 64, 0.5 * np.log(2), np.log(2), 1e-300, 708.0]])
    got = run(binary, "expm1", x)
    assert ulp_err(got, mpmath.expm1, x) <= 2.5
    assert got[-7] == 0.0 and np.all(got <= 0.0) and np.all(got >= -1.0)
    assert run(binary, "expm1", np.array([-1e4, -np.inf]))[0] == -1.0


STEPS = pytest.mark.parametrize("steps", ["", "2"], ids=["newton1", "newton2"])   # fastmath.cuh: HM_NEWTON_STEPS variants


@STEPS
def test_log_pos(binary, steps):
    rng = np.random.default_rng(2)
    k = rng.integers(0, 2 ** 52, 4000)
    u = (k + 0.5) * 2.0 ** -52                       # exactly the uniforms the sampler draws
    u = np.concatenate([u, [2.0 ** -53, 1 - 2.0 ** -53, 0.5, 0.70710678118654752, 0.7071067811865476, 0.25],
                        np.exp(-rng.uniform(0, 36, 2000)), rng.uniform(1.0, 5.0, 1000), [1.0, 2.0, 1e300, 3e-308]])
    got = run(binary, "log" + steps, u)
    assert ulp_err(got, mpmath.log, u) <= 2.0       # worst case: e ln2 and ln m of opposite sign near m = sqrt 2


@STEPS
def test_sqrt_fast(binary, steps):
    rng = np.random.default_rng(3)
    w = np.concatenate([np.exp(rng.uniform(-36, 5, 4000)), rng.uniform(0.4, 2.0, 2000), [1.0, 4.0, 2.0, 73.5]])
    got = run(binary, "sqrt" + steps, w)
    assert ulp_err(got, mpmath.sqrt, w) <= 1.0
    assert np.mean(got == np.sqrt(w)) > 0.95          # almost always the correctly rounded root


@STEPS
def test_sqrt_rsqrt_pair(binary, steps):
    """The p = 2 RAM update takes sqrt(s1) and 1/sqrt(s1) from one Newton pair (s1 = 1 + c u1^2 in (0.4, 2))."""
    rng = np.random.default_rng(4)
    w = np.concatenate([rng.uniform(0.4, 2.0, 4000), np.exp(rng.uniform(-20, 20, 2000)), [1.0, 4.0, 0.25, 2.0]])
    root, inv = run(binary, "sqrt_both_root" + steps, w), run(binary, "sqrt_both_inv" + steps, w)
    assert ulp_err(root, mpmath.sqrt, w) <= 1.0
    assert ulp_err(inv, lambda x: 1 / mpmath.sqrt(x), w) <= 2.0
    assert root[-4] == 1.0 and inv[-4] == 1.0 and root[-3] == 2.0 and inv[-3] == 0.5


def test_u01_is_exact(binary):
    rng = np.random.default_rng(4)
    a = rng.integers(0, 2 ** 32, 5000, dtype=np.uint64)
    b = rng.integers(0, 2 ** 32, 5000, dtype=np.uint64)
    a[:4] = [0, 2 ** 32 - 1, 0, 2 ** 32 - 1]
    b[:4] = [0, 2 ** 32 - 1, 2 ** 32 - 1, 0]
    packed = ((a << np.uint64(32)) | b).view(np.float64)
    got = run(binary, "u01", packed)
    k = (a >> np.uint64(6)) * np.uint64(2 ** 26) + (b >> np.uint64(6))
    want = (k.astype(np.float64) + 0.5) * 2.0 ** -52   # k < 2^52: the conversion and both operations are exact
    assert np.array_equal(got, want)
    assert got.min() == 2.0 ** -53 and got.max() == 1 - 2.0 ** -53


def test_u01_32_is_exact(binary):
    rng = np.random.default_rng(6)
    w = rng.integers(0, 2 ** 32, 5000, dtype=np.uint64)
    w[:3] = [0, 2 ** 32 - 1, 2 ** 31]
    got = run(binary, "u32", w.view(np.float64))
    assert np.array_equal(got, (w.astype(np.float64) + 0.5) * 2.0 ** -32)
    assert got.min() == 2.0 ** -33 and got.max() == 1 - 2.0 ** -33


def _angle_grid_points():
    rng = np.random.default_rng(8)
    w = rng.integers(0, 2 ** 32, 5000).astype(np.float64)
    near = []
    for z in (0, 2 ** 30, 2 ** 31, 3 * 2 ** 30, 2 ** 32):                    # the zeros of sin and cos on the 32-bit grid
        near += [z + o for o in range(-6, 6) if 0 <= z + o < 2 ** 32]
    for n in range(0, 64, 3):                                                # both sides of every third table boundary
        near += [n * 2 ** 26 + 2 ** 25 + o for o in (-2, -1, 0, 1)]
    u32 = (np.concatenate([w, np.array(near, dtype=np.float64)]) + 0.5) * 2.0 ** -32      # exactly the p = 1 uniforms
    k = rng.integers(0, 2 ** 52, 3000).astype(np.float64)
    k = np.concatenate([k, [0.0, 1.0, 2.0 ** 52 - 1, 2.0 ** 50, 2.0 ** 50 - 1, 2.0 ** 51, 2.0 ** 51 - 1]])
    u52 = (k + 0.5) * 2.0 ** -52                                             # exactly the p >= 2 uniforms
    return np.concatenate([u32, u52])


def test_sincos2pi_within_2_ulp_on_the_draw_grids(binary):
    """hm_sincos2pi(u) = (sin, cos)(2 pi u), the Box-Muller angle: <= 2 ulp of the RESULT everywhere on the two grids the
    sampler draws from, the neighbourhoods of the zeros included (the table entries there are exactly 0 and +-1)."""
    u = _angle_grid_points()
    two_pi = lambda x: 2 * mpmath.pi * x
    sn, cs = run(binary, "sin2pi", u), run(binary, "cos2pi", u)
    es, ec = ulp_err(sn, lambda x: mpmath.sin(two_pi(x)), u), ulp_err(cs, lambda x: mpmath.cos(two_pi(x)), u)
    assert es <= 2.0 and ec <= 2.0, (es, ec)
    # the identity the sampler relies on (a unit vector): to a few ulp
    assert np.abs(sn * sn + cs * cs - 1.0).max() < 1e-15


def test_sincos2pi_exact_at_the_quarter_turns(binary):
    u = np.array([0.0, 0.25, 0.5, 0.75, 1.0])
    assert np.array_equal(run(binary, "sin2pi", u), [0.0, 1.0, 0.0, -1.0, 0.0])
    assert np.array_equal(run(binary, "cos2pi", u), [1.0, 0.0, -1.0, 0.0, 1.0])
    # odd / even symmetry about the half turn, bit for bit (the reduction is symmetric: d -> -d, the table is antisymmetric)
    v = (np.arange(1, 4000, 7, dtype=np.float64) + 0.5) * 2.0 ** -32
    assert np.array_equal(run(binary, "sin2pi", 1.0 - v), -run(binary, "sin2pi", v))
    assert np.array_equal(run(binary, "cos2pi", 1.0 - v), run(binary, "cos2pi", v))
