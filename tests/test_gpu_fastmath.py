"""The DEVICE build of csrc/fastmath.cuh against the pins of tests/test_fastmath_host.py, function by function, through
cudahm_probe_math: the sampler's kernels call these very functions, and on the device the reciprocal and the reciprocal
square root start from MUFU seeds (about 20 good bits) that the host build can only imitate."""
import pytest

import test_fastmath_host as T
from paper_2105_08026_b200 import binding as B

pytestmark = pytest.mark.gpu

FN = {"exp": B.MATH_EXP, "expm1": B.MATH_EXPM1_NONPOS, "log": B.MATH_LOG, "sqrt": B.MATH_SQRT,
      "sqrt_both_root": B.MATH_SQRT_BOTH_ROOT, "sqrt_both_inv": B.MATH_SQRT_BOTH_INV,
      "sin2pi": B.MATH_SIN2PI, "cos2pi": B.MATH_COS2PI,
      "log2": B.MATH_LOG_2, "sqrt2": B.MATH_SQRT_2, "sqrt_both_root2": B.MATH_SQRT_BOTH_ROOT_2,
      "sqrt_both_inv2": B.MATH_SQRT_BOTH_INV_2}


def device(what, x):
    return B.probe_math(FN[what], x)


@pytest.mark.parametrize("pin", [T.test_exp_fast, T.test_expm1_nonpos, T.test_sincos2pi_within_2_ulp_on_the_draw_grids,
                                 T.test_sincos2pi_exact_at_the_quarter_turns], ids=lambda f: f.__name__[5:])
def test_device_build_meets_the_host_pin(pin):
    pin(device)


@pytest.mark.parametrize("steps", ["", "2"], ids=["newton1", "newton2"])
@pytest.mark.parametrize("pin", [T.test_log_pos, T.test_sqrt_fast, T.test_sqrt_rsqrt_pair], ids=lambda f: f.__name__[5:])
def test_device_build_meets_the_host_pin_in_both_newton_variants(pin, steps):
    pin(device, steps)
