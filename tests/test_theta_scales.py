"""The theta proposal scales of the input recipe (synth.THETA_COND_CHOL) against what they claim to
be: chol of the unit-N covariance of theta given the latents at the generating truth, recomputed through the oracle's
functions (tests/golden/make_theta_scales.py) at a small N, and against the closed forms where there are any."""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden"))
from make_theta_scales import conditional_cov_unit_n  # noqa: E402
from paper_2105_08026_b200 import synth  # noqa: E402


def _unpack(v, d):
    L = np.zeros((d, d))
    L[np.tril_indices(d)] = v
    return L


@pytest.mark.parametrize("model,d", [(0, 2), (1, 3), (2, 5), (3, 3), (4, 3), (5, 3)])
def test_stored_factors_are_the_conditional_covariance(model, d):
    L = _unpack(synth.THETA_COND_CHOL[model], d)
    C_stored = L @ L.T
    C = conditional_cov_unit_n(model, 3000 if model != 4 else 8000)
    sd, sd_s = np.sqrt(np.diag(C)), np.sqrt(np.diag(C_stored))
    # M4: ln l is informed by the few objects fainter than l, so its scale varies by tens of per cent between catalogs
    assert np.all(np.abs(sd_s / sd - 1) < (0.25 if model != 4 else 0.5)), (sd_s, sd)
    corr, corr_s = C / np.outer(sd, sd), C_stored / np.outer(sd_s, sd_s)
    assert np.all(np.abs(corr - corr_s) < (0.15 if model != 4 else 0.3)), (corr, corr_s)


def test_closed_forms():
    L0 = _unpack(synth.THETA_COND_CHOL[0], 2)
    np.testing.assert_allclose(L0 @ L0.T, np.diag([1.0, 0.5]), atol=2e-3)           # mu | chi: tau^2 / N; log tau | chi: 1 / (2N)
    L5 = _unpack(synth.THETA_COND_CHOL[5], 3)
    np.testing.assert_allclose(L5 @ L5.T, synth.NN3_CPOP, rtol=2e-3)                # mu | chi ~ N(chibar, C_pop / N)
    L3 = _unpack(synth.THETA_COND_CHOL[3], 3)
    XtX = np.array([[1.0, 1.5], [1.5, 3.0]])                                        # z ~ U(0, 3): E z = 1.5, E z^2 = 3
    np.testing.assert_allclose((L3 @ L3.T)[:2, :2], 0.09 * np.linalg.inv(XtX), rtol=5e-3)
    d = synth.theta_chol0(1, 300_000)
    assert d.shape == (6,) and abs(d[0] - 1.481 * 2.38 / np.sqrt(3 * 300_000)) < 1e-12
