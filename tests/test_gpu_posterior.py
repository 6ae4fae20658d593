"""Posterior agreement ON THE GPU (north_star: "posterior means and variances of theta agree within 4 Monte Carlo standard
errors"): free-running cudahm_run chains -- no oracle chain involved -- against the closed forms, exact grids and the
independent sampler that pin the oracle (tests/test_oracle_posterior.py P9, P11, P12; test_oracle_bb1.py; test_oracle_nn3.py:
the very same reference functions), at populations as large as each reference can be evaluated for.  The theta proposal
factor is the input recipe's (synth theta_chol0); theta acceptance must sit near the RAM target."""
import numpy as np
import pytest

from oracle import api as O
from paper_2105_08026_b200 import binding as B
from paper_2105_08026_b200 import synth
from test_oracle_bb1 import check_bb1_posterior
from test_oracle_nn3 import check_nn3_posterior
from test_oracle_nnp import check_nnp_posterior
from test_oracle_posterior import (check_binormal_posterior, check_linreg_posterior, check_normal1d_posterior,
                                   check_schechter_posterior)

pytestmark = pytest.mark.gpu


def _gpu_chain(model, inp, n, seed, burn, T, astar, precision=B.F64, thin=1):
    g = B.Sampler(model, n, seed=seed, precision=precision, target_accept_chi=astar, theta_mode=B.THETA_DEVICE_TAIL,
                  max_trace_rows=T // thin)
    g.set_data(inp["cols"])
    if inp["consts"] is not None:
        g.set_model_consts(inp["consts"])
    g.set_init(inp["theta0"], theta_chol0=inp["theta_chol0"])
    g.run(burn + T, burn, thin, sync=True)
    tr, st = g.get_theta_trace(), g.get_stats()
    assert tr.shape == (T // thin, g.dtheta)
    rate = st["theta_accepts"] / st["theta_proposals"]
    assert 0.10 < rate < 0.40, f"theta acceptance {rate:.3f}: the RAM adaptation of L_theta should home in on 0.234"
    g.close()
    return tr


def test_m0_theta_posterior_on_the_gpu():
    n = 2000
    inp = synth.make_normal1d(n, seed=135)
    check_normal1d_posterior(inp, _gpu_chain(B.M_NORMAL1D, inp, n, 135, 5000, 40000, 0.44))


def test_m1_theta_posterior_on_the_gpu():
    n = 2000
    inp = synth.make_thinned_schechter1d(n, seed=138)
    tr = _gpu_chain(B.M_THINNED_SCHECHTER1D, inp, n, 138, 10000, 60000, 0.44)
    o = O.Sampler(1, n, seed=138)                      # only for the oracle's pinned T(theta) in the amplitude check
    o.set_data(inp["cols"]); o.set_model_consts(inp["consts"]); o.set_init(inp["theta0"])
    check_schechter_posterior(inp, tr, o.theta_only, ngrid=41, nloc=401)


def test_m2_theta_posterior_on_the_gpu():
    n = 20000
    inp = synth.make_binormal2d(n, seed=137)
    check_binormal_posterior(inp, _gpu_chain(B.M_BINORMAL2D, inp, n, 137, 5000, 40000, 0.234), n_ref=36000)


@pytest.mark.parametrize("precision", [B.F64, B.F32_STATE_F64_REDUCE], ids=["f64", "f32"])
def test_m3_theta_posterior_on_the_gpu(precision):
    n = 20000
    inp = synth.make_linreg_me1d(n, seed=136, fp32=True)
    check_linreg_posterior(inp, _gpu_chain(B.M_LINREG_ME1D, inp, n, 136, 5000, 40000, 0.44, precision=precision), npts=41)


def test_m4_theta_posterior_on_the_gpu():
    n = 100
    inp = synth.make_bb1_fluxnoise1d(n, seed=41, truth=(-1.3, np.log(0.3), 0.0))
    check_bb1_posterior(inp, _gpu_chain(B.M_BB1_FLUXNOISE1D, inp, n, 41, 10000, 200000, 0.44), grid=(33, 65, 33))


def test_m5_theta_posterior_on_the_gpu():
    n = 20000
    inp = synth.make_normal3d_knowncov(n, seed=152)
    check_nn3_posterior(inp, _gpu_chain(B.M_NORMAL3D_KNOWNCOV, inp, n, 152, 5000, 40000, 0.234))


@pytest.mark.parametrize("p", [4, 5, 6])
def test_normal_family_theta_posterior_on_the_gpu(p):
    n = 20000
    inp = synth.make_normalpd_knowncov(n, seed=160 + p, p=p)
    check_nnp_posterior(inp, _gpu_chain(synth.nnp_model(p), inp, n, 160 + p, 8000, 40000, 0.234), p)
