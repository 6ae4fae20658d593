"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default block size, default
theta mode: the on-chip kernel for C2, the streaming persistent kernel for C3 / C4), against the oracle run on the
whole population.  fp64: a free-running stretch must reproduce the oracle's state element by element; fp32 (C4): one
iteration from identical state, with the expected handful of near-tie accept flips counted."""
import numpy as np
import pytest

from oracle import api as O
from paper_2105_08026_b200 import binding as B
from paper_2105_08026_b200 import synth

pytestmark = pytest.mark.gpu


def _pair(name, iters_moments=False):
    c = synth.CONFIGS[name]
    inp = synth.make_inputs(name)
    kw = dict(seed=c.seed, precision=c.precision, target_accept_chi=c.target_accept_chi,
              target_accept_theta=c.target_accept_theta, keep_chi_moments=c.keep_chi_moments)
    orc = O.Sampler(c.model, c.n_objects, **kw)
    gpu = B.Sampler(c.model, c.n_objects, theta_mode=B.THETA_DEVICE_TAIL, max_trace_rows=64, **kw)
    for s in (orc, gpu):
        s.set_data(inp["cols"])
        if inp["consts"] is not None:
            s.set_model_consts(inp["consts"])
        s.set_init(inp["theta0"])
    return c, orc, gpu


def test_c2_full_size_free_running():
    """C2 as benched: N = 3e5, thinned-Schechter model, moments on, on-chip kernel (148 x 640).  25 iterations
    = 7.5e6 decisions (near-tie probability ~1e-9 each) free-running against the oracle."""
    c, orc, gpu = _pair("C2")
    iters, burn, thin = 25, 5, 5
    orc.run(iters, burn, thin)
    gpu.run(iters, burn, thin, sync=True)
    st = gpu.get_stats()
    assert (st["grid_blocks"], st["block_threads"]) == (148, 640), "C2 must run the on-chip kernel on a 148-SM part"
    so, sg = orc.get_state(), gpu.get_state()
    np.testing.assert_allclose(sg["theta"], so["theta"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["chi"], so["chi"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["L"], so["L"], rtol=1e-9)
    mo, vo, ko = orc.get_chi_moments()
    mg, vg, kg = gpu.get_chi_moments()
    assert kg == ko == iters - burn
    np.testing.assert_allclose(mg, mo, rtol=1e-10, atol=1e-10)
    np.testing.assert_allclose(vg, vo, rtol=1e-8, atol=1e-13)
    sto = orc.get_stats()
    assert st["chi_accepts"] == sto["chi_accepts"] and st["nonfinite"] == sto["nonfinite"]
    assert st["theta_accepts"] == sto["theta_accepts"]


def test_c5_full_size_free_running():
    """C5, the paper's case study (BB1 population, N = 1e5) in the on-chip kernel; 12 iterations."""
    c, orc, gpu = _pair("C5")
    orc.run(12, 0, 1)
    gpu.run(12, 0, 1, sync=True)
    st = gpu.get_stats()
    assert st["block_threads"] == 640
    so, sg = orc.get_state(), gpu.get_state()
    np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["chi"], so["chi"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["L"], so["L"], rtol=1e-9)
    np.testing.assert_allclose(sg["L_theta"], so["L_theta"], rtol=1e-8, atol=1e-12)
    sto = orc.get_stats()
    assert st["chi_accepts"] == sto["chi_accepts"] and st["theta_accepts"] == sto["theta_accepts"]


def test_c6_full_size_free_running():
    """C6, the normal-normal benchmark at the paper's largest population (N = 3e4, p = 3) in the
    streaming persistent kernel; 40 iterations."""
    c, orc, gpu = _pair("C6")
    orc.run(40, 0, 1)
    gpu.run(40, 0, 1, sync=True)
    so, sg = orc.get_state(), gpu.get_state()
    np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["chi"], so["chi"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["L"], so["L"], rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(sg["L_theta"], so["L_theta"], rtol=1e-8, atol=1e-12)
    st, sto = gpu.get_stats(), orc.get_stats()
    assert st["chi_accepts"] == sto["chi_accepts"] and st["theta_accepts"] == sto["theta_accepts"]


def test_c3_full_size_free_running():
    """C3 as benched: N = 1e6, 2-D latent, streaming persistent kernel (148 x 512); 8 iterations."""
    c, orc, gpu = _pair("C3")
    orc.run(8, 0, 1)
    gpu.run(8, 0, 1, sync=True)
    st = gpu.get_stats()
    assert (st["grid_blocks"], st["block_threads"]) == (148, 512)
    assert (st["stage_steps"], st["l2_prefetch"]) == (0, 0), "C3 (state + data inside L2, p = 2) keeps the plain variant"
    so, sg = orc.get_state(), gpu.get_state()
    np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["chi"], so["chi"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["L"], so["L"], rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(sg["L_theta"], so["L_theta"], rtol=1e-8, atol=1e-12)
    assert st["chi_accepts"] == orc.get_stats()["chi_accepts"]


def test_c4_full_size_single_steps():
    """C4 as benched: N = 1e7, fp32 state / fp64 reductions.  fp32 log-density differences of ~1e-7 flip a few accept
    decisions per iteration (expected ~1e-6 per decision), so each iteration starts from the oracle's
    state: everything else must agree to fp32 rounding, the population sums to 1e-10-ish of their terms."""
    c, orc, gpu = _pair("C4")
    n = c.n_objects
    flips = 0
    for it in range(2):
        st = orc.get_state()
        gpu.set_state(st["chi"], st["L"], st["theta"], st["L_theta"], st["t"])
        orc.run(1, 0, 1)
        gpu.run(1, 0, 1, sync=True)
        so, sg = orc.get_state(), gpu.get_state()
        dchi = np.abs(sg["chi"][0] - so["chi"][0])
        moved = dchi > 2e-5 * np.maximum(1.0, np.abs(so["chi"][0]))
        flips += int(moved.sum())
        assert moved.sum() <= 200, f"{int(moved.sum())} accept decisions differ in one fp32 iteration of {n}"
        ok = ~moved
        np.testing.assert_allclose(sg["L"][0][ok], so["L"][0][ok], rtol=2e-5)
        # theta is decided from fp64 sums of fp64 population terms: only the flipped objects perturb it
        np.testing.assert_allclose(sg["theta"], so["theta"], rtol=1e-6, atol=1e-6)
    stg = gpu.get_stats()
    assert (stg["grid_blocks"], stg["block_threads"]) == (148, 512)
    assert (stg["stage_steps"], stg["l2_prefetch"]) == (2, 1), "C4 as benched: staged draws + L2 prefetch (DESIGN.md 8.7)"
    print(f"C4: {flips} near-tie accept flips in {2 * n} fp32 decisions")
