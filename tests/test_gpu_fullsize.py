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
        s.set_init(inp["theta0"], theta_chol0=inp["theta_chol0"])      # the recipe's theta proposal scale, as benched
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
    general on-chip kernel (resident_gen.cuh: 148 x 384); 40 iterations."""
    c, orc, gpu = _pair("C6")
    orc.run(40, 0, 1)
    gpu.run(40, 0, 1, sync=True)
    assert gpu.get_stats()["block_threads"] == 384, "C6 must run the general on-chip kernel"
    so, sg = orc.get_state(), gpu.get_state()
    np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["chi"], so["chi"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["L"], so["L"], rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(sg["L_theta"], so["L_theta"], rtol=1e-8, atol=1e-12)
    st, sto = gpu.get_stats(), orc.get_stats()
    assert st["chi_accepts"] == sto["chi_accepts"] and st["theta_accepts"] == sto["theta_accepts"]


def test_c3_full_size_free_running():
    """C3 as benched: N = 1e6, 2-D latent, streaming kernel with dedicated tail warps (148 x (384 + 128)); 8 iterations."""
    c, orc, gpu = _pair("C3")
    orc.run(8, 0, 1)
    gpu.run(8, 0, 1, sync=True)
    st = gpu.get_stats()
    assert (st["grid_blocks"], st["block_threads"]) == (148, 512)
    assert (st["dedicated_tail"], st["stage_steps"], st["l2_prefetch"]) == (1, 2, 0), "C3 as benched: k_persistent_dt (DESIGN.md 8.7b)"
    so, sg = orc.get_state(), gpu.get_state()
    np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["chi"], so["chi"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["L"], so["L"], rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(sg["L_theta"], so["L_theta"], rtol=1e-8, atol=1e-12)
    assert st["chi_accepts"] == orc.get_stats()["chi_accepts"]


def test_c4_full_size_single_steps():
    """C4 as benched: N = 1e7, fp32 state / fp64 reductions (SURVEY 8(c) protocol (ii) for fp32).  fp32 log targets differ
    by ~1e-7 relative between the two sides, which flips a few accept decisions per iteration (expected ~1e-6 per
    decision), so every iteration starts from the oracle's state.  Per iteration:
      - the launch configuration bench.py times (k_persistent<AHEAD>: staged draws + L2 prefetch) and the tapped
        k_sweep + k_tail pair give the SAME bits (state and theta), so the taps speak for the benched kernel;
      - flips are split into inside / outside the fp32 near-tie band (1e-4) and each must be explained by the measured
        difference of the two sides' log alpha (a decision can only differ if log u lies between them);
      - a_i, b_i of objects rejected on both sides (identical chi) agree to 1e-12; S and Delta equal the exactly rounded
        sums of the GPU's own terms to 1e-10 (the deterministic reduction at full size) and the oracle's sums up to what
        the terms moved by."""
    import math
    c, orc, gpu = _pair("C4")
    n = c.n_objects
    flips_in = flips_out = 0
    for it in range(2):
        st = orc.get_state()
        gpu.set_state(st["chi"], st["L"], st["theta"], st["L_theta"], st["t"])
        gpu.run(1, 0, 1, sync=True)
        sg = gpu.get_state()
        gpu.set_state(st["chi"], st["L"], st["theta"], st["L_theta"], st["t"])
        tg = gpu.debug_step(10 ** 12, 1)
        sd = gpu.get_state()
        for k in ("chi", "L", "theta", "L_theta"):
            assert np.array_equal(sg[k], sd[k]), f"benched kernel and tapped kernels differ in {k}"
        to = orc.step(10 ** 12, 1, taps=True)
        so = orc.get_state()
        assert np.array_equal(to["u"], tg["u"])
        with np.errstate(divide="ignore", invalid="ignore"):
            la_o = np.minimum(0.0, to["pi_prop"] - to["pi_cur"])
            la_g = np.minimum(0.0, tg["pi_prop"] - tg["pi_cur"])
            gap = np.abs(la_o - np.log(to["u"]))
        mism = to["accepted"] != tg["accepted"]
        inside = mism & (gap < 1e-4)
        flips_in += int(inside.sum())
        flips_out += int((mism & ~inside).sum())
        assert mism.sum() <= 200, f"{int(mism.sum())} accept decisions differ in one fp32 iteration of {n}"
        assert np.all(gap[mism] <= np.abs(la_g - la_o)[mism] * (1 + 1e-6) + 1e-6), "a flip the log-alpha difference does not explain"
        assert np.all(np.abs(tg["pi_cur"] - to["pi_cur"]) <= 1e-5 * np.maximum(1.0, np.abs(to["pi_cur"]))), "pi_cur (north_star fp32: 1e-5)"
        ok = ~mism
        np.testing.assert_allclose(sg["L"][0][ok], so["L"][0][ok], rtol=2e-5)
        rej = (to["accepted"] == 0) & (tg["accepted"] == 0)
        assert np.all(np.abs(tg["a"][rej] - to["a"][rej]) <= 1e-12 * np.maximum(1.0, np.abs(to["a"][rej]))), "a_i of rejected objects"
        assert np.all(np.abs(tg["b"][rej] - to["b"][rej]) <= 1e-9 * np.maximum(1.0, np.abs(to["b"][rej]))), "b_i of rejected objects (theta' to 1e-9)"
        S_ref, D_ref = math.fsum(tg["a"]), math.fsum(tg["b"] - tg["a"])
        dsum = float(np.abs(tg["b"] - tg["a"]).sum())
        assert abs(tg["S"] - S_ref) <= 1e-10 * abs(S_ref), "S against the exactly rounded sum of its terms"
        assert abs(tg["Delta"] - D_ref) <= 1e-10 * max(1.0, dsum), "Delta against the exactly rounded sum of its terms"
        assert abs(tg["S"] - to["S"]) <= 1e-10 * abs(to["S"]) + float(np.abs(tg["a"] - to["a"]).sum())
        assert abs(tg["Delta"] - to["Delta"]) <= 1e-10 * dsum + float(np.abs((tg["b"] - tg["a"]) - (to["b"] - to["a"])).sum())
        # theta is decided from fp64 sums of fp64 population terms: only the flipped objects perturb it
        np.testing.assert_allclose(sg["theta"], so["theta"], rtol=1e-6, atol=1e-6)
    stg = gpu.get_stats()
    assert (stg["grid_blocks"], stg["block_threads"]) == (148, 512)
    assert (stg["stage_steps"], stg["l2_prefetch"]) == (2, 1), "C4 as benched: staged draws + L2 prefetch (DESIGN.md 8.7)"
    print(f"C4: {flips_in} accept flips inside the fp32 near-tie band (1e-4), {flips_out} outside it, in {2 * n} fp32 decisions")
