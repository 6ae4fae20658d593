"""Helpers shared by the GPU parity tests: build an oracle and a CUDA sampler on the same seeded inputs and
compare their taps / states with the tolerances of BASELINE.json north_star."""
import numpy as np

from oracle import api as O
from paper_2105_08026_b200 import binding as B
from paper_2105_08026_b200 import synth

# north_star: per-object log-densities rel 1e-12 (fp64) / 1e-5 (fp32) with absolute floor tol*max(1,|pi|);
# population sum rel 1e-10; accept sequences identical except where |log alpha - log u| < 1e-9 (fp64).
TOL = {B.F64: dict(pi=1e-12, chi=1e-13, L=1e-12, pop=1e-12, tie=1e-9),
       B.F32_STATE_F64_REDUCE: dict(pi=1e-5, chi=2e-6, L=1e-5, pop=1e-5, tie=1e-4)}


def make_pair(model, n, seed, precision=B.F64, theta_mode=B.THETA_DEVICE_TAIL, astar=0.44, inputs=None, theta0=None,
              keep_moments=False, max_trace_rows=0, freeze_theta=False, block_threads=0, blocks_per_sm=0,
              want_oracle=True, flags=0, adapt_until=0, prior_mean=None, prior_sd=None):
    if inputs is None:
        maker = {0: synth.make_normal1d, 1: synth.make_thinned_schechter1d, 2: synth.make_binormal2d,
                 3: synth.make_linreg_me1d, 4: synth.make_bb1_fluxnoise1d,
                 5: synth.make_normal3d_knowncov}[model]
        kw = dict(fp32=True) if (precision == B.F32_STATE_F64_REDUCE and model in (0, 3)) else {}
        if model == 3 and precision == B.F64:
            kw = dict(fp32=False)
        inputs = maker(n, seed, **kw)
    th0 = inputs["theta0"] if theta0 is None else theta0
    orc = None
    if want_oracle:
        orc = O.Sampler(model, n, seed=seed, precision=precision, target_accept_chi=astar,
                        keep_chi_moments=keep_moments, freeze_theta=freeze_theta, adapt_until=adapt_until,
                        prior_mean=prior_mean, prior_sd=prior_sd)
        orc.set_data(inputs["cols"])
        if inputs["consts"] is not None:
            orc.set_model_consts(inputs["consts"])
        orc.set_init(th0)
    gpu = B.Sampler(model, n, seed=seed, precision=precision, theta_mode=theta_mode, target_accept_chi=astar,
                    keep_chi_moments=keep_moments, max_trace_rows=max_trace_rows, freeze_theta=freeze_theta,
                    block_threads=block_threads, blocks_per_sm=blocks_per_sm, flags=flags, adapt_until=adapt_until,
                    prior_mean=prior_mean, prior_sd=prior_sd)
    gpu.set_data(inputs["cols"])
    if inputs["consts"] is not None:
        gpu.set_model_consts(inputs["consts"])
    gpu.set_init(th0)
    return orc, gpu, inputs


def sync_gpu_to_oracle(orc, gpu):
    st = orc.get_state()
    gpu.set_state(st["chi"], st["L"], st["theta"], st["L_theta"], st["t"])
    return st


def close(a, b, rel, floor_scale=1.0):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    both_inf = np.isinf(a) & np.isinf(b) & (np.sign(a) == np.sign(b))
    with np.errstate(invalid="ignore"):
        ok = np.abs(a - b) <= rel * np.maximum(floor_scale, np.maximum(np.abs(a), np.abs(b)))
    return ok | both_inf


def compare_step(to, tg, precision, state_before, what=""):
    """Compare one iteration's taps (oracle `to`, GPU `tg`) from identical fed state.
    Returns the number of accept decisions that legitimately differ (near ties, inside the band)."""
    tol = TOL[precision]
    L0 = state_before["L"]
    scale = np.abs(L0).max(0) + np.abs(state_before["chi"]).max(0)        # natural size of a proposal step
    assert np.array_equal(to["u"], tg["u"]), f"{what}: accept uniforms must be bit-identical"
    d = np.abs(to["chi_prop"] - tg["chi_prop"]).max(0)
    # z differs by a few ulp of libm vs CUDA; when cos(2 pi u2) ~ 0 the ABSOLUTE error stays ~ulp * radius * L
    assert np.all(d <= tol["chi"] * 8 * np.maximum(scale, 1.0)), f"{what}: chi' max err {d.max():.3e}"
    assert np.all(close(to["pi_cur"], tg["pi_cur"], tol["pi"])), f"{what}: pi_cur"
    # pi_prop inherits d(pi)/d(chi) * delta(chi'): allow for it
    dp = np.abs(to["pi_prop"] - tg["pi_prop"])
    fin = np.isfinite(to["pi_prop"]) & np.isfinite(tg["pi_prop"])
    assert np.array_equal(np.isfinite(to["pi_prop"]), np.isfinite(tg["pi_prop"])) or (~fin).sum() <= 2, f"{what}: support"
    bound = tol["pi"] * np.maximum(1.0, np.abs(to["pi_prop"])) * 64
    assert np.all(dp[fin] <= bound[fin]), f"{what}: pi_prop max err {np.max(dp[fin] / bound[fin]):.2f}x"
    assert np.all(np.abs(to["alpha"] - tg["alpha"]) <= 64 * tol["pi"] * np.maximum(1.0, np.abs(to["pi_prop"]))), f"{what}: alpha"
    mism = to["accepted"] != tg["accepted"]
    with np.errstate(divide="ignore"):
        gap = np.abs(np.log(to["alpha"]) - np.log(to["u"]))
    assert np.all(gap[mism] < tol["tie"]), f"{what}: {int((gap[mism] >= tol['tie']).sum())} accept mismatches outside the tie band"
    same = ~mism
    assert np.all(close(to["L_new"], tg["L_new"], tol["L"] * 16, floor_scale=0.0) | (np.abs(to["L_new"] - tg["L_new"]) <= tol["L"] * 16 * np.abs(L0).max(0))), f"{what}: L_new"
    assert np.all(close(to["a"][same], tg["a"][same], tol["pop"] * 64)), f"{what}: a_i"
    assert np.all(close(to["b"][same], tg["b"][same], tol["pop"] * 64)), f"{what}: b_i"
    if not mism.any():
        # population sums: relative 1e-10 (north_star); Delta relative to the size of its terms
        assert abs(to["S"] - tg["S"]) <= 1e-10 * max(1.0, abs(to["S"])) * (1 if precision == B.F64 else 1e4), f"{what}: S"
        dsum = np.abs(to["b"] - to["a"]).sum()
        assert abs(to["Delta"] - tg["Delta"]) <= 1e-10 * max(1.0, dsum, abs(to["Delta"])) * (1 if precision == B.F64 else 1e4), f"{what}: Delta"
    return int(mism.sum())


def compare_theta_step(to, tg, what="", rel=1e-9):
    np.testing.assert_allclose(tg["theta_prop"], to["theta_prop"], rtol=rel, atol=rel, err_msg=f"{what}: theta'")
    assert tg["u_theta"] == to["u_theta"], f"{what}: theta accept uniform must be bit-identical"
    for k in ("T_cur", "T_prop", "lp_cur", "lp_prop"):
        assert np.all(close(to[k], tg[k], 1e-10)), f"{what}: {k} {to[k]} vs {tg[k]}"
