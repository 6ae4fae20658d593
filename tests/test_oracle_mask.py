"""Pins of the oracle's frozen-member hooks (member properties "which should be held
fixed over the course of posterior simulation"): the per-object update mask and the per-object adaptation counter."""
import numpy as np
import pytest

from mcmc_util import mean_and_var_with_mcse
from oracle import api as O
from paper_2105_08026_b200 import synth


def _sampler(n, seed, **kw):
    inp = synth.make_normal1d(n, seed)
    s = O.Sampler(0, n, seed=seed, target_accept_chi=0.44, **kw)
    s.set_data(inp["cols"])
    s.set_init(inp["theta0"] if "theta0" not in kw else kw["theta0"])
    return s, inp


def test_held_objects_keep_chi_and_L_bit_for_bit_and_the_rest_sample_the_conjugate_law():
    n, burn, T = 40, 1500, 24000
    inp = synth.make_normal1d(n, seed=91)
    theta = np.array([0.2, -0.1])
    s = O.Sampler(0, n, seed=91, target_accept_chi=0.44, freeze_theta=True, keep_chi_moments=True)
    s.set_data(inp["cols"]); s.set_init(theta)
    mask = (np.arange(n) % 3 != 0).astype(np.uint8)           # every third object is held fixed
    s.set_update_mask(mask)
    st0 = s.get_state()
    s.run(burn, burn_in=burn)
    chain = np.empty((T, n))
    for t in range(T):
        s.step(burn_in=burn)
        chain[t] = s.get_state()["chi"][0]
    st1 = s.get_state()
    held = mask == 0
    assert np.array_equal(st1["chi"][:, held], st0["chi"][:, held]) and np.array_equal(st1["L"][:, held], st0["L"][:, held])
    assert np.all(st1["L"][0, ~held] != st0["L"][0, ~held])
    assert np.array_equal(s.get_counters(), np.where(held, 0, burn + T).astype(np.uint32))
    y, sig = inp["cols"]
    tau = np.exp(theta[1])
    v2 = 1 / (1 / sig ** 2 + 1 / tau ** 2)
    m = (y / sig ** 2 + theta[0] / tau ** 2) * v2
    mean, mse, var, vse = mean_and_var_with_mcse(chain[:, ~held])
    assert np.all(np.abs(mean - m[~held]) <= 5 * mse) and np.all(np.abs(var - v2[~held]) <= 5 * vse + 1e-4)
    z = np.concatenate([(mean - m[~held]) / mse, (var - v2[~held]) / vse])
    assert np.sqrt(np.mean(z ** 2)) < 1.5
    # the moments of a held object are those of a constant; proposals count the updated objects only
    mm, vv, k = s.get_chi_moments()
    assert k == T and np.allclose(mm[0, held], st0["chi"][0, held], rtol=0, atol=1e-12) and np.all(vv[0, held] < 1e-20)
    stt = s.get_stats()
    assert stt["chi_proposals"] == (burn + T) * int((~held).sum())
    assert stt["chi_accepts"] / stt["chi_proposals"] == pytest.approx(0.44, abs=0.01)


def test_held_objects_stay_in_the_population_sums():
    """S = sum_i log f(chi_i; theta) and Delta run over ALL objects; the taps of a held object are the documented ones."""
    n = 200
    s, inp = _sampler(n, 92)
    s.run(5)
    mask = (np.arange(n) % 2).astype(np.uint8)
    s.set_update_mask(mask)
    st = s.get_state()
    tp = s.step(taps=True)
    held = mask == 0
    a = np.array([O.logpop(0, st["chi"][:, i], np.array(inp["cols"])[:, i], st["theta"]) for i in range(n)])
    assert np.array_equal(tp["a"][held], a[held])
    assert tp["S"] == pytest.approx(O.osum(tp["a"]), rel=1e-14)
    assert tp["Delta"] == pytest.approx(O.osum(tp["b"] - tp["a"]), rel=1e-12, abs=1e-12)
    assert np.all(tp["alpha"][held] == 0) and np.all(tp["u"][held] == 1) and np.all(tp["accepted"][held] == 0)
    assert np.array_equal(tp["chi_prop"][0, held], st["chi"][0, held]) and np.array_equal(tp["L_new"][:, held], st["L"][:, held])
    assert np.array_equal(tp["pi_prop"][held], tp["pi_cur"][held])
    # the updated objects draw exactly what they draw without a mask (streams are keyed by object, not by position)
    s2, _ = _sampler(n, 92)
    s2.run(5)
    tp2 = s2.step(taps=True)
    assert np.array_equal(tp["u"][~held], tp2["u"][~held]) and np.array_equal(tp["chi_prop"][0, ~held], tp2["chi_prop"][0, ~held])


def test_all_ones_mask_and_counter_reproduce_the_plain_chain_bit_for_bit():
    n = 150
    a, _ = _sampler(n, 93)
    b, _ = _sampler(n, 93, per_object_counter=True)
    b.set_update_mask(np.ones(n, np.uint8))
    a.run(300, 50, 5); b.run(300, 50, 5)
    sa, sb = a.get_state(), b.get_state()
    for k in ("chi", "L", "theta", "L_theta"):
        assert np.array_equal(sa[k], sb[k]), k
    assert np.array_equal(a.get_theta_trace(), b.get_theta_trace())
    assert np.all(b.get_counters() == 300)


def test_per_object_counter_sets_eta_from_the_objects_own_update_count():
    """Objects released after K held iterations adapt with eta = (c_i + 2)^(-2/3), c_i their OWN count (P4 iii closed form:
    L_new = L sqrt(1 + eta_i (alpha - alpha*))); with the global counter they would use (t + 1)^(-2/3)."""
    n, K = 64, 400
    for per_obj in (True, False):
        s, _ = _sampler(n, 94, per_object_counter=per_obj)
        mask = (np.arange(n) >= n // 2).astype(np.uint8)
        s.set_update_mask(mask)
        s.run(K)
        s.set_update_mask(None)
        st = s.get_state()
        c0 = s.get_counters()
        assert np.array_equal(c0, np.where(mask == 1, K, 0).astype(np.uint32))
        tp = s.step(taps=True)
        eta = (c0 + 2.0) ** (-2.0 / 3.0) if per_obj else np.full(n, (K + 2.0) ** (-2.0 / 3.0))
        want = st["L"][0] * np.sqrt(1.0 + eta * (tp["alpha"] - 0.44))
        np.testing.assert_allclose(tp["L_new"][0], want, rtol=1e-14)
        assert np.array_equal(s.get_counters(), c0 + 1)
    # set_state(t) sets every counter to t; set_counters overrides
    s.set_state(st["chi"], st["L"], st["theta"], st["L_theta"], 7)
    assert np.all(s.get_counters() == 7)
    s.set_counters(np.arange(n))
    assert np.array_equal(s.get_counters(), np.arange(n))
