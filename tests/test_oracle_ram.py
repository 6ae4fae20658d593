"""Pins P4/P5 of the oracle's RAM step (Eq. 2.6): the factor against numpy's Cholesky
of the right-hand side, the p=1 closed form, the determinant lemma, the SPD invariant along real
chains, and the long-run behaviour against the closed-form acceptance rate of 1-D random-walk Metropolis."""
import numpy as np
import pytest
from scipy import integrate, stats

from oracle import api as O
from paper_2105_08026_b200 import synth


def _unpack(Lp, p):
    L = np.zeros((p, p))
    k = 0
    for r in range(p):
        for c in range(r + 1):
            L[r, c] = Lp[k]
            k += 1
    return L


def _pack(L):
    p = L.shape[0]
    return np.array([L[r, c] for r in range(p) for c in range(r + 1)])


@pytest.mark.parametrize("p", [1, 2, 3, 5])
def test_ram_update_is_the_left_cholesky_factor_of_eq_2_6(p):
    g = np.random.default_rng(p)
    for trial in range(50):
        A = g.normal(size=(p, p))
        L = np.linalg.cholesky(A @ A.T + 0.1 * np.eye(p))
        z = g.normal(size=p)
        eta, alpha, astar = g.uniform(0.01, 0.7), g.uniform(0, 1), g.choice([0.234, 0.4, 0.44])
        c = eta * (alpha - astar)
        out = _unpack(O.ram_update(_pack(L), z, c), p)
        u = z / np.linalg.norm(z)
        rhs = L @ (np.eye(p) + c * np.outer(u, u)) @ L.T                     # Eq. 2.6 right-hand side
        np.testing.assert_allclose(out @ out.T, rhs, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(out, np.linalg.cholesky(rhs), rtol=1e-11, atol=1e-13)   # library routine
        assert np.all(np.diag(out) > 0) and np.allclose(out, np.tril(out))
        # matrix determinant lemma: det(I + c u u^T) = 1 + c
        assert np.prod(np.diag(out)) ** 2 == pytest.approx(np.prod(np.diag(L)) ** 2 * (1 + c), rel=1e-12)


def test_ram_update_p1_closed_form_and_sign():
    for L, z, c in ((1.0, 0.3, 0.2), (0.37, -2.0, -0.3), (5.0, 1e-8, 0.0)):
        assert O.ram_update([L], [z], c)[0] == pytest.approx(L * np.sqrt(1 + c), rel=1e-15)
    # alpha > alpha_* widens the proposal, alpha < alpha_* narrows it (adaptation toward the target rate)
    assert O.ram_update([1.0], [1.0], 0.5 * (1.0 - 0.44))[0] > 1.0 > O.ram_update([1.0], [1.0], 0.5 * (0.0 - 0.44))[0]


def test_rwm_acceptance_closed_form():
    """Random-walk Metropolis on N(0, v^2) with proposal sd s v accepts at rate (2/pi) atan(2/s); numerically."""
    for s in (1.0, 2.41758, 4.0):
        f = lambda d, x: stats.norm.pdf(x) * stats.norm.pdf(d, 0, s) * min(1.0, np.exp(0.5 * x * x - 0.5 * (x + d) ** 2))
        val = integrate.dblquad(f, -8, 8, -8 * s, 8 * s, epsabs=1e-7)[0]
        assert val == pytest.approx(2 / np.pi * np.arctan(2 / s), abs=2e-5)
    assert 2 / np.pi * np.arctan(2 / 2.41758) == pytest.approx(0.44, abs=1e-5)


def _conjugate_1d(inp, theta):
    y, sigma = inp["cols"][0], inp["cols"][1]
    mu, tau = theta[0], np.exp(theta[1])
    v2 = 1.0 / (1.0 / sigma ** 2 + 1.0 / tau ** 2)
    return (y / sigma ** 2 + mu / tau ** 2) * v2, v2


def test_ram_long_run_scale_and_acceptance_1d():
    """theta frozen, model M0: the target of object i is N(m_i, v_i^2), so RAM with alpha_* = 0.44 must drive
    S_i / v_i to 2/tan(0.44 pi/2) = 2.4176 and the mean acceptance to 0.44 (DESIGN.md pin P5)."""
    n, T = 400, 6000
    inp = synth.make_normal1d(n, seed=21)
    theta = np.array([0.1, -0.2])
    s = O.Sampler(0, n, seed=21, target_accept_chi=0.44, freeze_theta=True)
    s.set_data(inp["cols"]); s.set_init(theta)
    s.run(T // 2)
    acc0 = s.get_stats()["chi_accepts"]
    s.run(T - T // 2)
    st = s.get_state()
    _, v2 = _conjugate_1d(inp, theta)
    ratio = st["L"][0] / np.sqrt(v2)
    assert np.all(st["L"][0] > 0)
    assert ratio.mean() == pytest.approx(2.41758, abs=0.03)       # sd across chains ~0.05 at this T
    assert 0.02 < ratio.std() < 0.12
    rate = (s.get_stats()["chi_accepts"] - acc0) / (n * (T - T // 2))
    assert rate == pytest.approx(0.44, abs=0.004)
    assert np.array_equal(st["theta"], theta) and s.get_stats()["theta_proposals"] == 0


def test_ram_target_rate_is_respected_for_other_targets():
    n, T = 300, 5000
    inp = synth.make_normal1d(n, seed=22)
    s = O.Sampler(0, n, seed=22, target_accept_chi=0.3, freeze_theta=True)
    s.set_data(inp["cols"]); s.set_init([0.0, 0.0])
    s.run(T // 2); acc0 = s.get_stats()["chi_accepts"]; s.run(T - T // 2)
    assert (s.get_stats()["chi_accepts"] - acc0) / (n * (T - T // 2)) == pytest.approx(0.3, abs=0.005)


def test_first_update_uses_n_equals_2():
    """X_1, S_1 are the initial values, so the first RAM update is n = 2 (eta = 2^(-2/3)); S_1 = I."""
    inp = synth.make_normal1d(16, seed=23)
    s = O.Sampler(0, 16, seed=23, target_accept_chi=0.44, freeze_theta=True)
    s.set_data(inp["cols"]); s.set_init([0.0, 0.0])
    assert np.all(s.get_state()["L"] == 1.0)
    tp = s.step(taps=True)
    want = np.sqrt(1.0 + 2.0 ** (-2.0 / 3.0) * (tp["alpha"] - 0.44))
    np.testing.assert_allclose(tp["L_new"][0], want, rtol=1e-14)
    tp2 = s.step(taps=True)
    np.testing.assert_allclose(tp2["L_new"][0], want * np.sqrt(1.0 + 3.0 ** (-2.0 / 3.0) * (tp2["alpha"] - 0.44)), rtol=1e-14)


def test_spd_invariant_along_a_2d_chain():
    """L_i L_i^T stays symmetric positive definite (north_star's RAM invariant): packed factors keep a positive
    diagonal, and det grows by exactly (1 + c) each step."""
    n = 64
    inp = synth.make_binormal2d(n, seed=24)
    s = O.Sampler(2, n, seed=24, target_accept_chi=0.234)
    s.set_data(inp["cols"]); s.set_init(inp["theta0"])
    prev = s.get_state()["L"]
    for t in range(1, 400):
        tp = s.step(taps=True)
        L = s.get_state()["L"]
        assert np.all(L[0] > 0) and np.all(L[2] > 0) and np.all(np.isfinite(L))
        c = (t + 1.0) ** (-2.0 / 3.0) * (tp["alpha"] - 0.234)
        np.testing.assert_allclose((L[0] * L[2]) ** 2, (prev[0] * prev[2]) ** 2 * (1 + c), rtol=1e-11)
        prev = L
    Lth = s.get_state()["L_theta"]
    assert np.all(_unpack(Lth, 5).diagonal() > 0)


def test_accept_rule_and_alpha_definition():
    """alpha_n = min{1, pi(Y)/pi(X)} is the acceptance PROBABILITY, the move is taken iff u < alpha,
    and the proposal is Y = X + S U."""
    n = 200
    inp = synth.make_normal1d(n, seed=25)
    s = O.Sampler(0, n, seed=25, target_accept_chi=0.44, freeze_theta=True)
    s.set_data(inp["cols"]); s.set_init([0.0, 0.0])
    s.run(20)
    before = s.get_state()
    tp = s.step(taps=True)
    after = s.get_state()
    np.testing.assert_allclose(tp["alpha"], np.minimum(1.0, np.exp(tp["pi_prop"] - tp["pi_cur"])), rtol=1e-14)
    assert np.array_equal(tp["accepted"], (tp["u"] < tp["alpha"]).astype(np.int32))
    assert 0 < tp["accepted"].sum() < n
    draws = [O.plate_draws_f64(25, i, 21, 1) for i in range(n)]      # pinned in test_oracle_rng.py
    z = np.array([d[0][0] for d in draws])
    np.testing.assert_allclose(tp["chi_prop"][0], before["chi"][0] + before["L"][0] * z, rtol=1e-15)
    assert np.array_equal(tp["u"], np.array([d[1] for d in draws]))
    np.testing.assert_array_equal(after["chi"][0], np.where(tp["accepted"] == 1, tp["chi_prop"][0], before["chi"][0]))
    # pi is l_i * f: check against the separately pinned log-densities
    i = 7
    d = [inp["cols"][0][i], inp["cols"][1][i]]
    assert tp["pi_cur"][i] == O.loglik(0, [before["chi"][0, i]], d) + O.logpop(0, [before["chi"][0, i]], d, [0.0, 0.0])
    assert tp["a"][i] == O.logpop(0, [after["chi"][0, i]], d, [0.0, 0.0])
