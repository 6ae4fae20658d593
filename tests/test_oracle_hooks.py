"""Pins of the advanced-use hooks: a user prior on theta that overrides the
default uniform one, and a flag that freezes the RAM adaptation after a given iteration."""
import numpy as np

from mcmc_util import mean_and_var_with_mcse
from oracle import api as O
from paper_2105_08026_b200 import synth


def test_user_prior_shifts_the_posterior_as_the_exact_grid_says():
    """M0 with chi integrated out, y_i ~ N(mu, s_i^2 + tau^2): exact 2-D grid over (mu, log tau) with an informative
    normal prior on mu and on log tau multiplying the default uniform one."""
    n, burn, T = 60, 4000, 60000
    inp = synth.make_normal1d(n, seed=61)
    pm, psd = [0.8, -0.3], [0.15, 0.2]
    s = O.Sampler(0, n, seed=61, target_accept_chi=0.44, prior_mean=pm, prior_sd=psd)
    s.set_data(inp["cols"]); s.set_init(inp["theta0"])
    s.run(burn + T, burn_in=burn)
    tr = s.get_theta_trace()
    y, sig = inp["cols"]
    mu = np.linspace(-0.4, 1.4, 451); lam = np.linspace(-1.2, 0.6, 451)
    V = sig[None, None, :] ** 2 + np.exp(2 * lam)[None, :, None]
    lp = (-0.5 * np.log(V) - 0.5 * (y[None, None, :] - mu[:, None, None]) ** 2 / V).sum(-1)
    flat = lp.copy()
    lp += -0.5 * ((mu[:, None] - pm[0]) / psd[0]) ** 2 - 0.5 * ((lam[None, :] - pm[1]) / psd[1]) ** 2

    def moments(l):
        w = np.exp(l - l.max()); w /= w.sum()
        m0, m1 = (w.sum(1) * mu).sum(), (w.sum(0) * lam).sum()
        return np.array([m0, m1]), np.array([(w.sum(1) * (mu - m0) ** 2).sum(), (w.sum(0) * (lam - m1) ** 2).sum()])

    gm, gv = moments(lp)
    fm, _ = moments(flat)
    assert abs(gm[0] - fm[0]) > 0.1                                  # the prior really matters in this set-up
    mean, mse, var, vse = mean_and_var_with_mcse(tr)
    assert np.all(np.abs(mean - gm) <= 4 * mse + 1e-3), (mean, gm, mse)
    assert np.all(np.abs(var - gv) <= 4 * vse + 0.02 * gv), (var, gv, vse)
    # an infinite prior sd is no factor at all: identical chain to the default
    a = O.Sampler(0, n, seed=61, target_accept_chi=0.44, prior_mean=[3.0, 3.0], prior_sd=[np.inf, np.inf])
    b = O.Sampler(0, n, seed=61, target_accept_chi=0.44)
    for q in (a, b):
        q.set_data(inp["cols"]); q.set_init(inp["theta0"]); q.run(200, burn_in=0)
    assert np.array_equal(a.get_theta_trace(), b.get_theta_trace())


def test_adaptation_freeze():
    """adapt_until = K: identical to the default up to iteration K, proposal factors constant afterwards (eta_n = 0 in
    Eq. 2.6 gives S_n S_n^T = S S^T), and the frozen chain still samples the conjugate conditional."""
    n, K = 40, 1500
    inp = synth.make_normal1d(n, seed=62)
    th = np.array([0.1, np.log(0.8)])
    a = O.Sampler(0, n, seed=62, target_accept_chi=0.44, freeze_theta=True, adapt_until=K)
    b = O.Sampler(0, n, seed=62, target_accept_chi=0.44, freeze_theta=True)
    for q in (a, b):
        q.set_data(inp["cols"]); q.set_init(th); q.run(K)
    sa, sb = a.get_state(), b.get_state()
    assert np.array_equal(sa["chi"], sb["chi"]) and np.array_equal(sa["L"], sb["L"])
    L_K = sa["L"].copy()
    T = 30000
    chain = np.empty((T, n))
    for t in range(T):
        a.step()
        chain[t] = a.get_state()["chi"][0]
    np.testing.assert_allclose(a.get_state()["L"], L_K, rtol=1e-12)      # frozen (chol(L L^T) = L up to rounding)
    b.run(50)
    assert not np.allclose(b.get_state()["L"], L_K, rtol=1e-6)            # the default keeps adapting
    y, sg = inp["cols"]
    tau2 = np.exp(2 * th[1])
    v = 1.0 / (1.0 / sg ** 2 + 1.0 / tau2)
    m = (y / sg ** 2 + th[0] / tau2) * v
    mean, mse, var, vse = mean_and_var_with_mcse(chain)
    assert np.all(np.abs(mean - m) <= 5 * mse) and np.all(np.abs(var - v) <= 5 * vse)
    # theta factor: frozen as well
    c = O.Sampler(0, n, seed=62, target_accept_chi=0.44, adapt_until=100)
    c.set_data(inp["cols"]); c.set_init(inp["theta0"]); c.run(100)
    Lth = c.get_state()["L_theta"].copy()
    c.run(100)
    np.testing.assert_allclose(c.get_state()["L_theta"], Lth, rtol=1e-12)
