"""Pins of the oracle's normal-normal benchmark model (M5; Eq. 3.1-3.4): 3-vector
latents, known C_pop and sigma_j, theta = mu.  Everything about this model has a closed form: the densities are
scipy's, chi_i | mu, y_i is the conjugate normal, and mu | y ~ N(ybar, (C_pop + diag sigma^2)/N) under the uniform
hyperprior."""
import numpy as np
import pytest
from scipy import stats

from mcmc_util import mean_and_var_with_mcse
from oracle import api as O
from paper_2105_08026_b200 import synth

M5 = O.M_NORMAL3D_KNOWNCOV


def test_constants_are_the_papers():
    """Eq. 3.3-3.4 and the sigma_j of PAPER.md:164."""
    assert O.model_dims(5) == dict(p=3, dtheta=3, n_cols=3, n_consts=9)
    c = synth.NN3_CONSTS
    np.testing.assert_allclose(c[:3], [1.2, 0.4, 0.24])
    C = np.zeros((3, 3)); C[np.tril_indices(3)] = c[3:]; C = C + np.tril(C, -1).T
    D = np.diag([2.3, 0.45, 13.4]); R = np.array([[1, 0.3, -0.5], [0.3, 1, 0.54], [-0.5, 0.54, 1]])
    np.testing.assert_allclose(C, D @ R @ D, rtol=1e-15)
    assert np.all(np.linalg.eigvalsh(C) > 0)
    np.testing.assert_allclose(synth.NN3_MU, [1.2, -0.4, 3.4])


def test_densities_match_scipy():
    g = np.random.default_rng(0)
    c = synth.NN3_CONSTS
    C = synth.NN3_CPOP
    for _ in range(20):
        chi = synth.NN3_MU + np.linalg.cholesky(C) @ g.normal(size=3)
        mu = synth.NN3_MU + g.normal(size=3)
        y = chi + c[:3] * g.normal(size=3)
        want = stats.multivariate_normal.logpdf(chi, mu, C) + 0.5 * np.log(np.linalg.det(2 * np.pi * C))
        assert O.logpop(M5, chi, y, mu, c) == pytest.approx(want, rel=1e-12, abs=1e-12)
        wl = (stats.norm.logpdf(y, chi, c[:3]) + np.log(c[:3]) + 0.5 * np.log(2 * np.pi)).sum()
        assert O.loglik(M5, chi, y, c) == pytest.approx(wl, rel=1e-13, abs=1e-13)
    assert O.logprior(M5, [1.2, -0.4, 3.4]) == 0.0 and O.logprior(M5, [1.2, -1001.0, 3.4]) == -np.inf


def test_plate_stationary_law_is_the_conjugate_normal():
    """theta frozen: chi_i | mu, y_i ~ N(V (C^-1 mu + S^-1 y_i), V), V = (C^-1 + S^-1)^-1, S = diag sigma_j^2: the p = 3 RAM
    chain must land on it (means, variances and the cross moments), and accept at alpha_* = 0.234."""
    n, burn, T = 12, 5000, 60000
    inp = synth.make_normal3d_knowncov(n, seed=51)
    mu = synth.NN3_MU
    s = O.Sampler(M5, n, seed=51, target_accept_chi=0.234, freeze_theta=True)
    s.set_data(inp["cols"]); s.set_model_consts(inp["consts"]); s.set_init(mu)
    s.run(burn)
    a0 = s.get_stats()["chi_accepts"]
    chain = np.empty((T, 3, n))
    for t in range(T):
        s.step()
        chain[t] = s.get_state()["chi"]
    assert (s.get_stats()["chi_accepts"] - a0) / (T * n) == pytest.approx(0.234, abs=0.01)
    Ci, Si = np.linalg.inv(synth.NN3_CPOP), np.diag(1 / synth.NN3_SIGMA ** 2)
    V = np.linalg.inv(Ci + Si)
    y = np.array(inp["cols"])
    zs = []
    for i in range(n):
        m = V @ (Ci @ mu + Si @ y[:, i])
        x = chain[:, :, i]
        mean, mse, var, vse = mean_and_var_with_mcse(x)
        assert np.all(np.abs(mean - m) <= 5 * mse) and np.all(np.abs(var - np.diag(V)) <= 5 * vse), f"object {i}"
        zs += list((mean - m) / mse) + list((var - np.diag(V)) / vse)
        for a, b in ((0, 1), (0, 2), (1, 2)):
            cr = (x[:, a] - m[a]) * (x[:, b] - m[b])
            cm, cse, _, _ = mean_and_var_with_mcse(cr)
            assert abs(cm[0] - V[a, b]) <= 5 * cse[0], f"object {i} cov({a},{b})"
            zs.append((cm[0] - V[a, b]) / cse[0])
    assert np.sqrt(np.mean(np.square(zs))) < 1.5
    # the adapted proposal factor reproduces the SHAPE of the target: S S^T ~ k V with one k for all entries
    L = s.get_state()["L"]
    k = []
    for i in range(n):
        S_ = np.zeros((3, 3)); S_[np.tril_indices(3)] = L[:, i]
        k.append(np.diag(S_ @ S_.T) / np.diag(V))
    k = np.array(k)
    assert np.all(np.abs(k / k.mean(1, keepdims=True) - 1) < 0.5)


def check_nn3_posterior(inp, tr):
    """mu | y ~ N(ybar, (C_pop + diag sigma_j^2)/N) with the uniform hyperprior of PAPER.md:166."""
    y = np.array(inp["cols"])
    n = y.shape[1]
    S = (synth.NN3_CPOP + np.diag(synth.NN3_SIGMA ** 2)) / n
    mean, mse, var, vse = mean_and_var_with_mcse(tr)
    sd = np.sqrt(np.diag(S))
    assert np.all(np.abs(mean - y.mean(1)) <= 4 * mse + 0.01 * sd), (mean, y.mean(1), mse)
    assert np.all(np.abs(var - np.diag(S)) <= 4 * vse + 0.03 * np.diag(S)), (var, np.diag(S), vse)
    cr = (tr[:, 0] - y[0].mean()) * (tr[:, 2] - y[2].mean())
    cm, cse, _, _ = mean_and_var_with_mcse(cr)
    assert abs(cm[0] - S[0, 2]) <= 4 * cse[0] + 0.03 * sd[0] * sd[2]


def test_theta_posterior_is_the_closed_form():
    n, burn, T = 30, 20000, 150000
    inp = synth.make_normal3d_knowncov(n, seed=52)
    s = O.Sampler(M5, n, seed=52, target_accept_chi=0.234)
    s.set_data(inp["cols"]); s.set_model_consts(inp["consts"]); s.set_init(inp["theta0"])
    s.run(burn + T, burn_in=burn)
    check_nn3_posterior(inp, s.get_theta_trace())
