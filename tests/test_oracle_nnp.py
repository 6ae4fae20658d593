"""Pins of the oracle's normal-normal model for p = 4, 5, 6 (RAM for general dimension, PAPER.md:129-140
Eq. 2.6; PAPER.md:146-166 is the p = 3 instance, pinned in test_oracle_nn3.py).  As there: the densities are scipy's,
chi_i | mu, y_i is the conjugate normal, mu | y ~ N(ybar, (C_pop + diag sigma^2)/N); and the p x p RAM update keeps its
defining identity."""
import numpy as np
import pytest
from scipy import stats

from mcmc_util import mean_and_var_with_mcse
from oracle import api as O
from paper_2105_08026_b200 import synth

PS = [4, 5, 6]


@pytest.mark.parametrize("p", PS)
def test_dims_constants_and_densities(p):
    model = synth.nnp_model(p)
    assert O.model_dims(model) == dict(p=p, dtheta=p, n_cols=p, n_consts=p + p * (p + 1) // 2)
    c, C = synth.nnp_consts(p), synth.nnp_cpop(p)
    assert np.all(np.linalg.eigvalsh(C) > 0)
    np.testing.assert_allclose(synth.NNP_R[:3, :3], synth.NN3_R)          # the paper's Eq. 3.4 is the leading block
    np.testing.assert_allclose(synth.nnp_cpop(3), synth.NN3_CPOP)
    g = np.random.default_rng(p)
    for _ in range(20):
        chi = synth.NNP_MU[:p] + np.linalg.cholesky(C) @ g.normal(size=p)
        mu = synth.NNP_MU[:p] + g.normal(size=p)
        y = chi + c[:p] * g.normal(size=p)
        want = stats.multivariate_normal.logpdf(chi, mu, C) + 0.5 * np.log(np.linalg.det(2 * np.pi * C))
        assert O.logpop(model, chi, y, mu, c) == pytest.approx(want, rel=1e-11, abs=1e-11)
        wl = (stats.norm.logpdf(y, chi, c[:p]) + np.log(c[:p]) + 0.5 * np.log(2 * np.pi)).sum()
        assert O.loglik(model, chi, y, c) == pytest.approx(wl, rel=1e-13, abs=1e-13)
    th = synth.NNP_MU[:p].copy()
    assert O.logprior(model, th) == 0.0
    th[p - 1] = 1001.0
    assert O.logprior(model, th) == -np.inf


@pytest.mark.parametrize("p", PS)
def test_plate_stationary_law_is_the_conjugate_normal(p):
    """theta frozen: chi_i | mu, y_i ~ N(V (C^-1 mu + S^-1 y_i), V), V = (C^-1 + S^-1)^-1: means, variances, all cross moments;
    acceptance homes in on alpha_* = 0.234; L L^T stays symmetric positive definite (the RAM invariant) along the chain."""
    n, burn, T = 8, 15000, 60000
    model = synth.nnp_model(p)
    inp = synth.make_normalpd_knowncov(n, seed=60 + p, p=p)
    mu = synth.NNP_MU[:p]
    s = O.Sampler(model, n, seed=60 + p, target_accept_chi=0.234, freeze_theta=True)
    s.set_data(inp["cols"]); s.set_model_consts(inp["consts"]); s.set_init(mu)
    s.run(burn)
    a0 = s.get_stats()["chi_accepts"]
    chain = np.empty((T, p, n))
    for t in range(T):
        s.step()
        chain[t] = s.get_state()["chi"]
    # eta_n = n^(-2/3) closes in on alpha_* more slowly the more directions there are to learn
    assert (s.get_stats()["chi_accepts"] - a0) / (T * n) == pytest.approx(0.234, abs=0.02)
    Ci, Si = np.linalg.inv(synth.nnp_cpop(p)), np.diag(1 / synth.NNP_SIGMA[:p] ** 2)
    V = np.linalg.inv(Ci + Si)
    y = np.array(inp["cols"])
    zs = []
    for i in range(n):
        m = V @ (Ci @ mu + Si @ y[:, i])
        x = chain[:, :, i]
        mean, mse, var, vse = mean_and_var_with_mcse(x)
        assert np.all(np.abs(mean - m) <= 5 * mse) and np.all(np.abs(var - np.diag(V)) <= 5 * vse), f"object {i}"
        zs += list((mean - m) / mse) + list((var - np.diag(V)) / vse)
        for a in range(p):
            for b in range(a):
                cr = (x[:, a] - m[a]) * (x[:, b] - m[b])
                cm, cse, _, _ = mean_and_var_with_mcse(cr)
                assert abs(cm[0] - V[a, b]) <= 5 * cse[0], f"object {i} cov({a},{b})"
                zs.append((cm[0] - V[a, b]) / cse[0])
    assert np.sqrt(np.mean(np.square(zs))) < 1.5
    L = s.get_state()["L"]
    for i in range(n):
        S_ = np.zeros((p, p)); S_[np.tril_indices(p)] = L[:, i]
        assert np.all(np.diag(S_) > 0) and np.all(np.linalg.eigvalsh(S_ @ S_.T) > 0)


@pytest.mark.parametrize("p", PS)
def test_theta_posterior_is_the_closed_form(p):
    """mu | y ~ N(ybar, (C_pop + diag sigma_j^2)/N) with the uniform hyperprior of PAPER.md:166."""
    n, burn, T = 30, 20000, 120000
    model = synth.nnp_model(p)
    inp = synth.make_normalpd_knowncov(n, seed=70 + p, p=p)
    s = O.Sampler(model, n, seed=70 + p, target_accept_chi=0.234)
    s.set_data(inp["cols"]); s.set_model_consts(inp["consts"]); s.set_init(inp["theta0"], theta_chol0=inp["theta_chol0"])
    s.run(burn + T, burn_in=burn)
    check_nnp_posterior(inp, s.get_theta_trace(), p)


def check_nnp_posterior(inp, tr, p):
    y = np.array(inp["cols"])
    n = y.shape[1]
    S = (synth.nnp_cpop(p) + np.diag(synth.NNP_SIGMA[:p] ** 2)) / n
    mean, mse, var, vse = mean_and_var_with_mcse(tr)
    sd = np.sqrt(np.diag(S))
    assert np.all(np.abs(mean - y.mean(1)) <= 4 * mse + 0.01 * sd), (mean, y.mean(1), mse)
    assert np.all(np.abs(var - np.diag(S)) <= 4 * vse + 0.03 * np.diag(S)), (var, np.diag(S), vse)
    for a, b in ((0, p - 1), (1, 2)):
        cr = (tr[:, a] - y[a].mean()) * (tr[:, b] - y[b].mean())
        cm, cse, _, _ = mean_and_var_with_mcse(cr)
        assert abs(cm[0] - S[a, b]) <= 4 * cse[0] + 0.03 * sd[a] * sd[b]


@pytest.mark.parametrize("p", PS)
def test_ram_update_identity_general_p(p):
    """P4 for p = 4 .. 6: L_n L_n^T = L (I + c u u^T) L^T, lower-triangular, positive diagonal, determinant lemma."""
    g = np.random.default_rng(10 + p)
    for _ in range(50):
        A = g.normal(size=(p, p))
        L = np.linalg.cholesky(A @ A.T + 0.1 * np.eye(p))
        z = g.normal(size=p)
        c = g.uniform(-0.76, 0.63)
        Ln = np.zeros((p, p)); Ln[np.tril_indices(p)] = O.ram_update(L[np.tril_indices(p)], z, c)
        u = z / np.linalg.norm(z)
        M = L @ (np.eye(p) + c * np.outer(u, u)) @ L.T
        np.testing.assert_allclose(Ln @ Ln.T, M, rtol=1e-12, atol=1e-13 * np.abs(M).max())
        assert np.all(np.diag(Ln) > 0)
        assert np.prod(np.diag(Ln)) ** 2 == pytest.approx(np.prod(np.diag(L)) ** 2 * (1 + c), rel=1e-12)
