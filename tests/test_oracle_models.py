"""Pins P3 (log-densities), the Gauss-Legendre rule and the selection integral of the oracle against
library routines (scipy.stats / scipy.integrate / numpy.polynomial) and normalisation closed forms."""
import numpy as np
import pytest
from scipy import integrate, special, stats

from oracle import api as O
from paper_2105_08026_b200 import synth

LOG2PI = np.log(2 * np.pi)


def test_model_dims():
    assert O.model_dims(0) == dict(p=1, dtheta=2, n_cols=2, n_consts=0)
    assert O.model_dims(1) == dict(p=1, dtheta=3, n_cols=2, n_consts=6)
    assert O.model_dims(2) == dict(p=2, dtheta=5, n_cols=4, n_consts=0)
    assert O.model_dims(3) == dict(p=1, dtheta=3, n_cols=3, n_consts=0)


def test_gaussian_loglik_matches_scipy():
    g = np.random.default_rng(0)
    for _ in range(20):
        chi, y, s, z = g.normal(), g.normal(), g.uniform(0.1, 2), g.uniform(0, 3)
        want = stats.norm.logpdf(y, chi, s) + np.log(s) + 0.5 * LOG2PI          # constants in chi dropped
        assert O.loglik(0, [chi], [y, s]) == pytest.approx(want, rel=1e-13, abs=1e-14)
        assert O.loglik(3, [chi], [y, s, z]) == pytest.approx(want, rel=1e-13, abs=1e-14)
        c2, y2, s2 = g.normal(size=2), g.normal(size=2), g.uniform(0.05, 0.3, 2)
        want2 = (stats.norm.logpdf(y2, c2, s2) + np.log(s2) + 0.5 * LOG2PI).sum()
        assert O.loglik(2, c2, [y2[0], y2[1], s2[0], s2[1]]) == pytest.approx(want2, rel=1e-13)


def test_normal_population_matches_scipy_and_integrates_to_one():
    g = np.random.default_rng(1)
    for _ in range(10):
        mu, lam, chi, a, b, z = g.normal(), g.normal(0, 0.5), g.normal(), g.normal(), g.normal(), g.uniform(0, 3)
        tau = np.exp(lam)
        assert O.logpop(0, [chi], [0, 1], [mu, lam]) == pytest.approx(
            stats.norm.logpdf(chi, mu, tau) + 0.5 * LOG2PI, rel=1e-13, abs=1e-14)
        assert O.logpop(3, [chi], [0, 1, z], [a, b, lam]) == pytest.approx(
            stats.norm.logpdf(chi, a + b * z, tau) + 0.5 * LOG2PI, rel=1e-13, abs=1e-14)
    val, _ = integrate.quad(lambda x: np.exp(O.logpop(0, [x], [0, 1], [0.3, -0.4])), -10, 10, epsabs=1e-13)
    assert val == pytest.approx(np.sqrt(2 * np.pi), rel=1e-10)        # restores the dropped (2 pi)^-1/2
    val, _ = integrate.quad(lambda x: np.exp(O.logpop(3, [x], [0, 1, 2.0], [1.0, -0.5, np.log(0.3)])), -5, 5,
                            epsabs=1e-13, points=[0.0])
    assert val == pytest.approx(np.sqrt(2 * np.pi), rel=1e-10)


def test_binormal_population_matches_scipy():
    g = np.random.default_rng(2)
    for _ in range(20):
        m = g.normal(size=2); lam = g.normal(0, 0.5, 2); zeta = g.normal(0, 0.7); chi = g.normal(size=2)
        s = np.exp(lam); rho = np.tanh(zeta)
        cov = np.array([[s[0] ** 2, rho * s[0] * s[1]], [rho * s[0] * s[1], s[1] ** 2]])
        want = stats.multivariate_normal.logpdf(chi, m, cov) + LOG2PI
        got = O.logpop(2, chi, [0, 0, 1, 1], [m[0], m[1], lam[0], lam[1], zeta])
        assert got == pytest.approx(want, rel=1e-12, abs=1e-13)


def test_schechter_population_is_a_gamma_law_in_luminosity():
    """exp(f - a) dx = (L/L*)^(alpha+1) e^(-L/L*) dL/L: for alpha > -1 that is Gamma(alpha+1) times the gamma
    pdf of L with shape alpha+1 and scale L* (the paper: "essentially a gamma distribution")."""
    c = synth.SCHECHTER_CONSTS
    for alpha, xs, a in ((-0.5, 0.0, 1.0), (-0.2, 0.7, -2.0), (-0.9, -0.3, 5.0)):
        for x in (-3.0, -1.0, 0.1, 1.5, 3.0):
            Lum, Ls = np.exp(x), np.exp(xs)
            want = a + stats.gamma.logpdf(Lum, alpha + 1, scale=Ls) + np.log(Lum) + special.gammaln(alpha + 1)
            assert O.logpop(1, [x], [1e-3, 0.05], [alpha, xs, a], c) == pytest.approx(want, rel=1e-12, abs=1e-13)
    # steep slopes (alpha < -1, the configs' truth) are fine too: same formula, no gamma normaliser
    assert O.logpop(1, [0.4], [0, 0], [-1.2, 0.1, 2.0], c) == pytest.approx(2.0 - 0.2 * 0.3 - np.exp(0.3), rel=1e-14)
    # support: -inf outside [x_lo, x_hi]
    assert O.logpop(1, [c[2] - 1e-9], [0, 0], [-1.2, 0.0, 0.0], c) == -np.inf
    assert O.logpop(1, [c[3] + 1e-9], [0, 0], [-1.2, 0.0, 0.0], c) == -np.inf
    assert np.isfinite(O.logpop(1, [c[2]], [0, 0], [-1.2, 0.0, 0.0], c))


def test_schechter_flux_likelihood():
    c = synth.SCHECHTER_CONSTS
    for x, Fhat, r in ((0.0, 0.0301, 1.6), (-1.0, 0.0112, 1.2), (1.0, 0.05, 2.1)):
        g = 1 / (4 * np.pi * r * r)
        want = stats.norm.logpdf(Fhat, np.exp(x) * g, c[1]) + np.log(c[1]) + 0.5 * LOG2PI
        assert O.loglik(1, [x], [Fhat, g], c) == pytest.approx(want, rel=1e-11)


def test_logprior():
    assert O.logprior(0, [0.3, -1.0]) == 0.0
    assert O.logprior(0, [1001.0, 0.0]) == -np.inf and O.logprior(0, [0.0, -10.5]) == -np.inf
    assert O.logprior(3, [1.0, -0.5, -1.2]) == 0.0 and O.logprior(3, [1.0, -0.5, 11.0]) == -np.inf
    assert O.logprior(2, [0, 0.5, 0, -0.5, 0.3]) == 0.0 and O.logprior(2, [0, 0.5, 0, -0.5, 10.1]) == -np.inf
    # PAPER.md:284 Eq. 5.4: p(beta) = 0.903/(1+beta^2) on (-2, 0); the constant is dropped
    for al in (-1.9, -1.2, -0.1):
        assert O.logprior(1, [al, 0.0, 3.0]) == pytest.approx(stats.cauchy.logpdf(al) + np.log(np.pi), rel=1e-13)
    assert O.logprior(1, [0.0, 0.0, 3.0]) == -np.inf and O.logprior(1, [-2.0, 0.0, 3.0]) == -np.inf
    assert O.logprior(1, [-1.0, 21.0, 3.0]) == -np.inf and O.logprior(1, [-1.0, 0.0, 51.0]) == -np.inf
    assert O.logprior(0, [np.nan, 0.0]) == -np.inf
    # the prior constant of Eq. 5.4: 1/(phi_U - phi_L) = 1/atan(2) = 0.903
    assert 1 / np.arctan(2.0) == pytest.approx(0.903, abs=5e-4)


def test_f32_log_densities_track_f64():
    g = np.random.default_rng(3)
    for _ in range(50):
        chi, y, s, z = g.normal(), g.normal(), g.uniform(0.1, 1.0), g.uniform(0, 3)
        th = [1.0 + 0.1 * g.normal(), -0.5, np.log(0.3)]
        f32 = [float(np.float32(v)) for v in (chi, y, s, z)]
        a64 = O.loglik(3, [f32[0]], f32[1:]) + O.logpop(3, [f32[0]], f32[1:], [float(np.float32(t)) for t in th])
        a32 = O.loglik_f32(3, [chi], [y, s, z]) + O.logpop_f32(3, [chi], [y, s, z], th)
        assert a32 == pytest.approx(a64, rel=2e-6, abs=2e-6)


def test_gauss_legendre_matches_numpy():
    for n, a, b in ((5, -1.0, 1.0), (256, 1.0, 10 ** (1 / 3)), (1024, np.log(1e-4), np.log(30.0))):
        x, w = O.gauss_legendre(n, a, b)
        xr, wr = np.polynomial.legendre.leggauss(n)
        np.testing.assert_allclose(x, 0.5 * (b - a) * xr + 0.5 * (b + a), rtol=0, atol=2e-14 * max(1, abs(a), abs(b)))
        # numpy's end weights are only good to ~1e-9 relative at n=1024 (checked against mpmath); see the mpmath pin below
        np.testing.assert_allclose(w, 0.5 * (b - a) * wr, rtol=5e-9, atol=1e-17)
        assert np.all(np.diff(x) > 0) and w.sum() == pytest.approx(b - a, rel=1e-14)
    x, w = O.gauss_legendre(8, 0.0, 2.0)
    assert (w * x ** 15).sum() == pytest.approx(2.0 ** 16 / 16, rel=1e-13)      # exact to degree 2n-1
    # 40-digit roots/weights of P_64 from mpmath
    import mpmath as mp
    mp.mp.dps = 40
    x, w = O.gauss_legendre(64, -1.0, 1.0)
    for i in (0, 1, 20, 40, 63):
        xi = mp.findroot(lambda t: mp.legendre(64, t), mp.mpf(x[i]))
        dp = 64 * (xi * mp.legendre(64, xi) - mp.legendre(63, xi)) / (xi * xi - 1)
        assert abs(x[i] - float(xi)) < 2e-16 and w[i] == pytest.approx(float(2 / ((1 - xi * xi) * dp * dp)), rel=1e-14)


def _schechter_sampler(n=64):
    inp = synth.make_thinned_schechter1d(n, seed=5)
    s = O.Sampler(1, n, seed=5)
    s.set_data(inp["cols"]); s.set_model_consts(inp["consts"]); s.set_init(inp["theta0"])
    return s, inp


def test_selection_integral_against_adaptive_quadrature():
    """T(theta) = -A int dx phi(x) int dr h(r) Phi((F - F_lim)/sigma_F)  (Eq. 4.4 denominator, with
    eta of Eq. 5.10) -- the fixed 1,024 x 256 rule against scipy's adaptive integrators."""
    s, inp = _schechter_sampler()
    F_lim, sig, x_lo, x_hi, r_min, r_max = inp["consts"]
    vol = r_max ** 3 - r_min ** 3

    def G(x):
        f = lambda r: 3 * r * r / vol * stats.norm.cdf((np.exp(x) / (4 * np.pi * r * r) - F_lim) / sig)
        # the integrand has a step of width ~ sigma_F at the detection edge: tell quad where it is
        r_edge = np.sqrt(np.exp(x) / (4 * np.pi * F_lim))
        pts = [r_edge] if r_min < r_edge < r_max else None
        return integrate.quad(f, r_min, r_max, points=pts, epsabs=1e-14, epsrel=1e-12, limit=400)[0]

    xk, Wk = s.get_selection_table()
    xr, _ = np.polynomial.legendre.leggauss(1024)
    np.testing.assert_allclose(xk, 0.5 * (x_hi - x_lo) * xr + 0.5 * (x_hi + x_lo), atol=1e-13)
    _, wx = O.gauss_legendre(1024, x_lo, x_hi)
    for k in (0, 300, 520, 640, 700, 800, 1023):
        # outer weights: the oracle's rule, itself pinned to mpmath above (numpy's end weights are off by 1e-9)
        assert Wk[k] == pytest.approx(wx[k] * G(xk[k]), rel=1e-10, abs=1e-18)

    for th in ([-1.2, 0.0, 3.0], [-0.7, 0.4, 1.0], [-1.6, -0.5, 6.0]):
        phiG = lambda x: np.exp((th[0] + 1) * (x - th[1]) - np.exp(x - th[1])) * G(x)
        # G rises from 0 to 1 between ln(4 pi r_min^2 F_lim) and ln(4 pi r_max^2 F_lim)
        e1, e2 = np.log(4 * np.pi * r_min ** 2 * F_lim), np.log(4 * np.pi * r_max ** 2 * F_lim)
        I = integrate.quad(phiG, x_lo, x_hi, points=[e1 - 0.2, e1, e2, e2 + 0.2], epsabs=1e-13, epsrel=1e-10,
                           limit=400)[0]
        assert s.theta_only(th) == pytest.approx(-np.exp(th[2]) * I, rel=2e-9)


def test_theta_only_is_zero_for_models_without_selection():
    inp = synth.make_normal1d(8, 0)
    s = O.Sampler(0, 8)
    s.set_data(inp["cols"]); s.set_init(inp["theta0"])
    assert s.theta_only([0.1, 0.2]) == 0.0


def test_expected_detected_count_matches_the_simulation():
    """At the simulation truth A I(alpha, x*) is the expected number of detections: the generator's
    thinning fraction must reproduce it -- an end-to-end check that eta, h(r) and F = L/(4 pi r^2) are wired
    the same way in the simulator (numpy) and in the oracle's quadrature (C++)."""
    n = 40_000
    inp = synth.make_thinned_schechter1d(n, seed=11)
    s = O.Sampler(1, n, seed=0)
    s.set_data(inp["cols"]); s.set_model_consts(inp["consts"]); s.set_init(inp["theta0"])
    expected = -s.theta_only(inp["theta_true"])
    assert abs(expected - n) < 4.5 * np.sqrt(n / inp["detected_fraction"] * inp["detected_fraction"] * (1 - inp["detected_fraction"])) + 0.002 * n


def test_oracle_sum_is_correctly_rounded_enough():
    import math
    g = np.random.default_rng(4)
    v = g.normal(size=200_000) * 10.0 ** g.uniform(-6, 6, 200_000)
    assert O.osum(v) == pytest.approx(math.fsum(v), rel=1e-15, abs=1e-9 * 0)
    v = np.array([1e16, 1.0, -1e16, 1.0])
    assert O.osum(v) == 2.0
