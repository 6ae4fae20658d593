"""Seeded synthetic inputs for the five BASELINE.json configs (C0..C4) and the paper's BB1 case study (C5).

This module serves BOTH the CUDA path and the oracle and therefore holds none of the method's
arithmetic (no log-density, no RAM step, no Philox stream of the sampler): it only simulates
catalogs with the shape of the paper's workloads -- one latent per object, heteroscedastic Gaussian
member likelihoods, volume-uniform distances, flux-limited thinning -- with
BASELINE.json's parameter values.  The paper's own simulated catalogs are not available; these
stand in for them.  Random numbers: numpy's Philox bit generator, keyed by the
config's seed, so every call is reproducible on any machine.
"""
from dataclasses import dataclass

import numpy as np

M_NORMAL1D, M_THINNED_SCHECHTER1D, M_BINORMAL2D, M_LINREG_ME1D, M_BB1_FLUXNOISE1D, M_NORMAL3D_KNOWNCOV = 0, 1, 2, 3, 4, 5
M_NORMAL4D_KNOWNCOV, M_NORMAL5D_KNOWNCOV, M_NORMAL6D_KNOWNCOV = 6, 7, 8
F64, F32_STATE_F64_REDUCE = 0, 1


@dataclass(frozen=True)
class RunConfig:
    name: str
    model: int
    precision: int
    n_objects: int
    n_iter: int
    burn_in: int
    thin: int
    target_accept_chi: float
    target_accept_theta: float
    keep_chi_moments: bool
    seed: int


# BASELINE.json "configs" 0..4 (burn-in / thinning where BASELINE is silent: DESIGN.md section 7)
CONFIGS = {
    "C0": RunConfig("C0", M_NORMAL1D, F64, 1_000, 2_000, 500, 1, 0.44, 0.234, True, 0),
    "C1": RunConfig("C1", M_THINNED_SCHECHTER1D, F64, 100_000, 5_000, 1_000, 1, 0.44, 0.234, False, 1),
    "C2": RunConfig("C2", M_THINNED_SCHECHTER1D, F64, 300_000, 10_000, 2_000, 10, 0.44, 0.234, True, 2),
    "C3": RunConfig("C3", M_BINORMAL2D, F64, 1_000_000, 5_000, 1_000, 1, 0.234, 0.234, False, 3),
    "C4": RunConfig("C4", M_LINREG_ME1D, F32_STATE_F64_REDUCE, 10_000_000, 2_000, 500, 1, 0.44, 0.234, False, 4),
    # the paper's own case study (Table 5.1): BB1 population, N = 1e5
    "C5": RunConfig("C5", M_BB1_FLUXNOISE1D, F64, 100_000, 5_000, 1_000, 1, 0.44, 0.234, False, 5),
    # the normal-normal benchmark of PAPER.md:146-188 (3-vector latents, known C_pop) at the
    # largest population the paper ran (N = 3e4), p = 3 RAM with the general rank-one Cholesky update
    "C6": RunConfig("C6", M_NORMAL3D_KNOWNCOV, F64, 30_000, 5_000, 1_000, 1, 0.234, 0.234, False, 6),
}

# constants of the thinned point-process configs: {F_lim, sigma_F, x_lo, x_hi, r_min, r_max}
SCHECHTER_CONSTS = np.array([1e-3, 1e-4, np.log(1e-4), np.log(30.0), 1.0, 10.0 ** (1.0 / 3.0)])
SCHECHTER_TRUTH = (-1.2, 0.0)   # (alpha, x* = log L*)


# BB1 case study.  Units: luminosity in 1e10 L_sun (u_true = 1, l_true = 0.01), distance in
# Gpc (r_max = 1), flux in (1e10 L_sun)/Gpc^2, so F_fid = u/(4 pi r_max^2) = 1/(4 pi) (Eq. 5.2).
# nu = 5, alpha = 0.01.  The printed sigma_0 and F_th are inconsistent with "L = 20 u at r_max is
# just detectable" (reading R18); the text's statement is kept: F_th = 20 F_fid, and sigma_0 follows from
# F_th = nu sigma(F_th), i.e. sigma_0 = F_th sqrt(1 - nu^2 alpha^2)/nu (Eq. 5.9 with the nu^2 restored).
BB1_TRUTH = (-1.5, np.log(0.01), 0.0)          # (beta, ln l, ln u)           PAPER.md:262, Table 5.1
BB1_NU, BB1_ALPHA_NOISE = 5.0, 1e-2
BB1_FTH = 20.0 / (4.0 * np.pi)
BB1_SIGMA0 = BB1_FTH * np.sqrt(1.0 - (BB1_NU * BB1_ALPHA_NOISE) ** 2) / BB1_NU
# constants of the model: {sigma_0, alpha, x_lo, x_hi, r_min, r_max, F_th}
BB1_CONSTS = np.array([BB1_SIGMA0, BB1_ALPHA_NOISE, np.log(1e-5), np.log(30.0), 1e-4, 1.0, BB1_FTH])


# normal-normal benchmark (Eq. 3.3-3.4)
NN3_MU = np.array([1.2, -0.4, 3.4])
NN3_D = np.array([2.3, 0.45, 13.4])
NN3_R = np.array([[1.0, 0.3, -0.5], [0.3, 1.0, 0.54], [-0.5, 0.54, 1.0]])
NN3_SIGMA = np.array([1.2, 0.4, 0.24])
NN3_CPOP = NN3_D[:, None] * NN3_R * NN3_D[None, :]
# constants of the model: {sigma_1..3, packed lower triangle of C_pop}
NN3_CONSTS = np.concatenate([NN3_SIGMA, NN3_CPOP[np.tril_indices(3)]])


# Initial theta proposal factor handed to both samplers (SURVEY 8(c) S7 allows "diag(user scales)"; the library default
# 0.1 I is 100-1000 x the width of theta | chi at N >= 1e5 and eta_n = n^(-2/3) shrinks it too slowly).  The conditional
# law of theta given the latents narrows as N^(-1/2); its unit-N covariance C at the generating truth of each recipe
# below was computed once through the oracle (tests/golden/make_theta_scales.py: finite-difference Hessian of
# sum_i log f(chi_i; theta) + T(theta) + log prior) and is stored here as chol(C), packed lower-triangular row-major.
# theta_chol0 = (2.38 / sqrt(dtheta)) chol(C) / sqrt(N): the random-walk scaling at which a Gaussian target accepts
# about a quarter of the proposals, so the RAM adaptation of L_theta starts near its fixed point.
THETA_COND_CHOL = {
    M_NORMAL1D: [1.0, 0.0, 0.7071],
    M_THINNED_SCHECHTER1D: [1.481, -3.214, 2.542, 4.413, -1.182, 0.994],
    M_BINORMAL2D: [1.0, 0.182, 0.5786, 0.0, 0.0, 0.7139, 0.0, 0.0, 0.0648, 0.7075, 0.0, 0.0, 0.2177, 0.2020, 0.9663],
    M_LINREG_ME1D: [0.6, -0.3, 0.1732, 0.0, 0.0, 0.7071],
    M_BB1_FLUXNOISE1D: [2.038, -18.80, 17.98, -1.795, -0.185, 1.005],
    M_NORMAL3D_KNOWNCOV: [2.3, 0.135, 0.4293, -6.7, 9.6924, 6.3817],
}


def theta_chol0(model, n):
    d = {M_NORMAL1D: 2, M_THINNED_SCHECHTER1D: 3, M_BINORMAL2D: 5, M_LINREG_ME1D: 3, M_BB1_FLUXNOISE1D: 3,
         M_NORMAL3D_KNOWNCOV: 3}[model]
    return np.asarray(THETA_COND_CHOL[model], dtype=np.float64) * (2.38 / np.sqrt(d) / np.sqrt(max(int(n), 1)))


# the normal-normal model for p = 4, 5, 6 (RAM for general dimension): the paper's
# three components (Eq. 3.3-3.4) followed by up to three more; R is the leading p x p block of a fixed positive definite
# correlation matrix whose leading 3 x 3 block is the paper's Eq. 3.4
NNP_MU = np.array([1.2, -0.4, 3.4, 0.7, -2.1, 5.0])
NNP_D = np.array([2.3, 0.45, 13.4, 1.1, 0.8, 3.2])
NNP_SIGMA = np.array([1.2, 0.4, 0.24, 0.6, 0.3, 1.5])
NNP_R = np.array([[1.0, 0.3, -0.5, 0.2, -0.1, 0.15],
                  [0.3, 1.0, 0.54, -0.25, 0.2, 0.1],
                  [-0.5, 0.54, 1.0, -0.3, 0.1, -0.2],
                  [0.2, -0.25, -0.3, 1.0, 0.35, -0.15],
                  [-0.1, 0.2, 0.1, 0.35, 1.0, 0.25],
                  [0.15, 0.1, -0.2, -0.15, 0.25, 1.0]])


def nnp_model(p):
    return {3: M_NORMAL3D_KNOWNCOV, 4: M_NORMAL4D_KNOWNCOV, 5: M_NORMAL5D_KNOWNCOV, 6: M_NORMAL6D_KNOWNCOV}[int(p)]


def nnp_cpop(p):
    return NNP_D[:p, None] * NNP_R[:p, :p] * NNP_D[None, :p]


def nnp_consts(p):
    """{sigma_1 .. sigma_p, packed lower triangle of C_pop}"""
    return np.concatenate([NNP_SIGMA[:p], nnp_cpop(p)[np.tril_indices(p)]])


def _rng(seed):
    return np.random.Generator(np.random.Philox(key=int(seed)))


def _round_f32(cols):
    return [c.astype(np.float32).astype(np.float64) for c in cols]


def make_normal1d(n, seed=0, fp32=False):
    """C0: sigma_i ~ U(0.5,1.5); chi_i ~ N(0,1); y_i = chi_i + sigma_i eps."""
    g = _rng(seed)
    sigma = g.uniform(0.5, 1.5, n)
    chi = g.standard_normal(n)
    y = chi + sigma * g.standard_normal(n)
    cols = [y, sigma]
    if fp32:
        cols = _round_f32(cols)
    sd = float(np.std(cols[0])) if n > 1 else 1.0
    return dict(model=M_NORMAL1D, cols=cols, consts=None, chi_true=chi[None, :],
                theta_true=np.array([0.0, 0.0]),
                theta0=np.array([float(np.mean(cols[0])) if n else 0.0, np.log(max(sd, 1e-3))]),
                theta_chol0=theta_chol0(M_NORMAL1D, n))


def make_thinned_schechter1d(n, seed=1):
    """C1/C2: latent x = ln L from the density prop. to exp((alpha+1)x - e^x) on [x_lo, x_hi] (inverse CDF
    on a 200,001-point grid), V ~ U(1,10), r = V^(1/3), F = e^x/(4 pi r^2), Fhat = F + sigma_F eps, kept iff
    Fhat > F_lim.  Columns: Fhat_i and g_i = 1/(4 pi r_i^2)."""
    g = _rng(seed)
    F_lim, sig_F, x_lo, x_hi, r_min, r_max = SCHECHTER_CONSTS
    alpha, xstar = SCHECHTER_TRUTH
    grid = np.linspace(x_lo, x_hi, 200_001)
    dens = np.exp((alpha + 1.0) * (grid - xstar) - np.exp(grid - xstar))
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (dens[1:] + dens[:-1]) * np.diff(grid))])
    Z = cdf[-1]
    cdf /= Z
    xs, Fh, gs = [], [], []
    kept, drawn = 0, 0
    while kept < n:
        m = max(4096, int(1.2 * (n - kept) / 0.15))
        x = np.interp(g.uniform(size=m), cdf, grid)
        r = g.uniform(r_min ** 3, r_max ** 3, m) ** (1.0 / 3.0)
        gi = 1.0 / (4.0 * np.pi * r * r)
        Fhat = np.exp(x) * gi + sig_F * g.standard_normal(m)
        ok = np.flatnonzero(Fhat > F_lim)
        if kept + ok.size >= n:          # stop at exactly n detections; count the candidates used
            ok = ok[: n - kept]
            drawn += int(ok[-1]) + 1 if ok.size else 0
        else:
            drawn += m
        kept += ok.size
        xs.append(x[ok]); Fh.append(Fhat[ok]); gs.append(gi[ok])
    x, Fhat, gi = np.concatenate(xs), np.concatenate(Fh), np.concatenate(gs)
    a_true = float(np.log(max(drawn, 1) / Z))       # amplitude whose expected population count = candidates drawn
    return dict(model=M_THINNED_SCHECHTER1D, cols=[Fhat, gi], consts=SCHECHTER_CONSTS.copy(),
                chi_true=x[None, :], theta_true=np.array([alpha, xstar, a_true]),
                theta0=np.array([alpha + 0.05, xstar + 0.05, a_true + 0.05]),
                theta_chol0=theta_chol0(M_THINNED_SCHECHTER1D, n), detected_fraction=n / max(drawn, 1))


def make_bb1_fluxnoise1d(n, seed=5, truth=BB1_TRUTH):
    """C5, the paper's case study: L ~ BB1(beta, l, u) (Eq. 5.1), r uniform in volume on
    [r_min, r_max], F = L/(4 pi r^2), Fhat = F + sigma(F) eps with sigma(F)^2 = sigma_0^2 + (alpha F)^2 (Eq. 5.8), kept
    iff Fhat > F_th.  Only ~1e-3 of the population is detectable, so candidates are drawn where detection is
    possible at all: r <= R(x) = min(r_max, 3 r_det(x)), r_det = sqrt(L/(4 pi F_th)) (beyond 3 r_det the flux is below
    F_th/9, 40 sigma under the threshold), and x = ln L from the BB1 density times the probability of r <= R(x).
    That is the full process conditioned on an event every detection satisfies (up to Phi(-40))."""
    g = _rng(seed)
    sig0, a_n, x_lo, x_hi, r_min, r_max, F_th = BB1_CONSTS
    beta, ll, lu = truth
    grid = np.linspace(x_lo, x_hi, 400_001)
    Lum = np.exp(grid)
    dens = np.exp((beta + 1.0) * (grid - lu) - Lum / np.exp(lu)) * -np.expm1(-Lum / np.exp(ll))   # L f(L) / C
    R3 = np.minimum(r_max, 3.0 * np.sqrt(Lum / (4.0 * np.pi * F_th))) ** 3
    vfrac = np.clip((R3 - r_min ** 3) / (r_max ** 3 - r_min ** 3), 0.0, 1.0)
    w = dens * vfrac
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (w[1:] + w[:-1]) * np.diff(grid))])
    reach = cdf[-1] / np.trapezoid(dens, grid)          # share of the population drawn from at all
    cdf /= cdf[-1]
    xs, Fh, gs = [], [], []
    kept, drawn = 0, 0
    while kept < n:
        m = max(4096, int(1.2 * (n - kept) / 0.03))
        x = np.interp(g.uniform(size=m), cdf, grid)
        Rx = np.minimum(r_max, 3.0 * np.sqrt(np.exp(x) / (4.0 * np.pi * F_th)))
        r = (r_min ** 3 + g.uniform(size=m) * np.maximum(Rx ** 3 - r_min ** 3, 0.0)) ** (1.0 / 3.0)
        gi = 1.0 / (4.0 * np.pi * r * r)
        F = np.exp(x) * gi
        Fhat = F + np.sqrt(sig0 ** 2 + (a_n * F) ** 2) * g.standard_normal(m)
        ok = np.flatnonzero(Fhat > F_th)
        if kept + ok.size >= n:
            ok = ok[: n - kept]
            drawn += int(ok[-1]) + 1 if ok.size else 0
        else:
            drawn += m
        kept += ok.size
        xs.append(x[ok]); Fh.append(Fhat[ok]); gs.append(gi[ok])
    x, Fhat, gi = np.concatenate(xs), np.concatenate(Fh), np.concatenate(gs)
    th = np.array([beta, ll, lu])
    return dict(model=M_BB1_FLUXNOISE1D, cols=[Fhat, gi], consts=BB1_CONSTS.copy(), chi_true=x[None, :],
                theta_true=th, theta0=th + np.array([0.03, 0.1, 0.03]),
                theta_chol0=theta_chol0(M_BB1_FLUXNOISE1D, n), detected_fraction=reach * n / max(drawn, 1))


def make_normal3d_knowncov(n, seed=6):
    """C6, the normal-normal benchmark: chi_i ~ N3(mu, C_pop = D R D), y_ij = chi_ij + sigma_j eps."""
    g = _rng(seed)
    chi = NN3_MU[:, None] + np.linalg.cholesky(NN3_CPOP) @ g.standard_normal((3, n))
    y = chi + NN3_SIGMA[:, None] * g.standard_normal((3, n))
    return dict(model=M_NORMAL3D_KNOWNCOV, cols=[y[0].copy(), y[1].copy(), y[2].copy()], consts=NN3_CONSTS.copy(),
                chi_true=chi, theta_true=NN3_MU.copy(), theta0=NN3_MU + np.array([0.05, -0.02, 0.2]),
                theta_chol0=theta_chol0(M_NORMAL3D_KNOWNCOV, n))


def make_normalpd_knowncov(n, seed=7, p=4):
    """The normal-normal model with p-vector latents, p = 3 .. 6: chi_i ~ N_p(mu, C_pop), y_ij = chi_ij + sigma_j eps."""
    g = _rng(seed)
    C = nnp_cpop(p)
    chi = NNP_MU[:p, None] + np.linalg.cholesky(C) @ g.standard_normal((p, n))
    y = chi + NNP_SIGMA[:p, None] * g.standard_normal((p, n))
    # theta | chi ~ N(chibar, C_pop / N): the proposal factor of the recipe (see THETA_COND_CHOL)
    chol0 = np.linalg.cholesky(C)[np.tril_indices(p)] * (2.38 / np.sqrt(p) / np.sqrt(max(int(n), 1)))
    return dict(model=nnp_model(p), cols=[y[j].copy() for j in range(p)], consts=nnp_consts(p), chi_true=chi,
                theta_true=NNP_MU[:p].copy(), theta0=NNP_MU[:p] + 0.05 * NNP_D[:p] * np.array([1, -1, 1, -1, 1, -1])[:p],
                theta_chol0=chol0)


def make_binormal2d(n, seed=3, fp32=False):
    """C3: chi ~ N2(m, Sigma), m=(0,0.5), sds (1, e^-0.5), rho=0.3; per-axis sigma ~ U(0.05,0.3)."""
    g = _rng(seed)
    m = np.array([0.0, 0.5]); lam = np.array([0.0, -0.5]); rho = 0.3
    s = g.uniform(0.05, 0.3, (2, n))
    e = g.standard_normal((2, n))
    chi = np.empty((2, n))
    chi[0] = m[0] + np.exp(lam[0]) * e[0]
    chi[1] = m[1] + np.exp(lam[1]) * (rho * e[0] + np.sqrt(1 - rho * rho) * e[1])
    y = chi + s * g.standard_normal((2, n))
    cols = [y[0], y[1], s[0], s[1]]
    if fp32:
        cols = _round_f32(cols)
    th = np.array([m[0], m[1], lam[0], lam[1], np.arctanh(rho)])
    return dict(model=M_BINORMAL2D, cols=cols, consts=None, chi_true=chi, theta_true=th,
                theta0=th + np.array([0.05, -0.05, 0.05, 0.05, -0.05]), theta_chol0=theta_chol0(M_BINORMAL2D, n))


def make_linreg_me1d(n, seed=4, fp32=True):
    """C4: z ~ U(0,3); chi ~ N(1 - 0.5 z, 0.3^2); sigma = exp(ln 0.2 + 0.5 eps); y = chi + sigma eps'."""
    g = _rng(seed)
    z = g.uniform(0.0, 3.0, n)
    chi = 1.0 - 0.5 * z + 0.3 * g.standard_normal(n)
    sigma = np.exp(np.log(0.2) + 0.5 * g.standard_normal(n))
    y = chi + sigma * g.standard_normal(n)
    cols = [y, sigma, z]
    if fp32:
        cols = _round_f32(cols)
    th = np.array([1.0, -0.5, np.log(0.3)])
    return dict(model=M_LINREG_ME1D, cols=cols, consts=None, chi_true=chi[None, :], theta_true=th,
                theta0=th + np.array([0.02, -0.02, 0.05]), theta_chol0=theta_chol0(M_LINREG_ME1D, n))


def make_inputs(config_name, n_objects=None):
    """Inputs of config C0..C6; n_objects overrides N (reduced-size parity cases keep the recipe)."""
    c = CONFIGS[config_name]
    n = c.n_objects if n_objects is None else int(n_objects)
    if c.model == M_NORMAL1D:
        return make_normal1d(n, c.seed)
    if c.model == M_THINNED_SCHECHTER1D:
        return make_thinned_schechter1d(n, c.seed)
    if c.model == M_BINORMAL2D:
        return make_binormal2d(n, c.seed)
    if c.model == M_BB1_FLUXNOISE1D:
        return make_bb1_fluxnoise1d(n, c.seed)
    if c.model == M_NORMAL3D_KNOWNCOV:
        return make_normal3d_knowncov(n, c.seed)
    return make_linreg_me1d(n, c.seed, fp32=(c.precision == F32_STATE_F64_REDUCE))
