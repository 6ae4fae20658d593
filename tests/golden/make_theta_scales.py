"""Writes nothing the tests compare against: it PRINTS the constants stored in paper_2105_08026_b200/synth.py
(THETA_COND_CHOL), so that they can be regenerated.  For each model: the unit-N covariance C of theta given the latents at
the generating truth, from a central finite-difference Hessian of

    sum_i log f(chi_i; theta) + T(theta) + log prior(theta)          (the target of the theta step)

evaluated through the ORACLE's functions only (oracle_logpop, oracle_theta_only, oracle_logprior) on the synthetic latents,
then chol(C) packed row-major.  The closed forms it reproduces: M0 diag(tau^2, 1/2); M3 tau^2 (X^T X / N)^-1 and 1/2; M5 C_pop.

    python tests/golden/make_theta_scales.py [N]
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
from oracle import api as O  # noqa: E402
from paper_2105_08026_b200 import synth  # noqa: E402

MAKERS = {0: synth.make_normal1d, 1: synth.make_thinned_schechter1d, 2: synth.make_binormal2d,
          3: lambda n, s: synth.make_linreg_me1d(n, s, fp32=False), 4: synth.make_bb1_fluxnoise1d,
          5: synth.make_normal3d_knowncov}


def conditional_cov_unit_n(model, n, seed=7, h=2e-3):
    inp = MAKERS[model](n, seed)
    chi, cols, th0 = inp["chi_true"], np.array(inp["cols"]), np.array(inp["theta_true"], float)
    s = O.Sampler(model, n, seed=1)
    s.set_data(inp["cols"])
    if inp["consts"] is not None:
        s.set_model_consts(inp["consts"])
    s.set_init(th0)

    def F(th):
        v = sum(O.logpop(model, chi[:, i], cols[:, i], th, inp["consts"]) for i in range(n))
        return v + s.theta_only(th) + O.logprior(model, th)

    d = len(th0)
    H = np.zeros((d, d))
    f0 = F(th0)
    for a in range(d):
        for b in range(a, d):
            ea, eb = np.zeros(d), np.zeros(d)
            ea[a], eb[b] = h, h
            if a == b:
                H[a, a] = (F(th0 + ea) - 2 * f0 + F(th0 - ea)) / h ** 2
            else:
                H[a, b] = H[b, a] = (F(th0 + ea + eb) - F(th0 + ea - eb) - F(th0 - ea + eb) + F(th0 - ea - eb)) / (4 * h * h)
    return np.linalg.inv(-H) * n


if __name__ == "__main__":
    np.set_printoptions(precision=4, suppress=True, linewidth=150)
    n = int(sys.argv[1]) if len(sys.argv) > 1 else 20000
    for model in range(6):
        Cn = conditional_cov_unit_n(model, n)
        sd = np.sqrt(np.diag(Cn))
        print(f"model {model}: sd sqrt(N) = {sd}\n corr =\n{Cn / np.outer(sd, sd)}\n chol(C N) packed = "
              f"{np.linalg.cholesky(Cn)[np.tril_indices(len(sd))]}")
