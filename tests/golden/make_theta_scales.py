"""Conditional covariance of theta given the latents (at the generating truth) x N, per model: finite-difference
Hessian of sum_i log f(chi_i; theta) + T(theta) + log prior, evaluated through the oracle."""
import sys, numpy as np
sys.path.insert(0, "/root/repo")
from oracle import api as O
from paper_2105_08026_b200 import synth

def cond_cov(model, inp, n):
    chi = inp["chi_true"]; cols = np.array(inp["cols"]); th0 = np.array(inp["theta_true"], float)
    s = O.Sampler(model, n, seed=1)
    s.set_data(inp["cols"])
    if inp["consts"] is not None: s.set_model_consts(inp["consts"])
    s.set_init(th0)
    def F(th):
        v = sum(O.logpop(model, chi[:, i], cols[:, i], th, inp["consts"]) for i in range(n))
        return v + s.theta_only(th) + O.logprior(model, th)
    d = len(th0); h = np.full(d, 2e-3)
    H = np.zeros((d, d)); f0 = F(th0)
    for a in range(d):
        for b in range(a, d):
            ea = np.zeros(d); ea[a] = h[a]; eb = np.zeros(d); eb[b] = h[b]
            if a == b: H[a, a] = (F(th0 + ea) - 2 * f0 + F(th0 - ea)) / h[a] ** 2
            else:
                H[a, b] = H[b, a] = (F(th0 + ea + eb) - F(th0 + ea - eb) - F(th0 - ea + eb) + F(th0 - ea - eb)) / (4 * h[a] * h[b])
    C = np.linalg.inv(-H)
    return C * n

np.set_printoptions(precision=4, suppress=True, linewidth=150)
n = int(sys.argv[1]) if len(sys.argv) > 1 else 20000
for name, model, mk in (("M0", 0, synth.make_normal1d), ("M1", 1, synth.make_thinned_schechter1d), ("M2", 2, synth.make_binormal2d),
                        ("M3", 3, lambda n, s: synth.make_linreg_me1d(n, s, fp32=False)), ("M4", 4, synth.make_bb1_fluxnoise1d),
                        ("M5", 5, synth.make_normal3d_knowncov)):
    inp = mk(n, 7)
    C = cond_cov(model, inp, n)
    sd = np.sqrt(np.diag(C))
    print(name, "sd*sqrt(N):", sd, "\n corr:\n", C / np.outer(sd, sd))
    print(" chol(C N):", np.linalg.cholesky(C)[np.tril_indices(len(sd))])
