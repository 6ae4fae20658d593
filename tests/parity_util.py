"""Helpers shared by the GPU parity tests: build an oracle and a CUDA sampler on the same seeded inputs and compare their
taps / states.

Tolerances (DESIGN.md section 14 derives every one that is not north_star's own figure):
  north_star   per-object log-densities rel 1e-12 (fp64) / 1e-5 (fp32), floor tol * max(1, |pi|); population sum rel 1e-10;
               accept sequences identical except where |log alpha - log u| < 1e-9 (those are counted).
  fed state    every GPU tap is ALSO compared with the oracle's primitive evaluated at the GPU's own upstream taps
               (the oracle's log-densities at the GPU's chi', the closed form / defining identity of the RAM update at the
               GPU's alpha), so each stage is held to north_star's figure on identical inputs and no tolerance has to
               absorb the propagated few-ulp difference of the normals (device log / sqrt / sin-cos of fastmath.cuh against glibc's).
  propagated   the direct GPU-vs-oracle comparisons downstream of the normals use bounds computed from the measured
               upstream differences (first-order error propagation), not fixed multipliers.
"""
import ctypes as C
import math

import numpy as np

from oracle import api as O
from paper_2105_08026_b200 import binding as B
from paper_2105_08026_b200 import synth

EPS = 2.0 ** -52
EPS32 = 2.0 ** -23
# north_star figures
TOL = {B.F64: dict(pi=1e-12, tie=1e-9, eps=EPS), B.F32_STATE_F64_REDUCE: dict(pi=1e-5, tie=1e-4, eps=EPS32)}
# radius of a Box-Muller pair: sqrt(-2 ln u_min); u_min = 2^-33 (32-bit plate uniforms, p = 1), 2^-53 (52 bits), 2^-24 (fp32)
RAD_MAX = 8.6


def make_pair(model, n, seed, precision=B.F64, theta_mode=B.THETA_DEVICE_TAIL, astar=0.44, inputs=None, theta0=None,
              keep_moments=False, max_trace_rows=0, freeze_theta=False, block_threads=0, blocks_per_sm=0,
              want_oracle=True, flags=0, adapt_until=0, prior_mean=None, prior_sd=None, theta_chol0=None, **extra):
    if inputs is None:
        maker = {0: synth.make_normal1d, 1: synth.make_thinned_schechter1d, 2: synth.make_binormal2d,
                 3: synth.make_linreg_me1d, 4: synth.make_bb1_fluxnoise1d,
                 5: synth.make_normal3d_knowncov}.get(model)
        kw = dict(fp32=True) if (precision == B.F32_STATE_F64_REDUCE and model in (0, 3)) else {}
        if model == 3 and precision == B.F64:
            kw = dict(fp32=False)
        inputs = maker(n, seed, **kw) if maker else synth.make_normalpd_knowncov(n, seed, p=model - 2)
    th0 = inputs["theta0"] if theta0 is None else theta0
    orc = None
    if want_oracle:
        orc = O.Sampler(model, n, seed=seed, precision=precision, target_accept_chi=astar,
                        keep_chi_moments=keep_moments, freeze_theta=freeze_theta, adapt_until=adapt_until,
                        prior_mean=prior_mean, prior_sd=prior_sd, **extra)
        orc.set_data(inputs["cols"])
        if inputs["consts"] is not None:
            orc.set_model_consts(inputs["consts"])
        orc.set_init(th0, theta_chol0=theta_chol0)
    gpu = B.Sampler(model, n, seed=seed, precision=precision, theta_mode=theta_mode, target_accept_chi=astar,
                    keep_chi_moments=keep_moments, max_trace_rows=max_trace_rows, freeze_theta=freeze_theta,
                    block_threads=block_threads, blocks_per_sm=blocks_per_sm, flags=flags, adapt_until=adapt_until,
                    prior_mean=prior_mean, prior_sd=prior_sd, **extra)
    gpu.set_data(inputs["cols"])
    if inputs["consts"] is not None:
        gpu.set_model_consts(inputs["consts"])
    gpu.set_init(th0, theta_chol0=theta_chol0)
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


# ------------------------------------------------------------------------------------------------------------------
# the oracle's per-object primitives over a whole population (plain loops over oracle_loglik / oracle_logpop)
class OracleDensities:
    def __init__(self, model, precision, inputs):
        self.model, self.f32 = model, precision == B.F32_STATE_F64_REDUCE
        self.lib = O.lib()
        cols = np.asarray(inputs["cols"], dtype=np.float64)
        self.n = cols.shape[1]
        self.dt = np.float32 if self.f32 else np.float64
        self.ct = C.c_float if self.f32 else C.c_double
        self.data = np.ascontiguousarray(cols.T.astype(self.dt))                    # (N, ncols): one row per object
        self.data64 = np.ascontiguousarray(cols.T.astype(self.dt).astype(np.float64))
        self.consts = None if inputs["consts"] is None else np.ascontiguousarray(np.asarray(inputs["consts"], self.dt))
        self.consts64 = None if inputs["consts"] is None else np.ascontiguousarray(np.asarray(inputs["consts"], np.float64))

    @staticmethod
    def _rows(a, ct):
        base, stride = a.ctypes.data, a.strides[0]
        return [C.cast(base + i * stride, C.POINTER(ct)) for i in range(a.shape[0])]

    def target(self, chi, theta):
        """log l_i(chi_i) + log f(chi_i; theta) in the state precision (the oracle's own sum of its two functions)."""
        x = np.ascontiguousarray(np.asarray(chi, dtype=np.float64).T.astype(self.dt))
        th = np.ascontiguousarray(np.asarray(theta, dtype=self.dt))
        pc = None if self.consts is None else self.consts.ctypes.data_as(C.POINTER(self.ct))
        pt = th.ctypes.data_as(C.POINTER(self.ct))
        lk = self.lib.oracle_loglik_f32 if self.f32 else self.lib.oracle_loglik
        lp = self.lib.oracle_logpop_f32 if self.f32 else self.lib.oracle_logpop
        out = np.empty(self.n, dtype=self.dt)
        for i, (px, pd) in enumerate(zip(self._rows(x, self.ct), self._rows(self.data, self.ct))):
            out[i] = self.dt(lk(self.model, px, pd, pc)) + self.dt(lp(self.model, px, pd, pt, pc))
        return out.astype(np.float64)

    def pop(self, chi, theta):
        """log f(chi_i; theta) in fp64 (population terms are fp64 in both precisions, reading R13)."""
        x = np.ascontiguousarray(np.asarray(chi, dtype=np.float64).T)
        th = np.ascontiguousarray(np.asarray(theta, dtype=np.float64))
        pc = None if self.consts64 is None else self.consts64.ctypes.data_as(C.POINTER(C.c_double))
        pt = th.ctypes.data_as(C.POINTER(C.c_double))
        out = np.empty(self.n)
        for i, (px, pd) in enumerate(zip(self._rows(x, C.c_double), self._rows(self.data64, C.c_double))):
            out[i] = self.lib.oracle_logpop(self.model, px, pd, pt, pc)
        return out


def unpack(Lp, p):
    """(ntri, N) packed lower triangles -> (N, p, p)."""
    n = Lp.shape[1]
    M = np.zeros((n, p, p))
    k = 0
    for r in range(p):
        for c in range(r + 1):
            M[:, r, c] = Lp[k]
            k += 1
    return M


def compare_step(to, tg, precision, state_before, what="", ctx=None):
    """Compare one iteration's taps (oracle `to`, GPU `tg`) from identical fed state `state_before`.
    ctx = dict(model, inputs, astar[, eta_exponent, adapt_until]) enables the fed-state checks (see the module docstring).
    Returns the number of accept decisions that legitimately differ (near ties, inside the band)."""
    tol = TOL[precision]
    eps, tpi = tol["eps"], tol["pi"]
    chi0, L0 = state_before["chi"], state_before["L"]
    p = chi0.shape[0]
    Lm0 = unpack(L0, p)
    # 1. uniforms: dyadic rationals, bit for bit
    assert np.array_equal(to["u"], tg["u"]), f"{what}: accept uniforms must be bit-identical"
    # 2. chi' = chi + L z.  The normals differ by the rounding of two independent libms: |dz_k| <= 8 ulp x radius (log and
    #    sqrt of the radius <= 2 ulp each, cos / sin <= 2 ulp ABSOLUTE near their zeros, one product), radius <= RAD_MAX;
    #    the p products and sums add (p + 1) ulp of |chi'|.
    rowsum = np.abs(Lm0).sum(2).T                                                          # (p, N): sum_k |L_rk|
    bound_chi = 8 * eps * RAD_MAX * rowsum + (p + 1) * eps * np.maximum(np.abs(to["chi_prop"]), np.abs(chi0))
    d_chi = np.abs(to["chi_prop"] - tg["chi_prop"])
    assert np.all(d_chi <= bound_chi), f"{what}: chi' err / bound {np.max(d_chi / bound_chi):.2f}"
    # 3. log target at the (identical) current chi: north_star
    assert np.all(close(to["pi_cur"], tg["pi_cur"], tpi)), f"{what}: pi_cur"
    mism = to["accepted"] != tg["accepted"]
    if ctx is not None:
        od = ctx.get("_od")
        if od is None:
            od = ctx["_od"] = OracleDensities(ctx["model"], precision, ctx["inputs"])
        theta, theta_p = state_before["theta"], tg["theta_prop"]
        # 4. log target at the proposal: the oracle's functions AT THE GPU's chi' -- north_star's figure on identical
        #    input, support decision (finite / -inf) included
        pp_fed = od.target(tg["chi_prop"], theta)
        assert np.array_equal(np.isfinite(pp_fed), np.isfinite(tg["pi_prop"])), f"{what}: support at the GPU's chi'"
        assert np.all(close(pp_fed, tg["pi_prop"], tpi)), f"{what}: pi_prop at the GPU's chi'"
        # 5. alpha = exp(min(0, pi' - pi)) from the GPU's own two log targets: both exps <= 2 ulp, and the T-precision
        #    subtraction pi' - pi rounds once more (relative eps of the difference); the taps themselves may carry one more
        #    rounding each (M4: the normaliser log C is added back on the host), eps (|pi'| + |pi|) in the exponent
        with np.errstate(invalid="ignore", over="ignore"):
            la_g = np.minimum(0.0, tg["pi_prop"] - tg["pi_cur"])
            la_g = np.where(np.isnan(la_g), -np.inf, la_g)
            a_ref = np.exp(la_g)
        tiny = 1e-300 if precision == B.F64 else 2e-38                       # below the smallest normal number: no relative claim
        with np.errstate(invalid="ignore"):
            slack = np.where(np.isfinite(la_g), np.abs(la_g) + np.abs(tg["pi_prop"]) + np.abs(tg["pi_cur"]), 0.0)
            ok = np.abs(tg["alpha"] - a_ref) <= a_ref * (4 * eps + eps * slack) + tiny
        assert np.all(ok), f"{what}: alpha from the GPU's own log targets"
        # 7. RAM update at the GPU's alpha: p = 1 closed form L sqrt(1 + c) (P4 iii); p >= 2 the defining identity
        #    L_n L_n^T = L (I + c z z^T / |z|^2) L^T (Eq. 2.6) with L z = chi' - chi read off the GPU's taps
        t_next = state_before["t"] + 1
        frozen = ctx.get("adapt_until", 0) > 0 and t_next > ctx.get("adapt_until", 0)
        eta = 0.0 if frozen else float(t_next + 1) ** (-ctx.get("eta_exponent", 2.0 / 3.0))
        if precision == B.F32_STATE_F64_REDUCE:
            eta = float(np.float32(eta))
        cc = eta * (tg["alpha"] - (float(np.float32(ctx["astar"])) if precision != B.F64 else ctx["astar"]))
        if p == 1:
            ref = L0[0] * np.sqrt(1.0 + cc)
            assert np.all(np.abs(tg["L_new"][0] - ref) <= 6 * eps * np.abs(ref)), f"{what}: L_new closed form"
        else:
            Ln = unpack(tg["L_new"], p)
            v = (tg["chi_prop"] - chi0).T                                                  # (N, p) = L z as the GPU formed it
            z = np.linalg.solve(Lm0, v[:, :, None])[:, :, 0]
            M = Lm0 @ np.transpose(Lm0, (0, 2, 1)) + (cc / (z * z).sum(1))[:, None, None] * v[:, :, None] * v[:, None, :]
            R = Ln @ np.transpose(Ln, (0, 2, 1)) - M
            # v = chi' - chi carries the rounding of chi' (eps |chi'| absolute), amplified by |c| <= 1 in the rank-one term
            scale = np.abs(M).max((1, 2)) + np.abs(chi0).max(0) * np.abs(v).max(1) / np.maximum((z * z).sum(1), 1e-300)
            assert np.all(np.abs(R).max((1, 2)) <= 1e-12 * scale), f"{what}: L_n L_n^T identity {np.max(np.abs(R).max((1, 2)) / scale):.2e}"
            assert np.all(np.diagonal(Ln, axis1=1, axis2=2) > 0), f"{what}: diag(L_new) > 0"
        # 8. population terms at the GPU's own new chi, at theta (a_i) and the GPU's theta' (b_i): north_star, 1e-12
        chi_new_g = np.where(tg["accepted"][None, :] != 0, tg["chi_prop"], chi0)
        if precision != B.F64:
            chi_new_g = chi_new_g.astype(np.float32).astype(np.float64)
        a_fed, b_fed = od.pop(chi_new_g, theta), od.pop(chi_new_g, theta_p)
        assert np.all(close(a_fed, tg["a"], 1e-12)), f"{what}: a_i at the GPU's chi"
        assert np.all(close(b_fed, tg["b"], 1e-12)), f"{what}: b_i at the GPU's chi and theta'"
        # ... and directly against the oracle's where the input was identical (rejected on both sides): same figure
        rej = (to["accepted"] == 0) & (tg["accepted"] == 0)
        assert np.all(close(to["a"][rej], tg["a"][rej], 1e-12)), f"{what}: a_i of rejected objects"
        # 9. the deterministic reduction: the GPU's sums against the exactly rounded sums of the terms it summed
        S_ref, D_ref = math.fsum(a_fed), math.fsum(b_fed - a_fed)
        assert abs(tg["S"] - S_ref) <= 1e-10 * max(1.0, abs(S_ref)), f"{what}: S against fsum of its terms"
        assert abs(tg["Delta"] - D_ref) <= 1e-10 * max(1.0, float(np.abs(b_fed - a_fed).sum())), f"{what}: Delta against fsum of its terms"
    # direct comparisons downstream of the normals, with propagated bounds -----------------------------------------
    # pi_prop: |d pi| <= north_star's figure + |pi(chi'_gpu) - pi(chi'_oracle)| (the oracle's own function at both points)
    fin = np.isfinite(to["pi_prop"]) & np.isfinite(tg["pi_prop"])
    if ctx is not None:
        with np.errstate(invalid="ignore"):
            moved = np.abs(pp_fed - to["pi_prop"])
            ok = np.abs(tg["pi_prop"] - to["pi_prop"]) <= tpi * np.maximum(1.0, np.abs(to["pi_prop"])) + moved
        assert np.all(ok[fin]), f"{what}: pi_prop against the oracle's own"
        # a support decision may differ only where chi' itself straddles the boundary within its bound
        sup = np.isfinite(to["pi_prop"]) != np.isfinite(tg["pi_prop"])
        if sup.any():
            lo, hi = ctx["inputs"]["consts"][2], ctx["inputs"]["consts"][3]
            edge = np.minimum(np.abs(tg["chi_prop"][0] - lo), np.abs(tg["chi_prop"][0] - hi))
            assert np.all(edge[sup] <= bound_chi[0][sup]), f"{what}: support decisions differ away from the boundary"
    else:
        assert np.array_equal(np.isfinite(to["pi_prop"]), np.isfinite(tg["pi_prop"])), f"{what}: support"
    # alpha: |d alpha| <= alpha (|d pi'| + |d pi|) + 4 ulp (exp is its own derivative)
    with np.errstate(invalid="ignore"):
        dl = np.where(fin, np.abs(tg["pi_prop"] - to["pi_prop"]), 0.0) + np.abs(tg["pi_cur"] - to["pi_cur"])
    amax = np.maximum(to["alpha"], tg["alpha"])
    tiny = 1e-300 if precision == B.F64 else 2e-38
    with np.errstate(invalid="ignore"):
        size = np.where(fin, np.abs(to["pi_prop"] - to["pi_cur"]) + np.abs(to["pi_prop"]) + np.abs(to["pi_cur"]), 0.0)
    assert np.all((np.abs(to["alpha"] - tg["alpha"]) <= amax * (2 * dl + 8 * eps * (1 + size)) + tiny) | ~fin), f"{what}: alpha"
    # 6. accept decisions: identical outside the near-tie band (north_star), counted inside it
    with np.errstate(divide="ignore"):
        gap = np.abs(np.log(to["alpha"]) - np.log(to["u"]))
    assert np.all(gap[mism] < tol["tie"]), f"{what}: {int((gap[mism] >= tol['tie']).sum())} accept mismatches outside the tie band"
    # L_new against the oracle's form-and-factor route: d L <= (eta |d alpha| / (1 - alpha*) + 16 ulp) max|L| per object
    # (d sqrt(1 + c) = dc / (2 sqrt(1 + c)), 1 + c >= 1 - alpha*; the unit vector's few-ulp difference enters times |c| <= 1)
    da = np.abs(to["alpha"] - tg["alpha"])
    lmax = np.abs(L0).max(0)
    assert np.all(np.abs(to["L_new"] - tg["L_new"]) <= (2.0 * da + 16 * eps * (1 + RAD_MAX)) * lmax), f"{what}: L_new against the oracle's"
    if not mism.any():
        # population sums against the oracle's: relative 1e-10 (north_star; Delta relative to the size of its terms, it is a
        # sum of differences of either sign) plus what the terms themselves moved by (the new chi differs by the bound of 2.)
        moved_a = float(np.abs(tg["a"] - to["a"]).sum())
        moved_d = float(np.abs((tg["b"] - tg["a"]) - (to["b"] - to["a"])).sum())
        assert abs(to["S"] - tg["S"]) <= 1e-10 * max(1.0, abs(to["S"])) + moved_a, f"{what}: S"
        dsum = float(np.abs(to["b"] - to["a"]).sum())
        assert abs(to["Delta"] - tg["Delta"]) <= 1e-10 * max(1.0, dsum, abs(to["Delta"])) + moved_d, f"{what}: Delta"
    return int(mism.sum())


def compare_theta_step(to, tg, what="", rel=1e-9):
    np.testing.assert_allclose(tg["theta_prop"], to["theta_prop"], rtol=rel, atol=rel, err_msg=f"{what}: theta'")
    assert tg["u_theta"] == to["u_theta"], f"{what}: theta accept uniform must be bit-identical"
    for k in ("T_cur", "T_prop", "lp_cur", "lp_prop"):
        assert np.all(close(to[k], tg[k], 1e-10)), f"{what}: {k} {to[k]} vs {tg[k]}"
