"""The parity harness itself (tests/parity_util.py::compare_step), on the CPU: the oracle compared with itself must
pass every check, and a tap perturbed by a relative 1e-9 (far below the old multipliers, far above north_star's 1e-12)
must be caught by the fed-state checks."""
import copy

import numpy as np
import pytest

from oracle import api as O
from paper_2105_08026_b200 import synth

binding = pytest.importorskip("paper_2105_08026_b200.binding")
from parity_util import compare_step  # noqa: E402

CASES = [(0, 0, 0.44, synth.make_normal1d, {}), (1, 0, 0.44, synth.make_thinned_schechter1d, {}),
         (2, 0, 0.234, synth.make_binormal2d, {}), (3, 1, 0.44, synth.make_linreg_me1d, dict(fp32=True)),
         (4, 0, 0.44, synth.make_bb1_fluxnoise1d, {}), (5, 0, 0.234, synth.make_normal3d_knowncov, {}),
         (8, 0, 0.234, synth.make_normalpd_knowncov, dict(p=6))]


@pytest.mark.parametrize("model,precision,astar,maker,kw", CASES, ids=["M0", "M1", "M2", "M3f32", "M4", "M5", "p6"])
def test_oracle_against_itself_and_perturbed_taps(model, precision, astar, maker, kw):
    n = 257
    inp = maker(n, 5, **kw)
    o = O.Sampler(model, n, seed=5, precision=precision, target_accept_chi=astar)
    o.set_data(inp["cols"])
    if inp["consts"] is not None:
        o.set_model_consts(inp["consts"])
    o.set_init(inp["theta0"])
    o.run(7)
    st = o.get_state()
    to = o.step(taps=True)
    ctx = dict(model=model, inputs=inp, astar=astar)
    assert compare_step(to, to, precision, st, "self", ctx=ctx) == 0
    rel = 1e-9 if precision == 0 else 1e-3
    for key in ("pi_prop", "a", "b", "L_new", "pi_cur"):
        bad = copy.deepcopy(to)
        v = bad[key]
        idx = np.flatnonzero(np.isfinite(v.reshape(-1)) & (np.abs(v.reshape(-1)) > 1e-3))[3]
        v.reshape(-1)[idx] *= 1.0 + rel
        with pytest.raises(AssertionError):
            compare_step(to, bad, precision, st, "perturbed " + key, ctx=ctx)
