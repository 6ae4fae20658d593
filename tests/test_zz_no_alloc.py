"""cudahm_debug_step_noalloc: the tapped iteration whose tap scratch lives in the library's built-in device array (no
cudaMalloc in the call) against the existing cudahm_debug_step (cudaMalloc per call).  Same kernels, same launch shape, same
inputs => the taps must be IDENTICAL, which is stricter than any tolerance of the parity tests.  Collected last on purpose
(the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from parity_util import make_pair
from paper_2105_08026_b200 import binding as B

pytestmark = pytest.mark.gpu
ARRAYS = ("chi_prop", "pi_cur", "pi_prop", "alpha", "u", "accepted", "L_new", "a", "b", "theta_prop")
SCALARS = ("S", "Delta", "T_cur", "T_prop", "lp_cur", "lp_prop", "log_r", "alpha_theta", "u_theta", "accepted_theta")


def _twins(model, n, seed, astar, precision=B.F64):
    _, a, inp = make_pair(model, n, seed=seed, astar=astar, precision=precision, want_oracle=False, max_trace_rows=8)
    _, b, _ = make_pair(model, n, seed=seed, astar=astar, precision=precision, want_oracle=False, max_trace_rows=8, inputs=inp)
    a.run(6, 0, 10 ** 6, sync=True)
    b.run(6, 0, 10 ** 6, sync=True)
    return a, b


def _same(ta, tb, what):
    for k in ARRAYS:
        assert np.array_equal(ta[k], tb[k], equal_nan=True), f"{what}: {k}"
    for k in SCALARS:
        assert ta[k] == tb[k] or (ta[k] != ta[k] and tb[k] != tb[k]), f"{what}: {k} {ta[k]} vs {tb[k]}"


def test_no_alloc_entry_point_matches_the_allocating_one_on_two_calls_in_a_row():
    a, b = _twins(B.M_BINORMAL2D, 5003, 21, 0.234)                    # p = 2: 5 per-object tap columns + L
    assert 0 < b.debug_step_noalloc_bytes() <= B.NOALLOC_SCRATCH_BYTES
    for call in range(2):                                             # two calls in a row on the shared array
        _same(a.debug_step(10 ** 6, 1), b.debug_step_noalloc(10 ** 6, 1), f"M2 call {call}")
    for k in ("chi", "L", "theta", "L_theta", "t"):
        assert np.array_equal(a.get_state()[k], b.get_state()[k]), k
    # a SMALLER handle of another model and precision right after: the array still holds the M2 taps beyond its range
    c, d = _twins(B.M_LINREG_ME1D, 3001, 22, 0.44, precision=B.F32_STATE_F64_REDUCE)
    for call in range(2):
        _same(c.debug_step(10 ** 6, 1), d.debug_step_noalloc(10 ** 6, 1), f"M3 fp32 call {call}")
    # and the first handle again, interleaved with the allocating path on the same handle
    _same(a.debug_step(10 ** 6, 1), b.debug_step_noalloc(10 ** 6, 1), "M2 again")
    tb = b.debug_step(10 ** 6, 1)
    ta = a.debug_step_noalloc(10 ** 6, 1)
    _same(ta, tb, "paths swapped")
    assert a.get_stats()["chi_proposals"] == b.get_stats()["chi_proposals"]


def test_no_alloc_entry_point_refuses_what_does_not_fit_and_leaves_the_handle_usable():
    n = 100_000                                                       # p = 1: 68 B per object = 6.8 MB > 4 MiB
    _, g, _ = make_pair(B.M_NORMAL1D, n, seed=23, want_oracle=False)
    assert g.debug_step_noalloc_bytes() > B.NOALLOC_SCRATCH_BYTES
    before = g.get_state()
    with pytest.raises(B.CudahmError) as e:
        g.debug_step_noalloc()
    assert e.value.code == B.E_WORKSPACE and "CUDAHM_NOALLOC_SCRATCH_BYTES" in str(e.value)
    after = g.get_state()
    assert after["t"] == before["t"] and np.array_equal(after["chi"], before["chi"])
    g.debug_step()                                                    # the allocating path still serves it
    assert g.get_state()["t"] == before["t"] + 1
