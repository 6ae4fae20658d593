"""Long chains on every kernel variant: one cudahm_run call and the same chain split at random into many calls must
leave bit-identical state, trace and moments, with everything finite and the theta acceptance rate near its target.

A property that holds at any chain length (the draws are counter-based, SURVEY 8(c) / DESIGN.md R4, so the chain is
a pure function of (seed, t) however the calls are cut): it is what a lost barrier, a stale mailbox epoch, a ring
slot reused too early or a graph launched with stale parameters would break, and those show up only after many
iterations and many launches, well past the lengths the oracle comparisons in test_gpu_parity.py can afford."""
import numpy as np
import pytest

from paper_2105_08026_b200 import binding as B
from paper_2105_08026_b200 import synth

pytestmark = pytest.mark.gpu

# (config, population or 0 for the config's own, iterations, the block size the variant must report)
CASES = [
    ("C0", 0, 40_000, 640),          # on-chip p = 1, one slot in one block
    ("C0", 1, 20_000, 640),          # a single object
    ("C1", 75_777, 20_000, 640),     # first population past the sweep-side selection sum (2 slots per thread)
    ("C2", 0, 20_000, 640),          # on-chip p = 1 as benched
    ("C5", 33, 20_000, 640),         # one full warp plus one lane
    ("C6", 0, 20_000, 384),          # general on-chip kernel, one object per thread
    ("C6", 37_889, 10_000, 384),     # first population past one object per thread
    ("C3", 200_001, 10_000, 384),    # general on-chip kernel, p = 2, ragged
    ("C2", 303_105, 6_000, None),    # first population past the on-chip capacity: streaming kernel, staged draws
    ("C3", 0, 4_000, 512),           # streaming kernel with dedicated tail warps (384 + 128) as benched
    ("C4", 1_000_001, 6_000, None),  # fp32 streaming kernel, ragged
]


def _chain(c, n, inp, total, burn, thin, cuts):
    s = B.Sampler(c.model, n, seed=c.seed, precision=c.precision, theta_mode=B.THETA_DEVICE_TAIL,
                  target_accept_chi=c.target_accept_chi, target_accept_theta=c.target_accept_theta,
                  keep_chi_moments=c.keep_chi_moments, max_trace_rows=(total - burn) // thin + 1)
    s.set_data(inp["cols"])
    if inp["consts"] is not None:
        s.set_model_consts(inp["consts"])
    s.set_init(inp["theta0"], theta_chol0=inp["theta_chol0"])
    for k in cuts:
        s.run(k, burn, thin)
    s.sync()
    out = dict(state=s.get_state(), trace=s.get_theta_trace(), stats=s.get_stats(),
               moments=s.get_chi_moments() if c.keep_chi_moments else None)
    s.close()
    return out


@pytest.mark.parametrize("name,n_over,iters,block", CASES, ids=[f"{c[0]}-{c[1] or 'full'}" for c in CASES])
def test_long_chain_is_split_invariant(name, n_over, iters, block):
    c = synth.CONFIGS[name]
    n = n_over or c.n_objects
    inp = synth.make_inputs(name, n_objects=n)
    burn, thin = 500, 50
    total = burn + iters
    rng = np.random.default_rng(n + iters)
    cuts, left = [], total
    while left > 0:
        k = int(min(left, rng.choice([1, 2, 3, 7, 64, 1000, 5000])))
        cuts.append(k)
        left -= k
    a = _chain(c, n, inp, total, burn, thin, [total])
    b = _chain(c, n, inp, total, burn, thin, cuts)
    if block is not None:
        assert a["stats"]["block_threads"] == block, "the case no longer reaches the kernel variant it names"
    assert a["stats"]["dedicated_tail"] == int(name == "C3" and not n_over)
    # launch path: a handle's first persistent launch is direct, every later one goes through its one-node
    # graph with the parameters updated in place -- a graph call that fails makes the handle fall back to direct launches
    # for good, silently but for this count
    assert a["stats"]["graph_launches"] == 0 and b["stats"]["graph_launches"] == len(cuts) - 1
    assert a["state"]["t"] == b["state"]["t"] == total
    for key in ("chi", "L", "theta", "L_theta"):
        assert np.isfinite(a["state"][key]).all()
        assert np.array_equal(a["state"][key], b["state"][key]), key
    assert len(a["trace"]) == iters // thin and np.isfinite(a["trace"]).all()
    assert np.array_equal(a["trace"], b["trace"])
    for key in ("chi_accepts", "theta_accepts", "theta_proposals", "nonfinite"):
        assert a["stats"][key] == b["stats"][key], key
    if c.keep_chi_moments:
        (ma, va, ka), (mb, vb, kb) = a["moments"], b["moments"]
        assert ka == kb == iters and np.isfinite(va).all()
        assert np.array_equal(ma, mb) and np.array_equal(va, vb)
    # RAM steers the theta acceptance rate to its target (Sec. 3, the RAM recursion); a chain whose
    # decisions were corrupted drifts off it.  n = 1 has a one-object posterior far from the recipe's proposal scale.
    acc = a["stats"]["theta_accepts"] / a["stats"]["theta_proposals"]
    assert abs(acc - c.target_accept_theta) < (0.06 if n > 1 else 0.1), acc
