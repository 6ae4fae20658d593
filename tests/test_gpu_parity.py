"""GPU parity: the CUDA path (through the C ABI, include/cudahm.h) against the CPU oracle on the same seeded
inputs, element by element.  Tolerances are BASELINE.json north_star's (tests/parity_util.py::TOL):
per-object log-densities rel 1e-12 (fp64) / 1e-5 (fp32), population sum rel 1e-10, accept sequences identical
except inside the near-tie band |log alpha - log u| < 1e-9 (counted)."""
import numpy as np
import pytest

from parity_util import TOL, compare_step, compare_theta_step, make_pair, sync_gpu_to_oracle
from paper_2105_08026_b200 import binding as B

pytestmark = pytest.mark.gpu
NO_TRACE = 10 ** 12   # burn-in beyond any iteration: tapped steps append nothing to the theta trace

# (model, precision, alpha_*, N): sizes span several 16-byte vectors, several blocks and a ragged tail
CASES = [
    (B.M_NORMAL1D, B.F64, 0.44, 1000),
    (B.M_THINNED_SCHECHTER1D, B.F64, 0.44, 4099),
    (B.M_BINORMAL2D, B.F64, 0.234, 3001),
    (B.M_LINREG_ME1D, B.F64, 0.44, 2050),
    (B.M_NORMAL1D, B.F32_STATE_F64_REDUCE, 0.44, 4097),
    (B.M_LINREG_ME1D, B.F32_STATE_F64_REDUCE, 0.44, 10007),
    (B.M_BB1_FLUXNOISE1D, B.F64, 0.44, 4099),
    (B.M_NORMAL3D_KNOWNCOV, B.F64, 0.234, 3003),
    (B.M_NORMAL4D_KNOWNCOV, B.F64, 0.234, 2051),
    (B.M_NORMAL5D_KNOWNCOV, B.F64, 0.234, 1031),
    (B.M_NORMAL6D_KNOWNCOV, B.F64, 0.234, 1543),
]
IDS = ["M0-f64", "M1-f64", "M2-f64", "M3-f64", "M0-f32", "M3-f32", "M4-f64", "M5-f64", "p4-f64", "p5-f64", "p6-f64"]


@pytest.mark.parametrize("model,precision,astar,n", CASES, ids=IDS)
def test_single_step_fed_state(model, precision, astar, n):
    """One iteration from identical state: every tap of SURVEY 8(c) protocol (i)."""
    orc, gpu, inp = make_pair(model, n, seed=11 + model, precision=precision, astar=astar, block_threads=256)
    st = sync_gpu_to_oracle(orc, gpu)
    to, tg = orc.step(NO_TRACE, 1, taps=True), gpu.debug_step(NO_TRACE, 1)
    nm = compare_step(to, tg, precision, st, what=f"model {model}", ctx=dict(model=model, inputs=inp, astar=astar))
    compare_theta_step(to, tg, what=f"model {model}")
    assert nm == 0 or precision != B.F64, "an fp64 near tie in the very first step is (almost surely) a bug"
    if nm == 0:
        assert to["accepted_theta"] == tg["accepted_theta"]


@pytest.mark.parametrize("model,precision,astar,n", CASES, ids=IDS)
def test_lockstep_trajectory(model, precision, astar, n):
    """Protocol (ii): lock-step for 60 iterations with taps; accept sequences identical outside the tie band;
    the GPU is re-fed the oracle's state after every iteration in fp32 (per-decision disagreement is expected
    there) and only after a counted in-band divergence in fp64."""
    orc, gpu, inp = make_pair(model, n, seed=21 + model, precision=precision, astar=astar, block_threads=256)
    ties = 0
    ctx = dict(model=model, inputs=inp, astar=astar)
    st = sync_gpu_to_oracle(orc, gpu)
    for it in range(60):
        to, tg = orc.step(NO_TRACE, 1, taps=True), gpu.debug_step(NO_TRACE, 1)
        nm = compare_step(to, tg, precision, st, what=f"model {model} it {it}", ctx=ctx)
        compare_theta_step(to, tg, what=f"model {model} it {it}", rel=1e-9 if precision == B.F64 else 1e-6)
        ties += nm
        if precision == B.F64 and nm == 0 and to["accepted_theta"] == tg["accepted_theta"]:
            st = orc.get_state()
            sg = gpu.get_state()
            np.testing.assert_allclose(sg["chi"], st["chi"], rtol=1e-11, atol=1e-11)
            # an off-diagonal entry of L can nearly cancel: measure against the object's largest entry
            assert np.all(np.abs(sg["L"] - st["L"]) <= 1e-10 * np.abs(st["L"]).max(0)), "L"
            np.testing.assert_allclose(sg["theta"], st["theta"], rtol=1e-9, atol=1e-9)
            np.testing.assert_allclose(sg["L_theta"], st["L_theta"], rtol=1e-8, atol=1e-12)
            # keep the two strictly in lock step so rounding differences do not accumulate into a decision
            gpu.set_state(st["chi"], st["L"], st["theta"], st["L_theta"], st["t"])
        else:
            st = sync_gpu_to_oracle(orc, gpu)
    if precision == B.F64:
        assert ties <= 1, f"{ties} near ties in {60 * n} fp64 decisions (expected ~1e-9 each)"
    else:
        assert ties <= 60 * n * 1e-3


@pytest.mark.parametrize("mode", [B.THETA_HOST, B.THETA_GRAPH, B.THETA_DEVICE_TAIL], ids=["host", "graph", "tail"])
@pytest.mark.parametrize("model,astar,n", [(B.M_NORMAL1D, 0.44, 1000), (B.M_THINNED_SCHECHTER1D, 0.44, 3000),
                                             (B.M_BINORMAL2D, 0.234, 2000), (B.M_BB1_FLUXNOISE1D, 0.44, 3000),
                                             (B.M_NORMAL3D_KNOWNCOV, 0.234, 2001), (B.M_NORMAL4D_KNOWNCOV, 0.234, 1501),
                                             (B.M_NORMAL5D_KNOWNCOV, 0.234, 1201), (B.M_NORMAL6D_KNOWNCOV, 0.234, 1001)],
                         ids=["M0", "M1", "M2", "M4", "M5", "p4", "p5", "p6"])
def test_free_running_matches_oracle(model, astar, n, mode):
    """cudahm_run (no taps, no resync) for 120 iterations in every theta mode against oracle_run: same theta
    trace, same chi / L, same moments, same counters.  (~1e5 decisions at ~1e-9 tie probability each.)"""
    iters, burn, thin = 120, 20, 5
    orc, gpu, _ = make_pair(model, n, seed=31 + model, astar=astar, theta_mode=mode, keep_moments=True,
                            max_trace_rows=(iters - burn) // thin)
    orc.run(iters, burn, thin)
    gpu.run(iters, burn, thin, sync=True)
    so, sg = orc.get_state(), gpu.get_state()
    assert sg["t"] == so["t"] == iters
    tro, trg = orc.get_theta_trace(), gpu.get_theta_trace()
    assert trg.shape == tro.shape == ((iters - burn) // thin, gpu.dtheta)
    np.testing.assert_allclose(trg, tro, rtol=1e-8, atol=1e-8)
    np.testing.assert_allclose(sg["chi"], so["chi"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["L"], so["L"], rtol=1e-9)
    np.testing.assert_allclose(sg["L_theta"], so["L_theta"], rtol=1e-7, atol=1e-12)
    mo, vo, ko = orc.get_chi_moments()
    mg, vg, kg = gpu.get_chi_moments()
    assert kg == ko == iters - burn
    np.testing.assert_allclose(mg, mo, rtol=1e-10, atol=1e-10)
    np.testing.assert_allclose(vg, vo, rtol=1e-8, atol=1e-12)
    stg, sto = gpu.get_stats(), orc.get_stats()
    for k in ("iterations", "chi_accepts", "chi_proposals", "theta_accepts", "theta_proposals", "nonfinite",
              "moment_samples", "trace_rows"):
        assert stg[k] == sto[k], k
    assert stg["gpu_launches"] > 0


@pytest.mark.parametrize("mode", [B.THETA_HOST, B.THETA_GRAPH, B.THETA_DEVICE_TAIL], ids=["host", "graph", "tail"])
@pytest.mark.parametrize("model,astar,n,flags", [(B.M_NORMAL1D, 0.44, 1500, 0), (B.M_BINORMAL2D, 0.234, 2000, 0),
                                                   (B.M_NORMAL1D, 0.44, 1500, B.FLAG_STREAMING_ONLY)],
                         ids=["M0", "M2", "M0-streaming"])
def test_user_prior_and_adaptation_freeze_match_oracle(model, astar, n, flags, mode):
    """The advanced-use hooks: a user prior on theta (normal factors on some components) and
    adapt_until (eta_n = 0 from iteration 61 on), free-running against the oracle in every theta driver."""
    iters, burn, thin, K = 120, 20, 5, 60
    dt = 2 if model == B.M_NORMAL1D else 5
    pm = [0.3, -0.2, 0.0, 0.0, 0.0][:dt]
    psd = [0.05, np.inf, 0.1, np.inf, 0.2][:dt]
    orc, gpu, _ = make_pair(model, n, seed=71 + model, astar=astar, theta_mode=mode, max_trace_rows=(iters - burn) // thin,
                            adapt_until=K, prior_mean=pm, prior_sd=psd, flags=flags)
    orc.run(K, burn, thin)
    gpu.run(K, burn, thin, sync=True)
    L_K, Lth_K = gpu.get_state()["L"].copy(), gpu.get_state()["L_theta"].copy()
    np.testing.assert_allclose(L_K, orc.get_state()["L"], rtol=1e-9)
    orc.run(iters - K, burn, thin)
    gpu.run(iters - K, burn, thin, sync=True)
    so, sg = orc.get_state(), gpu.get_state()
    np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-8, atol=1e-8)
    np.testing.assert_allclose(sg["chi"], so["chi"], rtol=1e-9, atol=1e-9)
    assert np.array_equal(sg["L"], L_K) and np.array_equal(sg["L_theta"], Lth_K)      # frozen: bit for bit on the device
    np.testing.assert_allclose(sg["L"], so["L"], rtol=1e-9)
    stg, sto = gpu.get_stats(), orc.get_stats()
    assert stg["chi_accepts"] == sto["chi_accepts"] and stg["theta_accepts"] == sto["theta_accepts"]
    # the prior is felt: lp taps differ from the default's zero
    tg = gpu.debug_step(NO_TRACE, 1)
    to = orc.step(NO_TRACE, 1, taps=True)
    assert to["lp_cur"] != 0.0
    compare_theta_step(to, tg, what="hooks")


@pytest.mark.parametrize("model,astar,n", [(B.M_THINNED_SCHECHTER1D, 0.44, 4001), (B.M_BINORMAL2D, 0.234, 3000),
                                             (B.M_BB1_FLUXNOISE1D, 0.44, 2500)], ids=["M1", "M2", "M4"])
@pytest.mark.parametrize("on_device", [False, True], ids=["host-exchange", "device-exchange"])
def test_sharded_population_matches_oracle(model, astar, n, on_device):
    """the population split by object range over THREE handles (here on one GPU, launched one after the
    other), theta replicated, the shards' totals summed in rank order between the sweep and the theta step
    (cudahm_shard_sweep / cudahm_shard_decide) -- against the UNSHARDED oracle chain."""
    from paper_2105_08026_b200 import sharded
    iters, burn, thin = 100, 20, 5
    orc, _, inp = make_pair(model, n, seed=81 + model, astar=astar, keep_moments=True, theta_mode=B.THETA_HOST)
    orc.run(iters, burn, thin)
    parts = []
    for lo, hi in sharded.shard_ranges(n, 3):
        g = B.Sampler(model, hi - lo, seed=81 + model, theta_mode=B.THETA_HOST, target_accept_chi=astar, keep_chi_moments=True,
                      max_trace_rows=(iters - burn) // thin, object_offset=lo, n_objects_total=n)
        g.set_data([c[lo:hi] for c in inp["cols"]])
        if inp["consts"] is not None:
            g.set_model_consts(inp["consts"])
        g.set_init(inp["theta0"])
        parts.append(g)
    sharded.LocalShards(parts, device=on_device).run(iters, burn, thin)
    for g in parts:
        np.testing.assert_allclose(g.get_theta_trace(), orc.get_theta_trace(), rtol=1e-8, atol=1e-8)
        assert np.array_equal(g.get_theta_trace(), parts[0].get_theta_trace())
    so = orc.get_state()
    np.testing.assert_allclose(np.concatenate([g.get_state()["chi"] for g in parts], axis=1), so["chi"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(np.concatenate([g.get_state()["L"] for g in parts], axis=1), so["L"], rtol=1e-9)
    np.testing.assert_allclose(np.concatenate([g.get_chi_moments()[0] for g in parts], axis=1), orc.get_chi_moments()[0],
                               rtol=1e-10, atol=1e-10)
    st, sto = parts[0].get_stats(), orc.get_stats()
    assert st["chi_accepts"] == sto["chi_accepts"] and st["theta_accepts"] == sto["theta_accepts"] and st["iterations"] == iters
    # accepts are global on every shard, so proposals must be the WHOLE population's too (a rate above 1 otherwise)
    for g in parts:
        assert g.get_stats()["chi_proposals"] == sto["chi_proposals"] == iters * n


def test_single_shard_is_the_host_mode_run_bit_for_bit():
    from paper_2105_08026_b200 import sharded
    _, a, inp = make_pair(B.M_THINNED_SCHECHTER1D, 3000, seed=9, theta_mode=B.THETA_HOST, max_trace_rows=60, want_oracle=False)
    _, b, _ = make_pair(B.M_THINNED_SCHECHTER1D, 3000, seed=9, theta_mode=B.THETA_HOST, max_trace_rows=60, want_oracle=False,
                        inputs=inp)
    a.run(60, 0, 1, sync=True)
    sharded.LocalShards([b]).run(60, 0, 1)
    sa, sb = a.get_state(), b.get_state()
    for k in ("chi", "L", "theta", "L_theta"):
        assert np.array_equal(sa[k], sb[k]), k
    assert np.array_equal(a.get_theta_trace(), b.get_theta_trace())
    # device-tail handles refuse the call: sharded stepping is defined for THETA_HOST
    _, c, _ = make_pair(B.M_NORMAL1D, 100, seed=1, want_oracle=False)
    with pytest.raises(B.CudahmError):
        c.shard_sweep()


def test_bench_sharded_leg_runs():
    """`bench.py --sharded` (one shard on this box): the JSON line carries the metric, a positive rate and the launch
    count of a host-driven loop (two kernels per iteration)."""
    import json, os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--sharded", "--config", "C0", "--steps", "40",
                          "--warmup", "10"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["metric"] == "plate_ram_updates_per_s" and line["value"] > 0 and line["n_gpus"] == 1
    assert line["gpu_launches"] == 80 and line["config"]["theta_mode"] == "host"
    assert 0.2 < line["accept"]["chi"] < 0.7


def test_theta_modes_agree():
    """Same grid, same thread->object map, same reduction order in the three streaming drivers.  GRAPH and the
    plain-load streaming DEVICE_TAIL kernel run the theta step with the same device code => identical bits.  HOST
    runs it with the host libm (exp, pow, sincos differ from the device's by ulps); the on-chip kernel
    (resident.cuh) and the TMA-staged streaming kernel (stream_tma.cuh) own objects in other fixed orders: they
    agree to rounding, not bitwise."""
    out = []
    for mode, flags in ((B.THETA_HOST, 0), (B.THETA_GRAPH, 0),
                        (B.THETA_DEVICE_TAIL, B.FLAG_STREAMING_ONLY),
                        (B.THETA_DEVICE_TAIL, 0), (B.THETA_DEVICE_TAIL, B.FLAG_STREAMING_ONLY | B.FLAG_TMA_STAGING)):
        _, gpu, _ = make_pair(B.M_THINNED_SCHECHTER1D, 5000, seed=5, theta_mode=mode, max_trace_rows=130,
                              want_oracle=False, flags=flags)
        gpu.run(130, 0, 1, sync=True)
        s = gpu.get_state()
        out.append((s["chi"], s["L"], s["theta"], s["L_theta"], gpu.get_theta_trace()))
    for a, b in zip(out[1], out[2]):
        assert np.array_equal(a, b)
    for other in (out[0], out[3], out[4]):
        for a, b in zip(other, out[2]):
            np.testing.assert_allclose(a, b, rtol=1e-9, atol=1e-10)


@pytest.mark.parametrize("flags", [B.FLAG_STREAMING_ONLY | B.FLAG_TMA_STAGING, B.FLAG_STREAMING_ONLY], ids=["tma", "ldg"])
@pytest.mark.parametrize("model,astar,n", [(B.M_NORMAL1D, 0.44, 1000), (B.M_THINNED_SCHECHTER1D, 0.44, 3000),
                                             (B.M_LINREG_ME1D, 0.44, 150001), (B.M_BB1_FLUXNOISE1D, 0.44, 3000),
                                             (B.M_NORMAL3D_KNOWNCOV, 0.234, 2001)],
                         ids=["M0", "M1", "M3", "M4", "M5"])
def test_streaming_persistent_kernel_matches_oracle(model, astar, n, flags):
    """The HBM-streaming persistent kernel (what C3 / C4 and any population too large for shared memory run),
    forced on the small fp64 p=1 cases that would otherwise take the on-chip kernel."""
    iters, burn, thin = 100, 20, 5
    orc, gpu, _ = make_pair(model, n, seed=41 + model, astar=astar, keep_moments=True, precision=B.F64,
                            max_trace_rows=(iters - burn) // thin, flags=flags)
    orc.run(iters, burn, thin)
    gpu.run(iters, burn, thin, sync=True)
    so, sg = orc.get_state(), gpu.get_state()
    np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-8, atol=1e-8)
    np.testing.assert_allclose(sg["chi"], so["chi"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["L"], so["L"], rtol=1e-9)
    mo, vo, ko = orc.get_chi_moments()
    mg, vg, kg = gpu.get_chi_moments()
    assert kg == ko
    np.testing.assert_allclose(mg, mo, rtol=1e-10, atol=1e-10)
    stg, sto = gpu.get_stats(), orc.get_stats()
    assert stg["chi_accepts"] == sto["chi_accepts"] and stg["theta_accepts"] == sto["theta_accepts"]
    assert stg["block_threads"] != 640


@pytest.mark.parametrize("model,astar,n,precision", [(B.M_THINNED_SCHECHTER1D, 0.44, 200001, B.F64),
                                                       (B.M_BINORMAL2D, 0.234, 200001, B.F64),
                                                       (B.M_LINREG_ME1D, 0.44, 400003, B.F32_STATE_F64_REDUCE),
                                                       (B.M_NORMAL3D_KNOWNCOV, 0.234, 160001, B.F64)],
                         ids=["M1", "M2", "M3f32", "M5"])
@pytest.mark.parametrize("block", [256, 512, 1024])
def test_staged_draws_and_prefetch_do_not_change_the_chain(model, astar, n, precision, block):
    """k_persistent<AHEAD>: plate draws of the next iteration staged in shared memory during the exchange, next step's
    columns prefetched into L2.  Whatever the number of staged steps (none, some, more than the sweep has), with or
    without prefetch, the chain is the plain kernel's bit for bit; the plain kernel is checked against the oracle."""
    iters, burn, thin = 40, 10, 5
    n = n * (block // 256)                      # at least three steps per thread at every block size
    if block == 1024 and model == B.M_NORMAL3D_KNOWNCOV:
        pytest.skip("p = 3 at 64 registers per thread: not a configuration anything selects")
    variants = [B.flag_stage_steps(0) | B.FLAG_PREFETCH_OFF, B.flag_stage_steps(0) | B.FLAG_PREFETCH_ON,
                B.flag_stage_steps(1) | B.FLAG_PREFETCH_OFF, B.flag_stage_steps(2) | B.FLAG_PREFETCH_ON,
                B.flag_stage_steps(9) | B.FLAG_PREFETCH_ON, 0]
    ref, inp, orc = None, None, None
    for k, fl in enumerate(variants):
        o, gpu, inp = make_pair(model, n, seed=77 + model, astar=astar, keep_moments=True, precision=precision,
                                max_trace_rows=(iters - burn) // thin, flags=fl | B.FLAG_STREAMING_ONLY,
                                block_threads=block, blocks_per_sm=1, inputs=inp, want_oracle=(k == 0 and block == 256))
        gpu.run(iters, burn, thin, sync=True)
        st, tr, mom = gpu.get_state(), gpu.get_theta_trace(), gpu.get_chi_moments()
        assert gpu.get_stats()["block_threads"] == block
        assert gpu.get_stats()["grid_blocks"] * block * (2 if precision == B.F64 else 4) * 2 < n   # at least 3 steps
        gpu.close()
        if k == 0:
            ref, orc = (st, tr, mom), o
        else:
            for key in ("chi", "L", "theta", "L_theta"):
                assert np.array_equal(ref[0][key], st[key]), (key, hex(fl))
            assert np.array_equal(ref[1], tr) and np.array_equal(ref[2][0], mom[0]) and np.array_equal(ref[2][1], mom[1])
    if precision == B.F64 and orc is not None:
        orc.run(iters, burn, thin)
        so = orc.get_state()
        np.testing.assert_allclose(ref[0]["chi"], so["chi"], rtol=1e-9, atol=1e-9)
        np.testing.assert_allclose(ref[1], orc.get_theta_trace(), rtol=1e-8, atol=1e-8)


def test_resume_is_bit_exact():
    """Counter-based streams: run(70) + run(50) == run(120), and get_state/set_state round-trips."""
    _, g1, inp = make_pair(B.M_BINORMAL2D, 3000, seed=8, astar=0.234, max_trace_rows=120, want_oracle=False)
    g1.run(120, 0, 1, sync=True)
    _, g2, _ = make_pair(B.M_BINORMAL2D, 3000, seed=8, astar=0.234, max_trace_rows=120, inputs=inp, want_oracle=False)
    g2.run(70, 0, 1)
    g2.run(50, 0, 1, sync=True)
    s1, s2 = g1.get_state(), g2.get_state()
    for k in ("chi", "L", "theta", "L_theta"):
        assert np.array_equal(s1[k], s2[k]), k
    assert np.array_equal(g1.get_theta_trace(), g2.get_theta_trace())
    _, g3, _ = make_pair(B.M_BINORMAL2D, 3000, seed=8, astar=0.234, max_trace_rows=120, inputs=inp, want_oracle=False)
    g3.run(70, 0, 1, sync=True)
    mid = g3.get_state()
    _, g4, _ = make_pair(B.M_BINORMAL2D, 3000, seed=8, astar=0.234, max_trace_rows=120, inputs=inp, want_oracle=False)
    g4.set_state(mid["chi"], mid["L"], mid["theta"], mid["L_theta"], mid["t"])
    g4.run(50, 0, 1, sync=True)
    s4 = g4.get_state()
    for k in ("chi", "L", "theta", "L_theta"):
        assert np.array_equal(s1[k], s4[k]), k


@pytest.mark.parametrize("n", [0, 1, 2, 3, 31, 33, 1023, 1025])
@pytest.mark.parametrize("precision", [B.F64, B.F32_STATE_F64_REDUCE], ids=["f64", "f32"])
def test_ragged_and_degenerate_sizes(n, precision):
    """Empty, single-object and ragged-tail populations (vector tails, partial warps)."""
    orc, gpu, inp = make_pair(B.M_NORMAL1D, n, seed=3, precision=precision, astar=0.44, max_trace_rows=16)
    if n > 0:
        st = sync_gpu_to_oracle(orc, gpu)
        to, tg = orc.step(taps=True), gpu.debug_step()
        compare_step(to, tg, precision, st, what=f"N={n}", ctx=dict(model=B.M_NORMAL1D, inputs=inp, astar=0.44))
        sync_gpu_to_oracle(orc, gpu)
    gpu.run(8, 0, 1, sync=True)
    orc.run(8, 0, 1)
    if precision == B.F64:
        np.testing.assert_allclose(gpu.get_theta_trace()[-8:], orc.get_theta_trace()[-8:], rtol=1e-9, atol=1e-9)
    assert gpu.get_stats()["iterations"] == orc.get_stats()["iterations"]


@pytest.mark.parametrize("model", [B.M_NORMAL3D_KNOWNCOV, B.M_NORMAL4D_KNOWNCOV, B.M_NORMAL5D_KNOWNCOV, B.M_NORMAL6D_KNOWNCOV],
                         ids=["p3", "p4", "p5", "p6"])
@pytest.mark.parametrize("n", [1, 2, 3, 5, 63, 65, 513])
def test_ragged_sizes_p3(n, model):
    """The p >= 3 path (general rank-one update, ceil(p/2) Box-Muller pairs per object) on ragged and tiny populations."""
    orc, gpu, inp = make_pair(model, n, seed=4, astar=0.234, max_trace_rows=16)
    st = sync_gpu_to_oracle(orc, gpu)
    to, tg = orc.step(taps=True), gpu.debug_step()
    compare_step(to, tg, B.F64, st, what=f"N={n}", ctx=dict(model=model, inputs=inp, astar=0.234))
    sync_gpu_to_oracle(orc, gpu)
    gpu.run(8, 0, 1, sync=True)
    orc.run(8, 0, 1)
    np.testing.assert_allclose(gpu.get_theta_trace()[-8:], orc.get_theta_trace()[-8:], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(gpu.get_state()["L"], orc.get_state()["L"], rtol=1e-9, atol=1e-12)


def test_frozen_theta_conjugate_conditional():
    """theta frozen: chi_i | theta, y_i ~ N((y/s^2 + mu/tau^2) v, v), v = 1/(1/s^2 + 1/tau^2) (closed form, P6):
    the on-device moments must land on it, and the RAM scale on 2.4176 sd (P5)."""
    from paper_2105_08026_b200 import synth
    n, iters, burn = 4096, 6000, 1000
    inp = synth.make_normal1d(n, 17)
    th = np.array([0.1, np.log(0.8)])
    _, gpu, _ = make_pair(B.M_NORMAL1D, n, seed=17, astar=0.44, inputs=inp, theta0=th, keep_moments=True,
                          freeze_theta=True, want_oracle=False)
    gpu.run(iters, burn, 1, sync=True)
    y, s = inp["cols"]
    tau2 = np.exp(2 * th[1])
    v = 1.0 / (1.0 / s ** 2 + 1.0 / tau2)
    m = (y / s ** 2 + th[0] / tau2) * v
    mean, var, k = gpu.get_chi_moments()
    assert k == iters - burn
    zs = (mean[0] - m) / np.sqrt(v)
    # ESS ~ k/4.5 for a tuned 1-D random-walk Metropolis: sd of the mean ~ 0.03 sd units
    assert np.abs(zs).max() < 0.2 and abs(zs.mean()) < 0.005
    assert abs(np.mean(var[0] / v) - 1.0) < 0.02
    L = gpu.get_state()["L"][0]
    assert abs(np.mean(L / np.sqrt(v)) - 2.41758) < 0.06
    st = gpu.get_stats()
    assert abs(st["chi_accepts"] / st["chi_proposals"] - 0.44) < 0.01


def test_config0_posterior_against_oracle_and_closed_form():
    """BASELINE config 0 as stated (N=1000, 2000 iterations, 500 burn-in, seed 0): GPU and oracle theta
    posteriors agree within 4 MCSE (they are in fact the same chain to rounding)."""
    from mcmc_util import mean_and_var_with_mcse
    from paper_2105_08026_b200 import synth
    c = synth.CONFIGS["C0"]
    inp = synth.make_inputs("C0")
    orc, gpu, _ = make_pair(c.model, c.n_objects, seed=c.seed, astar=c.target_accept_chi, inputs=inp,
                            keep_moments=True, max_trace_rows=c.n_iter - c.burn_in)
    orc.run(c.n_iter, c.burn_in, c.thin)
    gpu.run(c.n_iter, c.burn_in, c.thin, sync=True)
    tg, to = gpu.get_theta_trace(), orc.get_theta_trace()
    assert tg.shape == to.shape == (1500, 2)
    mg, seg, vg, sevg = mean_and_var_with_mcse(tg)
    mo, seo, vo, sevo = mean_and_var_with_mcse(to)
    assert np.all(np.abs(mg - mo) <= 4 * np.hypot(seg, seo))
    assert np.all(np.abs(vg - vo) <= 4 * np.hypot(sevg, sevo))
    # closed form: mu | tau, y ~ N(sum w y / sum w, 1/sum w), w = 1/(sigma^2 + tau^2), at the posterior-mean tau
    y, s = inp["cols"]
    w = 1.0 / (s ** 2 + np.exp(2 * mg[1]))
    assert abs(mg[0] - (w * y).sum() / w.sum()) <= 4 * seg[0] + 0.01


def test_two_on_chip_handles_of_one_model_with_different_sizes():
    """cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the function, not the handle: creating a SMALL handle of
    the same model after a LARGE one must not lower the large one's limit (both run the on-chip kernel)."""
    _, big, inp_b = make_pair(B.M_THINNED_SCHECHTER1D, 120_000, seed=3, want_oracle=False, max_trace_rows=8)
    _, small, _ = make_pair(B.M_THINNED_SCHECHTER1D, 2_000, seed=4, want_oracle=False, max_trace_rows=8)
    assert big.get_stats()["block_threads"] == small.get_stats()["block_threads"] == 640
    small.run(4, 0, 1, sync=True)
    big.run(4, 0, 1, sync=True)            # launches with the larger shared-memory request after the small handle's
    small.run(4, 0, 1, sync=True)
    _, ref, _ = make_pair(B.M_THINNED_SCHECHTER1D, 120_000, seed=3, want_oracle=False, max_trace_rows=8, inputs=inp_b)
    ref.run(4, 0, 1, sync=True)
    assert np.array_equal(ref.get_state()["chi"], big.get_state()["chi"])
    assert big.get_stats()["iterations"] == 4 and small.get_stats()["iterations"] == 8


def test_graph_cache_is_dropped_when_the_model_constants_change():
    """THETA_GRAPH caches an executable graph whose nodes hold the model constants by value: set_model_consts on a live
    handle (then set_init and a run long enough to replay the graph) must give the chain of a fresh handle."""
    from paper_2105_08026_b200 import synth
    n, iters = 3000, 120
    inp = synth.make_normal3d_knowncov(n, 5)
    consts2 = inp["consts"].copy()
    consts2[:3] *= 1.5                                       # other measurement errors: another target
    _, a, _ = make_pair(B.M_NORMAL3D_KNOWNCOV, n, seed=5, astar=0.234, theta_mode=B.THETA_GRAPH, inputs=inp,
                        max_trace_rows=iters, want_oracle=False)
    a.run(iters, 0, 1, sync=True)                            # graph captured with the first constants
    a.set_model_consts(consts2)
    a.set_init(inp["theta0"])
    a.run(iters, 0, 1, sync=True)
    inp2 = dict(inp, consts=consts2)
    _, b, _ = make_pair(B.M_NORMAL3D_KNOWNCOV, n, seed=5, astar=0.234, theta_mode=B.THETA_GRAPH, inputs=inp2,
                        max_trace_rows=iters, want_oracle=False)
    b.run(iters, 0, 1, sync=True)
    assert np.array_equal(a.get_theta_trace(), b.get_theta_trace())
    assert np.array_equal(a.get_state()["chi"], b.get_state()["chi"])


def test_theta0_outside_the_prior_support_is_refused():
    _, g, inp = make_pair(B.M_NORMAL1D, 100, seed=1, want_oracle=False)
    with pytest.raises(B.CudahmError) as e:
        g.set_init(np.array([0.0, 50.0]))                    # |log tau| <= 10 is the prior box
    assert e.value.code == B.E_NONFINITE
    g.set_init(inp["theta0"])
    g.run(3, 0, 1, sync=True)


@pytest.mark.parametrize("mode", [B.THETA_HOST, B.THETA_GRAPH, B.THETA_DEVICE_TAIL], ids=["host", "graph", "tail"])
@pytest.mark.parametrize("model,astar,n,precision", [(B.M_NORMAL1D, 0.44, 3001, B.F64), (B.M_BINORMAL2D, 0.234, 2501, B.F64),
                                                       (B.M_LINREG_ME1D, 0.44, 4099, B.F32_STATE_F64_REDUCE)],
                         ids=["M0", "M2", "M3f32"])
def test_update_mask_and_per_object_counter_match_oracle(model, astar, n, precision, mode):
    """Frozen members: a third of the objects held fixed for 60 iterations, then
    released (their own update counts lag, so their eta_n is larger), 60 more; free-running against the oracle in every theta
    driver.  Held objects keep chi and L bit for bit, stay in the population sums, and consume no proposals."""
    K1, K2, burn, thin = 60, 60, 20, 5
    orc, gpu, inp = make_pair(model, n, seed=91 + model, astar=astar, precision=precision, theta_mode=mode, keep_moments=True,
                              max_trace_rows=(K1 + K2 - burn) // thin, update_mask=True, per_object_counter=True)
    mask = (np.arange(n) % 3 != 1).astype(np.uint8)
    held = mask == 0
    s0 = gpu.get_state()
    orc.set_update_mask(mask)
    gpu.set_update_mask(mask)
    if precision == B.F64:
        orc.run(K1, burn, thin)
        gpu.run(K1, burn, thin, sync=True)
    else:                               # fp32: lock-step from the oracle's state (near-tie flips are expected, see C4)
        for _ in range(K1):
            st = sync_gpu_to_oracle(orc, gpu)
            orc.set_counters(orc.get_counters()); gpu.set_counters(orc.get_counters())
            orc.run(1, burn, thin); gpu.run(1, burn, thin, sync=True)
    s1, o1 = gpu.get_state(), orc.get_state()
    assert np.array_equal(s1["chi"][:, held], s0["chi"][:, held]) and np.array_equal(s1["L"][:, held], s0["L"][:, held])
    assert np.array_equal(gpu.get_counters(), orc.get_counters())
    assert np.array_equal(gpu.get_counters(), np.where(held, 0, K1).astype(np.uint32))
    if precision == B.F64:
        np.testing.assert_allclose(s1["chi"], o1["chi"], rtol=1e-9, atol=1e-9)
        np.testing.assert_allclose(s1["L"], o1["L"], rtol=1e-9)
        assert gpu.get_stats()["chi_proposals"] == orc.get_stats()["chi_proposals"] == K1 * int(mask.sum())
        assert gpu.get_stats()["chi_accepts"] == orc.get_stats()["chi_accepts"]
    # a tapped step with the mask on: held objects report the documented taps and stay in S and Delta
    st = sync_gpu_to_oracle(orc, gpu)
    gpu.set_counters(orc.get_counters())
    to, tg = orc.step(NO_TRACE, 1, taps=True), gpu.debug_step(NO_TRACE, 1)
    for k in ("chi_prop", "L_new"):
        assert np.array_equal(tg[k][:, held], st[k.replace("chi_prop", "chi").replace("L_new", "L")][:, held])
    assert np.all(tg["alpha"][held] == 0) and np.all(tg["u"][held] == 1) and np.all(tg["accepted"][held] == 0)
    assert np.array_equal(tg["pi_prop"][held], tg["pi_cur"][held])
    tol = 1e-12 if precision == B.F64 else 1e-5
    assert np.all(np.abs(tg["a"][held] - to["a"][held]) <= 1e-12 * np.maximum(1.0, np.abs(to["a"][held])))
    assert np.array_equal(tg["u"][~held], to["u"][~held])
    assert np.all(np.abs(tg["pi_cur"] - to["pi_cur"]) <= tol * np.maximum(1.0, np.abs(to["pi_cur"])))
    import math
    assert abs(tg["S"] - math.fsum(tg["a"])) <= 1e-10 * max(1.0, abs(tg["S"]))
    # release: the held objects now adapt with eta from their OWN count (1 -> n = 2 ...), the others with theirs
    sync_gpu_to_oracle(orc, gpu)
    gpu.set_counters(orc.get_counters())
    orc.set_update_mask(None); gpu.set_update_mask(None)
    if precision == B.F64:
        orc.run(K2 - 1, burn, thin)
        gpu.run(K2 - 1, burn, thin, sync=True)
        s2, o2 = gpu.get_state(), orc.get_state()
        np.testing.assert_allclose(s2["chi"], o2["chi"], rtol=1e-9, atol=1e-9)
        np.testing.assert_allclose(s2["L"], o2["L"], rtol=1e-9)
        np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-8, atol=1e-8)
        mo, _, ko = orc.get_chi_moments()
        mg, _, kg = gpu.get_chi_moments()
        assert kg == ko
        np.testing.assert_allclose(mg, mo, rtol=1e-10, atol=1e-10)
    else:
        orc.run(1, burn, thin); gpu.run(1, burn, thin, sync=True)
        s2, o2 = gpu.get_state(), orc.get_state()
        same = np.abs(s2["chi"][0] - o2["chi"][0]) <= 2e-5 * np.maximum(1.0, np.abs(o2["chi"][0]))
        assert (~same).sum() <= 3
        np.testing.assert_allclose(s2["L"][0][same], o2["L"][0][same], rtol=2e-5)
    assert np.array_equal(gpu.get_counters(), orc.get_counters())
    assert np.all(s2["L"][:, held] != s1["L"][:, held])
    assert gpu.get_stats()["block_threads"] != 640


def test_mask_calls_need_the_config_switches():
    _, g, _ = make_pair(B.M_NORMAL1D, 100, seed=1, want_oracle=False)
    with pytest.raises(B.CudahmError) as e:
        g.set_update_mask(np.ones(100, np.uint8))
    assert e.value.code == B.E_STATE
    with pytest.raises(B.CudahmError):
        g.get_counters()
    # an all-ones mask + counter on the HOLD kernels is the plain chain bit for bit
    _, a, inp = make_pair(B.M_BINORMAL2D, 3000, seed=8, astar=0.234, max_trace_rows=50, want_oracle=False, flags=B.FLAG_STREAMING_ONLY)
    _, b, _ = make_pair(B.M_BINORMAL2D, 3000, seed=8, astar=0.234, max_trace_rows=60, want_oracle=False, inputs=inp,
                        update_mask=True, per_object_counter=True)
    a.run(50, 0, 1, sync=True); b.run(50, 0, 1, sync=True)
    for k in ("chi", "L", "theta", "L_theta"):
        assert np.array_equal(a.get_state()[k], b.get_state()[k]), k
    assert np.array_equal(a.get_theta_trace(), b.get_theta_trace())
    mask_dev = __import__("torch").ones(3000, dtype=__import__("torch").uint8, device="cuda")
    mask_dev[::2] = 0
    b.set_update_mask(mask_dev)
    b.run(3, 0, 1, sync=True)
    assert b.get_stats()["chi_proposals"] == 50 * 3000 + 3 * 1500


@pytest.mark.parametrize("model,precision,astar,n", [(B.M_BINORMAL2D, B.F64, 0.234, 150_001), (B.M_NORMAL3D_KNOWNCOV, B.F64, 0.234, 30_000),
                                                       (B.M_NORMAL6D_KNOWNCOV, B.F64, 0.234, 9_001),
                                                       (B.M_LINREG_ME1D, B.F32_STATE_F64_REDUCE, 0.44, 400_003)],
                         ids=["M2", "M5", "p6", "M3f32"])
def test_general_on_chip_kernel_is_the_streaming_chain(model, precision, astar, n):
    """resident_gen.cuh keeps p >= 2 and fp32 populations in shared memory and runs update_vec itself from there: per object
    the same arithmetic as the streaming kernel, so chi / L / moments agree to the rounding of the (differently ordered)
    population sums, over several slots per thread and a ragged tail."""
    iters, burn, thin = 60, 10, 5
    out, inp = [], None
    for flags in (0, B.FLAG_STREAMING_ONLY):
        _, g, inp = make_pair(model, n, seed=55 + model, precision=precision, astar=astar, keep_moments=True,
                              max_trace_rows=(iters - burn) // thin, want_oracle=False, flags=flags, inputs=inp)
        g.run(iters, burn, thin, sync=True)
        st = g.get_state()
        out.append((st["chi"], st["L"], g.get_theta_trace(), g.get_chi_moments()[0], g.get_stats()))
        g.close()
    assert out[0][4]["block_threads"] == 384 and out[1][4]["block_threads"] != 384
    if precision == B.F64:
        np.testing.assert_allclose(out[0][2], out[1][2], rtol=1e-9, atol=1e-10)
        np.testing.assert_allclose(out[0][0], out[1][0], rtol=1e-9, atol=1e-10)
        np.testing.assert_allclose(out[0][1], out[1][1], rtol=1e-9, atol=1e-12)
        np.testing.assert_allclose(out[0][3], out[1][3], rtol=1e-10, atol=1e-10)
        assert out[0][4]["chi_accepts"] == out[1][4]["chi_accepts"]
    else:      # fp32: theta differs by the rounding of the sums, which flips a few near-tie decisions over 60 iterations
        np.testing.assert_allclose(out[0][2], out[1][2], rtol=1e-4, atol=1e-4)
        assert abs(out[0][4]["chi_accepts"] - out[1][4]["chi_accepts"]) <= 1e-4 * iters * n


@pytest.mark.parametrize("mode", [B.THETA_HOST, B.THETA_DEVICE_TAIL], ids=["host", "device"])
def test_m4_proposal_with_vanishing_selection_integral_is_rejected(mode):
    """DESIGN.md reading R26 on the GPU, device tail (k_tail through debug_step) and host tail (THETA_HOST run): a theta'
    inside the prior box whose selection sum underflows to 0 is rejected, as in the oracle -- not accepted on -N log 0."""
    n = 60
    orc, gpu, inp = make_pair(B.M_BB1_FLUXNOISE1D, n, seed=43, theta_mode=mode, max_trace_rows=0)
    st = orc.get_state()
    theta = np.array([st["theta"][0], -29.0, st["theta"][2]])
    chol = np.array([1e-3, 0.0, 1e-3, 0.0, 0.0, 12.0])
    hit = 0
    for t in range(400):
        orc.set_state(st["chi"], st["L"], theta, chol, t)
        gpu.set_state(st["chi"], st["L"], theta, chol, t)
        to = orc.step(NO_TRACE, 1, taps=True)
        if mode == B.THETA_HOST:
            gpu.run(1, NO_TRACE, 1, sync=True)
            acc_g = int(not np.array_equal(gpu.get_state()["theta"], theta))
        else:
            tg = gpu.debug_step(NO_TRACE, 1)
            acc_g = tg["accepted_theta"]
            np.testing.assert_allclose(tg["theta_prop"], to["theta_prop"], rtol=1e-9, atol=1e-9)
        if np.isfinite(to["lp_prop"]) and to["theta_prop"][2] < -21.0:
            assert to["accepted_theta"] == 0 and acc_g == 0
            hit += 1
        elif abs(to["log_r"]) > 1e-6 or not np.isfinite(to["log_r"]):
            assert acc_g == to["accepted_theta"]
    assert hit >= 5, hit


@pytest.mark.parametrize("mode", [B.THETA_HOST, B.THETA_GRAPH, B.THETA_DEVICE_TAIL], ids=["host", "graph", "tail"])
def test_trace_and_moment_counts_across_split_runs_crossing_burn_in(mode):
    """cudahm_run checks the trace capacity from HOST mirrors of the row and moment counts (no device read-back before the
    launch): split runs that cross burn-in with thinning, a zero-length run and a tapped step in between must leave the
    same counts, trace and moments as the oracle; a run that would overflow the trace is refused with nothing launched."""
    n, burn, thin = 1500, 20, 7
    chunks = [7, 1, 13, 0, 29, 50]                      # 100 iterations: rows at t = 27, 34, ..., 97 -> 11
    rows_total = (sum(chunks) + 1 - burn) // thin        # + 1: the tapped step below
    orc, gpu, _ = make_pair(B.M_NORMAL1D, n, seed=61, theta_mode=mode, keep_moments=True, max_trace_rows=rows_total)
    done = 0
    for k, c in enumerate(chunks):
        orc.run(c, burn, thin)
        gpu.run(c, burn, thin, sync=True)
        done += c
        if k == 2:                                       # a tapped step through the other kernels, in between
            orc.step(burn, thin)
            gpu.debug_step(burn, thin)
            done += 1
        sg, so = gpu.get_stats(), orc.get_stats()
        for key in ("iterations", "trace_rows", "moment_samples"):
            assert sg[key] == so[key], (key, k)
        assert sg["trace_rows"] == max(0, (done - burn) // thin) and sg["moment_samples"] == max(0, done - burn)
    assert gpu.get_theta_trace().shape == (rows_total, 2)
    np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-8, atol=1e-8)
    mg, vg, kg = gpu.get_chi_moments()
    mo, vo, ko = orc.get_chi_moments()
    assert kg == ko == done - burn
    np.testing.assert_allclose(mg, mo, rtol=1e-10, atol=1e-10)
    before = gpu.get_state()
    with pytest.raises(B.CudahmError) as e:              # 7 more iterations would add a 12th row
        gpu.run(7, burn, thin)
    assert e.value.code == B.E_INVALID and "trace" in str(e.value)
    after = gpu.get_state()
    assert after["t"] == before["t"] and np.array_equal(after["chi"], before["chi"])
    gpu.run(2, burn, thin, sync=True)                    # still room for iterations that add no row (t = 103 < 104)
    assert gpu.get_stats()["trace_rows"] == rows_total


@pytest.mark.parametrize("n", [150_529, 200_001])
def test_dedicated_tail_kernel_at_its_smallest_populations(n):
    """k_persistent_dt (M2, default block size, streaming forced) at the smallest population cudahm_create gives it (below
    150,529 objects -- fewer than 148 blocks of 512 x 2 -- the default block is 256 threads and the plain kernel runs) and with a ragged second step: the one-off wait
    for theta' is a block barrier inside the update and must be reached warp-uniformly.  Free-running against the oracle."""
    iters, burn, thin = 30, 10, 5
    orc, gpu, _ = make_pair(B.M_BINORMAL2D, n, seed=47, astar=0.234, keep_moments=True, max_trace_rows=(iters - burn) // thin,
                            flags=B.FLAG_STREAMING_ONLY)
    assert gpu.get_stats()["dedicated_tail"] == 1
    _, small, _ = make_pair(B.M_BINORMAL2D, n - 2, seed=47, astar=0.234, want_oracle=False, flags=B.FLAG_STREAMING_ONLY)
    assert small.get_stats()["dedicated_tail"] == (1 if n - 2 >= 150_529 else 0)
    orc.run(iters, burn, thin)
    gpu.run(iters, burn, thin, sync=True)
    so, sg = orc.get_state(), gpu.get_state()
    np.testing.assert_allclose(gpu.get_theta_trace(), orc.get_theta_trace(), rtol=1e-8, atol=1e-8)
    np.testing.assert_allclose(sg["chi"], so["chi"], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(sg["L"], so["L"], rtol=1e-9, atol=1e-12)
    assert gpu.get_stats()["chi_accepts"] == orc.get_stats()["chi_accepts"]


@pytest.mark.parametrize("model,precision,n,streaming", [
    (B.M_LINREG_ME1D, B.F32_STATE_F64_REDUCE, 400_001, True),     # fp32 streaming kernel, three ragged steps per thread
    (B.M_LINREG_ME1D, B.F32_STATE_F64_REDUCE, 50_001, False),     # fp32 state in the general on-chip kernel
    (B.M_NORMAL1D, B.F32_STATE_F64_REDUCE, 400_001, True),
    (B.M_BINORMAL2D, B.F64, 200_001, True),                       # fp64 streaming kernel (update inside the per-object loop)
], ids=["M3f32-stream", "M3f32-onchip", "M0f32-stream", "M2f64-stream"])
def test_moments_are_the_welford_moments_of_the_gpu_chain(model, precision, n, streaming):
    """The running chi moments against the definition (PAPER.md:337-341 reports posterior means and standard deviations of
    the member properties; Welford: mean_k = mean_{k-1} + (x - mean_{k-1}) / k, M2 += (x - mean_{k-1})(x - mean_k)),
    recomputed on the host in fp64 from the chi the GPU chain itself visits -- one iteration per call, chi read back after
    each.  Independent of fp32 near-tie decisions (the chain is the GPU's own), so it pins the accumulation exactly:
    the fp32 kernels update the moments after the per-object loop (kernels.cuh, MomentsAfterLoop), the fp64 ones inside."""
    burn, post = 3, 9
    _, gpu, _ = make_pair(model, n, seed=123 + model, precision=precision, astar=0.44 if model != B.M_BINORMAL2D else 0.234,
                          keep_moments=True, want_oracle=False, flags=B.FLAG_STREAMING_ONLY if streaming else 0,
                          block_threads=256 if streaming else 0, blocks_per_sm=1 if streaming else 0)
    p = gpu.p
    mean, m2 = np.zeros((p, n)), np.zeros((p, n))
    for t in range(1, burn + post + 1):
        gpu.run(1, burn, 1, sync=True)
        if t > burn:
            x = gpu.get_state()["chi"]                 # float64 view of the (fp32 or fp64) state: exact
            k = t - burn
            d = x - mean
            mean = mean + d * (1.0 / k)
            m2 = m2 + d * (x - mean)
    st = gpu.get_stats()
    assert st["block_threads"] == (256 if streaming else 384)
    mg, vg, kg = gpu.get_chi_moments()
    assert kg == post
    # a fused multiply-add on the device against two roundings here: a few ulp of the mean, relative to the spread for M2
    np.testing.assert_allclose(mg, mean, rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(vg, m2 / (post - 1), rtol=1e-11, atol=1e-14)
    assert (vg > 0).mean() > 0.1                       # objects moved (p = 2 accepts few proposals this early): not a 0 = 0 check
