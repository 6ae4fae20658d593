"""Small runs of every kernel variant, meant to be executed under compute-sanitizer on a GPU box:

    compute-sanitizer --tool memcheck  python tests/sanitizer_smoke.py
    compute-sanitizer --tool racecheck python tests/sanitizer_smoke.py

(one tool per call; see profiles/r01e_sanitizer.md for the recorded outcome).  Not collected by pytest."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2105_08026_b200 import binding as B  # noqa: E402
from paper_2105_08026_b200 import synth  # noqa: E402


def run(model, n, precision=B.F64, theta_mode=B.THETA_DEVICE_TAIL, flags=0, iters=6, astar=0.44):
    maker = {0: synth.make_normal1d, 1: synth.make_thinned_schechter1d, 2: synth.make_binormal2d,
             3: synth.make_linreg_me1d, 4: synth.make_bb1_fluxnoise1d, 5: synth.make_normal3d_knowncov}[model]
    kw = {}
    if model == 3:
        kw = dict(fp32=(precision != B.F64))
    if model == 0 and precision != B.F64:
        kw = dict(fp32=True)
    inp = maker(n, 5, **kw)
    s = B.Sampler(model, n, seed=5, precision=precision, theta_mode=theta_mode, target_accept_chi=astar,
                  keep_chi_moments=True, max_trace_rows=iters + 1, flags=flags)
    s.set_data(inp["cols"])
    if inp["consts"] is not None:
        s.set_model_consts(inp["consts"])
    s.set_init(inp["theta0"])
    s.debug_step()
    s.run(iters, 1, 1, sync=True)
    st = s.get_stats()
    assert st["iterations"] == iters + 1 and np.isfinite(s.get_theta_trace()).all()
    s.get_chi_moments()
    s.close()
    print(f"ok model {model} n {n} precision {precision} mode {theta_mode} flags {flags}: grid "
          f"{st['grid_blocks']}x{st['block_threads']}", flush=True)


if __name__ == "__main__":
    run(B.M_THINNED_SCHECHTER1D, 2500)                                   # on-chip kernel, ragged last block
    run(B.M_NORMAL1D, 700)                                               # on-chip kernel, generic population terms
    run(B.M_THINNED_SCHECHTER1D, 2500, flags=B.FLAG_STREAMING_ONLY)      # streaming persistent kernel
    run(B.M_BINORMAL2D, 2100, astar=0.234)                               # streaming, p = 2
    run(B.M_LINREG_ME1D, 4100, precision=B.F32_STATE_F64_REDUCE)         # streaming, fp32 state
    run(B.M_BINORMAL2D, 2100, astar=0.234, flags=B.FLAG_TMA_STAGING)     # TMA-staged streaming kernel
    run(B.M_THINNED_SCHECHTER1D, 2500, theta_mode=B.THETA_GRAPH, iters=55)   # k_sweep + k_tail, graph replay
    run(B.M_NORMAL1D, 700, theta_mode=B.THETA_HOST)                      # host theta step
    run(B.M_BB1_FLUXNOISE1D, 1900)                                       # on-chip kernel, BB1 case-study model
    run(B.M_NORMAL3D_KNOWNCOV, 1500, astar=0.234)                        # streaming, p = 3 (general rank-one update)
