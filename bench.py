#!/usr/bin/env python
"""bench.py -- plate-level RAM updates/s and Gibbs iterations/s of the CUDA path.

A "step" is one Gibbs iteration = one pass of the whole hot path over all N objects
of the workload.  Default workload: BASELINE.json configs[2] (C2: thinned-Schechter model, N = 3e5, fp64,
chi moments on device, theta chain thinned by 10) -- the configuration BASELINE.json's metric is quoted on.
`--warmup W` iterations run untimed as burn-in, then EXACTLY `--steps K` post-burn-in iterations are timed with
CUDA events on the sampler's stream, bracketed by barrier + synchronize; rank 0 prints ONE JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C0..C6] [--theta-mode tail|graph|host]
    python bench.py --impl reference ...      # the CPU oracle, as it stands, on the same config / metric

Multi-GPU: the path does not shard without a per-iteration exchange (the theta step needs the global sum), and
BASELINE.json says one GPU only: `--gpus N` (under torchrun) runs N independent replicas (different seeds), no
data-path collective; value = all ranks' updates / max-over-ranks device time ("replicas only").
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2105_08026_b200 import synth  # noqa: E402  (seeded inputs only: no method arithmetic)

METRIC = "plate_ram_updates_per_s"
UNIT = "updates/s"
# algorithmic bytes per object per iteration: state read+write and
# data read; + running-moment read+write (fp64 mean and M2 per component) once past burn-in
ALG_BYTES = {"C0": (48, 32), "C1": (48, 32), "C2": (48, 32), "C3": (112, 64), "C4": (28, 32), "C5": (48, 32),
             "C6": (240, 96)}     # p = 3: chi 3 + L 6 doubles read and written, 3 data doubles read
MODES = {"host": 0, "graph": 1, "tail": 2}
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel PER LAUNCH of K iterations, as (bytes per launch that do
# not depend on K, bytes per iteration), from the committed `ncu --set full` captures under profiles/ (r02_*_ncu.md):
#   C2  on-chip kernel: 14.63 MB at K = 20 (the driver's launch) and 14.72 MB at K = 300 -- the state load; nothing per iteration
#   C3  streaming kernel (dedicated tail warps), 60 iterations: 220.1 MB = 3.7 MB per iteration (the 104 MB working set is
#       served from L2: hit rate 96 %; 3.7-5.6 MB per iteration from capture to capture)
#   C4  streaming kernel, 30 iterations: 8,335.9 MB = 277.9 MB per iteration (= the algorithmic 280 MB: nothing is re-read)
#   C6  general on-chip kernel, 300 iterations: 3.25 MB, taken as the per-launch state load
# A config without a capture reports traffic = null.
NCU_DRAM_BYTES = {"C2": (14.63e6, 0.0), "C3": (0.0, 220.09e6 / 60), "C4": (0.0, 8335.89e6 / 30), "C6": (3.25e6, 0.0)}
# warp-level instructions executed per 32 object-updates (smsp__inst_executed.sum / (N K / 32)) and fp64-pipe activity from
# the same captures.  They give the compute floor reported beside the HBM one: issue slots (4 warp-instructions / clk / SM).
NCU_WARP_INSTR_PER_32 = {"C2": (389, 37.6), "C3": (392, 42.3), "C4": (138, 12.0), "C6": (1223, 14.9)}
N_SMS, SM_CLOCK_HZ = 148, 1.965e9


def workload_label(name):
    if name == "C5":
        return "C5: the paper's own case study (PAPER.md section 5.3, Table 5.1: BB1 population, N = 1e5); not a BASELINE.json config"
    if name == "C6":
        return "C6: the paper's normal-normal benchmark (PAPER.md section 3: 3-vector latents, N = 3e4); not a BASELINE.json config"
    return f"{name}: BASELINE.json configs[{int(name[1])}]"


def config_entry(cfg_name, c, n, W):
    """`config` of the JSON line: the same keys in the CUDA arm and in the --impl reference arm."""
    return {"workload": workload_label(cfg_name), "n_objects": n, "burn_in": W, "thin": c.thin,
            "chi_moments": bool(c.keep_chi_moments),
            "model": ["normal1d", "thinned_schechter1d", "binormal2d", "linreg_me1d", "bb1_fluxnoise1d",
                      "normal3d_knowncov", "normalpd_knowncov"][c.model]}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8000)
    ap.add_argument("--warmup", type=int, default=2000)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", default="C2", choices=sorted(synth.CONFIGS))
    ap.add_argument("--theta-mode", default="tail", choices=sorted(MODES))
    ap.add_argument("--n-objects", type=int, default=0, help="override N (parity-size experiments)")
    ap.add_argument("--no-extras", action="store_true", help="skip cpu_baseline, floors and the side configs")
    ap.add_argument("--sharded", action="store_true",
                    help="ONE chain over a population of N objects PER GPU sharded by object range (SURVEY 8(e)): "
                         "all-gather of five doubles per rank and iteration; default for --gpus > 1 is independent replicas")
    ap.add_argument("--block-threads", type=int, default=0)
    ap.add_argument("--blocks-per-sm", type=int, default=0)
    ap.add_argument("--flags", type=int, default=0, help="cudahm_config.flags (CUDAHM_FLAG_*), for experiments")
    return ap.parse_args()


def load_peaks():
    """MEASURED_PEAKS.json (driver-written) or the profiling guide's stated fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons DURING the timed region (NVML; nvidia-smi as a fallback)."""

    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "hw_power_brake": 0x80}
    NOTE = {"sw_power_cap": 0x4}

    def __init__(self, index):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _once(self):
        if self.nv is not None:
            self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
            r = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)) if hasattr(
                self.nv, "nvmlDeviceGetCurrentClocksEventReasons") else int(
                self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            for name, bit in {**self.BAD, **self.NOTE}.items():
                if r & bit:
                    self.reasons.add(name)
        else:
            import subprocess
            out = subprocess.run(["nvidia-smi", f"--id={self.index}", "--query-gpu=clocks.sm,clocks.max.sm,"
                                  "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                                  "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap",
                                  "--format=csv,noheader,nounits"], capture_output=True, text=True).stdout
            f = [x.strip() for x in out.strip().split(",")]
            if len(f) >= 6:
                self.samples.append(float(f[0]))
                self.max_mhz = float(f[1])
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[2:6]):
                    if v.lower().startswith("active"):
                        self.reasons.add(name)

    def _loop(self):
        while not self._stop.is_set():
            try:
                self._once()
            except Exception:
                pass
            self._stop.wait(0.002 if self.nv is not None else 0.2)

    def start(self):
        self._thr = threading.Thread(target=self._loop, daemon=True)
        self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join()
        try:
            self._once()
        except Exception:
            pass
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ----------------------------------------------------------------------------------------------------------
def make_workload(cfg_name, n_override=0, seed_offset=0):
    c = synth.CONFIGS[cfg_name]
    n = n_override or c.n_objects
    if c.model == synth.M_NORMAL1D:
        inp = synth.make_normal1d(n, c.seed + seed_offset)
    elif c.model == synth.M_THINNED_SCHECHTER1D:
        inp = synth.make_thinned_schechter1d(n, c.seed + seed_offset)
    elif c.model == synth.M_BINORMAL2D:
        inp = synth.make_binormal2d(n, c.seed + seed_offset)
    elif c.model == synth.M_BB1_FLUXNOISE1D:
        inp = synth.make_bb1_fluxnoise1d(n, c.seed + seed_offset)
    elif c.model == synth.M_NORMAL3D_KNOWNCOV:
        inp = synth.make_normal3d_knowncov(n, c.seed + seed_offset)
    else:
        inp = synth.make_linreg_me1d(n, c.seed + seed_offset, fp32=(c.precision == synth.F32_STATE_F64_REDUCE))
    return c, n, inp


def make_gpu_sampler(c, n, inp, args, seed, max_trace_rows, device, cols=None):
    from paper_2105_08026_b200 import binding as B
    s = B.Sampler(c.model, n, device=device, seed=seed, precision=c.precision, theta_mode=MODES[args.theta_mode],
                  target_accept_chi=c.target_accept_chi, target_accept_theta=c.target_accept_theta,
                  keep_chi_moments=c.keep_chi_moments, max_trace_rows=max_trace_rows,
                  block_threads=args.block_threads, blocks_per_sm=args.blocks_per_sm, flags=getattr(args, "flags", 0))
    s.set_data(inp["cols"] if cols is None else cols)
    if inp["consts"] is not None:
        s.set_model_consts(inp["consts"])
    s.set_init(inp["theta0"], theta_chol0=make_theta_chol0(inp, n))
    return s


def trace_rows_needed(total_iters, burn_in, thin):
    return max(0, (total_iters - burn_in) // thin) + 1


REPEATS = 5     # best and median of 5


def make_theta_chol0(inp, n):
    """The theta proposal factor the workload recipe supplies; None = the library default."""
    f = inp.get("theta_chol0")
    return None if f is None else np.asarray(f, dtype=np.float64)


def warm_up(s, W, thin):
    """The W untimed warm-up iterations, as three cudahm_run calls (W - 2, 1, 1) where W allows: the library submits a
    handle's first persistent launch directly, builds its one-node graph at the second and pays the graph's first in-place
    parameter update at the third -- the timed regions then see the steady launch path."""
    parts = [W - 2, 1, 1] if W >= 3 else [W]
    for k in parts:
        if k > 0:
            s.run(k, W, thin)
    s.sync()


def time_gpu(cfg_name, args, device, rank, world, barrier, with_clocks=True, repeats=REPEATS):
    """W burn-in iterations untimed, then `repeats` timed regions of EXACTLY K iterations each, back to back, each timed
    on the device with CUDA events on the sampler's stream (inputs resident in HBM).  ms = the median region."""
    import torch
    c, n, inp = make_workload(cfg_name, args.n_objects if cfg_name == args.config else 0, seed_offset=rank)
    W, K = args.warmup, args.steps
    dt = np.float64 if c.precision == synth.F64 else np.float32
    dev_cols = [torch.from_numpy(np.ascontiguousarray(col, dtype=dt)).to(device) for col in inp["cols"]]
    s = make_gpu_sampler(c, n, inp, args, c.seed + rank, trace_rows_needed(W + repeats * K, W, c.thin), device, cols=dev_cols)
    warm_up(s, W, c.thin)                               # burn-in = warm-up (adaptation, caches, clocks, launch path)
    l0 = s.get_stats()["gpu_launches"]
    stream = s.stream
    clk = ClockSampler(torch.device(device).index or 0) if with_clocks else None
    if clk:
        clk.start()
    times = []
    for _ in range(repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        torch.cuda.synchronize(device)
        with torch.cuda.stream(stream):
            e0.record(stream)
            s.run(K, W, c.thin)
            e1.record(stream)
        torch.cuda.synchronize(device)
        barrier()
        times.append(e0.elapsed_time(e1))
    clocks = clk.stop() if clk else None
    ms = float(np.median(times))
    st = s.get_stats()
    tr = s.get_theta_trace()
    res = dict(cfg=c, n=n, ms=ms, times=times, launches=(st["gpu_launches"] - l0) // repeats, stats=st, clocks=clocks,
               trace=tr, inputs=inp, lib_ms=st["last_run_ms"])
    s.close()
    return res


def timing_entry(times, K):
    return {"protocol": f"{len(times)} timed regions of exactly {K} Gibbs iterations each, back to back after the warm-up; "
                        "CUDA events on the sampler's stream; value and ms_per_step are the MEDIAN region",
            "region_ms": [float(t) for t in times], "best_us_per_iter": min(times) * 1e3 / K,
            "median_us_per_iter": float(np.median(times)) * 1e3 / K}


def fixed_cost_per_run(cfg_name, args, device):
    """Fixed cost of one cudahm_run (launch, state load / write-back of the on-chip kernel, first front): device time of a
    K1-iteration run minus K1 x the marginal iteration time, the latter from a K2-iteration run (best of 3 each)."""
    import copy
    import torch
    c, n, inp = make_workload(cfg_name, 0, 0)
    K1, K2, W = 20, 2020, max(args.warmup, 5)
    a = copy.copy(args)
    a.n_objects = 0
    s = make_gpu_sampler(c, n, inp, a, c.seed, trace_rows_needed(W + 3 * (K1 + K2), W, c.thin), device)
    warm_up(s, W, c.thin)
    best = {}
    for K in (K1, K2, K1, K2, K1, K2):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(device)
        with torch.cuda.stream(s.stream):
            e0.record(s.stream)
            s.run(K, W, c.thin)
            e1.record(s.stream)
        torch.cuda.synchronize(device)
        best[K] = min(best.get(K, 1e30), e0.elapsed_time(e1) * 1e3)
    s.close()
    per_iter = (best[K2] - best[K1]) / (K2 - K1)
    return {"fixed_us_per_run": best[K1] - K1 * per_iter, "marginal_us_per_iter": per_iter,
            "how": f"best of 3: t({K1} iterations) = {best[K1]:.1f} us, t({K2}) = {best[K2]:.1f} us on {cfg_name}; fixed = t({K1}) - {K1} x "
                   "(t(K2) - t(K1)) / (K2 - K1): cooperative launch, load of the state into shared memory, first front, "
                   "write-back"}


def time_e2e(cfg_name, args, device, rank):
    """The same job through the public API with HOST buffers: H2D of the data columns (pinned), burn-in + timed
    iterations, D2H of the thinned theta trace and the chi moments -- all inside the timed region."""
    import torch
    c, n, inp = make_workload(cfg_name, args.n_objects if cfg_name == args.config else 0, seed_offset=rank)
    W, K = args.warmup, args.steps
    dt = np.float64 if c.precision == synth.F64 else np.float32
    pinned = [torch.from_numpy(np.ascontiguousarray(col, dtype=dt)).pin_memory() for col in inp["cols"]]
    host_cols = [p.numpy() for p in pinned]
    rows = trace_rows_needed(W + K, W, c.thin)
    s = make_gpu_sampler(c, n, inp, args, c.seed + rank, rows, device)   # allocation + table set-up: outside
    # result buffers in pinned host memory, allocated before the clock starts (like the input buffers)
    out_mean = torch.empty((s.p, n), dtype=torch.float64).pin_memory().numpy() if c.keep_chi_moments else None
    out_var = torch.empty((s.p, n), dtype=torch.float64).pin_memory().numpy() if c.keep_chi_moments else None
    torch.cuda.synchronize(device)
    t0 = time.perf_counter()
    s.set_data(host_cols)                    # H2D
    s.set_init(inp["theta0"], theta_chol0=make_theta_chol0(inp, n))
    s.run(W + K, W, c.thin)
    tr = s.get_theta_trace()                 # D2H (synchronises)
    d2h = tr.nbytes
    if c.keep_chi_moments:
        mean, var, _ = s.get_chi_moments(out_mean, out_var)   # D2H
        d2h += mean.nbytes + var.nbytes
    torch.cuda.synchronize(device)
    sec = time.perf_counter() - t0
    h2d = sum(p.numel() * p.element_size() for p in pinned)
    s.close()
    return dict(sec=sec, n=n, iters=W + K, h2d=h2d, d2h=d2h)


def kernel_label(st):
    """Which persistent kernel a THETA_DEVICE_TAIL run launched (cudahm_get_stats says)."""
    if st["block_threads"] == 640:
        return "k_resident"
    if st["block_threads"] == 384:
        return "k_resident_gen"
    if st.get("dedicated_tail", 0):
        return f"k_persistent_dt (dedicated tail warps, own-staged draw steps {st['stage_steps']})"
    if st.get("stage_steps", 0) or st.get("l2_prefetch", 0):
        return f"k_persistent<AHEAD> (staged draw steps {st['stage_steps']}, L2 prefetch {'on' if st['l2_prefetch'] else 'off'})"
    return "k_persistent"


def roofline_entry(cfg_name, c, n, K, W, ms, peak, peak_src, kernel=None):
    """HBM roofline on ALGORITHMIC bytes (the bound north_star names) plus the two compute floors of the same kernel:
    issue slots and the fp64 pipe, from ncu instruction counts where a capture exists (north_star: "the slower of bytes
    moved at HBM peak and the op count at the pipe peak")."""
    base, mom = ALG_BYTES[cfg_name]
    per_obj = base + (mom if c.keep_chi_moments else 0)     # the timed iterations are all past burn-in
    bytes_per_iter = per_obj * n
    achieved = bytes_per_iter * K / (ms * 1e-3) / 1e9
    us = ms * 1e3 / K
    hbm_floor = bytes_per_iter / (peak * 1e9) * 1e6
    out = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
           "traffic": (NCU_DRAM_BYTES[cfg_name][0] + NCU_DRAM_BYTES[cfg_name][1] * K)
                      if (n == c.n_objects and cfg_name in NCU_DRAM_BYTES) else None,
           "peak_source": peak_src, "kernel": kernel,
           "launches_timed": 1, "iterations_per_launch": K, "alg_bytes_per_object_iter": per_obj,
           "alg_bytes_per_iter": bytes_per_iter, "alg_bytes_per_launch": bytes_per_iter * K,
           "us_per_iter": us, "floors_us_per_iter": {"hbm": hbm_floor}}
    ins = NCU_WARP_INSTR_PER_32.get(cfg_name) if n == c.n_objects else None
    if ins:
        issue = ins[0] * (n / 32.0) / (4.0 * N_SMS * SM_CLOCK_HZ) * 1e6
        out["floors_us_per_iter"]["issue_slots"] = issue
        out["warp_instructions_per_32_updates"] = ins[0]
        out["fp64_pipe_active_pct_ncu"] = ins[1]
        out["frac_of_slowest_floor"] = max(hbm_floor, issue) / us
    return out


# ----------------------------------------------------------------------------------------------------------
def time_oracle(cfg_name, n_sample, iters, burn_in, seed_offset=0):
    """The CPU oracle as it stands (single thread, never tuned) on the first n_sample objects' worth of the
    workload: `iters` Gibbs iterations.  Returns seconds.  The ONLY place bench.py executes oracle/."""
    from oracle import api as O
    c, n, inp = make_workload(cfg_name, n_sample, seed_offset)
    o = O.Sampler(c.model, n, seed=c.seed, precision=c.precision, target_accept_chi=c.target_accept_chi,
                  target_accept_theta=c.target_accept_theta, keep_chi_moments=c.keep_chi_moments)
    o.set_data(inp["cols"])
    if inp["consts"] is not None:
        o.set_model_consts(inp["consts"])
    o.set_init(inp["theta0"], theta_chol0=make_theta_chol0(inp, n))
    t0 = time.perf_counter()
    o.run(iters, burn_in, c.thin)
    sec = time.perf_counter() - t0
    o.close()
    return sec, n


def cpu_baseline(cfg_name, n, budget_s=12.0):
    """Bounded sample: full-N iterations of the oracle, count chosen for about `budget_s` seconds of CPU work."""
    sec, _ = time_oracle(cfg_name, n, 3, 0)
    per_it = sec / 3
    iters = int(max(3, min(2000, budget_s / max(per_it, 1e-9))))
    sec, _ = time_oracle(cfg_name, n, iters, 0)
    return {"value": n * iters / sec, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{iters} Gibbs iterations of the full {cfg_name} workload (N={n}), moments on from iteration 1, "
                      f"{sec:.1f} s on one host core (oracle/liboracle.so, g++ -O2, single thread)",
            "gibbs_iters_per_s": iters / sec}


def aggregate(local_ms, local_units, dist=None):
    """Whole-job throughput: all ranks' units / MAX over ranks of the device time.  `dist` is torch.distributed
    (initialised) or None for a single process."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_units / (local_ms * 1e-3), local_ms, local_units
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([local_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return u.item() / (t.item() * 1e-3), t.item(), u.item()


def run_reference(args, rank):
    """--impl reference: the oracle on the same config / metric; each step is one Gibbs iteration over a bounded
    sample of the workload (the first n_s objects' recipe) so the whole run ends within a few minutes."""
    if rank != 0:
        return
    c = synth.CONFIGS[args.config]
    n_full = args.n_objects or c.n_objects
    W, K = args.warmup, args.steps
    probe_n = min(n_full, 20000)
    sec, _ = time_oracle(args.config, probe_n, 5, 0)
    per_update = sec / (5 * probe_n)
    n_s = int(min(n_full, max(100, 75.0 / (per_update * (W + K)))))
    sw, _ = time_oracle(args.config, n_s, W, W) if W > 0 else (0.0, n_s)
    # timed: K post-burn-in steps (run W+K with burn-in W, subtract the separately timed warm-up leg)
    st, _ = time_oracle(args.config, n_s, W + K, W)
    sec_k = max(st - sw, 1e-9)
    value = n_s * K / sec_k
    sample = (f"each step = one Gibbs iteration over a {n_s}-object sample of {args.config} (same recipe, seed); "
              f"{W}+{K} iterations, single host thread")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
            "warmup": W, "ms_per_step": sec_k * 1e3 / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if c.precision == synth.F64 else "f32 state / f64 reductions",
            "data": "synthetic",
            "config": config_entry(args.config, c, n_full, W),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                             "sample_objects": n_s},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gibbs_iters_per_s": K / sec_k, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_sharded(args, device, rank, world, dist, barrier, peak, peak_src):
    """ONE Metropolis-within-Gibbs chain over world x N objects, sharded by object range over the ranks (weak scaling:
    N objects per GPU).  theta is replicated; per iteration every rank sweeps its shard (cudahm_shard_sweep), the ranks
    all-gather their five totals over NCCL and sum them in rank order, and every rank takes the identical theta
    decision (cudahm_shard_decide).  The host sits in the loop (launch + D2H + sync + all-gather per iteration), so
    this pays for populations whose sweep takes much longer than that (~1e7 objects per GPU and up)."""
    import torch
    from paper_2105_08026_b200 import binding as B
    from paper_2105_08026_b200 import sharded
    c, n, inp = make_workload(args.config, args.n_objects, seed_offset=rank)   # each rank simulates its own shard
    W, K = args.warmup, args.steps
    stride = n + (n & 1)
    th0 = torch.from_numpy(np.array(inp["theta0"], dtype=np.float64)).to(device)
    if world > 1:
        dist.broadcast(th0, 0)                                  # the initial theta must be the same everywhere
    th0 = th0.cpu().numpy()
    if c.model == synth.M_THINNED_SCHECHTER1D:
        th0[2] += np.log(world)                                 # the amplitude counts the whole population
    s = B.Sampler(c.model, n, device=device, seed=c.seed, precision=c.precision, theta_mode=B.THETA_HOST,
                  target_accept_chi=c.target_accept_chi, target_accept_theta=c.target_accept_theta,
                  keep_chi_moments=c.keep_chi_moments, max_trace_rows=trace_rows_needed(W + K, W, c.thin),
                  object_offset=rank * stride, n_objects_total=world * stride)
    s.set_data(inp["cols"])
    if inp["consts"] is not None:
        s.set_model_consts(inp["consts"])
    s.set_init(th0)
    drv = sharded.DistributedShard(s, dist, device) if world > 1 else sharded.LocalShards([s], device=True)
    drv.run(W, W, c.thin)
    l0 = s.get_stats()["gpu_launches"]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize(device)
    with torch.cuda.stream(s.stream):
        e0.record(s.stream)
        drv.run(K, W, c.thin)
        e1.record(s.stream)
    torch.cuda.synchronize(device)
    barrier()
    value, ms, _ = aggregate(e0.elapsed_time(e1), float(n) * K, dist if world > 1 else None)
    st = s.get_stats()
    if rank == 0:
        rf = roofline_entry(args.config, c, n, K, W, ms, peak, peak_src, "k_sweep")
        rf.update(launches_timed=K, iterations_per_launch=1, alg_bytes_per_launch=rf["alg_bytes_per_iter"], traffic=None)
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if c.precision == synth.F64 else "f32 state / f64 reductions", "data": "synthetic",
            "config": {"workload": workload_label(args.config), "n_objects_per_gpu": n, "n_objects_total": world * n,
                       "parallelism": f"one chain sharded by object range over {world} gpu(s); one device-side all-gather of 5 doubles per rank and iteration, one 40-byte-per-rank read-back",
                       "theta_mode": "host", "grid": [st["grid_blocks"], st["block_threads"]]},
            "gibbs_iters_per_s": K / (ms * 1e-3), "gpu_launches": int(st["gpu_launches"] - l0), "roofline": rf,
            "accept": {"chi": st["chi_accepts"] / max(1, st["chi_proposals"]),
                       "theta": st["theta_accepts"] / max(1, st["theta_proposals"])}}), flush=True)
    s.close()


# ----------------------------------------------------------------------------------------------------------
def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return 0

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback (use --impl reference for the oracle)")
    from paper_2105_08026_b200 import binding as B
    B.load()                                        # fails loudly if libcudahm.so has not been built
    device = f"cuda:{local_rank}"
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device(device))

    def barrier():
        if world > 1:
            dist.barrier()

    peak, peak_src = load_peaks()
    if args.sharded:
        run_sharded(args, device, rank, world, dist, barrier, peak, peak_src)
        if world > 1:
            dist.destroy_process_group()
        return 0
    W, K = args.warmup, args.steps
    r = time_gpu(args.config, args, device, rank, world, barrier)
    c, n = r["cfg"], r["n"]
    value, ms, units = aggregate(r["ms"], float(n) * K, dist if world > 1 else None)
    e = time_e2e(args.config, args, device, rank)
    e_value, e_ms, _ = aggregate(e["sec"] * 1e3, float(e["n"]) * e["iters"], dist if world > 1 else None)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if c.precision == synth.F64 else "f32 state / f64 reductions", "data": "synthetic",
        "config": config_entry(args.config, c, n, W),
        "launch": {"theta_mode": args.theta_mode, "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "grid": [r["stats"]["grid_blocks"], r["stats"]["block_threads"]],
                   "l2": ("inputs larger than L2: every iteration streams the whole state through HBM"
                          if n * ALG_BYTES[args.config][0] > 126e6 else
                          "streaming persistent kernel on a working set SMALLER than L2 (the sampler iterates over the "
                          "same objects inside one launch, so there is nothing to flush between iterations): the state "
                          "is served from L2, roofline.achieved divides the ALGORITHMIC bytes by the time"
                          if r["stats"]["block_threads"] not in (640, 384) else
                          "state resident ON CHIP by design: the sampler iterates K times over the same objects "
                          "inside one persistent launch and keeps them in shared memory, so there is nothing to "
                          "flush between iterations; roofline.achieved divides the ALGORITHMIC bytes by the time "
                          "(roofline.traffic is what actually reached DRAM); other_configs.C4 is the HBM-streaming "
                          "config, whose inputs are larger than L2")},
        "timing": timing_entry(r["times"], K),
        "gibbs_iters_per_s": K * world / (ms * 1e-3),
        "e2e": {"value": e_value, "unit": UNIT, "h2d_bytes_per_step": e["h2d"] / e["iters"],
                "d2h_bytes_per_step": e["d2h"] / e["iters"], "seconds": e_ms * 1e-3,
                "what": "set_data(host cols, H2D) + set_init + run(W+K) + get_theta_trace + get_chi_moments (D2H)"},
        "gpu_launches": int(r["launches"]),
        "clocks": r["clocks"],
        "roofline": roofline_entry(args.config, c, n, K, W, r["ms"], peak, peak_src,
                                   kernel_label(r["stats"]) if args.theta_mode == "tail" else "k_sweep"),
        "accept": {"chi": r["stats"]["chi_accepts"] / max(1, r["stats"]["chi_proposals"]),
                   "theta": r["stats"]["theta_accepts"] / max(1, r["stats"]["theta_proposals"])},
        "theta_mean": [float(x) for x in r["trace"].mean(0)] if len(r["trace"]) else None,
    }
    if rank == 0 and world == 1 and not args.no_extras:
        line.update(extras(args, device, peak, peak_src, n))
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def extras(args, device, peak, peak_src, n):
    """Rank 0, N=1 only: latency floors, ALU peaks, the other theta drivers, the flushed-L2 sweep, the larger
    configs (HBM-bound) and the CPU oracle baseline."""
    import copy
    import torch
    from paper_2105_08026_b200 import binding as B
    out = {}
    st = torch.cuda.current_stream(device)
    floors = {}
    for name, kind in (("launch_pair", B.FLOOR_LAUNCH), ("graph_pair", B.FLOOR_GRAPH),
                       ("grid_barrier", B.FLOOR_GRID_BARRIER), ("host_sync", B.FLOOR_HOST_SYNC)):
        floors[name] = B.probe_floor(kind, 2000, 0, 0, st)
    out["floors_us_per_iter"] = floors
    out["alu_peaks_tera_fma_per_s"] = {"fp64": B.probe_fma_peak(0, st), "fp32": B.probe_fma_peak(1, st)}
    modes = {}
    for m in ("graph", "host"):
        a = copy.copy(args)
        a.theta_mode, a.steps, a.warmup = m, min(args.steps, 2000), min(args.warmup, 500)
        r = time_gpu(args.config, a, device, 0, 1, lambda: None, with_clocks=False, repeats=1)
        modes[m] = {"us_per_iter": r["ms"] * 1e3 / a.steps, "updates_per_s": r["n"] * a.steps / (r["ms"] * 1e-3),
                    "gpu_launches": int(r["launches"])}
    out["other_theta_modes"] = modes
    out["fixed_cost"] = fixed_cost_per_run(args.config, args, device)
    side = {}
    # every BASELINE.json config (C0 .. C4; C2 also at its steady state: burn-in 2,000 + 8,000 timed iterations in one
    # launch) plus the paper's own two workloads (C5: BB1 case study, C6: normal-normal benchmark), each as 3 timed regions
    for label, cfg_name, k, w in (("C0", "C0", 1500, 500), ("C1", "C1", 2000, 1000), ("C2_steady", "C2", 8000, 2000),
                                  ("C3", "C3", 600, 200), ("C4", "C4", 300, 100), ("C5", "C5", 3000, 1000),
                                  ("C6", "C6", 3000, 1000)):
        a = copy.copy(args)
        a.steps, a.warmup, a.n_objects = k, w, 0
        r = time_gpu(cfg_name, a, device, 0, 1, lambda: None, with_clocks=False, repeats=3)
        kern = kernel_label(r["stats"])
        rf = roofline_entry(cfg_name, r["cfg"], r["n"], k, w, r["ms"], peak, peak_src, kern)
        side[label] = {"workload": workload_label(cfg_name), "n_objects": r["n"], "steps": k, "warmup": w,
                       "updates_per_s": r["n"] * k / (r["ms"] * 1e-3),
                       "gibbs_iters_per_s": k / (r["ms"] * 1e-3), "roofline": rf, "timing": timing_entry(r["times"], k),
                       "grid": [r["stats"]["grid_blocks"], r["stats"]["block_threads"]],
                       "accept": {"chi": r["stats"]["chi_accepts"] / max(1, r["stats"]["chi_proposals"]),
                                  "theta": r["stats"]["theta_accepts"] / max(1, r["stats"]["theta_proposals"])}}
    out["other_configs"] = side
    out["cpu_baseline"] = cpu_baseline(args.config, n)
    return out


if __name__ == "__main__":
    sys.exit(main())
