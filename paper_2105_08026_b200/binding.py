"""Thin ctypes binding of libcudahm.so (include/cudahm.h): argument marshalling only.

PyTorch is used for device memory (one uint8 workspace tensor per sampler) and the CUDA stream;
every step of the sampler runs in the library's kernels.  There is no CPU fallback: if the library
has not been built (`python -m paper_2105_08026_b200.build`) or no CUDA device is present, calls fail.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libcudahm.so")

OK, E_INVALID, E_STATE, E_CUDA, E_WORKSPACE, E_UNSUPPORTED, E_NONFINITE = 0, -1, -2, -3, -4, -5, -6
M_NORMAL1D, M_THINNED_SCHECHTER1D, M_BINORMAL2D, M_LINREG_ME1D, M_BB1_FLUXNOISE1D, M_NORMAL3D_KNOWNCOV = 0, 1, 2, 3, 4, 5
M_NORMAL4D_KNOWNCOV, M_NORMAL5D_KNOWNCOV, M_NORMAL6D_KNOWNCOV = 6, 7, 8
F64, F32_STATE_F64_REDUCE = 0, 1
THETA_HOST, THETA_GRAPH, THETA_DEVICE_TAIL = 0, 1, 2
FLAG_STREAMING_ONLY, FLAG_TMA_STAGING = 1, 2
FLAG_PREFETCH_OFF, FLAG_PREFETCH_ON, FLAG_TIME_RUNS = 4, 8, 16


def flag_stage_steps(n):
    """CUDAHM_FLAG_STAGE_STEPS(n): exactly n steps of plate draws staged ahead of the sweep (0 = off)."""
    return ((int(n) + 1) << 8) & 0xff00
FLOOR_LAUNCH, FLOOR_GRAPH, FLOOR_GRID_BARRIER, FLOOR_HOST_SYNC = 0, 1, 2, 3
NOALLOC_SCRATCH_BYTES = 4 << 20       # CUDAHM_NOALLOC_SCRATCH_BYTES

EXPORTS = ["cudahm_model_dims", "cudahm_workspace_bytes", "cudahm_create", "cudahm_destroy", "cudahm_set_data",
           "cudahm_set_model_consts", "cudahm_set_init", "cudahm_run", "cudahm_debug_step", "cudahm_debug_step_noalloc",
           "cudahm_debug_step_noalloc_bytes",
           "cudahm_get_theta_trace", "cudahm_get_chi_moments", "cudahm_get_stats", "cudahm_get_state",
           "cudahm_set_state", "cudahm_sync", "cudahm_last_error", "cudahm_shard_sweep", "cudahm_shard_decide", "cudahm_shard_combine", "cudahm_shard_sweep_device",
           "cudahm_shard_decide_gathered", "cudahm_set_update_mask", "cudahm_get_counters", "cudahm_set_counters",
           "cudahm_probe_floor", "cudahm_probe_fma_peak", "cudahm_probe_math"]

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class Config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("model", C.c_int32), ("precision", C.c_int32),
                ("theta_mode", C.c_int32), ("n_objects", C.c_int64), ("p", C.c_int32), ("dtheta", C.c_int32),
                ("n_data_cols", C.c_int32), ("freeze_theta", C.c_int32), ("seed", C.c_uint64),
                ("target_accept_chi", C.c_double), ("target_accept_theta", C.c_double),
                ("eta_exponent", C.c_double), ("init_scale_chi", C.c_double), ("keep_chi_moments", C.c_int32),
                ("block_threads", C.c_int32), ("blocks_per_sm", C.c_int32), ("flags", C.c_int32),
                ("max_trace_rows", C.c_int64), ("adapt_until", C.c_int64),
                ("prior_mean", C.c_double * 8), ("prior_isd", C.c_double * 8),
                ("object_offset", C.c_int64), ("n_objects_total", C.c_int64),
                ("update_mask", C.c_int32), ("per_object_counter", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("iterations", "chi_accepts", "chi_proposals", "theta_accepts",
                                         "theta_proposals", "nonfinite", "moment_samples", "trace_rows",
                                         "gpu_launches")] + \
               [("grid_blocks", C.c_int32), ("block_threads", C.c_int32), ("last_run_ms", C.c_double),
                ("stage_steps", C.c_int32), ("l2_prefetch", C.c_int32), ("dedicated_tail", C.c_int32), ("graph_launches", C.c_int32)]


class Taps(C.Structure):
    _fields_ = [("chi_prop", _dp), ("pi_cur", _dp), ("pi_prop", _dp), ("alpha", _dp), ("u", _dp),
                ("accepted", _ip), ("L_new", _dp), ("a", _dp), ("b", _dp), ("theta_prop", C.c_double * 8),
                ("S", C.c_double), ("Delta", C.c_double), ("T_cur", C.c_double), ("T_prop", C.c_double),
                ("lp_cur", C.c_double), ("lp_prop", C.c_double), ("log_r", C.c_double),
                ("alpha_theta", C.c_double), ("u_theta", C.c_double), ("accepted_theta", C.c_int32),
                ("pad_", C.c_int32)]


_lib = None


def load():
    """dlopen the in-tree library; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2105_08026_b200.build` "
                           "(nvcc, sm_100a); there is no CPU fallback")
    L = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    L.cudahm_model_dims.argtypes = [C.c_int] + [C.POINTER(C.c_int)] * 4
    L.cudahm_workspace_bytes.argtypes = [C.POINTER(Config)]
    L.cudahm_workspace_bytes.restype = C.c_size_t
    L.cudahm_create.argtypes = [C.POINTER(Config), vp, C.c_size_t, vp, C.POINTER(vp)]
    L.cudahm_destroy.argtypes = [vp]
    L.cudahm_destroy.restype = None
    L.cudahm_set_data.argtypes = [vp, C.POINTER(vp), C.c_int, C.c_int]
    L.cudahm_set_model_consts.argtypes = [vp, _dp, C.c_int]
    L.cudahm_set_init.argtypes = [vp, vp, C.c_int, _dp, _dp]
    L.cudahm_run.argtypes = [vp, C.c_int64, C.c_int64, C.c_int32]
    L.cudahm_debug_step.argtypes = [vp, C.c_int64, C.c_int32, C.POINTER(Taps)]
    L.cudahm_debug_step_noalloc.argtypes = [vp, C.c_int64, C.c_int32, C.POINTER(Taps)]
    L.cudahm_debug_step_noalloc_bytes.argtypes = [vp]
    L.cudahm_debug_step_noalloc_bytes.restype = C.c_size_t
    L.cudahm_get_theta_trace.argtypes = [vp, _dp, C.c_int64, C.POINTER(C.c_int64)]
    L.cudahm_get_chi_moments.argtypes = [vp, _dp, _dp, C.c_int64, C.POINTER(C.c_int64)]
    L.cudahm_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.cudahm_get_state.argtypes = [vp, vp, vp, _dp, _dp, C.POINTER(C.c_int64)]
    L.cudahm_set_state.argtypes = [vp, vp, vp, _dp, _dp, C.c_int64]
    L.cudahm_shard_sweep.argtypes = [vp, C.c_int64, C.c_int32, _dp]
    L.cudahm_shard_decide.argtypes = [vp, C.c_int64, C.c_int32, _dp]
    L.cudahm_shard_combine.argtypes = [_dp, C.c_int, _dp]
    L.cudahm_shard_sweep_device.argtypes = [vp, C.c_int64, C.c_int32, vp]
    L.cudahm_shard_decide_gathered.argtypes = [vp, C.c_int64, C.c_int32, vp, C.c_int]
    L.cudahm_set_update_mask.argtypes = [vp, vp, C.c_int]
    L.cudahm_get_counters.argtypes = [vp, vp]
    L.cudahm_set_counters.argtypes = [vp, vp]
    L.cudahm_sync.argtypes = [vp]
    L.cudahm_last_error.argtypes = [vp]
    L.cudahm_last_error.restype = C.c_char_p
    L.cudahm_probe_floor.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, _dp]
    L.cudahm_probe_fma_peak.argtypes = [vp, C.c_int, _dp]
    L.cudahm_probe_math.argtypes = [vp, C.c_int, _dp, _dp, C.c_longlong]
    _lib = L
    return L


class CudahmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"cudahm error {code}: {msg}")
        self.code = code


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def model_dims(model):
    v = [C.c_int() for _ in range(4)]
    rc = load().cudahm_model_dims(model, *[C.byref(x) for x in v])
    if rc:
        raise CudahmError(rc, load().cudahm_last_error(None).decode())
    return dict(p=v[0].value, dtheta=v[1].value, n_cols=v[2].value, n_consts=v[3].value)


def make_config(model, n_objects, seed=0, precision=F64, theta_mode=THETA_DEVICE_TAIL, target_accept_chi=0.4,
                target_accept_theta=0.234, eta_exponent=2.0 / 3.0, init_scale_chi=1.0, freeze_theta=False,
                keep_chi_moments=False, max_trace_rows=0, block_threads=0, blocks_per_sm=0, flags=0, adapt_until=0,
                prior_mean=None, prior_sd=None, object_offset=0, n_objects_total=0, update_mask=False,
                per_object_counter=False):
    d = model_dims(model)
    cfg = Config(C.sizeof(Config), model, precision, theta_mode, int(n_objects), d["p"], d["dtheta"], d["n_cols"],
                  int(freeze_theta), seed, target_accept_chi, target_accept_theta, eta_exponent, init_scale_chi,
                  int(keep_chi_moments), block_threads, blocks_per_sm, int(flags), int(max_trace_rows), int(adapt_until))
    if prior_mean is not None:          # user prior: independent normal factors on theta (sd = inf: none)
        for j, (m, sd) in enumerate(zip(prior_mean, prior_sd)):
            cfg.prior_mean[j] = float(m)
            cfg.prior_isd[j] = 0.0 if not np.isfinite(sd) else 1.0 / float(sd)
    cfg.object_offset, cfg.n_objects_total = int(object_offset), int(n_objects_total)
    cfg.update_mask, cfg.per_object_counter = int(update_mask), int(per_object_counter)
    return cfg


def shard_combine(totals_by_rank):
    """cudahm_shard_combine: the rank-order sum of the shards' totals (n_ranks x 5 host doubles -> 5); no device needed."""
    t = np.ascontiguousarray(np.asarray(totals_by_rank, dtype=np.float64).reshape(-1, 5))
    out = np.empty(5)
    rc = load().cudahm_shard_combine(_d(t), t.shape[0], _d(out))
    if rc:
        raise CudahmError(rc, load().cudahm_last_error(None).decode())
    return out


def workspace_bytes(cfg):
    return int(load().cudahm_workspace_bytes(C.byref(cfg)))


class Sampler:
    """One cudahm_sampler.  Same call names as include/cudahm.h; numpy in, numpy out."""

    def __init__(self, model, n_objects, device="cuda:0", stream=None, **kw):
        import torch
        self._torch = torch
        self.lib = load()
        self.cfg = make_config(model, n_objects, **kw)
        self.N, self.p, self.dtheta = int(n_objects), self.cfg.p, self.cfg.dtheta
        self.ntri = self.p * (self.p + 1) // 2
        self.ntri_theta = self.dtheta * (self.dtheta + 1) // 2
        self.dtype = np.float64 if self.cfg.precision == F64 else np.float32
        nbytes = workspace_bytes(self.cfg)
        if nbytes == 0:
            raise CudahmError(E_INVALID, "invalid configuration")
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self._h = C.c_void_p()
            rc = self.lib.cudahm_create(C.byref(self.cfg), C.c_void_p(self.workspace.data_ptr()), nbytes,
                                        C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        if rc:
            raise CudahmError(rc, self.lib.cudahm_last_error(None).decode())
        self._run = self.lib.cudahm_run

    def _ck(self, rc):
        if rc:
            raise CudahmError(rc, self.lib.cudahm_last_error(self._h).decode())

    def _dev(self):
        return self._torch.cuda.device(self.device)

    def close(self):
        if getattr(self, "_h", None):
            with self._dev():
                self.lib.cudahm_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_data(self, cols):
        """cols: host arrays (cast to the state precision) or CUDA torch tensors of the state precision."""
        torch = self._torch
        on_dev = all(isinstance(c, torch.Tensor) and c.is_cuda for c in cols)
        if on_dev:
            keep = [c.contiguous() for c in cols]
            ptrs = [c.data_ptr() for c in keep]
        else:
            keep = [np.ascontiguousarray(np.asarray(c), dtype=self.dtype) for c in cols]
            assert all(k.shape == (self.N,) for k in keep)
            ptrs = [k.ctypes.data for k in keep]
        arr = (C.c_void_p * len(ptrs))(*ptrs)
        with self._dev():
            self._ck(self.lib.cudahm_set_data(self._h, arr, len(ptrs), int(on_dev)))

    def set_model_consts(self, v):
        v = np.ascontiguousarray(np.asarray(v, dtype=np.float64))
        with self._dev():
            self._ck(self.lib.cudahm_set_model_consts(self._h, _d(v), v.size))

    def set_init(self, theta0, chi0=None, theta_chol0=None):
        th = np.ascontiguousarray(np.asarray(theta0, dtype=np.float64))
        c0 = None if chi0 is None else np.ascontiguousarray(np.asarray(chi0).reshape(-1), dtype=self.dtype)
        l0 = None if theta_chol0 is None else np.ascontiguousarray(np.asarray(theta_chol0, dtype=np.float64))
        with self._dev():
            self._ck(self.lib.cudahm_set_init(self._h, None if c0 is None else C.c_void_p(c0.ctypes.data), 0,
                                              _d(th), _d(l0)))

    def set_update_mask(self, mask):
        """mask: N bytes (1 = update, 0 = hold fixed), host array or CUDA uint8 tensor; None = update everything."""
        torch = self._torch
        with self._dev():
            if mask is None:
                self._ck(self.lib.cudahm_set_update_mask(self._h, None, 0))
            elif isinstance(mask, torch.Tensor) and mask.is_cuda:
                m = mask.contiguous()
                assert m.dtype == torch.uint8 and m.numel() == self.N
                self._ck(self.lib.cudahm_set_update_mask(self._h, C.c_void_p(m.data_ptr()), 1))
            else:
                m = np.ascontiguousarray(np.asarray(mask, dtype=np.uint8))
                assert m.shape == (self.N,)
                self._ck(self.lib.cudahm_set_update_mask(self._h, C.c_void_p(m.ctypes.data), 0))

    def get_counters(self):
        out = np.empty(self.N, dtype=np.uint32)
        with self._dev():
            self._ck(self.lib.cudahm_get_counters(self._h, C.c_void_p(out.ctypes.data)))
        return out

    def set_counters(self, c):
        c = np.ascontiguousarray(np.asarray(c, dtype=np.uint32))
        assert c.shape == (self.N,)
        with self._dev():
            self._ck(self.lib.cudahm_set_counters(self._h, C.c_void_p(c.ctypes.data)))

    def run(self, n_iter, burn_in=0, thin=1, sync=False):
        # no torch device context here: cudahm_run makes the handle's device current itself, and the context manager's
        # two device switches are 3 us of host time between the caller's stream position and the launch
        rc = self._run(self._h, n_iter, burn_in, thin)
        if rc:
            self._ck(rc)
        if sync:
            self.sync()

    def sync(self):
        with self._dev():
            self._ck(self.lib.cudahm_sync(self._h))

    def shard_sweep(self, burn_in=0, thin=1):
        """One sweep over this handle's objects: {S, Delta, Tq, n_accept, n_nonfinite} of this shard (THETA_HOST)."""
        tot = np.empty(5)
        with self._dev():
            self._ck(self.lib.cudahm_shard_sweep(self._h, burn_in, thin, _d(tot)))
        return tot

    def shard_decide(self, totals_global, burn_in=0, thin=1):
        """The theta step of the iteration just swept, from the totals summed over all shards."""
        tot = np.ascontiguousarray(totals_global, dtype=np.float64)
        with self._dev():
            self._ck(self.lib.cudahm_shard_decide(self._h, burn_in, thin, _d(tot)))

    def shard_sweep_device(self, totals_dev_ptr, burn_in=0, thin=1):
        """One sweep over this handle's objects; its five totals are left in the DEVICE buffer at totals_dev_ptr."""
        with self._dev():
            self._ck(self.lib.cudahm_shard_sweep_device(self._h, burn_in, thin, C.c_void_p(int(totals_dev_ptr))))

    def shard_decide_gathered(self, gathered_dev_ptr, n_ranks, burn_in=0, thin=1):
        """The theta step from the DEVICE array gathered[n_ranks][5] (rank order), combined inside the library."""
        with self._dev():
            self._ck(self.lib.cudahm_shard_decide_gathered(self._h, burn_in, thin, C.c_void_p(int(gathered_dev_ptr)), int(n_ranks)))

    def debug_step(self, burn_in=0, thin=1):
        N, p = self.N, self.p
        out = dict(chi_prop=np.empty((p, N)), pi_cur=np.empty(N), pi_prop=np.empty(N), alpha=np.empty(N),
                   u=np.empty(N), accepted=np.empty(N, dtype=np.int32), L_new=np.empty((self.ntri, N)),
                   a=np.empty(N), b=np.empty(N))
        tp = Taps()
        for k in ("chi_prop", "pi_cur", "pi_prop", "alpha", "u", "L_new", "a", "b"):
            setattr(tp, k, _d(out[k]))
        tp.accepted = out["accepted"].ctypes.data_as(_ip)
        with self._dev():
            self._ck(self.lib.cudahm_debug_step(self._h, burn_in, thin, C.byref(tp)))
        out["theta_prop"] = np.array(tp.theta_prop[: self.dtheta])
        for k in ("S", "Delta", "T_cur", "T_prop", "lp_cur", "lp_prop", "log_r", "alpha_theta", "u_theta",
                  "accepted_theta"):
            out[k] = getattr(tp, k)
        return out

    def debug_step_noalloc(self, burn_in=0, thin=1):
        """cudahm_debug_step_noalloc: the same tapped iteration with its tap scratch in the library's built-in device array
        (no cudaMalloc in the call); raises CudahmError(E_WORKSPACE) if the population does not fit NOALLOC_SCRATCH_BYTES."""
        N, p = self.N, self.p
        out = dict(chi_prop=np.empty((p, N)), pi_cur=np.empty(N), pi_prop=np.empty(N), alpha=np.empty(N),
                   u=np.empty(N), accepted=np.empty(N, dtype=np.int32), L_new=np.empty((self.ntri, N)),
                   a=np.empty(N), b=np.empty(N))
        tp = Taps()
        for k in ("chi_prop", "pi_cur", "pi_prop", "alpha", "u", "L_new", "a", "b"):
            setattr(tp, k, _d(out[k]))
        tp.accepted = out["accepted"].ctypes.data_as(_ip)
        with self._dev():
            self._ck(self.lib.cudahm_debug_step_noalloc(self._h, burn_in, thin, C.byref(tp)))
        out["theta_prop"] = np.array(tp.theta_prop[: self.dtheta])
        for k in ("S", "Delta", "T_cur", "T_prop", "lp_cur", "lp_prop", "log_r", "alpha_theta", "u_theta",
                  "accepted_theta"):
            out[k] = getattr(tp, k)
        return out

    def debug_step_noalloc_bytes(self):
        return int(self.lib.cudahm_debug_step_noalloc_bytes(self._h))

    def get_theta_trace(self):
        n = C.c_int64()
        with self._dev():
            self._ck(self.lib.cudahm_get_theta_trace(self._h, None, 0, C.byref(n)))
            out = np.empty((n.value, self.dtheta))
            self._ck(self.lib.cudahm_get_theta_trace(self._h, _d(out), n.value, C.byref(n)))
        return out

    def get_chi_moments(self, mean=None, var=None):
        """mean, var: optional caller buffers (p, N) float64, e.g. pinned host memory; allocated here if omitted."""
        mean = np.empty((self.p, self.N)) if mean is None else mean
        var = np.empty((self.p, self.N)) if var is None else var
        assert mean.shape == var.shape == (self.p, self.N) and mean.dtype == var.dtype == np.float64
        assert mean.flags.c_contiguous and var.flags.c_contiguous
        n = C.c_int64()
        with self._dev():
            self._ck(self.lib.cudahm_get_chi_moments(self._h, _d(mean), _d(var), self.N, C.byref(n)))
        return mean, var, n.value

    def get_stats(self):
        s = Stats()
        with self._dev():
            self._ck(self.lib.cudahm_get_stats(self._h, C.byref(s)))
        return {k: getattr(s, k) for k, _ in Stats._fields_}

    def get_state(self):
        chi, L = np.empty((self.p, self.N), self.dtype), np.empty((self.ntri, self.N), self.dtype)
        th, Lth = np.empty(self.dtheta), np.empty(self.ntri_theta)
        t = C.c_int64()
        with self._dev():
            self._ck(self.lib.cudahm_get_state(self._h, C.c_void_p(chi.ctypes.data), C.c_void_p(L.ctypes.data),
                                               _d(th), _d(Lth), C.byref(t)))
        return dict(chi=chi.astype(np.float64), L=L.astype(np.float64), theta=th, L_theta=Lth, t=t.value)

    def set_state(self, chi=None, L=None, theta=None, L_theta=None, t=0):
        c = None if chi is None else np.ascontiguousarray(np.asarray(chi), dtype=self.dtype)
        l = None if L is None else np.ascontiguousarray(np.asarray(L), dtype=self.dtype)
        th = None if theta is None else np.ascontiguousarray(np.asarray(theta, dtype=np.float64))
        lt = None if L_theta is None else np.ascontiguousarray(np.asarray(L_theta, dtype=np.float64))
        with self._dev():
            self._ck(self.lib.cudahm_set_state(self._h, None if c is None else C.c_void_p(c.ctypes.data),
                                               None if l is None else C.c_void_p(l.ctypes.data), _d(th), _d(lt), t))


def probe_floor(kind, n_iter=2000, grid_blocks=0, block_threads=0, stream=None):
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    out = C.c_double()
    rc = load().cudahm_probe_floor(C.c_void_p(st.cuda_stream), kind, n_iter, grid_blocks, block_threads, C.byref(out))
    if rc:
        raise CudahmError(rc, "probe_floor failed")
    return out.value


def probe_fma_peak(dtype, stream=None):
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    out = C.c_double()
    rc = load().cudahm_probe_fma_peak(C.c_void_p(st.cuda_stream), dtype, C.byref(out))
    if rc:
        raise CudahmError(rc, "probe_fma_peak failed")
    return out.value


# cudahm_probe.h: CUDAHM_MATH_*
MATH_EXP, MATH_EXPM1_NONPOS, MATH_LOG, MATH_SQRT, MATH_SQRT_BOTH_ROOT, MATH_SQRT_BOTH_INV, MATH_SIN2PI, MATH_COS2PI = range(8)
MATH_LOG_2, MATH_SQRT_2, MATH_SQRT_BOTH_ROOT_2, MATH_SQRT_BOTH_INV_2 = range(8, 12)   # the two-Newton-step variants


def probe_math(fn, x, stream=None):
    """y = fn(x) evaluated by the DEVICE build of csrc/fastmath.cuh (cudahm_probe_math); x: float64 array."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty_like(x)
    rc = load().cudahm_probe_math(C.c_void_p(st.cuda_stream), int(fn), _d(x), _d(y), x.size)
    if rc:
        raise CudahmError(rc, "probe_math failed")
    return y
