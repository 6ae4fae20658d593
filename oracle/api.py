"""ctypes binding of oracle/liboracle.so.  TEST INFRASTRUCTURE ONLY (see oracle/oracle.h).

Importable only from tests/, __graft_entry__.smoke() and bench.py's CPU-baseline legs.  Argument
marshalling only; every number comes from the C++ oracle.
"""
import ctypes as C

import numpy as np

from . import build as _build

M_NORMAL1D, M_THINNED_SCHECHTER1D, M_BINORMAL2D, M_LINREG_ME1D, M_BB1_FLUXNOISE1D = 0, 1, 2, 3, 4
M_NORMAL3D_KNOWNCOV, M_NORMAL4D_KNOWNCOV, M_NORMAL5D_KNOWNCOV, M_NORMAL6D_KNOWNCOV = 5, 6, 7, 8
F64, F32_STATE_F64_REDUCE = 0, 1
KIND_PLATE, KIND_THETA = 0, 1

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class Config(C.Structure):
    _fields_ = [("model", C.c_int32), ("precision", C.c_int32), ("n_objects", C.c_int64),
                ("seed", C.c_uint64), ("target_accept_chi", C.c_double),
                ("target_accept_theta", C.c_double), ("eta_exponent", C.c_double),
                ("init_scale_chi", C.c_double), ("freeze_theta", C.c_int32),
                ("keep_chi_moments", C.c_int32), ("adapt_until", C.c_int64),
                ("prior_mean", C.c_double * 8), ("prior_isd", C.c_double * 8),
                ("object_offset", C.c_int64), ("n_objects_total", C.c_int64),
                ("per_object_counter", C.c_int32), ("pad_", C.c_int32)]


class Taps(C.Structure):
    _fields_ = [("chi_prop", _dp), ("pi_cur", _dp), ("pi_prop", _dp), ("alpha", _dp), ("u", _dp),
                ("accepted", _ip), ("L_new", _dp), ("a", _dp), ("b", _dp),
                ("theta_prop", C.c_double * 8),
                ("S", C.c_double), ("Delta", C.c_double), ("T_cur", C.c_double), ("T_prop", C.c_double),
                ("lp_cur", C.c_double), ("lp_prop", C.c_double), ("log_r", C.c_double),
                ("alpha_theta", C.c_double), ("u_theta", C.c_double),
                ("accepted_theta", C.c_int32), ("pad_", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("iterations", "chi_accepts", "chi_proposals", "theta_accepts",
                                         "theta_proposals", "nonfinite", "moment_samples", "trace_rows")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.oracle_create.argtypes = [C.POINTER(Config), C.POINTER(C.c_void_p)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_destroy.restype = None
        L.oracle_set_data.argtypes = [C.c_void_p, C.POINTER(_dp), C.c_int]
        L.oracle_set_model_consts.argtypes = [C.c_void_p, _dp, C.c_int]
        L.oracle_set_init.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.oracle_set_update_mask.argtypes = [C.c_void_p, C.POINTER(C.c_uint8)]
        L.oracle_get_counters.argtypes = [C.c_void_p, C.POINTER(C.c_uint32)]
        L.oracle_set_counters.argtypes = [C.c_void_p, C.POINTER(C.c_uint32)]
        L.oracle_run.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_int32]
        L.oracle_step.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.POINTER(Taps)]
        L.oracle_shard_sweep.argtypes = [C.c_void_p, C.c_int64, C.c_int32, _dp]
        L.oracle_shard_decide.argtypes = [C.c_void_p, C.c_int64, C.c_int32, _dp]
        L.oracle_get_theta_trace.argtypes = [C.c_void_p, _dp, C.c_int64, C.POINTER(C.c_int64)]
        L.oracle_get_chi_moments.argtypes = [C.c_void_p, _dp, _dp, C.c_int64, C.POINTER(C.c_int64)]
        L.oracle_get_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, C.POINTER(C.c_int64)]
        L.oracle_set_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, C.c_int64]
        L.oracle_get_stats.argtypes = [C.c_void_p, C.POINTER(Stats)]
        L.oracle_theta_only.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_get_selection_table.argtypes = [C.c_void_p, _dp, _dp, C.c_int, C.POINTER(C.c_int)]
        L.oracle_model_dims.argtypes = [C.c_int] + [C.POINTER(C.c_int)] * 4
        u32p = C.POINTER(C.c_uint32)
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_philox4x32_10.restype = None
        L.oracle_stream_words.argtypes = [C.c_uint64, C.c_int, C.c_uint64, C.c_uint32, C.c_uint32, u32p]
        L.oracle_stream_words.restype = None
        L.oracle_uniform_f64.argtypes = [C.c_uint64, C.c_int, C.c_uint64, C.c_uint32, C.c_uint32]
        L.oracle_uniform_f64.restype = C.c_double
        L.oracle_normals_f64.argtypes = [C.c_uint64, C.c_int, C.c_uint64, C.c_uint32, C.c_int, _dp]
        L.oracle_normals_f64.restype = None
        fp = C.POINTER(C.c_float)
        L.oracle_draws_f32.argtypes = [C.c_uint64, C.c_int, C.c_uint64, C.c_uint32, fp, fp]
        L.oracle_draws_f32.restype = None
        L.oracle_plate_draws_f64.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_int, _dp, _dp]
        L.oracle_plate_draws_f64.restype = None
        L.oracle_plate_draws_f32.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_int, fp, fp]
        L.oracle_plate_draws_f32.restype = None
        L.oracle_loglik.argtypes = [C.c_int, _dp, _dp, _dp]
        L.oracle_loglik.restype = C.c_double
        L.oracle_logpop.argtypes = [C.c_int, _dp, _dp, _dp, _dp]
        L.oracle_logpop.restype = C.c_double
        L.oracle_loglik_f32.argtypes = [C.c_int, fp, fp, fp]
        L.oracle_loglik_f32.restype = C.c_float
        L.oracle_logpop_f32.argtypes = [C.c_int, fp, fp, fp, fp]
        L.oracle_logpop_f32.restype = C.c_float
        L.oracle_logprior.argtypes = [C.c_int, _dp]
        L.oracle_logprior.restype = C.c_double
        L.oracle_ram_update.argtypes = [C.c_int, _dp, _dp, C.c_double, _dp]
        L.oracle_ram_update.restype = None
        L.oracle_gauss_legendre.argtypes = [C.c_int, C.c_double, C.c_double, _dp, _dp]
        L.oracle_gauss_legendre.restype = None
        L.oracle_bb1_log_norm.argtypes = [C.c_double] * 3
        L.oracle_bb1_log_norm.restype = C.c_double
        L.oracle_bb1_selection_integral_2d.argtypes = [_dp, _dp]
        L.oracle_bb1_selection_integral_2d.restype = C.c_double
        L.oracle_sum.argtypes = [_dp, C.c_int64]
        L.oracle_sum.restype = C.c_double
        _lib = L
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _arr(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle: {what} failed with code {rc}")


def model_dims(model):
    v = [C.c_int() for _ in range(4)]
    _check(lib().oracle_model_dims(model, *[C.byref(x) for x in v]), "model_dims")
    return dict(p=v[0].value, dtheta=v[1].value, n_cols=v[2].value, n_consts=v[3].value)


class Sampler:
    """Thin handle around oracle_sampler; same call names as the CUDA library."""

    def __init__(self, model, n_objects, seed=0, precision=F64, target_accept_chi=0.4,
                 target_accept_theta=0.234, eta_exponent=2.0 / 3.0, init_scale_chi=1.0,
                 freeze_theta=False, keep_chi_moments=False, adapt_until=0, prior_mean=None, prior_sd=None,
                 object_offset=0, n_objects_total=0, per_object_counter=False, update_mask=False):
        self.dims = model_dims(model)
        self.N = int(n_objects)
        self.p, self.dtheta = self.dims["p"], self.dims["dtheta"]
        self.ntri = self.p * (self.p + 1) // 2
        self.ntri_theta = self.dtheta * (self.dtheta + 1) // 2
        self.cfg = Config(model, precision, self.N, seed, target_accept_chi, target_accept_theta,
                          eta_exponent, init_scale_chi, int(freeze_theta), int(keep_chi_moments), int(adapt_until))
        if prior_mean is not None:
            for j, (m, sd) in enumerate(zip(prior_mean, prior_sd)):
                self.cfg.prior_mean[j] = float(m)
                self.cfg.prior_isd[j] = 0.0 if not np.isfinite(sd) else 1.0 / float(sd)
        self.cfg.object_offset, self.cfg.n_objects_total = int(object_offset), int(n_objects_total)
        self.cfg.per_object_counter = int(per_object_counter)
        self._h = C.c_void_p()
        _check(lib().oracle_create(C.byref(self.cfg), C.byref(self._h)), "create")

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_data(self, cols):
        cols = [_arr(c) for c in cols]
        assert all(c.shape == (self.N,) for c in cols)
        ptrs = (_dp * len(cols))(*[_d(c) for c in cols])
        _check(lib().oracle_set_data(self._h, ptrs, len(cols)), "set_data")

    def set_model_consts(self, v):
        v = _arr(v)
        _check(lib().oracle_set_model_consts(self._h, _d(v), v.size), "set_model_consts")

    def set_update_mask(self, mask):
        """mask: N bytes (1 = update, 0 = hold fixed) or None (update everything)."""
        if mask is None:
            _check(lib().oracle_set_update_mask(self._h, None), "set_update_mask")
            return
        m = np.ascontiguousarray(np.asarray(mask, dtype=np.uint8))
        assert m.shape == (self.N,)
        _check(lib().oracle_set_update_mask(self._h, m.ctypes.data_as(C.POINTER(C.c_uint8))), "set_update_mask")

    def get_counters(self):
        out = np.empty(self.N, dtype=np.uint32)
        _check(lib().oracle_get_counters(self._h, out.ctypes.data_as(C.POINTER(C.c_uint32))), "get_counters")
        return out

    def set_counters(self, c):
        c = np.ascontiguousarray(np.asarray(c, dtype=np.uint32))
        assert c.shape == (self.N,)
        _check(lib().oracle_set_counters(self._h, c.ctypes.data_as(C.POINTER(C.c_uint32))), "set_counters")

    def set_init(self, theta0, chi0=None, theta_chol0=None):
        th = _arr(theta0)
        c0 = None if chi0 is None else _arr(chi0).reshape(-1)
        l0 = None if theta_chol0 is None else _arr(theta_chol0)
        _check(lib().oracle_set_init(self._h, _d(c0), _d(th), _d(l0)), "set_init")

    def run(self, n_iter, burn_in=0, thin=1):
        _check(lib().oracle_run(self._h, n_iter, burn_in, thin), "run")

    def step(self, burn_in=0, thin=1, taps=False):
        """One Gibbs iteration; with taps=True returns a dict of per-object and scalar taps."""
        if not taps:
            _check(lib().oracle_step(self._h, burn_in, thin, None), "step")
            return None
        N, p = self.N, self.p
        out = dict(chi_prop=np.empty((p, N)), pi_cur=np.empty(N), pi_prop=np.empty(N), alpha=np.empty(N),
                   u=np.empty(N), accepted=np.empty(N, dtype=np.int32), L_new=np.empty((self.ntri, N)),
                   a=np.empty(N), b=np.empty(N))
        tp = Taps()
        for k in ("chi_prop", "pi_cur", "pi_prop", "alpha", "u", "L_new", "a", "b"):
            setattr(tp, k, _d(out[k]))
        tp.accepted = out["accepted"].ctypes.data_as(_ip)
        _check(lib().oracle_step(self._h, burn_in, thin, C.byref(tp)), "step")
        out["theta_prop"] = np.array(tp.theta_prop[: self.dtheta])
        for k in ("S", "Delta", "T_cur", "T_prop", "lp_cur", "lp_prop", "log_r", "alpha_theta", "u_theta",
                  "accepted_theta"):
            out[k] = getattr(tp, k)
        return out

    def get_theta_trace(self):
        n = C.c_int64()
        _check(lib().oracle_get_theta_trace(self._h, None, 0, C.byref(n)), "get_theta_trace")
        out = np.empty((n.value, self.dtheta))
        _check(lib().oracle_get_theta_trace(self._h, _d(out), n.value, C.byref(n)), "get_theta_trace")
        return out

    def get_chi_moments(self):
        mean, var = np.empty((self.p, self.N)), np.empty((self.p, self.N))
        n = C.c_int64()
        _check(lib().oracle_get_chi_moments(self._h, _d(mean), _d(var), self.N, C.byref(n)), "get_chi_moments")
        return mean, var, n.value

    def get_state(self):
        chi, L = np.empty((self.p, self.N)), np.empty((self.ntri, self.N))
        th, Lth = np.empty(self.dtheta), np.empty(self.ntri_theta)
        t = C.c_int64()
        _check(lib().oracle_get_state(self._h, _d(chi), _d(L), _d(th), _d(Lth), C.byref(t)), "get_state")
        return dict(chi=chi, L=L, theta=th, L_theta=Lth, t=t.value)

    def set_state(self, chi=None, L=None, theta=None, L_theta=None, t=0):
        a = [None if x is None else _arr(x) for x in (chi, L, theta, L_theta)]
        _check(lib().oracle_set_state(self._h, _d(a[0]), _d(a[1]), _d(a[2]), _d(a[3]), t), "set_state")

    def get_stats(self):
        s = Stats()
        _check(lib().oracle_get_stats(self._h, C.byref(s)), "get_stats")
        return {k: getattr(s, k) for k, _ in Stats._fields_}

    def shard_sweep(self, burn_in=0, thin=1):
        tot = np.empty(5)
        _check(lib().oracle_shard_sweep(self._h, burn_in, thin, _d(tot)), "shard_sweep")
        return tot

    def shard_decide(self, totals_global, burn_in=0, thin=1):
        tot = _arr(totals_global)
        _check(lib().oracle_shard_decide(self._h, burn_in, thin, _d(tot)), "shard_decide")

    def theta_only(self, theta):
        th, out = _arr(theta), C.c_double()
        _check(lib().oracle_theta_only(self._h, _d(th), C.byref(out)), "theta_only")
        return out.value

    def get_selection_table(self):
        xk, Wk, n = np.empty(1024), np.empty(1024), C.c_int()
        _check(lib().oracle_get_selection_table(self._h, _d(xk), _d(Wk), 1024, C.byref(n)), "selection_table")
        return xk[: n.value], Wk[: n.value]


# ---- stateless primitives -------------------------------------------------------------------------
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def stream_words(seed, kind, obj, t, d):
    o = (C.c_uint32 * 4)()
    lib().oracle_stream_words(seed, kind, obj, t, d, o)
    return [int(x) for x in o]


def uniform_f64(seed, kind, obj, t, d):
    return lib().oracle_uniform_f64(seed, kind, obj, t, d)


def normals_f64(seed, kind, obj, t, n):
    z = np.empty(n)
    lib().oracle_normals_f64(seed, kind, obj, t, n, _d(z))
    return z


def draws_f32(seed, kind, obj, t):
    z = (C.c_float * 2)()
    u = C.c_float()
    lib().oracle_draws_f32(seed, kind, obj, t, z, C.byref(u))
    return np.float32(z[0]), np.float32(z[1]), np.float32(u.value)


def plate_draws_f64(seed, i, t, p):
    """(z[0..p-1], accept uniform) of object i at iteration t."""
    z = np.zeros(max(p, 2))
    u = C.c_double()
    lib().oracle_plate_draws_f64(seed, i, t, p, _d(z), C.byref(u))
    return z[:p].copy(), u.value


def plate_draws_f32(seed, i, t, p):
    z = (C.c_float * 2)()
    u = C.c_float()
    lib().oracle_plate_draws_f32(seed, i, t, p, z, C.byref(u))
    return np.array([z[k] for k in range(p)], dtype=np.float32), np.float32(u.value)


def loglik(model, chi, data_i, consts=None):
    c = None if consts is None else _arr(consts)
    return lib().oracle_loglik(model, _d(_arr(chi)), _d(_arr(data_i)), _d(c))


def logpop(model, chi, data_i, theta, consts=None):
    c = None if consts is None else _arr(consts)
    return lib().oracle_logpop(model, _d(_arr(chi)), _d(_arr(data_i)), _d(_arr(theta)), _d(c))


def _f(a):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float32))
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


def loglik_f32(model, chi, data_i, consts=None):
    k = [_f(x) for x in (chi, data_i)]
    c = (None, None) if consts is None else _f(consts)
    return lib().oracle_loglik_f32(model, k[0][1], k[1][1], c[1])


def logpop_f32(model, chi, data_i, theta, consts=None):
    k = [_f(x) for x in (chi, data_i, theta)]
    c = (None, None) if consts is None else _f(consts)
    return lib().oracle_logpop_f32(model, k[0][1], k[1][1], k[2][1], c[1])


def logprior(model, theta):
    return lib().oracle_logprior(model, _d(_arr(theta)))


def ram_update(L_packed, z, c):
    z = _arr(z)
    Lp = _arr(L_packed)
    out = np.empty_like(Lp)
    lib().oracle_ram_update(z.size, _d(Lp), _d(z), c, _d(out))
    return out


def gauss_legendre(n, a, b):
    x, w = np.empty(n), np.empty(n)
    lib().oracle_gauss_legendre(n, a, b, _d(x), _d(w))
    return x, w


def bb1_log_norm(beta, l, u):
    return lib().oracle_bb1_log_norm(beta, l, u)


def bb1_selection_integral_2d(theta, consts):
    return lib().oracle_bb1_selection_integral_2d(_d(_arr(theta)), _d(_arr(consts)))


def osum(v):
    v = _arr(v)
    return lib().oracle_sum(_d(v), v.size)
