"""Thin Python binding of libnsgw.so (include/nsgw.h): argument marshalling only.

torch is used for device memory and streams; every step of the hot path runs in the library's CUDA kernels.
There is no CPU fallback: if the shared library is missing or no CUDA device is present, calls raise.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libnsgw.so")

MAX_DIM, MAX_DET = 16, 4


class NsConfig(C.Structure):
    _fields_ = [
        ("struct_version", C.c_int32), ("like_kind", C.c_int32), ("ndim", C.c_int32),
        ("n_live", C.c_int32), ("n_delete", C.c_int32), ("naccept", C.c_int32), ("maxmcmc", C.c_int32),
        ("walks0", C.c_double), ("delay", C.c_double),
        ("prior_kind", C.c_int32 * MAX_DIM), ("prior_lo", C.c_double * MAX_DIM), ("prior_hi", C.c_double * MAX_DIM),
        ("periodic", C.c_int32 * MAX_DIM),
        ("n_det", C.c_int32), ("n_freq", C.c_int32), ("f_min", C.c_double), ("df", C.c_double),
        ("det_vertex", (C.c_double * 3) * MAX_DET), ("det_xarm", (C.c_double * 3) * MAX_DET), ("det_yarm", (C.c_double * 3) * MAX_DET),
        ("gmst", C.c_double),
        ("toy_mean", C.c_double * MAX_DIM), ("toy_prec", C.c_double * (MAX_DIM * MAX_DIM)), ("toy_lognorm", C.c_double),
        ("phenom_table_host", C.POINTER(C.c_double)),
    ]


class NsStats(C.Structure):
    _fields_ = [
        ("iteration", C.c_int64), ("logl_star", C.c_double), ("logx", C.c_double), ("logz", C.c_double), ("h", C.c_double),
        ("dlogz", C.c_double), ("live_frac_log", C.c_double), ("walk_len", C.c_int32), ("pad0", C.c_int32),
        ("walks_next", C.c_double), ("accept_mean", C.c_double), ("accept_min", C.c_int32), ("accept_max", C.c_int32),
        ("n_eval", C.c_int64), ("n_oob", C.c_int64), ("n_stuck", C.c_int64), ("n_eval_total", C.c_int64),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "pad0"}


class NsState(C.Structure):
    _fields_ = [("struct_version", C.c_int32), ("pad0", C.c_int32), ("iteration", C.c_int64), ("n_eval_total", C.c_int64),
                ("logx", C.c_double), ("logz", C.c_double), ("h", C.c_double), ("walks", C.c_double), ("seed", C.c_uint64)]


EXPORTS = ["ns_init", "ns_free", "ns_last_error", "gw_loglike_batch", "gw_loglike_batch_host", "gw_waveform", "ns_prior_transform_batch",
           "ns_loglike_u_batch", "ns_walk_batch", "ns_step", "ns_run", "ns_run_many", "ns_slice_batch", "ns_relbin_setup", "ns_relbin_get", "gw_loglike_relbin_batch", "ns_get_live", "ns_finalize_evidence", "ns_posterior", "ns_posterior_resample",
           "nsgw_measure_fp64_peak", "nsgw_launch_count", "nsgw_profile_enable", "nsgw_profile_read", "nsgw_set_option",
           "ns_get_state", "ns_set_state", "nsgw_sweep_occupancy", "gw_loglike_batch_noalloc"]

# nsgw_set_option keys (include/nsgw.h)
NOALLOC_MAX_ROWS, NOALLOC_MAX_BINS = 4096, 16384     # gw_loglike_batch_noalloc (include/nsgw.h)
OPT_BINS_KERNEL, OPT_WALK_SPEC, OPT_LIKELIHOOD, OPT_INNER_KERNEL, OPT_SLICE_STEPS, OPT_WALK_STAGE, OPT_WALK_KERNEL, OPT_HOST_ZERO_COPY = 0, 1, 2, 3, 4, 5, 6, 7

_lib = None


def lib():
    """Loads libnsgw.so (fails loudly if it has not been built: run `python -m paper_2509_04336_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} is missing: build it with `python -m paper_2509_04336_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        L.ns_last_error.restype = C.c_char_p
        L.ns_last_error.argtypes = [C.c_void_p]
        L.ns_run.restype = C.c_int64
        L.ns_run_many.restype = C.c_int64
        L.nsgw_launch_count.restype = C.c_int64
        L.ns_free.restype = None
        L.ns_free.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _ptr(t):
    if t is None:
        return C.c_void_p(0)
    assert t.is_cuda and t.is_contiguous(), "device pointers must be contiguous CUDA tensors"
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _f64(x, device="cuda"):
    return torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64)).to(device)


def make_config(spec, sampler=None):
    """spec / sampler: plain dicts as produced by paper_2509_04336_b200.workloads."""
    c = NsConfig()
    c.struct_version = 1
    c.like_kind = int(spec["like_kind"])
    D = c.ndim = int(spec["ndim"])
    s = sampler or {}
    c.n_live = int(s.get("n_live", 0))
    c.n_delete = int(s.get("n_delete", 0))
    c.naccept = int(s.get("naccept", 60))
    c.maxmcmc = int(s.get("maxmcmc", 5000))
    c.walks0 = float(s.get("walks0", 100.0))
    c.delay = float(s.get("delay", -1.0))
    for d in range(D):
        c.prior_kind[d] = int(spec["prior_kind"][d])
        c.prior_lo[d] = float(spec["prior_lo"][d])
        c.prior_hi[d] = float(spec["prior_hi"][d])
        c.periodic[d] = int(spec["periodic"][d])
    c.n_det = int(spec.get("n_det", 0))
    c.n_freq = int(spec.get("n_freq", 0))
    c.f_min = float(spec.get("f_min", 0.0))
    c.df = float(spec.get("df", 0.0))
    c.gmst = float(spec.get("gmst", 0.0))
    for i in range(c.n_det):
        for j in range(3):
            c.det_vertex[i][j] = float(spec["det_vertex"][i][j])
            c.det_xarm[i][j] = float(spec["det_xarm"][i][j])
            c.det_yarm[i][j] = float(spec["det_yarm"][i][j])
    if "toy_mean" in spec:
        prec = np.asarray(spec["toy_prec"], dtype=np.float64).reshape(D, D)
        for i in range(D):
            c.toy_mean[i] = float(spec["toy_mean"][i])
            for j in range(D):
                c.toy_prec[i * D + j] = prec[i, j]
        c.toy_lognorm = float(spec["toy_lognorm"])
    keep = None
    if spec.get("phenom_table") is not None:
        keep = np.ascontiguousarray(spec["phenom_table"], dtype=np.float64).reshape(19 * 11)
        c.phenom_table_host = keep.ctypes.data_as(C.POINTER(C.c_double))
    return c, keep


class NsgwError(RuntimeError):
    pass


class Handle:
    """RAII wrapper of ns_handle.  All array arguments are CUDA float64 tensors unless stated."""

    def __init__(self, spec, sampler=None, live_u=None, strain=None, psd=None, seed=1):
        L = lib()
        if not torch.cuda.is_available():
            raise NsgwError("no CUDA device: libnsgw has no CPU fallback")
        cfg, keep = make_config(spec, sampler)
        self.cfg = cfg
        self.ndim, self.n_det, self.n_freq = cfg.ndim, cfg.n_det, cfg.n_freq
        self.n_live, self.n_delete = cfg.n_live, cfg.n_delete
        self._h = C.c_void_p(0)
        if strain is None and spec.get("strain") is not None:
            strain = _f64(spec["strain"])
        if psd is None and spec.get("psd") is not None:
            psd = _f64(spec["psd"])
        if live_u is not None and not torch.is_tensor(live_u):
            live_u = _f64(live_u)
        rc = L.ns_init(C.byref(self._h), C.byref(cfg), _ptr(live_u), _ptr(strain), _ptr(psd), C.c_uint64(seed), _stream())
        if rc != 0:
            raise NsgwError(f"ns_init failed ({rc}): {L.ns_last_error(None).decode()}")

    def _check(self, rc, what):
        if rc < 0:
            raise NsgwError(f"{what} failed ({rc}): {lib().ns_last_error(self._h).decode()}")
        return rc

    def close(self):
        if getattr(self, "_h", None) and self._h.value and _lib is not None:
            _lib.ns_free(self._h)
            self._h = C.c_void_p(0)

    __del__ = close

    # ---- likelihood ------------------------------------------------------------------------------
    def gw_loglike_batch(self, theta, parts=False, out=None, parts_out=None):
        B = theta.shape[0]
        logl = out if out is not None else torch.empty(B, dtype=torch.float64, device="cuda")
        pr = parts_out if parts_out is not None else (torch.empty(B, 2 * self.n_det, dtype=torch.float64, device="cuda") if parts else None)
        self._check(lib().gw_loglike_batch(self._h, _ptr(theta), C.c_int64(B), _ptr(logl), _ptr(pr), _stream()), "gw_loglike_batch")
        return (logl, pr) if parts else logl

    def gw_loglike_batch_host(self, theta_host, out_host):
        """theta_host [B, 11], out_host [B]: CPU float64 tensors (pinned for asynchronous copies).  Synchronises."""
        assert (not theta_host.is_cuda) and (not out_host.is_cuda) and theta_host.is_contiguous() and out_host.is_contiguous()
        assert theta_host.dtype == torch.float64 and out_host.dtype == torch.float64
        B = theta_host.shape[0]
        self._check(lib().gw_loglike_batch_host(self._h, C.c_void_p(theta_host.data_ptr()), C.c_int64(B),
                                                C.c_void_p(out_host.data_ptr()), _stream()), "gw_loglike_batch_host")
        return out_host

    def gw_loglike_batch_noalloc(self, theta, out):
        """gw_loglike_batch with the kernels' scratch in the library's fixed device array: no allocation inside the call (the
        caller passes `out` [B]).  B <= NOALLOC_MAX_ROWS, n_freq <= NOALLOC_MAX_BINS, else NsgwError; calls that overlap on the
        GPU race on the shared array."""
        assert theta.dtype == torch.float64 and out.dtype == torch.float64 and out.shape[0] == theta.shape[0]
        self._check(lib().gw_loglike_batch_noalloc(self._h, _ptr(theta), C.c_int64(theta.shape[0]), _ptr(out), _stream()),
                    "gw_loglike_batch_noalloc")
        return out

    def gw_waveform(self, theta):
        out = torch.empty(self.n_det, self.n_freq, 2, dtype=torch.float64, device="cuda")
        self._check(lib().gw_waveform(self._h, _ptr(theta), _ptr(out), _stream()), "gw_waveform")
        return out

    def prior_transform_batch(self, u):
        th = torch.empty_like(u)
        self._check(lib().ns_prior_transform_batch(self._h, _ptr(u), C.c_int64(u.shape[0]), _ptr(th), _stream()), "ns_prior_transform_batch")
        return th

    def loglike_u_batch(self, u):
        logl = torch.empty(u.shape[0], dtype=torch.float64, device="cuda")
        self._check(lib().ns_loglike_u_batch(self._h, _ptr(u), C.c_int64(u.shape[0]), _ptr(logl), _stream()), "ns_loglike_u_batch")
        return logl

    # ---- walk --------------------------------------------------------------------------------------
    def walk_batch(self, donors_u, u, logl, logl_star, walk_len, seed, stream_id, slot0=0, trace=False, counters=True):
        """In place on u / logl.  Returns dict of counters (+ trace)."""
        B = u.shape[0]
        na = torch.zeros(B, dtype=torch.int32, device="cuda") if counters else None
        ne = torch.zeros(B, dtype=torch.int32, device="cuda") if counters else None
        no = torch.zeros(B, dtype=torch.int32, device="cuda") if counters else None
        fl = torch.zeros(B, walk_len, dtype=torch.uint8, device="cuda") if trace else None
        tl = torch.zeros(B, walk_len, dtype=torch.float64, device="cuda") if trace else None
        self._check(lib().ns_walk_batch(self._h, _ptr(donors_u), C.c_int32(donors_u.shape[0]), _ptr(u), _ptr(logl), C.c_int64(B),
                                        C.c_double(logl_star), C.c_int32(walk_len), C.c_uint64(seed), C.c_uint32(stream_id),
                                        C.c_int64(slot0), _ptr(na), _ptr(ne), _ptr(no), _ptr(fl), _ptr(tl), _stream()), "ns_walk_batch")
        out = dict(n_accept=na, n_eval=ne, n_oob=no)
        if trace:
            out["flags"], out["trace_logl"] = fl, tl
        return out

    def slice_batch(self, lc, u, logl, logl_star, n_steps, seed, stream_id, slot0=0, trace=False):
        """In place on u / logl (hit-and-run slice sampling, R:L25).  Returns dict of counters (+ trace)."""
        B = u.shape[0]
        cnt = {k: torch.zeros(B, dtype=torch.int32, device="cuda") for k in ("n_eval", "n_oob", "n_expand", "n_shrink", "n_stuck")}
        te = torch.zeros(B, n_steps, dtype=torch.int32, device="cuda") if trace else None
        tl = torch.zeros(B, n_steps, dtype=torch.float64, device="cuda") if trace else None
        self._check(lib().ns_slice_batch(self._h, _ptr(lc), _ptr(u), _ptr(logl), C.c_int64(B), C.c_double(logl_star), C.c_int32(n_steps),
                                         C.c_uint64(seed), C.c_uint32(stream_id), C.c_int64(slot0), _ptr(cnt["n_eval"]),
                                         _ptr(cnt["n_oob"]), _ptr(cnt["n_expand"]), _ptr(cnt["n_shrink"]), _ptr(cnt["n_stuck"]),
                                         _ptr(te), _ptr(tl), _stream()), "ns_slice_batch")
        out = dict(cnt)
        if trace:
            out["trace_evals"], out["trace_logl"] = te, tl
        return out

    # ---- sampler -----------------------------------------------------------------------------------
    def step(self, want_stats=True, dead=None):
        st = NsStats()
        self._check(lib().ns_step(self._h, C.byref(st) if want_stats else None, _ptr(dead), _stream()), "ns_step")
        return st.as_dict() if want_stats else None

    def run(self, term_kind, term_tol, max_iter, dead=None):
        st = NsStats()
        n = self._check(lib().ns_run(self._h, C.c_int32(term_kind), C.c_double(term_tol), C.c_int64(max_iter), C.byref(st), _ptr(dead),
                                     _stream()), "ns_run")
        return int(n), st.as_dict()

    def get_live(self):
        u = torch.empty(self.n_live, self.ndim, dtype=torch.float64, device="cuda")
        l = torch.empty(self.n_live, dtype=torch.float64, device="cuda")
        self._check(lib().ns_get_live(self._h, _ptr(u), _ptr(l), _stream()), "ns_get_live")
        return u, l

    def get_state(self):
        """ns_get_state: (NsState, live_u, live_logl) -- everything a resumed run needs."""
        st = NsState()
        u = torch.empty(self.n_live, self.ndim, dtype=torch.float64, device="cuda")
        l = torch.empty(self.n_live, dtype=torch.float64, device="cuda")
        self._check(lib().ns_get_state(self._h, C.byref(st), _ptr(u), _ptr(l), _stream()), "ns_get_state")
        return st, u, l

    def set_state(self, st, live_u, live_logl):
        self._check(lib().ns_set_state(self._h, C.byref(st), _ptr(live_u), _ptr(live_logl), _stream()), "ns_set_state")

    def sweep_occupancy(self, rows):
        f, c = C.c_double(), C.c_int32()
        self._check(lib().nsgw_sweep_occupancy(self._h, C.c_int64(rows), C.byref(f), C.byref(c)), "nsgw_sweep_occupancy")
        return f.value, c.value

    def profile_enable(self, on=True):
        self._check(lib().nsgw_profile_enable(self._h, C.c_int32(1 if on else 0)), "nsgw_profile_enable")

    # ---- relative binning ---------------------------------------------------------------------------
    def relbin_setup(self, theta0, chi=1.0, eps=0.5, edges=None):
        th = (C.c_double * 11)(*[float(x) for x in theta0])
        nb = C.c_int32()
        if edges is not None:
            ed = (C.c_int32 * len(edges))(*[int(x) for x in edges])
            rc = lib().ns_relbin_setup(self._h, th, C.c_double(chi), C.c_double(eps), ed, C.c_int32(len(edges)), C.byref(nb), _stream())
        else:
            rc = lib().ns_relbin_setup(self._h, th, C.c_double(chi), C.c_double(eps), None, C.c_int32(0), C.byref(nb), _stream())
        self._check(rc, "ns_relbin_setup")
        self.rb_n_bins = nb.value
        return nb.value

    def relbin_get(self):
        import numpy as np
        nb, nd = self.rb_n_bins, self.n_det
        ed = (C.c_int32 * (nb + 1))()
        sm = (C.c_double * (nd * nb * 6))()
        self._check(lib().ns_relbin_get(self._h, ed, sm, _stream()), "ns_relbin_get")
        a = np.array(sm)
        A0 = a[: nd * nb * 2].reshape(nd, nb, 2)
        A1 = a[nd * nb * 2: nd * nb * 4].reshape(nd, nb, 2)
        B0 = a[nd * nb * 4: nd * nb * 5].reshape(nd, nb)
        B1 = a[nd * nb * 5:].reshape(nd, nb)
        return np.array(ed), A0, A1, B0, B1

    def gw_loglike_relbin_batch(self, theta, parts=False, out=None):
        B = theta.shape[0]
        logl = out if out is not None else torch.empty(B, dtype=torch.float64, device="cuda")
        pr = torch.empty(B, 2 * self.n_det, dtype=torch.float64, device="cuda") if parts else None
        self._check(lib().gw_loglike_relbin_batch(self._h, _ptr(theta), C.c_int64(B), _ptr(logl), _ptr(pr), _stream()),
                    "gw_loglike_relbin_batch")
        return (logl, pr) if parts else logl

    def set_option(self, key, value):
        self._check(lib().nsgw_set_option(self._h, C.c_int32(key), C.c_int32(value)), "nsgw_set_option")

    def profile_read(self):
        ms, n = C.c_double(), C.c_int64()
        self._check(lib().nsgw_profile_read(self._h, C.byref(ms), C.byref(n)), "nsgw_profile_read")
        return ms.value, n.value

    def finalize_evidence(self):
        a, b, c = C.c_double(), C.c_double(), C.c_double()
        self._check(lib().ns_finalize_evidence(self._h, C.byref(a), C.byref(b), C.byref(c), _stream()), "ns_finalize_evidence")
        return a.value, b.value, c.value

    def posterior(self, dead=None, theta_ref=None, want_theta=True):
        """ns_posterior: rows = dead (device [n_dead, ndim+3], optional) + the live points.  Returns a dict with theta [N, ndim]
        (device), logp [N] (device), logz, ess and cl [ndim] (NumPy; NaN without theta_ref)."""
        import numpy as np
        n_dead = 0 if dead is None else int(dead.shape[0])
        N = n_dead + self.n_live
        theta = torch.empty((N, self.ndim), dtype=torch.float64, device="cuda") if (want_theta or theta_ref is not None) else None
        logp = torch.empty(N, dtype=torch.float64, device="cuda")
        summ = (C.c_double * (2 + self.ndim))()
        ref = None
        if theta_ref is not None:
            ref = (C.c_double * self.ndim)(*[float(x) for x in theta_ref])
        self._check(lib().ns_posterior(self._h, _ptr(dead), C.c_int64(n_dead), _ptr(theta), _ptr(logp), ref, summ, _stream()), "ns_posterior")
        return {"theta": theta, "logp": logp, "logz": summ[0], "ess": summ[1], "cl": np.array(summ[2:2 + self.ndim])}

    def posterior_resample(self, logp, n_out, seed, theta=None):
        """ns_posterior_resample: systematic resampling of the weighted rows.  Returns (idx [n_out] int64 device, theta rows or None)."""
        N = int(logp.shape[0])
        cum = torch.empty(N, dtype=torch.float64, device="cuda")
        idx = torch.empty(n_out, dtype=torch.int64, device="cuda")
        out = torch.empty((n_out, self.ndim), dtype=torch.float64, device="cuda") if theta is not None else None
        self._check(lib().ns_posterior_resample(self._h, _ptr(logp), _ptr(theta), C.c_int64(N), C.c_int64(n_out), C.c_uint64(seed),
                                                _ptr(cum), _ptr(idx), _ptr(out), _stream()), "ns_posterior_resample")
        return idx, out


def run_many(handles, term_kind, term_tol, max_iter, dead=None):
    """ns_run_many: steps the handles' samplers concurrently (one stream each).  Returns (iterations per run, stats per run)."""
    n = len(handles)
    hs = (C.c_void_p * n)(*[h._h for h in handles])
    st = (NsStats * n)()
    its = (C.c_int64 * n)()
    dd = None
    if dead is not None:
        dd = (C.c_void_p * n)(*[C.c_void_p(d.data_ptr()) if d is not None else C.c_void_p(0) for d in dead])
    rc = lib().ns_run_many(hs, C.c_int32(n), C.c_int32(term_kind), C.c_double(term_tol), C.c_int64(max_iter), st, its, dd)
    if rc < 0:
        msgs = "; ".join(lib().ns_last_error(h._h).decode() for h in handles)
        raise NsgwError(f"ns_run_many failed ({rc}): {msgs}")
    return [int(x) for x in its], [s_.as_dict() for s_ in st]


def measure_fp64_peak(iters=1 << 18):
    t = C.c_double()
    rc = lib().nsgw_measure_fp64_peak(C.c_int64(iters), C.byref(t), _stream())
    if rc != 0:
        raise NsgwError(f"nsgw_measure_fp64_peak failed ({rc})")
    return t.value


def launch_count():
    return int(lib().nsgw_launch_count())
