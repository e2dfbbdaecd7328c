"""ctypes front end of liboracle.so -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from paper_2509_04336_b200 (the CUDA path) and the CUDA path imports nothing from here.
Every function is a thin call into oracle.cpp, whose header lists what pins each part, except the posterior weights and the
systematic resampling at the end of this file (readings R:L26, R:L27), written out here in NumPy/math.fsum and pinned by
tests/test_oracle_posterior.py.
"""
import math

import ctypes as C
import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())

c_d_p = C.POINTER(C.c_double)


class Problem(C.Structure):
    _fields_ = [
        ("like_kind", C.c_int32), ("ndim", C.c_int32),
        ("prior_kind", C.c_int32 * 16), ("prior_lo", C.c_double * 16), ("prior_hi", C.c_double * 16),
        ("periodic", C.c_int32 * 16),
        ("n_det", C.c_int32), ("n_freq", C.c_int32), ("f_min", C.c_double), ("df", C.c_double),
        ("det_vertex", (C.c_double * 3) * 4), ("det_xarm", (C.c_double * 3) * 4), ("det_yarm", (C.c_double * 3) * 4),
        ("gmst", C.c_double),
        ("toy_mean", C.c_double * 16), ("toy_prec", C.c_double * 256), ("toy_lognorm", C.c_double),
        ("phenom_table", (C.c_double * 11) * 19),
        ("strain", c_d_p), ("psd", c_d_p),
        ("relbin", C.c_void_p),
    ]


class SamplerCfg(C.Structure):
    _fields_ = [("n_live", C.c_int32), ("n_delete", C.c_int32), ("naccept", C.c_int32), ("maxmcmc", C.c_int32),
                ("walks0", C.c_double), ("delay", C.c_double)]


class Stats(C.Structure):
    _fields_ = [("iteration", C.c_int64), ("logl_star", C.c_double), ("logx", C.c_double), ("logz", C.c_double),
                ("h", C.c_double), ("dlogz", C.c_double), ("live_frac_log", C.c_double), ("walk_len", C.c_int32),
                ("walks_next", C.c_double), ("accept_mean", C.c_double), ("accept_min", C.c_int32),
                ("accept_max", C.c_int32), ("n_eval", C.c_int64), ("n_oob", C.c_int64), ("n_stuck", C.c_int64),
                ("n_eval_total", C.c_int64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def _dp(a):
    return a.ctypes.data_as(c_d_p) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class OracleProblem:
    """Holds an orc_problem plus the numpy arrays it points to.  `spec` is the plain dict made by
    paper_2509_04336_b200.workloads (inputs only: priors, detector geometry, grid, table, strain, psd)."""

    def __init__(self, spec):
        p = Problem()
        p.like_kind = int(spec["like_kind"])
        D = p.ndim = int(spec["ndim"])
        for d in range(D):
            p.prior_kind[d] = int(spec["prior_kind"][d])
            p.prior_lo[d] = float(spec["prior_lo"][d])
            p.prior_hi[d] = float(spec["prior_hi"][d])
            p.periodic[d] = int(spec["periodic"][d])
        p.n_det = int(spec.get("n_det", 0))
        p.n_freq = int(spec.get("n_freq", 0))
        p.f_min = float(spec.get("f_min", 0.0))
        p.df = float(spec.get("df", 0.0))
        p.gmst = float(spec.get("gmst", 0.0))
        for i in range(p.n_det):
            for j in range(3):
                p.det_vertex[i][j] = float(spec["det_vertex"][i][j])
                p.det_xarm[i][j] = float(spec["det_xarm"][i][j])
                p.det_yarm[i][j] = float(spec["det_yarm"][i][j])
        if "toy_mean" in spec:
            for d in range(D):
                p.toy_mean[d] = float(spec["toy_mean"][d])
            prec = _f64(spec["toy_prec"]).reshape(D, D)
            for i in range(D):
                for j in range(D):
                    p.toy_prec[i * D + j] = prec[i, j]
            p.toy_lognorm = float(spec["toy_lognorm"])
        if spec.get("phenom_table") is not None:
            tab = _f64(spec["phenom_table"]).reshape(19, 11)
            for i in range(19):
                for j in range(11):
                    p.phenom_table[i][j] = tab[i, j]
        self.strain = _f64(spec["strain"]) if spec.get("strain") is not None else None
        self.psd = _f64(spec["psd"]) if spec.get("psd") is not None else None
        p.strain = _dp(self.strain)
        p.psd = _dp(self.psd)
        self.p = p
        self.ndim = D
        self.n_det = p.n_det
        self.n_freq = p.n_freq

    def set_data(self, strain, psd):
        self.strain = _f64(strain)
        self.psd = _f64(psd)
        self.p.strain = _dp(self.strain)
        self.p.psd = _dp(self.psd)

    # ---- pieces -------------------------------------------------------------------------------
    def prior_transform(self, u):
        u = _f64(u).reshape(-1, self.ndim)
        th = np.empty_like(u)
        _lib.orc_prior_transform(C.byref(self.p), _dp(u), C.c_int64(u.shape[0]), _dp(th))
        return th

    def detector_response(self, det, ra, dec, psi):
        out = np.empty(3)
        _lib.orc_detector_response(C.byref(self.p), C.c_int(det), C.c_double(ra), C.c_double(dec), C.c_double(psi), _dp(out))
        return out  # F+, Fx, dt

    def amp_phase(self, theta, f):
        theta = _f64(theta)
        f = _f64(f)
        amp = np.empty_like(f)
        psi = np.empty_like(f)
        _lib.orc_amp_phase(C.byref(self.p), _dp(theta), _dp(f), C.c_int64(f.size), _dp(amp), _dp(psi))
        return amp, psi

    def phenomd_info(self, theta):
        out = np.empty(29)
        _lib.orc_phenomd_info(C.byref(self.p), _dp(_f64(theta)), _dp(out))
        keys = ["Frd", "Fdamp", "Fpeak", "t0", "C1int", "C2int", "C1mr", "C2mr", "M", "eta"]
        d = dict(zip(keys, out[:10]))
        d["Lambda"] = out[10:].copy()
        return d

    def waveform(self, theta):
        out = np.empty((self.n_det, self.n_freq, 2))
        _lib.orc_waveform(C.byref(self.p), _dp(_f64(theta)), _dp(out))
        return out

    def gw_loglike(self, theta, parts=False, threads=0):
        theta = _f64(theta).reshape(-1, 11)
        B = theta.shape[0]
        logl = np.empty(B)
        pr = np.empty((B, 2 * self.n_det)) if parts else None
        _lib.orc_gw_loglike(C.byref(self.p), _dp(theta), C.c_int64(B), _dp(logl), _dp(pr), C.c_int(threads))
        return (logl, pr) if parts else logl

    # ---- hit-and-run slice sampling inner kernel (DESIGN.md R:L25) --------------------------------------
    def slice_walk(self, Lc, u, logl, logl_star, S, seed, stream_id, slot0=0, trace=False, threads=0):
        """Copies of u / logl are evolved by S slice steps each; Lc [ndim, ndim] lower-triangular direction factor."""
        u = _f64(u).reshape(-1, self.ndim).copy()
        logl = _f64(logl).copy()
        Lc = _f64(Lc).reshape(self.ndim, self.ndim)
        B = u.shape[0]
        cnt = {k: np.zeros(B, dtype=np.int32) for k in ("n_eval", "n_oob", "n_expand", "n_shrink", "n_stuck")}
        te = np.zeros((B, S), dtype=np.int32) if trace else None
        tl = np.zeros((B, S)) if trace else None
        ip = lambda a: a.ctypes.data_as(C.POINTER(C.c_int32)) if a is not None else None
        _lib.orc_slice_walk(C.byref(self.p), _dp(Lc), _dp(u), _dp(logl), C.c_int64(B), C.c_double(logl_star), C.c_int32(S),
                            C.c_uint64(seed), C.c_uint32(stream_id), C.c_int64(slot0), ip(cnt["n_eval"]), ip(cnt["n_oob"]),
                            ip(cnt["n_expand"]), ip(cnt["n_shrink"]), ip(cnt["n_stuck"]), ip(te), _dp(tl), C.c_int(threads))
        out = dict(u=u, logl=logl, **cnt)
        if trace:
            out["trace_evals"], out["trace_logl"] = te, tl
        return out

    # ---- relative binning (DESIGN.md R:L24) ----------------------------------------------------------
    def relbin(self, theta0, chi=1.0, eps=0.5):
        return OracleRelBin(self, theta0, chi, eps)

    def live_cholesky(self, pts):
        pts = _f64(pts).reshape(-1, self.ndim)
        Lc = np.zeros((self.ndim, self.ndim))
        _lib.orc_live_cholesky(C.byref(self.p), _dp(pts), C.c_int32(pts.shape[0]), _dp(Lc))
        return Lc

    def use_relbin(self, rb):
        """Routes loglike_u, walk and the sampler through the relative-binning likelihood `rb` (None: back to the exact one)."""
        self._rb_in_use = rb                      # keep it alive
        self.p.relbin = rb.h if rb is not None else None

    def loglike_u(self, u, threads=0):
        u = _f64(u).reshape(-1, self.ndim)
        logl = np.empty(u.shape[0])
        _lib.orc_loglike_u(C.byref(self.p), _dp(u), C.c_int64(u.shape[0]), _dp(logl), C.c_int(threads))
        return logl

    def walk(self, surv_u, u, logl, logl_star, W, seed, stream_id, slot0=0, trace=False, threads=0):
        surv_u = _f64(surv_u).reshape(-1, self.ndim)
        u = _f64(u).reshape(-1, self.ndim).copy()
        logl = _f64(logl).copy()
        B = u.shape[0]
        na = np.zeros(B, np.int32)
        ne = np.zeros(B, np.int32)
        no = np.zeros(B, np.int32)
        fl = np.zeros((B, W), np.uint8) if trace else None
        tl = np.zeros((B, W)) if trace else None
        ip = C.POINTER(C.c_int32)
        _lib.orc_walk(C.byref(self.p), _dp(surv_u), C.c_int32(surv_u.shape[0]), _dp(u), _dp(logl), C.c_int64(B),
                      C.c_double(logl_star), C.c_int32(W), C.c_uint64(seed), C.c_uint32(stream_id), C.c_int64(slot0),
                      na.ctypes.data_as(ip), ne.ctypes.data_as(ip), no.ctypes.data_as(ip),
                      fl.ctypes.data_as(C.POINTER(C.c_uint8)) if trace else None, _dp(tl), C.c_int(threads))
        out = dict(u=u, logl=logl, n_accept=na, n_eval=ne, n_oob=no)
        if trace:
            out["flags"] = fl
            out["trace_logl"] = tl
        return out


class OracleSampler:
    def __init__(self, prob: OracleProblem, n_live, n_delete, naccept, maxmcmc=5000, walks0=100.0, delay=-1.0,
                 live_u=None, seed=1, threads=0):
        self.prob = prob
        self.cfg = SamplerCfg(n_live, n_delete, naccept, maxmcmc, walks0, delay)
        lu = _f64(live_u) if live_u is not None else None
        _lib.orc_state_create.restype = C.c_void_p
        self.h = C.c_void_p(_lib.orc_state_create(C.byref(prob.p), C.byref(self.cfg), _dp(lu), C.c_uint64(seed), C.c_int(threads)))
        self.n_live, self.n_delete, self.ndim = n_live, n_delete, prob.ndim

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.orc_state_free(self.h)
            self.h = None

    def use_slice_kernel(self, n_slice):
        """Replacements by n_slice hit-and-run slice steps (R:L25) instead of the acceptance walk (n_slice = 0: back to the walk)."""
        _lib.orc_state_set_inner(self.h, C.c_int32(1 if n_slice > 0 else 0), C.c_int32(n_slice))

    def live(self):
        u = np.empty((self.n_live, self.ndim))
        l = np.empty(self.n_live)
        _lib.orc_state_get_live(self.h, _dp(u), _dp(l))
        return u, l

    def step(self, want_dead=False):
        st = Stats()
        dead = np.empty((self.n_delete, self.ndim + 3)) if want_dead else None
        _lib.orc_step(self.h, C.byref(st), _dp(dead))
        return (st.as_dict(), dead) if want_dead else st.as_dict()

    def run(self, term_kind, tol, max_iter, want_dead=False):
        st = Stats()
        dead = np.empty((max_iter * self.n_delete, self.ndim + 3)) if want_dead else None
        _lib.orc_run.restype = C.c_int64
        n = _lib.orc_run(self.h, C.c_int32(term_kind), C.c_double(tol), C.c_int64(max_iter), C.byref(st), _dp(dead))
        if want_dead:
            return n, st.as_dict(), dead[: n * self.n_delete]
        return n, st.as_dict()

    def finalize(self):
        a, b, c = C.c_double(), C.c_double(), C.c_double()
        _lib.orc_finalize(self.h, C.byref(a), C.byref(b), C.byref(c))
        return a.value, b.value, c.value  # logZ, err, H


class OracleRelBin:
    """Relative-binning summary data about a fiducial theta0 and the approximate likelihood built on them."""

    def __init__(self, problem, theta0, chi, eps):
        self.P = problem
        _lib.orc_relbin_create.restype = C.c_void_p
        self.h = C.c_void_p(_lib.orc_relbin_create(C.byref(problem.p), _dp(_f64(theta0)), C.c_double(chi), C.c_double(eps)))
        if not self.h.value:
            raise ValueError("orc_relbin_create failed (unphysical theta0 or bad chi/eps)")
        _lib.orc_relbin_nbins.restype = C.c_int32
        self.n_bins = int(_lib.orc_relbin_nbins(self.h))

    def __del__(self):
        if getattr(self, "h", None) and self.h.value:
            _lib.orc_relbin_free(self.h)
            self.h = C.c_void_p(0)

    def edges(self):
        e = np.empty(self.n_bins + 1, dtype=np.int32)
        _lib.orc_relbin_edges(self.h, e.ctypes.data_as(C.POINTER(C.c_int32)))
        return e

    def summary(self):
        nd, nb = self.P.n_det, self.n_bins
        A0, A1 = np.empty((nd, nb, 2)), np.empty((nd, nb, 2))
        B0, B1 = np.empty((nd, nb)), np.empty((nd, nb))
        _lib.orc_relbin_summary(self.h, _dp(A0), _dp(A1), _dp(B0), _dp(B1))
        return A0, A1, B0, B1

    def loglike(self, theta, parts=False, threads=0):
        theta = _f64(theta).reshape(-1, 11)
        B = theta.shape[0]
        logl = np.empty(B)
        pr = np.empty((B, 2 * self.P.n_det)) if parts else None
        _lib.orc_relbin_loglike(C.byref(self.P.p), self.h, _dp(theta), C.c_int64(B), _dp(logl), _dp(pr), C.c_int(threads))
        return (logl, pr) if parts else logl


# ---- free functions ---------------------------------------------------------------------------
def philox(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) for x in key])
    o = (C.c_uint32 * 4)()
    _lib.orc_philox(c, k, o)
    return [int(x) for x in o]


_lib.orc_u53.restype = C.c_double
_lib.orc_mulhi32.restype = C.c_uint32
_lib.orc_gamma_draw.restype = C.c_double
_lib.orc_neff.restype = C.c_double


def u53(hi, lo):
    return _lib.orc_u53(C.c_uint32(hi), C.c_uint32(lo))


def mulhi32(w, m):
    return _lib.orc_mulhi32(C.c_uint32(w), C.c_uint32(m))


def gamma_draw(n_free, seed, t, j, stream_id, m):
    a, b, one = C.c_int32(), C.c_int32(), C.c_int32()
    g = _lib.orc_gamma_draw(C.c_int(n_free), C.c_uint64(seed), C.c_uint32(t), C.c_uint32(j), C.c_uint32(stream_id),
                            C.c_int32(m), C.byref(a), C.byref(b), C.byref(one))
    return g, a.value, b.value, bool(one.value)


def draw_live(ndim, n, seed):
    u = np.empty((n, ndim))
    _lib.orc_draw_live(C.c_int32(ndim), C.c_int64(n), C.c_uint64(seed), _dp(u))
    return u


def argsort(x):
    x = _f64(x)
    idx = np.empty(x.size, np.int32)
    _lib.orc_argsort(_dp(x), C.c_int64(x.size), idx.ctypes.data_as(C.POINTER(C.c_int32)))
    return idx


def evidence_update(logl_i, n_i, logx, logz, h):
    lx, lz, hh, lw = C.c_double(logx), C.c_double(logz), C.c_double(h), C.c_double()
    _lib.orc_evidence_update(C.c_double(logl_i), C.c_double(n_i), C.byref(lx), C.byref(lz), C.byref(hh), C.byref(lw))
    return lx.value, lz.value, hh.value, lw.value


def neff(n, k):
    return _lib.orc_neff(C.c_int32(n), C.c_int32(k))


# ---- posterior weights ("posterior samples as a natural by-product", "weights ... calculated using the prior volumes
#      enclosed between successive dead points and the likelihoods"; DESIGN reading R:L26) ---------------------------------------
def posterior_rows(dead, live_u, live_logl, logx):
    """The sample set of a run: the recorded dead points ([n_dead, D+3] rows u.., logL, log w, n_i as orc_step writes them)
    followed by the live points in ascending logL, whose widths continue the shrinkage from logx with n_i = n, n-1, .., 1
    (R:L17: log w_i = logX_{i-1} + log(1 - exp(-1/n_i)), logX_i = logX_{i-1} - 1/n_i).  Returns u [N, D], logL [N], log w [N]."""
    live_u = _f64(live_u)
    live_logl = _f64(live_logl)
    n, D = live_u.shape
    dead = np.zeros((0, D + 3)) if dead is None else _f64(dead).reshape(-1, D + 3)
    order = argsort(live_logl)
    lw = np.empty(n)
    lx = float(logx)
    for j in range(n):
        nj = float(n - j)
        lw[j] = lx + math.log(-math.expm1(-1.0 / nj))
        lx -= 1.0 / nj
    u = np.concatenate([dead[:, :D], live_u[order]])
    logl = np.concatenate([dead[:, D], live_logl[order]])
    logw = np.concatenate([dead[:, D + 1], lw])
    return u, logl, logw


def posterior_weights(logl, logw):
    """log p_i = logL_i + log w_i - logZ with logZ = log sum_i L_i w_i over the rows (R:L26).  Returns (log p, logZ)."""
    t = _f64(logl) + _f64(logw)
    m = float(np.max(t))
    logz = m + math.log(math.fsum(np.exp(t - m).tolist()))
    return t - logz, logz


def posterior(prob, dead, live_u, live_logl, logx, theta_ref=None):
    """Weighted posterior sample of a run (R:L26): theta = prior transform of every row, log p, logZ over the rows, Kish's
    effective sample size 1 / sum p_i^2 and, for a reference point, the credible level of each parameter
    CL_d = sum_i p_i [theta_i,d < theta_ref,d] (the statistic a PP test histograms)."""
    u, logl, logw = posterior_rows(dead, live_u, live_logl, logx)
    logp, logz = posterior_weights(logl, logw)
    theta = prob.prior_transform(u)
    pw = np.exp(logp)
    out = {"theta": theta, "logp": logp, "logz": logz, "ess": 1.0 / math.fsum((pw * pw).tolist())}
    if theta_ref is not None:
        ref = _f64(theta_ref)
        out["cl"] = np.array([math.fsum(pw[theta[:, d] < ref[d]].tolist()) for d in range(theta.shape[1])])
    return out


def posterior_resample(logp, n_out, seed):
    """Equal-weight posterior sample by systematic resampling (reading R:L27): one uniform U = u53(w0, w1) from the Philox block
    with counter (0, 0, 0, 4 << 24) and key = seed; positions t_j = (j + U) / n_out, j = 0..n_out-1; C_i = p_0 + .. + p_i in row
    order; row of draw j = the first i with C_i > t_j C_{N-1}.  Row i is drawn floor(n_out p_i) or ceil(n_out p_i) times.
    Returns (idx [n_out] int64, U)."""
    w = philox([0, 0, 0, 4 << 24], [seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF])
    U = u53(w[0], w[1])
    cum = np.cumsum(np.exp(_f64(logp)))
    t = (np.arange(n_out) + U) / n_out
    idx = np.searchsorted(cum, t * cum[-1], side="right")
    return np.minimum(idx, cum.size - 1).astype(np.int64), U
