"""Seeded synthetic INPUT generators shared by the CUDA path and the CPU oracle.

This module holds inputs only -- prior boxes, detector geometry, frequency grids, the analytic PSD shape,
coloured Gaussian noise, the surrogate fit table and the sampler settings of the five BASELINE.json
configs -- and none of the method's arithmetic (no waveform, no likelihood, no prior transform, no walk).
Wherever an input needs the method itself (the injected signal in the strain), the caller passes that in as a
callback: tests pass the oracle's waveform, bench.py's product leg passes the CUDA library's.

The paper's workloads (bilby-injected BBH signals in O4-design noise; priors of Table 1,
P:157-170; n_live/num_delete of P:196) are not available offline; these shapes and distributions
stand in for them.  DESIGN.md section 4 states the recipe.
"""
import math
import numpy as np

# like_kind / prior kinds (plain integers of the C-ABI; include/nsgw.h)
LIKE_GAUSS, LIKE_TAYLORF2, LIKE_PHENOMD, LIKE_SHELL = 0, 1, 2, 3
UNIFORM, POWERLAW2, SINE, COSINE, FIXED = 0, 1, 2, 3, 4

PARAM_NAMES = ["Mc", "q", "chi1", "chi2", "dL", "theta_jn", "psi", "phase", "tc", "ra", "dec"]

# Earth-fixed detector geometry (public LIGO/Virgo values): vertex [m], x-arm, y-arm unit vectors.
DETECTORS = {
    "H1": ((-2.16141492636e6, -3.83469517889e6, 4.60035022664e6),
           (-0.22389266154, 0.79983062746, 0.55690487831),
           (-0.91397818574, 0.02609403989, -0.40492342125)),
    "L1": ((-7.42760447238e4, -5.49628371971e6, 3.22425701744e6),
           (-0.95457412153, -0.14158077340, -0.26218911324),
           (0.29774156894, -0.48791033647, -0.82054461286)),
    "V1": ((4.54637409900e6, 8.42989697626e5, 4.37857696241e6),
           (-0.70045821479, 0.20848948619, 0.68256166277),
           (-0.05379255368, -0.96908180549, 0.24080451708)),
}
PSD_FACTOR = {"H1": 1.0, "L1": 1.0, "V1": 2.25}
GMST = 2.0
DATA_SEED = 20250904

# Surrogate fit table [19][11] (rows rho1..3, v2, gamma1..3, sigma1..4, beta1..3, alpha1..5; columns
# lambda00, lambda10, then nine spin columns = 0).  Synthetic constants of this build (DESIGN.md A.2).
_SURR = [
    (3931.9, -17395.8), (-40105.5, 112253.0), (83208.4, -191237.7), (0.81498, 2.57476),
    (0.0069274, 0.0302047), (1.010344, 0.000899), (1.308162, -0.005538),
    (2096.55, 1463.75), (-10114.06, -44631.0), (22933.66, 230960.0), (-14621.7, -377812.9),
    (97.8975, -42.6597), (-3.28270, -9.05138), (-2.51564e-5, 1.97503e-5),
    (43.3151, 638.633), (-0.0702021, -0.162698), (9.59881, -397.054), (-0.0298949, 1.40221),
    (0.997441, -0.00788445),
]


def surrogate_table():
    t = np.zeros((19, 11))
    for i, (a, b) in enumerate(_SURR):
        t[i, 0], t[i, 1] = a, b
    return t


def analytic_psd(f):
    """aLIGO-design-like analytic one-sided PSD shape S_a(f) [1/Hz] (positive on 20-2048 Hz)."""
    x = np.asarray(f, dtype=np.float64) / 215.0
    return 1e-49 * (x ** -4.14 - 5.0 * x ** -2 + 111.0 * (1.0 - x ** 2 + 0.5 * x ** 4) / (1.0 + 0.5 * x ** 2))


def freq_grid(f_min, f_max, T):
    df = 1.0 / T
    n = int(round((f_max - f_min) / df)) + 1
    return f_min, df, n


def gw_priors(mc_lo, mc_hi):
    kind = [UNIFORM, UNIFORM, UNIFORM, UNIFORM, POWERLAW2, SINE, UNIFORM, UNIFORM, UNIFORM, UNIFORM, COSINE]
    lo = [mc_lo, 0.125, -0.99, -0.99, 100.0, 0.0, 0.0, 0.0, -0.1, 0.0, -math.pi / 2]
    hi = [mc_hi, 1.0, 0.99, 0.99, 5000.0, math.pi, math.pi, 2 * math.pi, 0.1, 2 * math.pi, math.pi / 2]
    periodic = [0, 0, 0, 0, 0, 0, 1, 1, 0, 1, 0]  # psi, phase, ra
    return kind, lo, hi, periodic


def gw_spec(like_kind, dets, T, f_max, mc_range, f_min=20.0):
    """Problem description (no data yet) for a GW config."""
    f0, df, n = freq_grid(f_min, f_max, T)
    kind, lo, hi, per = gw_priors(*mc_range)
    return dict(
        like_kind=like_kind, ndim=11, prior_kind=kind, prior_lo=lo, prior_hi=hi, periodic=per,
        n_det=len(dets), n_freq=n, f_min=f0, df=df, gmst=GMST, det_names=list(dets),
        det_vertex=[DETECTORS[d][0] for d in dets], det_xarm=[DETECTORS[d][1] for d in dets],
        det_yarm=[DETECTORS[d][2] for d in dets], phenom_table=surrogate_table(), strain=None, psd=None,
    )


def noise(spec, psd, seed=DATA_SEED):
    """Coloured Gaussian noise n_k = sqrt(S_k/(4 df)) (g1 + i g2), shape [n_det, n_freq, 2]."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    g = rng.standard_normal((spec["n_det"], spec["n_freq"], 2))
    return g * np.sqrt(psd / (4.0 * spec["df"]))[:, :, None]


def make_data(spec, theta_inj, snr, waveform_fn, seed=DATA_SEED, with_noise=True):
    """Fills spec['psd'] and spec['strain'].  waveform_fn(spec_with_psd, theta) -> h[n_det, n_freq, 2] is the
    caller's implementation of the detector-frame signal (oracle in tests, CUDA library in bench.py).
    The PSD is kappa * S_a(f) (V1: 2.25 S_a) with kappa chosen so the injection's optimal network SNR
    sqrt(sum_det 4 df sum_k |h|^2/S) equals `snr` exactly."""
    f = spec["f_min"] + spec["df"] * np.arange(spec["n_freq"])
    base = np.stack([PSD_FACTOR[d] * analytic_psd(f) for d in spec["det_names"]])
    spec = dict(spec)
    spec["psd"] = base
    h = np.asarray(waveform_fn(spec, np.asarray(theta_inj, dtype=np.float64)))
    rho2 = 4.0 * spec["df"] * float(np.sum((h[..., 0] ** 2 + h[..., 1] ** 2) / base))
    kappa = rho2 / snr ** 2
    spec["psd"] = base * kappa
    spec["kappa"] = kappa
    spec["theta_inj"] = np.asarray(theta_inj, dtype=np.float64)
    spec["strain"] = h + (noise(spec, spec["psd"], seed) if with_noise else 0.0)
    return spec


def uniforms(n, ndim, seed):
    """Unit-cube rows for likelihood microbenchmarks (config 2): plain seeded uniforms in (0,1)."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    return rng.random((n, ndim)) * (1.0 - 2e-12) + 1e-12


def uniform_rows(lo, hi, ndim, seed):
    """Rows lo..hi-1 of an index-keyed stream of unit-cube rows: row i is the same whatever range it is drawn in, so a
    multi-GPU run that shards rows by global index sees exactly the rows of a single-GPU run (numpy Philox, counter
    advanced to the row)."""
    # numpy's Philox yields 4 doubles per counter step: start at the enclosing block boundary and slice
    bg = np.random.Philox(key=seed)
    first = (lo * ndim) // 4
    bg.advance(first)
    rng = np.random.Generator(bg)
    skip = lo * ndim - 4 * first
    flat = rng.random(skip + (hi - lo) * ndim)[skip:]
    return flat.reshape(hi - lo, ndim) * (1.0 - 2e-12) + 1e-12


# ------------------------------------------------------------------------------------------------------
# BASELINE.json configs
# ------------------------------------------------------------------------------------------------------
INJ_C3 = [28.0, 0.8, 0.3, -0.2, 800.0, 0.40, 2.66, 1.30, 0.0, 1.38, -1.21]   # Table 2 angles
INJ_C4 = [10.0, 0.7, -0.34, 0.01, 500.0, 1.30, 1.83, 5.21, 0.0, 1.07, -1.01]  # Table 4


def givens_cov():
    """Config-1 covariance: Q diag(0.05, 0.36667, 0.68333, 1.0) Q^T, Q = product of Givens rotations over the
    pairs (i<j) in lexicographic order, angle 0.3 + 0.4 t for t = 1..6."""
    Q = np.eye(4)
    t = 0
    for i in range(4):
        for j in range(i + 1, 4):
            t += 1
            a = 0.3 + 0.4 * t
            G = np.eye(4)
            G[i, i] = G[j, j] = math.cos(a)
            G[i, j] = -math.sin(a)
            G[j, i] = math.sin(a)
            Q = Q @ G
    lam = np.array([0.05, 0.36667, 0.68333, 1.0])
    return Q @ np.diag(lam) @ Q.T, lam


def config1():
    """Toy NS: 4-D correlated normalised Gaussian in the box [-10,10]^4 (closed form logZ = -4 ln 20)."""
    cov, lam = givens_cov()
    prec = np.linalg.inv(cov)
    lognorm = -0.5 * (4 * math.log(2 * math.pi) + float(np.sum(np.log(lam))))
    spec = dict(like_kind=LIKE_GAUSS, ndim=4, prior_kind=[UNIFORM] * 4, prior_lo=[-10.0] * 4, prior_hi=[10.0] * 4,
                periodic=[0] * 4, toy_mean=[0.0] * 4, toy_prec=prec, toy_lognorm=lognorm, n_det=0, n_freq=0)
    sampler = dict(n_live=200, n_delete=50, naccept=20, maxmcmc=5000, walks0=100.0, delay=-1.0, term_kind=0, term_tol=0.01)
    return spec, sampler, dict(logz_exact=-4.0 * math.log(20.0))


def config2(waveform_fn, with_noise=True):
    """Likelihood microbench: TaylorF2, H1+L1, 4 s, 20-1024 Hz (4017 bins), SNR 20."""
    spec = gw_spec(LIKE_TAYLORF2, ["H1", "L1"], 4.0, 1024.0, (20.0, 40.0))
    return make_data(spec, INJ_C3, 20.0, waveform_fn, with_noise=with_noise)


def config3(waveform_fn):
    spec = gw_spec(LIKE_PHENOMD, ["H1", "L1"], 4.0, 1024.0, (20.0, 40.0))
    spec = make_data(spec, INJ_C3, 20.0, waveform_fn)
    sampler = dict(n_live=1000, n_delete=500, naccept=60, maxmcmc=5000, walks0=100.0, delay=-1.0, term_kind=0, term_tol=0.1)
    return spec, sampler


def config4(waveform_fn):
    spec = gw_spec(LIKE_PHENOMD, ["H1", "L1"], 8.0, 2048.0, (8.0, 20.0))
    spec = make_data(spec, INJ_C4, 15.0, waveform_fn)
    sampler = dict(n_live=1400, n_delete=700, naccept=60, maxmcmc=5000, walks0=100.0, delay=-1.0, term_kind=1, term_tol=1e-3)
    return spec, sampler


# unit-cube image of INJ_C4 under the config-4/5 prior box (checked against the oracle's transform in tests)
U_INJ_C4 = [1.0 / 6.0, 0.575 / 0.875, 0.65 / 1.98, 1.0 / 1.98, (500.0 ** 3 - 100.0 ** 3) / (5000.0 ** 3 - 100.0 ** 3),
            0.5 * (1.0 - math.cos(1.30)), 1.83 / math.pi, 5.21 / (2 * math.pi), 0.5, 1.07 / (2 * math.pi),
            0.5 * (1.0 + math.sin(-1.01))]
C5_SIGMA = [0.01, 0.1, 0.15, 0.2, 0.1, 0.1, 0.15, 0.25, 0.005, 0.02, 0.02]


def config5(waveform_fn):
    spec = gw_spec(LIKE_PHENOMD, ["H1", "L1", "V1"], 16.0, 2048.0, (8.0, 20.0))
    return make_data(spec, INJ_C4, 15.0, waveform_fn)


def config5_live(spec, n, seed=5, u_inj=U_INJ_C4):
    """Live set of n unit-cube points scattered about the injection's unit-cube image: u_inj + sigma * z,
    periodic dims wrapped, the rest clipped into (0,1)."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    z = rng.standard_normal((n, 11))
    u = np.asarray(u_inj)[None, :] + np.asarray(C5_SIGMA)[None, :] * z
    per = np.asarray(spec["periodic"], dtype=bool)
    u[:, per] = u[:, per] - np.floor(u[:, per])
    u[:, ~per] = np.clip(u[:, ~per], 1e-9, 1.0 - 1e-9)
    return u


def shell_spec(ndim, periodic=None):
    """Cube-shell test likelihood L(u) = -max_d |u_d - 1/2| (walk-uniformity / volume pins)."""
    return dict(like_kind=LIKE_SHELL, ndim=ndim, prior_kind=[UNIFORM] * ndim, prior_lo=[0.0] * ndim, prior_hi=[1.0] * ndim,
                periodic=list(periodic) if periodic is not None else [0] * ndim, n_det=0, n_freq=0)


def fix_dims(spec, free, theta_fixed):
    """Copy of a GW spec with every parameter outside `free` FIXED at theta_fixed (periodic flags cleared on fixed dims)."""
    spec = dict(spec)
    kinds, lo, hi, per = list(spec["prior_kind"]), list(spec["prior_lo"]), list(spec["prior_hi"]), list(spec["periodic"])
    for d in range(spec["ndim"]):
        if d not in free:
            kinds[d] = FIXED
            lo[d] = hi[d] = float(theta_fixed[d])
            per[d] = 0
    spec["prior_kind"], spec["prior_lo"], spec["prior_hi"], spec["periodic"] = kinds, lo, hi, per
    return spec


def pp_problem_set(spec, n_inj, seed, waveform_fn, prior_transform_fn):
    """Stand-in for the paper's 100-injection study: n_inj signals drawn from the prior of `spec` (which carries its PSD),
    each in its own noise realisation.  Row i of the Philox(seed) uniforms goes through the caller's prior transform
    (prior_transform_fn(spec, u[n, ndim]) -> theta[n, ndim]) and waveform (waveform_fn(spec, theta) -> h[n_det, n_freq, 2]); the
    strain is h + noise(seed + 1 + i).  Returns (list of specs, theta[n_inj, ndim])."""
    u = uniforms(n_inj, spec["ndim"], seed)
    theta = np.asarray(prior_transform_fn(spec, u), dtype=np.float64)
    out = []
    for i in range(n_inj):
        s = dict(spec)
        s["theta_inj"] = theta[i].copy()
        s["strain"] = np.asarray(waveform_fn(spec, theta[i])) + noise(spec, spec["psd"], seed + 1 + i)
        out.append(s)
    return out, theta
