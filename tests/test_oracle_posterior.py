"""Pins of the oracle's posterior weights (oracle.posterior*, reading R:L26) against what the mathematics fixes:
a closed-form 1-D posterior reached by ideal shrinkage (quadrature bound), Kish's formula on hand-made rows, and the analytic
Gaussian posterior of config 1 (moments and marginal CDFs), also when the run is stopped early so that most of the mass sits
in the final live points."""
import math

import numpy as np

from oracle import oracle as O
from paper_2509_04336_b200 import workloads as W


def _ideal_run_1d(n, n_dead, scale):
    """Ideal nested sampling of L(x) = exp(-x/scale), x ~ U(0,1): X = x, the i-th dead point sits exactly at the expected
    shrinkage X_i = exp(-i/n) and the final live points at X_N exp(-(1/n + 1/(n-1) + ..)) (the widths R:L17 assigns)."""
    logx_prev = -np.arange(n_dead) / n
    x_dead = np.exp(-(np.arange(n_dead) + 1.0) / n)
    dead = np.stack([x_dead, -x_dead / scale, logx_prev + math.log(-math.expm1(-1.0 / n)), np.full(n_dead, float(n))], axis=1)
    logx = -n_dead / n
    steps = np.cumsum(1.0 / (n - np.arange(n)))
    x_live = np.exp(logx - steps)          # ascending logL = descending x
    rng = np.random.default_rng(3)
    perm = rng.permutation(n)              # the live set is stored in no particular order
    return dead, x_live[perm][:, None], (-x_live / scale)[perm], logx


def _spec_1d():
    return dict(like_kind=W.LIKE_GAUSS, ndim=1, prior_kind=[W.UNIFORM], prior_lo=[0.0], prior_hi=[1.0], periodic=[0],
                toy_mean=[0.0], toy_prec=np.eye(1), toy_lognorm=0.0, n_det=0, n_freq=0)


def test_ideal_shrinkage_reaches_the_closed_form_posterior():
    n, scale = 2000, 0.1
    P = O.OracleProblem(_spec_1d())
    z_exact = scale * (1.0 - math.exp(-1.0 / scale))
    for n_dead in (16000, 3000, 0):        # late stop, early stop (live points carry 22 % of X), live points only
        dead, lu, ll, logx = _ideal_run_1d(n, n_dead, scale)
        for ref in (0.02, 0.07, 0.2, 0.5):
            out = O.posterior(P, dead, lu, ll, logx, theta_ref=[ref])
            cdf = (1.0 - math.exp(-ref / scale)) / (1.0 - math.exp(-1.0 / scale))
            # widths sit to the right of each point (w_i = X_{i-1} - X_i): first-order quadrature, error <= max width / scale
            bound = 3.0 / n / scale if n_dead else 0.06
            assert abs(out["cl"][0] - cdf) < bound, (n_dead, ref, out["cl"][0], cdf)
        if n_dead:
            assert abs(out["logz"] - math.log(z_exact)) < 2.0 / n / scale
        assert abs(math.fsum(np.exp(out["logp"]).tolist()) - 1.0) < 1e-13
        assert out["theta"].shape == (n_dead + n, 1)
        assert np.all(np.diff(out["theta"][:, 0]) < 0)       # rows run inwards: dead points first, live points ascending logL


def test_rows_use_the_live_count_sawtooth():
    # three live points after logX = -1: widths X(1 - e^{-1/3}), X e^{-1/3}(1 - e^{-1/2}), X e^{-1/3-1/2}(1 - e^{-1})
    lu = np.array([[0.3], [0.1], [0.2]])
    ll = np.array([-3.0, -1.0, -2.0])
    u, logl, logw = O.posterior_rows(None, lu, ll, -1.0)
    assert np.array_equal(u[:, 0], [0.3, 0.2, 0.1]) and np.array_equal(logl, [-3.0, -2.0, -1.0])
    x = math.exp(-1.0)
    want = [x * (1 - math.exp(-1 / 3)), x * math.exp(-1 / 3) * (1 - math.exp(-0.5)), x * math.exp(-1 / 3 - 0.5) * (1 - math.exp(-1.0))]
    assert np.allclose(np.exp(logw), want, rtol=1e-14, atol=0)
    assert abs(sum(want) - x * (1 - math.exp(-1 / 3 - 0.5 - 1.0))) < 1e-16      # telescopes to X - X_final


def test_kish_effective_sample_size_and_levels_by_hand():
    P = O.OracleProblem(_spec_1d())
    # rows with L w = 3, 1 (dead) and no further mass: p = (0.75, 0.25)
    dead = np.array([[0.8, math.log(6.0), math.log(0.5), 2.0], [0.4, math.log(4.0), math.log(0.25), 1.0]])
    logp, logz = O.posterior_weights(dead[:, 1], dead[:, 2])
    assert np.allclose(np.exp(logp), [0.75, 0.25], rtol=1e-15) and abs(logz - math.log(4.0)) < 1e-15
    # through posterior(): one live point far below in likelihood so that it adds nothing
    out = O.posterior(P, dead, np.array([[0.1]]), np.array([-800.0]), math.log(0.25), theta_ref=[0.5])
    assert abs(out["ess"] - 1.0 / (0.75 ** 2 + 0.25 ** 2)) < 1e-12
    assert abs(out["cl"][0] - 0.25) < 1e-15        # theta < 0.5: the second row (0.4) and the massless live point
    # N equal weights: ESS = N
    lp, _ = O.posterior_weights(np.zeros(37), np.full(37, -2.0))
    assert abs(1.0 / np.sum(np.exp(lp) ** 2) - 37.0) < 1e-12


def _config1_posteriors(max_iter, seeds):
    spec, smp, _ = W.config1()
    P = O.OracleProblem(spec)
    cov, _ = W.givens_cov()
    ref = np.array([0.1, -0.3, 0.4, 0.2])
    means, seconds, cls, esss, dz = [], [], [], [], []
    for seed in seeds:
        S = O.OracleSampler(P, smp["n_live"], smp["n_delete"], smp["naccept"], smp["maxmcmc"], smp["walks0"], smp["delay"], seed=seed)
        nit, st, dead = S.run(smp["term_kind"], smp["term_tol"], max_iter, want_dead=True)
        lu, ll = S.live()
        out = O.posterior(P, dead, lu, ll, st["logx"], theta_ref=ref)
        pw = np.exp(out["logp"])
        means.append(pw @ out["theta"])
        seconds.append((out["theta"] * pw[:, None]).T @ out["theta"])
        cls.append(out["cl"])
        esss.append(out["ess"])
        dz.append(out["logz"] - S.finalize()[0])
    return cov, ref, np.array(means), np.mean(seconds, axis=0), np.array(cls), np.array(esss), np.array(dz)


def test_config1_gaussian_posterior_moments_and_marginal_cdfs():
    seeds = range(1, 25)
    cov, ref, means, second, cls, esss, dz = _config1_posteriors(500, seeds)
    # the rows' evidence is the sampler's own final evidence (same terms, other summation order)
    assert np.max(np.abs(dz)) < 1e-10
    sig = np.sqrt(np.diag(cov))
    se = sig / math.sqrt(np.mean(esss) * len(means))
    assert np.all(np.abs(means.mean(axis=0)) < 4.5 * se), (means.mean(axis=0), se)
    assert np.allclose(second, cov, atol=0.06 * float(np.max(sig)) ** 2, rtol=0.08), second - cov
    cdf = np.array([0.5 * (1 + math.erf(r / s / math.sqrt(2))) for r, s in zip(ref, sig)])
    assert np.all(np.abs(cls.mean(axis=0) - cdf) < 4.5 * 0.5 / np.sqrt(np.mean(esss) * len(cls))), (cls.mean(axis=0), cdf)
    assert 300 < np.mean(esss) < 3000


def test_config1_posterior_when_stopped_early():
    # 28 iterations: X = 0.75^28 = 3.2e-4, about ten times the Gaussian's own volume ((2 pi)^2 |Sigma|^(1/2) / 20^4 = 2.7e-5 of
    # the box): the contour is at r = 3 sigma and 94 % of the posterior mass (P(chi2_4 < 9)) is carried by the final live points' rows
    seeds = range(1, 61)
    cov, ref, means, second, cls, esss, dz = _config1_posteriors(28, seeds)
    assert np.max(np.abs(dz)) < 1e-10
    sig = np.sqrt(np.diag(cov))
    assert np.mean(esss) < 80
    cdf = np.array([0.5 * (1 + math.erf(r / s / math.sqrt(2))) for r, s in zip(ref, sig)])
    assert np.all(np.abs(cls.mean(axis=0) - cdf) < 5.0 * 0.5 / np.sqrt(np.mean(esss) * len(cls))), (cls.mean(axis=0), cdf)
    assert np.allclose(second, cov, atol=0.25 * float(np.max(sig)) ** 2), second - cov


def _toy_pp_specs(n_inj, seed):
    """PP law on the Gaussian toy: theta_inj ~ U(box), observed d = theta_inj + eps, eps ~ N(0, Sigma); the likelihood of theta
    is N(d; theta, Sigma), so the credible levels of theta_inj under the posterior are uniform."""
    spec, smp, _ = W.config1()
    cov, _ = W.givens_cov()
    rng = np.random.Generator(np.random.Philox(key=seed))
    th = rng.uniform(-10.0, 10.0, size=(n_inj, 4))
    d = th + rng.multivariate_normal(np.zeros(4), cov, size=n_inj)
    specs = []
    for i in range(n_inj):
        s = dict(spec)
        s["toy_mean"] = list(d[i])
        specs.append(s)
    return specs, th, smp


def test_pp_law_on_the_gaussian_toy():
    from scipy import stats
    specs, th, smp = _toy_pp_specs(120, 41)
    cl = np.empty((len(specs), 4))
    for i, s in enumerate(specs):
        P = O.OracleProblem(s)
        S = O.OracleSampler(P, smp["n_live"], smp["n_delete"], smp["naccept"], smp["maxmcmc"], smp["walks0"], smp["delay"], seed=1000 + i)
        nit, st, dead = S.run(smp["term_kind"], smp["term_tol"], 500, want_dead=True)
        lu, ll = S.live()
        cl[i] = O.posterior(P, dead, lu, ll, st["logx"], theta_ref=th[i])["cl"]
    pv = [stats.kstest(cl[:, d], "uniform").pvalue for d in range(4)]
    assert min(pv) > 0.01 / 4, pv
    assert np.all(np.abs(cl.mean(axis=0) - 0.5) < 4.0 / math.sqrt(12 * len(specs)))
    # posteriors too narrow / too wide pile the levels up at the ends / in the middle: the variance of uniform levels is 1/12
    assert np.all(np.abs(cl.var(axis=0) - 1 / 12) < 0.035)


def test_systematic_resampling_invariants():
    rng = np.random.default_rng(11)
    logp, _ = O.posterior_weights(rng.normal(0, 3, 500), rng.normal(-5, 2, 500))
    p = np.exp(logp)
    for n_out, seed in ((1000, 1), (137, 2), (5000, 2 ** 40 + 3)):
        idx, U = O.posterior_resample(logp, n_out, seed)
        assert 0.0 < U < 1.0 and idx.shape == (n_out,) and np.all(np.diff(idx) >= 0)
        cnt = np.bincount(idx, minlength=p.size)
        # systematic resampling: every row is drawn floor(n p) or ceil(n p) times
        assert np.all(cnt >= np.floor(n_out * p - 1e-9)) and np.all(cnt <= np.ceil(n_out * p + 1e-9))
        assert cnt.sum() == n_out
    # different seeds move the comb; the same seed repeats it
    a, Ua = O.posterior_resample(logp, 1000, 5)
    b, Ub = O.posterior_resample(logp, 1000, 6)
    c, Uc = O.posterior_resample(logp, 1000, 5)
    assert Ua != Ub and Ua == Uc and np.array_equal(a, c) and not np.array_equal(a, b)
    # equal weights, as many draws as rows: every row exactly once, whatever U
    lp = np.full(64, -math.log(64.0))
    assert np.array_equal(O.posterior_resample(lp, 64, 9)[0], np.arange(64))
    # a single draw is the U-quantile of the cumulative weights
    i1, U1 = O.posterior_resample(logp, 1, 3)
    cum = np.cumsum(p)
    assert cum[i1[0]] > U1 * cum[-1] and (i1[0] == 0 or cum[i1[0] - 1] <= U1 * cum[-1])
    # the uniform is the RNG contract's: block (0, 0, 0, 4 << 24) under key = seed
    w = O.philox([0, 0, 0, 4 << 24], [3, 0])
    assert U1 == O.u53(w[0], w[1])
