"""Pins for the oracle's sampler: top-k, evidence bookkeeping (eq. 3-5), walk uniformity, closed-form and brute-force logZ."""
import math

import numpy as np
import pytest
from scipy import stats

from oracle import oracle as O
from paper_2509_04336_b200 import workloads as W


def test_topk_is_stable_argsort():
    rng = np.random.default_rng(0)
    x = rng.normal(size=1000)
    x[::7] = x[3]                      # ties
    np.testing.assert_array_equal(O.argsort(x), np.argsort(x, kind="stable"))


def test_shrinkage_eq5_and_neff_eq7():
    # P:126-138 eq. 3-5: one batch shrinks log X by sum_{i<k} 1/(n-i) ~ ln(n/(n-k));  P:140-149: n_GPU ~ 1.4 n_CPU
    for n, k in [(1400, 700), (1000, 500), (200, 50), (100, 1)]:
        logx, logz, h = 0.0, -math.inf, 0.0
        for i in range(k):
            logx, logz, h, lw = O.evidence_update(-1.0, n - i, logx, logz, h)
        exact = -math.fsum(1.0 / (n - i) for i in range(k))
        assert abs(logx - exact) < 1e-13
        assert abs(logx + math.log(n / (n - k))) < 1.0 / (n - k)
    assert abs(O.neff(1400, 700) - 700 / math.log(2)) < 1e-9 and abs(O.neff(1400, 700) - 1009.9) < 0.05
    assert abs(O.neff(1000, 500) - 721.3) < 0.05
    assert abs(1400 / 1000 - 2 * math.log(2)) < 0.02          # eq. 7 as used in P:196


def test_constant_likelihood_evidence_closed_form():
    # L = e^c everywhere: Z = e^c (1 - X_end), H = -ln(1 - X_end); weights are X_{i-1} - X_i (R:L17)
    c, n = 2.5, 50
    logx, logz, h = 0.0, -math.inf, 0.0
    wsum = 0.0
    for it in range(40):
        for i in range(25):
            x_before = math.exp(logx)
            logx, logz, h, lw = O.evidence_update(c, n - i, logx, logz, h)
            assert abs(math.exp(lw) - (x_before - math.exp(logx))) < 1e-15
            wsum += math.exp(lw)
    xend = math.exp(logx)
    assert abs(wsum - (1 - xend)) < 1e-12
    assert abs(logz - (c + math.log1p(-xend))) < 1e-12
    assert abs(h - (-math.log1p(-xend))) < 1e-10


def _shell_run(D, n, k, naccept, periodic, nbatch, seed):
    spec = W.shell_spec(D, periodic)
    P = O.OracleProblem(spec)
    S = O.OracleSampler(P, n, k, naccept, maxmcmc=5000, walks0=50.0, seed=seed)
    out = []
    for b in range(nbatch):
        u0, l0 = S.live()
        st, dead = S.step(want_dead=True)
        u1, l1 = S.live()
        changed = np.where(l1 != l0)[0]
        out.append((st, dead, l1[changed]))
    return out


def test_walk_uniformity_and_volume_on_cube_shells():
    # L(u) = -max|u - 1/2|: X(L) = (2r)^D exactly.  New points must be uniform inside the shell: (r/r*)^D ~ U(0,1);
    # the estimated log X of each dead point must be unbiased (BJ: E[log X_i] = -sum 1/n_i).
    D, n, k = 5, 400, 200
    ratios, bias = [], []
    for seed in range(4):
        runs = _shell_run(D, n, k, 20, [0, 1, 0, 0, 1], 10, seed + 1)
        logx_est = 0.0
        for st, dead, lnew in runs:
            rstar = -st["logl_star"]
            ratios.append(((-lnew) / rstar) ** D)
            r_dead = -dead[:, D]
            logx_true = D * np.log(2 * r_dead)
            est_after = dead[:, D + 1] * 0 + np.cumsum(-1.0 / dead[:, D + 2]) + logx_est
            bias.append(np.mean(est_after - logx_true))
            logx_est = est_after[-1]
            assert abs(logx_est - st["logx"]) < 1e-12
    ratios = np.concatenate(ratios)
    assert ratios.max() < 1.0
    assert stats.kstest(ratios, "uniform").pvalue > 1e-3
    assert abs(ratios.mean() - 0.5) < 4 * 0.2887 / math.sqrt(ratios.size)
    # per-run sd of log X after b batches ~ sqrt(b k/(n (n-k))); the mean over batches and seeds is well inside 0.1
    assert abs(np.mean(bias)) < 0.1


def test_walk_length_adaptation_hits_naccept():
    runs = _shell_run(6, 300, 150, 20, [0] * 6, 14, 7)
    acc = [st["accept_mean"] for st, _, _ in runs[6:]]
    assert abs(np.mean(acc) - 20) < 3.0            # mean accepted steps per walk settles at naccept
    assert all(st["walk_len"] <= 5000 for st, _, _ in runs)


def test_config1_gaussian_logz_closed_form():
    spec, smp, truth = W.config1()
    P = O.OracleProblem(spec)
    pulls, errs = [], []
    for seed in range(1, 13):
        S = O.OracleSampler(P, smp["n_live"], smp["n_delete"], smp["naccept"], smp["maxmcmc"], smp["walks0"], smp["delay"], seed=seed)
        nit, st = S.run(smp["term_kind"], smp["term_tol"], 500)
        logz, err, h = S.finalize()
        assert 30 < nit < 90
        assert abs(h - 8.5) < 1.5
        pulls.append((logz - truth["logz_exact"]) / err)
        errs.append(err)
    pulls = np.array(pulls)
    assert abs(np.mean(errs) - 0.22) < 0.04
    assert np.all(np.abs(pulls) < 4.0)
    assert abs(pulls.mean()) < 3.0 / math.sqrt(len(pulls))
    assert 0.4 < pulls.std() < 1.8


def test_logz_2d_clipped_gaussian_quadrature():
    # box clips the Gaussian at +-1.5 sigma: logZ by brute-force quadrature on a 2048^2 grid
    cov = np.array([[1.0, 0.6], [0.6, 0.8]])
    prec = np.linalg.inv(cov)
    lognorm = -0.5 * (2 * math.log(2 * math.pi) + math.log(np.linalg.det(cov)))
    lo, hi = [-1.5, -1.5 * math.sqrt(0.8)], [1.5, 1.5 * math.sqrt(0.8)]
    spec = dict(like_kind=W.LIKE_GAUSS, ndim=2, prior_kind=[0, 0], prior_lo=lo, prior_hi=hi, periodic=[0, 0],
                toy_mean=[0.0, 0.0], toy_prec=prec, toy_lognorm=lognorm, n_det=0, n_freq=0)
    g = (np.arange(2048) + 0.5) / 2048
    X, Y = np.meshgrid(lo[0] + (hi[0] - lo[0]) * g, lo[1] + (hi[1] - lo[1]) * g, indexing="ij")
    q = prec[0, 0] * X * X + 2 * prec[0, 1] * X * Y + prec[1, 1] * Y * Y
    logz_quad = math.log(np.mean(np.exp(lognorm - 0.5 * q)))
    P = O.OracleProblem(spec)
    pulls = []
    for seed in range(1, 9):
        S = O.OracleSampler(P, 200, 100, 20, seed=seed)
        S.run(0, 0.01, 300)
        logz, err, _ = S.finalize()
        pulls.append((logz - logz_quad) / err)
    assert np.all(np.abs(pulls) < 4.0) and abs(np.mean(pulls)) < 3 / math.sqrt(8)


def test_logz_2d_gw_quadrature():
    # GW likelihood with only (dL, theta_jn) free, the rest FIXED at the injection: 192^2 midpoint quadrature of
    # exp(logL) over the unit square (prior measure is uniform in u) vs nested sampling
    def wf(spec, th):
        return O.OracleProblem(spec).waveform(th)
    spec = W.gw_spec(W.LIKE_TAYLORF2, ["H1", "L1"], 4.0, 96.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 8.0, wf)
    kinds, lo, hi = list(spec["prior_kind"]), list(spec["prior_lo"]), list(spec["prior_hi"])
    for d in range(11):
        if d not in (4, 5):
            kinds[d] = W.FIXED
            lo[d] = hi[d] = W.INJ_C3[d]
    spec["prior_kind"], spec["prior_lo"], spec["prior_hi"] = kinds, lo, hi
    spec["periodic"] = [0] * 11
    P = O.OracleProblem(spec)
    G = 192
    g = (np.arange(G) + 0.5) / G
    u = np.full((G * G, 11), 0.5)
    u[:, 4] = np.repeat(g, G)
    u[:, 5] = np.tile(g, G)
    ll = P.loglike_u(u)
    m = ll.max()
    logz_quad = m + math.log(np.mean(np.exp(ll - m)))
    pulls = []
    for seed in range(1, 4):
        S = O.OracleSampler(P, 200, 100, 20, seed=seed)
        S.run(0, 0.01, 200)
        logz, err, _ = S.finalize()
        pulls.append((logz - logz_quad) / err)
    assert np.all(np.abs(pulls) < 4.0), (pulls, logz_quad)


# ---- walk-length tuning ("same logic as bilby to target a desired number of accepted proposals", P:116 delay as a function of
#      the batch size; readings R:L13, R:L14): the recurrence on accept counts that are known without running any arithmetic ----
def _flat_sampler(n, k, naccept, maxmcmc, walks0, delay=-1.0, seed=1):
    """Constant likelihood (zero precision matrix): no proposal ever satisfies logL' > L*, so every walker accepts exactly 0 steps."""
    D = 3
    spec = dict(like_kind=W.LIKE_GAUSS, ndim=D, prior_kind=[W.UNIFORM] * D, prior_lo=[0.0] * D, prior_hi=[1.0] * D,
                periodic=[1] * D, toy_mean=[0.0] * D, toy_prec=np.zeros((D, D)), toy_lognorm=0.0, n_det=0, n_freq=0)
    return O.OracleSampler(O.OracleProblem(spec), n, k, naccept, maxmcmc=maxmcmc, walks0=walks0, delay=delay, seed=seed)


def test_walk_length_recurrence_by_hand():
    # (a) k = n/2: delay = max(100/(10*50) - 1, 0) = 0.  0 accepts -> floor 0.5: r = 0.5/10; naccept/r = 5*10/0.5 = 100 -> walks 100
    S = _flat_sampler(100, 50, naccept=5, maxmcmc=5000, walks0=10.0)
    st = S.step()
    assert st["walk_len"] == 10 and st["accept_mean"] == 0.0 and st["n_stuck"] == 50 and st["n_oob"] == 0 and st["n_eval"] == 500
    assert st["walks_next"] == 100.0
    # second step: W = 100, 0 accepts: 5*100/0.5 = 1000 (delay 0: no memory of the 100)
    st = S.step()
    assert st["walk_len"] == 100 and st["walks_next"] == 1000.0
    # (b) the maxmcmc cap: the same with maxmcmc = 60 -> 60, and the next walk has exactly 60 steps
    S = _flat_sampler(100, 50, naccept=5, maxmcmc=60, walks0=10.0)
    assert S.step()["walks_next"] == 60.0
    st = S.step()
    assert st["walk_len"] == 60 and st["n_eval"] == 50 * 60 and st["walks_next"] == 60.0
    # (c) sequential limit k = 1: delay = 100/10 - 1 = 9 (bilby's n_live/10 - 1): (10*9 + 100)/10 = 19
    S = _flat_sampler(100, 1, naccept=5, maxmcmc=5000, walks0=10.0)
    st = S.step()
    assert st["walk_len"] == 10 and abs(st["walks_next"] - 19.0) < 1e-12
    # then W = 19: naccept/r = 5*19/0.5 = 190; (19*9 + 190)/10 = 36.1
    st = S.step()
    assert st["walk_len"] == 19 and abs(st["walks_next"] - 36.1) < 1e-12
    # (d) the smoothing uses the REAL-valued walks, the rate uses the integer W: walks0 = 10.7 -> W = 10; (10.7*9 + 100)/10 = 19.63
    S = _flat_sampler(100, 1, naccept=5, maxmcmc=5000, walks0=10.7)
    st = S.step()
    assert st["walk_len"] == 10 and abs(st["walks_next"] - 19.63) < 1e-12
    # (e) explicit delay 2 with k = n/2: (10*2 + 100)/3 = 40; in-between batch k = 20 of 1000: delay = 1000/200 - 1 = 4: (10*4 + 100)/5 = 28
    assert abs(_flat_sampler(100, 50, 5, 5000, 10.0, delay=2.0).step()["walks_next"] - 40.0) < 1e-12
    assert abs(_flat_sampler(1000, 20, 5, 5000, 10.0).step()["walks_next"] - 28.0) < 1e-12


def test_walk_length_recurrence_with_accepts():
    # cube shell, all dims periodic (no out-of-bounds steps): the reported counts are integers, the update from them is by hand:
    # walks' = min((walks*delay + naccept*W/max(0.5, mean)) / (delay + 1), maxmcmc) in exact rational arithmetic
    from fractions import Fraction as Fr
    spec = W.shell_spec(3, [1, 1, 1])
    for n, k, maxmcmc in ((60, 30, 5000), (60, 3, 5000), (60, 30, 45)):
        S = O.OracleSampler(O.OracleProblem(spec), n, k, 4, maxmcmc=maxmcmc, walks0=20.0, seed=5)
        walks = Fr(20)
        delay = max(Fr(n, 10 * k) - 1, Fr(0))
        for it in range(4):
            st = S.step()
            Wl = max(1, min(int(walks), maxmcmc))
            assert st["walk_len"] == Wl and st["n_oob"] == 0 and st["n_eval"] == k * Wl
            total = round(st["accept_mean"] * k)
            assert abs(total - st["accept_mean"] * k) < 1e-9 and total > 0
            mean = max(Fr(1, 2), Fr(total, k))
            walks = min((walks * delay + 4 * Wl / mean) / (delay + 1), Fr(maxmcmc))
            assert abs(st["walks_next"] - float(walks)) <= 1e-12 * float(walks), (n, k, it, st["walks_next"], float(walks))
