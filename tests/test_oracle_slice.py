"""Pins of the oracle's hit-and-run slice-sampling inner kernel (oracle/oracle.cpp, reading R:L25): the kernel must leave
the uniform distribution on the likelihood-constrained region invariant and reach it from a point, for an isotropic region (cube
shells: closed-form radial law), for an elongated one (Gaussian ellipsoid with the covariance's Cholesky factor as direction
factor: closed-form law of the quadratic form) and with periodic dimensions; plus the book-keeping invariants of a slice step.
"""
import math

import numpy as np
from scipy import stats

from oracle import oracle as O
from paper_2509_04336_b200 import workloads as W


def test_slice_uniform_in_cube_shell_from_a_single_point():
    D = 6
    spec = W.shell_spec(D)
    P = O.OracleProblem(spec)
    rstar = 0.2                                   # region: |u - 1/2|_inf < 0.2, L* = -0.2
    B, S = 3000, 25
    u0 = np.full((B, D), 0.5) + 0.01              # every walker starts at the same interior point
    l0 = P.loglike_u(u0)
    res = P.slice_walk(np.eye(D) * 0.15, u0, l0, -rstar, S, 123, (6 << 24) | 1, trace=True)
    assert np.all(res["logl"] > -rstar) and np.all(res["n_stuck"] == 0)
    r = np.abs(res["u"] - 0.5).max(1)
    x = (r / rstar) ** D                          # uniform in the cube of half-width r*  <=>  (r/r*)^D ~ U(0,1)
    assert stats.kstest(x, "uniform").pvalue > 1e-3
    # every coordinate separately uniform on (0.3, 0.7)
    for d in range(D):
        assert stats.kstest((res["u"][:, d] - 0.3) / 0.4, "uniform").pvalue > 1e-4
    # book-keeping: evaluations add up; a step costs at least the two bracket ends (when in the cube) and one candidate
    assert np.array_equal(res["trace_evals"].sum(1), res["n_eval"])
    assert np.all(res["trace_evals"] + 0 >= 1)
    assert np.all(res["trace_logl"] > -rstar)
    assert res["n_expand"].sum() > 0 and res["n_shrink"].sum() > 0


def test_slice_uniform_in_gaussian_ellipsoid_with_cholesky_directions():
    spec, smp, _ = W.config1()
    P = O.OracleProblem(spec)
    cov, lam = W.givens_cov()
    # region {theta: theta^T Sigma^-1 theta < c}: logL > L* with L* = lognorm - c/2
    c = 4.0
    lstar = spec["toy_lognorm"] - 0.5 * c
    Lc = np.linalg.cholesky(cov) / 20.0           # unit-cube coordinates: theta = 20 u - 10
    B, S = 3000, 30
    u0 = np.full((B, 4), 0.5)
    u0[:, 0] += 1e-3
    l0 = P.loglike_u(u0)
    res = P.slice_walk(Lc, u0, l0, lstar, S, 77, (6 << 24) | 2)
    th = 20.0 * res["u"] - 10.0
    q = np.einsum("bi,ij,bj->b", th, np.linalg.inv(cov), th)
    assert np.all(q < c)
    # uniform in a 4-D ellipsoid: (q/c)^(D/2) ~ U(0,1)
    assert stats.kstest((q / c) ** 2, "uniform").pvalue > 1e-3
    # directions: the principal-axis coordinates are uncorrelated and scale with sqrt(eigenvalue)
    evals, evecs = np.linalg.eigh(cov)
    pc = th @ evecs
    ratio = pc.var(0) / evals
    assert ratio.max() / ratio.min() < 1.25
    # a badly scaled (isotropic, too wide) direction factor still samples correctly, at a higher cost in shrink steps
    res2 = P.slice_walk(np.eye(4) * 0.5, u0, l0, lstar, S, 78, (6 << 24) | 2)
    th2 = 20.0 * res2["u"] - 10.0
    q2 = np.einsum("bi,ij,bj->b", th2, np.linalg.inv(cov), th2)
    assert stats.kstest((q2 / c) ** 2, "uniform").pvalue > 1e-3
    assert res2["n_shrink"].mean() > res["n_shrink"].mean()


def test_slice_periodic_dimensions_and_fixed_dimensions():
    D = 5
    spec = W.shell_spec(D, [1, 0, 1, 0, 0])
    spec["prior_kind"] = [W.UNIFORM, W.UNIFORM, W.UNIFORM, W.UNIFORM, W.FIXED]
    P = O.OracleProblem(spec)
    B, S = 2000, 20
    u0 = np.full((B, D), 0.5)
    u0[:, 4] = 0.55                               # FIXED dimension: never moves; it contributes |0.05| to the shell norm
    l0 = P.loglike_u(u0)
    rstar = 0.45
    res = P.slice_walk(np.eye(D) * 0.3, u0, l0, -rstar, S, 5, (6 << 24) | 3)
    assert np.all(res["u"][:, 4] == 0.55)
    assert np.all((res["u"] >= 0.0) & (res["u"] < 1.0)) and np.all(res["logl"] > -rstar)
    for d in range(4):
        assert stats.kstest((res["u"][:, d] - 0.05) / 0.9, "uniform").pvalue > 1e-4


def test_slice_same_seed_same_chain_and_slot_keys_the_stream():
    spec = W.shell_spec(4)
    P = O.OracleProblem(spec)
    u0 = np.full((8, 4), 0.45)
    l0 = P.loglike_u(u0)
    a = P.slice_walk(np.eye(4) * 0.2, u0, l0, -0.3, 10, 9, 3)
    b = P.slice_walk(np.eye(4) * 0.2, u0, l0, -0.3, 10, 9, 3)
    assert np.array_equal(a["u"], b["u"])
    assert len({tuple(r) for r in a["u"]}) == 8           # same start, different slots: different chains
    c = P.slice_walk(np.eye(4) * 0.2, u0[3:5], l0[3:5], -0.3, 10, 9, 3, slot0=3)
    assert np.array_equal(c["u"], a["u"][3:5])            # the chain depends on the slot, not on the batch it is in


def test_live_cholesky_is_the_factor_of_the_sample_covariance():
    spec = W.shell_spec(5)
    spec["prior_kind"] = [W.UNIFORM, W.UNIFORM, W.FIXED, W.UNIFORM, W.UNIFORM]
    P = O.OracleProblem(spec)
    rng = np.random.default_rng(1)
    A = rng.normal(size=(5, 5))
    pts = 0.5 + 0.05 * rng.normal(size=(400, 5)) @ A.T
    Lc = P.live_cholesky(pts)
    free = [0, 1, 3, 4]
    C = np.cov(pts.T)[np.ix_(free, free)]
    np.testing.assert_allclose((Lc @ Lc.T)[np.ix_(free, free)], C, rtol=1e-9, atol=1e-15)
    assert np.all(Lc[2] == 0) and np.all(Lc[:, 2] == 0) and np.allclose(Lc, np.tril(Lc))
    np.testing.assert_allclose(Lc[np.ix_(free, free)], np.linalg.cholesky(C), rtol=1e-8, atol=1e-14)


def test_slice_sampler_gaussian_logz_closed_form_and_shrinkage():
    """The whole sampler with the slice kernel inside (directions from the survivors' covariance): config-1 evidence against the
    closed form, and the cube-shell volume law E[log X] (BJ pins of the acceptance-walk sampler, repeated for this kernel)."""
    spec, smp, ref = W.config1()
    P = O.OracleProblem(spec)
    pulls = []
    for seed in range(1, 7):
        S = O.OracleSampler(P, smp["n_live"], smp["n_delete"], smp["naccept"], smp["maxmcmc"], smp["walks0"], smp["delay"], seed=seed)
        S.use_slice_kernel(20)
        n, st = S.run(0, 0.01, 500)
        logz, err, _ = S.finalize()
        assert st["walk_len"] == 20 and st["accept_min"] >= 19      # every slice step moves the point
        pulls.append((logz - ref["logz_exact"]) / err)
    pulls = np.array(pulls)
    assert np.all(np.abs(pulls) < 3.5) and abs(pulls.mean()) < 1.5, pulls
    # cube shells: the true volume of each dead point is (2r)^D
    D = 6
    sspec = W.shell_spec(D)
    Ps = O.OracleProblem(sspec)
    bias = []
    for seed in range(1, 5):
        S = O.OracleSampler(Ps, 400, 200, 10, 500, 20.0, -1.0, seed=seed)
        S.use_slice_kernel(12)
        tot = []
        for it in range(12):
            st, dead = S.step(want_dead=True)
            r = -dead[:, D]
            logx_true = D * np.log(2 * r)
            logx_est = dead[:, D + 1] - np.log(-np.expm1(-1.0 / dead[:, D + 2]))     # logw = logX_prev + log(1 - e^{-1/n})
            tot.append(np.mean(logx_est - logx_true))
        bias.append(np.mean(tot[4:]))
    assert abs(np.mean(bias)) < 0.12, bias
