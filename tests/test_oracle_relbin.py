"""Pins of the oracle's relative-binning likelihood (oracle/oracle.cpp, reading R:L24) against what the mathematics
fixes: it is EXACT whenever h(theta)/h0 is constant in frequency (the d_L, phase and -- for one detector -- amplitude directions),
its summary data partition the exact inner products, it is second order in the bin width for a pure time shift (closed-form bound),
it converges to the exact likelihood as eps -> 0, and near the fiducial point its error is far below the nested-sampling tolerance.
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2509_04336_b200 import workloads as W


def wf(spec, th):
    return O.OracleProblem(spec).waveform(th)


@pytest.fixture(scope="module", params=[W.LIKE_TAYLORF2, W.LIKE_PHENOMD])
def prob(request):
    spec = W.gw_spec(request.param, ["H1", "L1"], 4.0, 512.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 14.0, wf)
    return spec, O.OracleProblem(spec)


def test_edges_and_bin_count(prob):
    spec, P = prob
    rb = P.relbin(W.INJ_C3, chi=1.0, eps=0.5)
    e = rb.edges()
    assert e[0] == 0 and e[-1] == spec["n_freq"] - 1 and np.all(np.diff(e) > 0)
    # bin count: floor(Delta_tot / eps) with Delta(f) = 2 pi chi sum sgn(g) (f/f*)^g -- evaluated here with exact rationals of the
    # end points: at f_max the gamma>0 terms are 1 and the gamma<0 ones -(f_max/f_min)^g; at f_min the reverse
    f_lo, f_hi = spec["f_min"], spec["f_min"] + (spec["n_freq"] - 1) * spec["df"]
    x = f_hi / f_lo
    d_hi = 3.0 - x ** (-5.0 / 3.0) - x ** (-2.0 / 3.0)
    d_lo = x ** -1.0 + x ** (-5.0 / 3.0) + x ** (-7.0 / 3.0) - 2.0
    n_expected = int(math.floor(2.0 * math.pi * (d_hi - d_lo) / 0.5))
    assert rb.n_bins <= n_expected and rb.n_bins >= n_expected - 3       # duplicates at the coarse low end may merge a few bins
    # halving eps doubles the number of bins (to within the merged ones)
    assert abs(P.relbin(W.INJ_C3, eps=0.25).n_bins - 2 * n_expected) <= 6
    # bins are narrow at low frequency (fast phase evolution) and wide at high frequency
    w = np.diff(e)
    assert w[:5].mean() < w[-5:].mean()


def test_summary_data_partition_the_exact_inner_products(prob):
    spec, P = prob
    rb = P.relbin(W.INJ_C3)
    A0, A1, B0, B1 = rb.summary()
    logl, parts = P.gw_loglike(np.array([W.INJ_C3]), parts=True)
    for d in range(2):
        # sum_b A0 = <d, h0> (complex; its real part is the exact <d,h>), sum_b B0 = <h0, h0>: every grid bin in exactly one bin
        assert abs(A0[d, :, 0].sum() - parts[0, 2 * d]) < 1e-10 * abs(parts[0, 2 * d])
        assert abs(B0[d].sum() - parts[0, 2 * d + 1]) < 1e-12 * parts[0, 2 * d + 1]
        # first moments about the bin centres are small compared with (bin width) x zeroth moments
        e = rb.edges()
        wid = np.diff(spec["f_min"] + e * spec["df"])
        assert np.all(np.abs(B1[d]) <= 0.5 * wid * B0[d] + 1e-30)


def test_exact_at_the_fiducial_point_and_along_constant_ratio_directions(prob):
    spec, P = prob
    rb = P.relbin(W.INJ_C3)
    th = np.array([W.INJ_C3] * 5)
    th[1, 4] = 1234.5                      # d_L: r = d_L0 / d_L
    th[2, 7] = W.INJ_C3[7] + 0.83          # phase: r = exp(-2 i dphi)
    th[3, 4], th[3, 7] = 333.0, 5.9        # both
    th[4, 7] = W.INJ_C3[7] + math.pi       # phase + pi: the same waveform
    exact, pe = P.gw_loglike(th, parts=True)
    approx, pa = rb.loglike(th, parts=True)
    scale = np.abs(pe[:, 0::2]).sum(1) + 0.5 * pe[:, 1::2].sum(1)
    assert np.max(np.abs(approx - exact) / scale) < 1e-11
    np.testing.assert_allclose(pa, pe, rtol=0, atol=1e-11 * scale.max())
    assert abs(approx[4] - approx[0]) < 1e-9


def test_time_shift_is_second_order_in_bin_width_and_bounded(prob):
    """h(theta) = h0 exp(-2 pi i f dt): linear interpolation of r inside a bin of width w has error <= (2 pi dt w)^2 / 8 in |r|,
    so |<d,h>_rb - <d,h>| <= max_b (2 pi dt w_b)^2/8 * sum_b sum_k |d h0|/S  and the error scales as dt^2."""
    spec, P = prob
    rb = P.relbin(W.INJ_C3, eps=0.5)
    e = rb.edges()
    wmax = np.diff(spec["f_min"] + e * spec["df"]).max()
    h0 = P.waveform(W.INJ_C3)
    d = np.asarray(spec["strain"])
    S = np.asarray(spec["psd"])
    l1 = 4 * spec["df"] * (np.hypot(d[..., 0], d[..., 1]) * np.hypot(h0[..., 0], h0[..., 1]) / S).sum()
    hh0 = 4 * spec["df"] * ((h0[..., 0] ** 2 + h0[..., 1] ** 2) / S).sum()
    errs = []
    for dt in (2e-4, 4e-4, 8e-4):
        th = np.array([W.INJ_C3])
        th[0, 8] += dt
        exact = P.gw_loglike(th)[0]
        approx = rb.loglike(th)[0]
        bound_r = (2 * math.pi * dt * wmax) ** 2 / 8
        assert abs(approx - exact) <= bound_r * l1 + (2 * bound_r + bound_r ** 2) * 0.5 * hh0
        errs.append(abs(approx - exact))
    # doubling dt multiplies the error by ~4 (second order), certainly by more than 2.5 and less than 6
    assert 2.5 < errs[1] / errs[0] < 6.0 and 2.5 < errs[2] / errs[1] < 6.0


def test_converges_with_eps_and_is_accurate_near_the_fiducial_point(prob):
    spec, P = prob
    rng = np.random.default_rng(12)
    # posterior-like scatter about the injection (unit-cube sigmas of the config-5 recipe, halved)
    u0 = np.array([0.4, 0.771, 0.652, 0.399, 0.0041, 0.0395, 0.8467, 0.2069, 0.5, 0.2196, 0.0317])
    u = u0[None, :] + rng.normal(0, 1, (400, 11)) * np.array(W.C5_SIGMA) * 0.1
    per = np.array(spec["periodic"], bool)
    u[:, per] -= np.floor(u[:, per])
    u[:, ~per] = np.clip(u[:, ~per], 1e-6, 1 - 1e-6)
    th = P.prior_transform(u)
    exact = P.gw_loglike(th)
    keep = exact > exact.max() - 60.0          # the region a sampler resolves
    bulk = exact > exact.max() - 12.0          # the posterior bulk
    assert keep.sum() > 40 and bulk.sum() > 5
    errs, errs_bulk = [], []
    for eps in (1.0, 0.5, 0.25, 0.125):
        d = np.abs(P.relbin(W.INJ_C3, eps=eps).loglike(th) - exact)
        errs.append(d[keep].max())
        errs_bulk.append(d[bulk].max())
    # second-order convergence: every halving of eps divides the error by ~4 (ask for > 3)
    assert errs[1] < errs[0] / 3 and errs[2] < errs[1] / 3 and errs[3] < errs[2] / 3
    # default eps = 0.5: the error in the posterior bulk is far below the dlogZ tolerance (0.1) of the runs
    assert errs_bulk[1] < 0.05 and errs[1] < 0.3 and errs[3] < 0.02


def test_unphysical_theta_and_bad_arguments(prob):
    spec, P = prob
    rb = P.relbin(W.INJ_C3)
    th = np.array([W.INJ_C3] * 2)
    th[1, 1] = 1.7
    out = rb.loglike(th)
    assert np.isfinite(out[0]) and np.isneginf(out[1])
    with pytest.raises(ValueError):
        P.relbin(th[1])
    with pytest.raises(ValueError):
        P.relbin(W.INJ_C3, eps=0.0)


def test_sampler_routes_through_relbin_when_asked(prob):
    spec, P = prob
    rb = P.relbin(W.INJ_C3)
    u = W.uniforms(50, 11, 3)
    exact = P.loglike_u(u)
    P.use_relbin(rb)
    try:
        np.testing.assert_array_equal(P.loglike_u(u), rb.loglike(P.prior_transform(u)))
        # a short run on the approximate likelihood works end to end and uses the same code path
        S = O.OracleSampler(P, 60, 30, 5, 40, 10.0, -1.0, seed=2)
        st = S.step()
        assert st["n_eval"] > 0 and np.isfinite(st["logz"])
    finally:
        P.use_relbin(None)
    np.testing.assert_array_equal(P.loglike_u(u), exact)
