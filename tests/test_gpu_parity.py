"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (DESIGN.md section 3 'T'):
  logL:       |dlogL| <= 1e-10 * max(1, |<d,h>| + <h,h>/2)     (BJ: 1e-10 relative, made well-conditioned)
  decisions:  identical except where |logL - L*| < 1e-8 or a proposal coordinate lies within 1e-12 of a bound
  integer / index work (Philox words, ranks, counters): bit-exact
"""
import math

import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2509_04336_b200 import workloads as W

pytestmark = pytest.mark.gpu


def wf(spec, th):
    return O.OracleProblem(spec).waveform(th)


def dev(x):
    return torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64)).cuda()


@pytest.fixture(scope="module")
def nsgw():
    from paper_2509_04336_b200 import nsgw as N
    assert torch.cuda.is_available()
    return N


@pytest.fixture(scope="module")
def c2():
    return W.config2(wf)


@pytest.fixture(scope="module")
def c3():
    return W.config3(wf)


def _check_logl(logl_g, parts_g, logl_o, parts_o, n_det):
    scale = np.maximum(1.0, np.abs(parts_o[:, 0::2]).sum(1) + 0.5 * parts_o[:, 1::2].sum(1))
    err = np.abs(logl_g - logl_o) / scale
    assert np.all(np.isfinite(logl_g) == np.isfinite(logl_o))
    assert np.nanmax(err) < 1e-10, np.nanmax(err)
    np.testing.assert_allclose(parts_g, parts_o, rtol=0, atol=1e-10 * scale.max())
    return np.nanmax(err)


def test_prior_transform_parity(nsgw, c2):
    h = nsgw.Handle(c2)
    u = W.uniforms(3001, 11, 11)
    th_g = h.prior_transform_batch(dev(u)).cpu().numpy()
    th_o = O.OracleProblem(c2).prior_transform(u)
    np.testing.assert_allclose(th_g, th_o, rtol=1e-15, atol=4e-15)   # FMA contraction + libm differences: a few ulp


def test_live_draw_is_bitwise_philox(nsgw):
    spec, smp, _ = W.config1()
    h = nsgw.Handle(spec, smp, seed=0x1234567890ABCDEF)
    u_g, l_g = h.get_live()
    u_o = O.draw_live(4, smp["n_live"], 0x1234567890ABCDEF)
    assert np.array_equal(u_g.cpu().numpy(), u_o)                      # Philox words + u01: bit-exact
    l_o = O.OracleProblem(spec).loglike_u(u_o)
    np.testing.assert_allclose(l_g.cpu().numpy(), l_o, rtol=1e-13)


KERNELS = [1, 2]   # NSGW_OPT_BINS_KERNEL: 1 = CTA per particle (pair), bins strided over threads (k_bins), 2 = lane per particle (k_bins_lp*)


@pytest.mark.parametrize("kern", KERNELS)
@pytest.mark.parametrize("B", [1, 515, 1027, 4101])
def test_taylorf2_loglike_parity(nsgw, c2, B, kern):
    # config-2 shape: 2 detectors x 4017 bins (3 full 1024-bin chunks + a ragged one); B spans the launch shapes
    # (P=1, P=2; sub-batches of 8 with ragged tails)
    h = nsgw.Handle(c2)
    h.set_option(0, kern)
    P = O.OracleProblem(c2)
    th = P.prior_transform(W.uniforms(B, 11, 100 + B))
    logl_o, parts_o = P.gw_loglike(th, parts=True)
    logl_g, parts_g = h.gw_loglike_batch(dev(th), parts=True)
    _check_logl(logl_g.cpu().numpy(), parts_g.cpu().numpy(), logl_o, parts_o, 2)


def test_taylorf2_injection_and_unphysical(nsgw, c2):
    h = nsgw.Handle(c2)
    P = O.OracleProblem(c2)
    th = np.array([W.INJ_C3] * 4)
    th[1, 1] = 1.5; th[2, 4] = -1.0; th[3, 2] = float("nan")
    lo = P.gw_loglike(th)
    for kern in KERNELS:
        h.set_option(0, kern)
        lg = h.gw_loglike_batch(dev(th)).cpu().numpy()
        assert abs(lg[0] - lo[0]) < 1e-10 * 400 and np.all(np.isneginf(lg[1:])) and np.all(np.isneginf(lo[1:]))
    assert h.gw_loglike_batch(dev(np.zeros((0, 11)))).numel() == 0     # empty batch


@pytest.mark.parametrize("model", ["taylorf2", "phenomd"])
def test_host_entry_paths_agree(nsgw, c2, c3, model):
    # gw_loglike_batch_host: pinned buffers used in place (theta fetched over the host link by the set-up kernel, logL stored into the
    # caller's buffer), the same with the copies forced, and pageable buffers -- all bit for bit the device call
    spec = c2 if model == "taylorf2" else c3[0]
    h = nsgw.Handle(spec)
    for B in (1, 700, 5000):
        u = W.uniforms(B, 11, 300 + B)
        th = h.prior_transform_batch(dev(u))
        th[B // 2, 1] = 1.5                                   # an unphysical row: -inf
        ref = h.gw_loglike_batch(th).cpu()
        th_pin, out_pin = th.cpu().pin_memory(), torch.full((B,), float("nan"), dtype=torch.float64).pin_memory()
        h.gw_loglike_batch_host(th_pin, out_pin)
        assert torch.equal(out_pin, ref)
        h.set_option(nsgw.OPT_HOST_ZERO_COPY, 0)
        out2 = torch.full((B,), float("nan"), dtype=torch.float64).pin_memory()
        h.gw_loglike_batch_host(th_pin, out2)
        h.set_option(nsgw.OPT_HOST_ZERO_COPY, 1)
        assert torch.equal(out2, ref)
        out3 = torch.full((B,), float("nan"), dtype=torch.float64)          # pageable
        h.gw_loglike_batch_host(th.cpu(), out3)
        assert torch.equal(out3, ref)


@pytest.mark.parametrize("kern", KERNELS)
@pytest.mark.parametrize("B", [3, 515, 4101])
def test_phenomd_loglike_parity_config3_shape(nsgw, c3, B, kern):
    spec, _ = c3
    h = nsgw.Handle(spec)
    h.set_option(0, kern)
    P = O.OracleProblem(spec)
    th = P.prior_transform(W.uniforms(B, 11, 200 + B))
    th[0] = W.INJ_C3
    logl_o, parts_o = P.gw_loglike(th, parts=True)
    logl_g, parts_g = h.gw_loglike_batch(dev(th), parts=True)
    _check_logl(logl_g.cpu().numpy(), parts_g.cpu().numpy(), logl_o, parts_o, 2)


def test_phenomd_builtin_table_equals_explicit(nsgw, c3):
    spec, _ = c3
    th = dev(O.OracleProblem(spec).prior_transform(W.uniforms(64, 11, 9)))
    a = nsgw.Handle(spec).gw_loglike_batch(th)
    b = nsgw.Handle(dict(spec, phenom_table=None)).gw_loglike_batch(th)
    assert torch.equal(a, b)


@pytest.mark.parametrize("kern", KERNELS)
def test_phenomd_spin_table_parity(nsgw, kern):
    # a fit table with non-zero spin columns and gamma2 < 1 exercises the chi_PN polynomial and the other Fpeak branch
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1", "V1"], 4.0, 512.0, (20.0, 40.0))
    tab = W.surrogate_table()
    rng = np.random.default_rng(3)
    tab[:, 2:] = tab[:, :1] * rng.normal(0, 0.02, (19, 9))
    tab[5, :] = 0; tab[5, 0] = 0.8
    spec["phenom_table"] = tab
    spec = W.make_data(spec, W.INJ_C3, 25.0, wf)
    P = O.OracleProblem(spec)
    th = P.prior_transform(W.uniforms(130, 11, 77))
    logl_o, parts_o = P.gw_loglike(th, parts=True)
    h = nsgw.Handle(spec)
    h.set_option(0, kern)
    logl_g, parts_g = h.gw_loglike_batch(dev(th), parts=True)
    _check_logl(logl_g.cpu().numpy(), parts_g.cpu().numpy(), logl_o, parts_o, 3)


@pytest.mark.parametrize("kern", KERNELS)
def test_phenomd_three_detector_long_segment_parity(nsgw, kern):
    # config-5 shape: 3 detectors x 32449 bins (16 s at 4096 Hz)
    spec = W.config5(wf)
    assert spec["n_freq"] == 32449 and spec["n_det"] == 3
    P = O.OracleProblem(spec)
    u = W.config5_live(spec, 96)
    th = P.prior_transform(u)
    logl_o, parts_o = P.gw_loglike(th, parts=True)
    h = nsgw.Handle(spec)
    h.set_option(0, kern)
    logl_g, parts_g = h.gw_loglike_batch(dev(th), parts=True)
    _check_logl(logl_g.cpu().numpy(), parts_g.cpu().numpy(), logl_o, parts_o, 3)


@pytest.mark.parametrize("kind", [W.LIKE_TAYLORF2, W.LIKE_PHENOMD])
@pytest.mark.parametrize("dets,f_max,T", [(["H1"], 64.0, 4.0),            # one detector, 177 bins (fewer than a CTA has threads)
                                          (["L1"], 20.25, 4.0),           # 2 bins: degenerate grid
                                          (["H1", "L1", "V1"], 85.0, 2.0),  # three detectors, 131 bins (one ragged tile)
                                          (["V1", "H1"], 532.5, 2.0)])    # 1026 bins: tiles of 256 plus a 2-bin tail
def test_loglike_edge_grids_parity(nsgw, kind, dets, f_max, T):
    spec = W.gw_spec(kind, dets, T, f_max, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 9.0, wf)
    P = O.OracleProblem(spec)
    th = P.prior_transform(W.uniforms(300, 11, 31))
    logl_o, parts_o = P.gw_loglike(th, parts=True)
    for kern in KERNELS:
        h = nsgw.Handle(spec)
        h.set_option(0, kern)
        logl_g, parts_g = h.gw_loglike_batch(dev(th), parts=True)
        _check_logl(logl_g.cpu().numpy(), parts_g.cpu().numpy(), logl_o, parts_o, len(dets))


def test_walk_single_detector_and_three_detectors(nsgw):
    rng = np.random.default_rng(21)
    for dets in (["H1"], ["H1", "L1", "V1"]):
        spec = W.gw_spec(W.LIKE_PHENOMD, dets, 4.0, 128.0, (20.0, 40.0))
        spec = W.make_data(spec, W.INJ_C3, 10.0, wf)
        P = O.OracleProblem(spec)
        h = nsgw.Handle(spec)
        m, B, Wlen = 120, 33, 9
        u_inj = np.array([0.4, 0.771, 0.652, 0.399, 0.0041, 0.0395, 0.8467, 0.2069, 0.5, 0.2196, 0.0317])
        donors = u_inj[None, :] + rng.normal(0, 1, (m, 11)) * np.array(W.C5_SIGMA) * 0.5
        per = np.array(spec["periodic"], bool)
        donors[:, per] -= np.floor(donors[:, per])
        donors[:, ~per] = np.clip(donors[:, ~per], 1e-6, 1 - 1e-6)
        ld = P.loglike_u(donors)
        lstar = float(np.median(ld))
        start = rng.integers(0, m, B)
        u0, l0 = donors[start].copy(), ld[start].copy()
        res_o = P.walk(donors, u0, l0, lstar, Wlen, 99, (5 << 24) | 1, slot0=0, trace=True)
        ug, lg_ = dev(u0), dev(l0)
        res_g = h.walk_batch(dev(donors), ug, lg_, lstar, Wlen, 99, (5 << 24) | 1, slot0=0, trace=True)
        clean, n_exc, n_steps = _compare_traces(res_g, res_o, lstar, Wlen, replay=(spec, P, donors, u0, 99, (5 << 24) | 1, 0))
        assert n_exc <= 2
        for key in ("n_accept", "n_eval", "n_oob"):
            assert np.array_equal(res_g[key].cpu().numpy()[clean], res_o[key][clean])
        np.testing.assert_allclose(ug.cpu().numpy()[clean], res_o["u"][clean], rtol=0, atol=1e-13)


@pytest.mark.parametrize("kind", [W.LIKE_TAYLORF2, W.LIKE_PHENOMD])
def test_waveform_parity(nsgw, kind):
    spec = W.gw_spec(kind, ["H1", "L1", "V1"], 4.0, 1024.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 20.0, wf)
    h_o = O.OracleProblem(spec).waveform(W.INJ_C3)
    h_g = nsgw.Handle(spec).gw_waveform(dev(W.INJ_C3)).cpu().numpy()
    amp = np.sqrt(h_o[..., 0] ** 2 + h_o[..., 1] ** 2).max()
    assert np.abs(h_g - h_o).max() < 5e-12 * amp


# ------------------------------------------------------------------------------------------------------
# Walk: decision parity on shared Philox streams (teacher-forced trace)
# ------------------------------------------------------------------------------------------------------
def _replay_proposal(spec, donors, u0, flags_o, seed, sid, slot, t_stop):
    """The oracle chain of one walker replayed in NumPy from its own draws (O.gamma_draw: a, b, gamma of step t) and its own trace
    (which steps were accepted) up to step t_stop: returns that step's proposal after the periodic wrap and its signed distance to
    the nearest non-periodic bound (negative outside the cube)."""
    kinds, per = np.asarray(spec["prior_kind"]), np.asarray(spec["periodic"], bool)
    free = kinds != W.FIXED
    cur = np.array(u0, dtype=np.float64)
    for t in range(t_stop + 1):
        g, a, b, _ = O.gamma_draw(int(free.sum()), seed, t, slot, sid, donors.shape[0])
        prop = np.where(free, cur + g * (donors[a] - donors[b]), cur)
        prop = np.where(per & free, prop - np.floor(prop), prop)
        if t == t_stop:
            chk = free & ~per
            margin = float(np.min(np.minimum(prop[chk], 1.0 - prop[chk]))) if chk.any() else 1.0
            return prop, margin
        if flags_o[t] & 2:
            cur = prop
    raise AssertionError


def _compare_traces(res_g, res_o, lstar, W_, replay=None):
    """Teacher-forced trace comparison.  A walker's first mismatching step must be excusable: both sides evaluated
    and a logL within 1e-8 of L*, or the out-of-bounds bit differs AND the proposal lies within 1e-12 of a non-periodic bound
    (replay = (spec, P, donors, u0, seed, sid, slot0) lets the test look at that coordinate).  Evaluated logL: the scaled 1e-10 bar."""
    fg, fo = res_g["flags"].cpu().numpy(), res_o["flags"]
    lg, lo = res_g["trace_logl"].cpu().numpy(), res_o["trace_logl"]
    B = fg.shape[0]
    n_excused, n_steps = 0, 0
    clean = np.ones(B, bool)
    for r in range(B):
        for t in range(W_):
            n_steps += 1
            if fg[r, t] != fo[r, t]:
                near = (fg[r, t] & 4) and (fo[r, t] & 4) and (abs(lg[r, t] - lstar) < 1e-8 or abs(lo[r, t] - lstar) < 1e-8)
                edge = False
                if not near and ((fg[r, t] ^ fo[r, t]) & 1) and replay is not None:
                    spec, _, donors, u0, seed, sid, slot0 = replay
                    _, margin = _replay_proposal(spec, donors, u0[r], fo[r], seed, sid, slot0 + r, t)
                    edge = abs(margin) < 1e-12
                assert near or edge, (r, t, fg[r, t], fo[r, t], lg[r, t], lo[r, t])
                n_excused += 1
                clean[r] = False
                break
            if fg[r, t] & 4:
                err = abs(lg[r, t] - lo[r, t])
                if np.isinf(lo[r, t]) or np.isinf(lg[r, t]):
                    assert lg[r, t] == lo[r, t], (r, t, lg[r, t], lo[r, t])
                elif err > 1e-10 * max(1.0, abs(lo[r, t])):
                    # cancellation between <d,h> and <h,h>/2: the bar is 1e-10 of their scale, which needs the proposal itself
                    assert replay is not None, (r, t, lg[r, t], lo[r, t])
                    spec, P, donors, u0, seed, sid, slot0 = replay
                    prop, _ = _replay_proposal(spec, donors, u0[r], fo[r], seed, sid, slot0 + r, t)
                    if spec["like_kind"] in (W.LIKE_TAYLORF2, W.LIKE_PHENOMD):
                        _, parts = P.gw_loglike(P.prior_transform(prop), parts=True)
                        scale = max(1.0, float(np.abs(parts[0, 0::2]).sum() + 0.5 * parts[0, 1::2].sum()))
                    else:
                        scale = max(1.0, abs(lo[r, t]))
                    assert err <= 1e-10 * scale, (r, t, lg[r, t], lo[r, t], scale)
    return clean, n_excused, n_steps


# spec = speculative chunk length of k_walk_gw (NSGW_OPT_WALK_SPEC): 1 = one step at a time, 8 = eight steps evaluated at once
# and the ones after an acceptance discarded, 3 = chunks that do not divide the walk length.  Results must not depend on it.
@pytest.mark.parametrize("kind,B,Wlen,spec_len", [(W.LIKE_TAYLORF2, 37, 12, 8), (W.LIKE_TAYLORF2, 37, 12, 1),
                                                  (W.LIKE_PHENOMD, 2051, 3, 8), (W.LIKE_PHENOMD, 70, 10, 3),
                                                  (W.LIKE_PHENOMD, 70, 10, 0),
                                                  # batch sizes that select the 96- and 64-thread walker CTAs (5 and 8 per SM)
                                                  (W.LIKE_PHENOMD, 700, 4, 0), (W.LIKE_TAYLORF2, 900, 4, 0)])
def test_walk_decision_parity(nsgw, kind, B, Wlen, spec_len):
    spec = W.gw_spec(kind, ["H1", "L1"], 4.0, 256.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 12.0, wf)
    P = O.OracleProblem(spec)
    h = nsgw.Handle(spec)
    h.set_option(1, spec_len)
    rng = np.random.default_rng(4)
    m = 300
    u_inj = np.array([0.4, 0.771, 0.652, 0.399, 0.0041, 0.0395, 0.8467, 0.2069, 0.5, 0.2196, 0.0317])
    donors = u_inj[None, :] + rng.normal(0, 1, (m, 11)) * np.array(W.C5_SIGMA) * 0.5
    per = np.array(spec["periodic"], bool)
    donors[:, per] -= np.floor(donors[:, per])
    donors[:, ~per] = np.clip(donors[:, ~per], 1e-6, 1 - 1e-6)
    ld = P.loglike_u(donors)
    lstar = float(np.median(ld))
    start = rng.integers(0, m, B)
    u0, l0 = donors[start].copy(), ld[start].copy()
    seed, sid = 0xC0FFEE12345, (5 << 24) | 17
    res_o = P.walk(donors, u0, l0, lstar, Wlen, seed, sid, slot0=3, trace=True)
    ug, lg_ = dev(u0), dev(l0)
    res_g = h.walk_batch(dev(donors), ug, lg_, lstar, Wlen, seed, sid, slot0=3, trace=True)
    clean, n_exc, n_steps = _compare_traces(res_g, res_o, lstar, Wlen, replay=(spec, P, donors, u0, seed, sid, 3))
    assert n_exc <= max(2, n_steps // 2000)
    # walkers whose every decision matched: identical counters, end points equal to rounding
    for key in ("n_accept", "n_eval", "n_oob"):
        assert np.array_equal(res_g[key].cpu().numpy()[clean], res_o[key][clean])
    np.testing.assert_allclose(ug.cpu().numpy()[clean], res_o["u"][clean], rtol=0, atol=1e-13)
    np.testing.assert_allclose(lg_.cpu().numpy()[clean], res_o["logl"][clean], rtol=0, atol=1e-9 * max(1.0, abs(lstar)))
    fl = res_o["flags"]
    assert (fl & 1).any() and (fl & 2).any() and ((fl & 4) > (fl & 2) * 2).any()      # the case exercises oob, accept and reject


@pytest.mark.parametrize("wk", [0, 1, 3])
def test_walk_speculation_is_invisible(nsgw, wk):
    """wk = NSGW_OPT_WALK_KERNEL (0: automatic = rounds swept by k_bins at this size, 1: one CTA per walker, 3: rounds swept by the
    lane-per-row kernel).  The speculative chunk length is a scheduling choice: end points, logL, counters and the whole trace are bit-identical
    for every value (the discarded steps are redone from the accepted point with the same Philox counters)."""
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1", "V1"], 4.0, 256.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 12.0, wf)
    h = nsgw.Handle(spec)
    h.set_option(6, wk)
    rng = np.random.default_rng(11)
    m, B, Wlen = 200, 130, 37
    u_inj = np.array([0.4, 0.771, 0.652, 0.399, 0.0041, 0.0395, 0.8467, 0.2069, 0.5, 0.2196, 0.0317])
    donors = u_inj[None, :] + rng.normal(0, 1, (m, 11)) * np.array(W.C5_SIGMA) * 0.5
    per = np.array(spec["periodic"], bool)
    donors[:, per] -= np.floor(donors[:, per])
    donors[:, ~per] = np.clip(donors[:, ~per], 1e-6, 1 - 1e-6)
    ld = h.loglike_u_batch(dev(donors)).cpu().numpy()
    lstar = float(np.quantile(ld, 0.2))
    start = rng.integers(0, m, B)
    ref = None
    for spec_len in (1, 2, 5, 8, 32, 0):
        h.set_option(1, spec_len)
        ug, lg_ = dev(donors[start]), dev(ld[start])
        res = h.walk_batch(dev(donors), ug, lg_, lstar, Wlen, 77, (5 << 24) | 3, slot0=0, trace=True)
        cur = [ug.cpu().numpy(), lg_.cpu().numpy()] + [res[k].cpu().numpy() for k in ("n_accept", "n_eval", "n_oob", "flags")]
        tl = res["trace_logl"].cpu().numpy()
        cur.append(np.where(np.isnan(tl), -1.0, tl))
        if ref is None:
            ref = cur
            assert ref[2].sum() > B and (ref[5] & 1).any()      # accepts and out-of-bounds steps both occur
        else:
            for x, y in zip(ref, cur):
                assert np.array_equal(x, y)


def test_walk_toy_and_shell_parity(nsgw):
    for spec in (W.config1()[0], W.shell_spec(6, [0, 1, 0, 0, 1, 0])):
        P = O.OracleProblem(spec)
        D = spec["ndim"]
        h = nsgw.Handle(spec)
        donors = O.draw_live(D, 150, 5)
        ld = P.loglike_u(donors)
        lstar = float(np.quantile(ld, 0.3))
        keep = np.where(ld > lstar)[0]
        donors = donors[keep]
        u0, l0 = donors[:67].copy(), ld[keep][:67].copy()
        res_o = P.walk(donors, u0, l0, lstar, 40, 99, 123, trace=True)
        ug, lg_ = dev(u0), dev(l0)
        res_g = h.walk_batch(dev(donors), ug, lg_, lstar, 40, 99, 123, trace=True)
        clean, n_exc, _ = _compare_traces(res_g, res_o, lstar, 40, replay=(spec, P, donors, u0, 99, 123, 0))
        assert n_exc == 0
        np.testing.assert_allclose(ug.cpu().numpy(), res_o["u"], rtol=0, atol=1e-13)
        assert np.array_equal(res_g["n_accept"].cpu().numpy(), res_o["n_accept"])


# ------------------------------------------------------------------------------------------------------
# ns_step / ns_run
# ------------------------------------------------------------------------------------------------------
def _sorted_live(u, l):
    o = np.lexsort((u[:, 0], l))
    return u[o], l[o]


def _step_parity(nsgw, spec, smp, nsteps, seed, tol_l, relbin_theta0=None, slice_steps=0):
    """Step-for-step comparison on the same seed and live points.  Integer work (walk length, counters) must be identical;
    floating-point state agrees to rounding drift.  Near-tied logL (a gamma = 1 proposal from a donor lands on another donor
    to 1 ulp) may be ranked in either order, so live sets are compared as sets (sorted by logL), not slot by slot."""
    P = O.OracleProblem(spec)
    if relbin_theta0 is not None:
        P.use_relbin(P.relbin(relbin_theta0))         # both sides sample the relative-binning likelihood (R:L24)
    S = O.OracleSampler(P, smp["n_live"], smp["n_delete"], smp["naccept"], smp["maxmcmc"], smp["walks0"], smp["delay"], seed=seed)
    u0, _ = S.live()
    h = nsgw.Handle(spec, smp, live_u=u0, seed=seed)
    if relbin_theta0 is not None:
        h.relbin_setup(relbin_theta0)
        h.set_option(2, 1)
    if slice_steps:
        S.use_slice_kernel(slice_steps)                # both sides replace points by hit-and-run slice steps (R:L25)
        h.set_option(4, slice_steps)
        h.set_option(3, 1)
    D, k = spec["ndim"], smp["n_delete"]
    for it in range(nsteps):
        dead_g = torch.empty(k, D + 3, dtype=torch.float64, device="cuda")
        st_g = h.step(dead=dead_g)
        st_o, dead_o = S.step(want_dead=True)
        for key in ("iteration", "walk_len", "accept_min", "accept_max", "n_eval", "n_oob", "n_stuck", "n_eval_total"):
            assert st_g[key] == st_o[key], (it, key, st_g[key], st_o[key])
        for key in ("logl_star", "logx", "logz", "h", "dlogz", "live_frac_log", "walks_next", "accept_mean"):
            # H's running update cancels terms of size |logZ|: allow 1e-9
            tol = 1e-9 if key == "h" else 1e-12 * max(1.0, abs(st_o[key])) + tol_l
            assert abs(st_g[key] - st_o[key]) <= tol, (it, key, st_g[key], st_o[key])
        np.testing.assert_allclose(dead_g.cpu().numpy(), dead_o, rtol=0, atol=tol_l + 1e-10)
        ug, lg_ = h.get_live()
        ug, lg_ = _sorted_live(ug.cpu().numpy(), lg_.cpu().numpy())
        uo, lo = _sorted_live(*S.live())
        np.testing.assert_allclose(lg_, lo, rtol=0, atol=tol_l + 1e-10)
        # rows whose logL is separated from its neighbours by more than the tolerance are uniquely ordered
        sep = np.ones(len(lo), bool)
        gap = np.diff(lo) > 1e-7
        sep[1:] &= gap
        sep[:-1] &= gap
        np.testing.assert_allclose(ug[sep], uo[sep], rtol=0, atol=1e-10)
    zg = h.finalize_evidence()
    zo = S.finalize()
    np.testing.assert_allclose(zg, zo, rtol=0, atol=1e-9 + tol_l)


def test_ns_step_parity_toy(nsgw):
    spec, smp, _ = W.config1()
    _step_parity(nsgw, spec, smp, 12, 21, 1e-11)


def test_ns_step_parity_shell_periodic(nsgw):
    spec = W.shell_spec(5, [0, 1, 0, 0, 1])
    smp = dict(n_live=333, n_delete=111, naccept=15, maxmcmc=400, walks0=33.0, delay=-1.0)
    _step_parity(nsgw, spec, smp, 8, 5, 0.0)


def test_ns_step_parity_gw(nsgw):
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 200.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 10.0, wf)
    smp = dict(n_live=90, n_delete=45, naccept=8, maxmcmc=40, walks0=10.0, delay=-1.0)
    _step_parity(nsgw, spec, smp, 4, 8, 1e-8)


def test_config1_full_runs_closed_form_logz(nsgw):
    spec, smp, truth = W.config1()
    pulls = []
    for seed in range(1, 41):
        h = nsgw.Handle(spec, smp, seed=seed)
        nit, st = h.run(smp["term_kind"], smp["term_tol"], 500)
        logz, err, H = h.finalize_evidence()
        assert 30 < nit < 90 and st["dlogz"] < smp["term_tol"]
        pulls.append((logz - truth["logz_exact"]) / err)
    pulls = np.array(pulls)
    assert np.all(np.abs(pulls) < 4.5)
    assert abs(pulls.mean()) < 3.0 / math.sqrt(len(pulls))
    assert 0.6 < pulls.std() < 1.5


def test_config1_run_vs_oracle_run(nsgw):
    # same seed: the first iterations reproduce the oracle decision for decision (checked by _step_parity above); a full run
    # is a chaotic Markov chain, so 1-ulp libm differences eventually flip a decision and only statistical agreement is defined:
    # logZ within the combined error (BJ).
    spec, smp, _ = W.config1()
    P = O.OracleProblem(spec)
    S = O.OracleSampler(P, smp["n_live"], smp["n_delete"], smp["naccept"], smp["maxmcmc"], smp["walks0"], smp["delay"], seed=77)
    n_o, st_o = S.run(0, 0.01, 500)
    h = nsgw.Handle(spec, smp, seed=77)
    n_g, st_g = h.run(0, 0.01, 500)
    assert abs(n_g - n_o) <= 3 and abs(st_g["n_eval_total"] - st_o["n_eval_total"]) < 0.05 * st_o["n_eval_total"]
    (zg, eg, _), (zo, eo, _) = h.finalize_evidence(), S.finalize()
    assert abs(zg - zo) < 3 * math.hypot(eg, eo)


def test_bench_configuration_sampled_parity(nsgw, c2):
    """BASELINE config 2 at full size in the launch configuration bench.py times (B = 65536 rows of the index-keyed stream,
    automatic kernel choice = k_bins_lp): 192 sampled rows against the oracle, and every row against the other kernel."""
    B = 65536
    h = nsgw.Handle(c2)
    u = dev(W.uniform_rows(0, B, 11, seed=2))
    theta = h.prior_transform_batch(u)
    logl, parts = h.gw_loglike_batch(theta, parts=True)
    logl, parts = logl.cpu().numpy(), parts.cpu().numpy()
    assert np.all(np.isfinite(logl))
    idx = np.unique(np.concatenate([np.arange(0, B, 347), [0, 127, 128, 255, 256, B - 257, B - 256, B - 1]]))
    P = O.OracleProblem(c2)
    lo, po = P.gw_loglike(theta.cpu().numpy()[idx], parts=True)
    _check_logl(logl[idx], parts[idx], lo, po, 2)
    h.set_option(0, 1)
    l1, p1 = h.gw_loglike_batch(theta, parts=True)
    scale = np.maximum(1.0, np.abs(parts[:, 0::2]).sum(1) + 0.5 * parts[:, 1::2].sum(1))
    assert np.max(np.abs(l1.cpu().numpy() - logl) / scale) < 2e-11
    # the identical call is bit-reproducible (fixed reduction order, no atomics)
    h.set_option(0, 0)
    assert np.array_equal(h.gw_loglike_batch(theta).cpu().numpy(), logl)


def test_phenomd_config4_shape_parity(nsgw):
    # config-4 shape: Mc in [8, 20], 8 s at 4096 Hz, 16225 bins x 2 detectors
    spec, _ = W.config4(wf)
    assert spec["n_freq"] == 16225 and spec["n_det"] == 2
    P = O.OracleProblem(spec)
    th = P.prior_transform(W.uniforms(48, 11, 404))
    logl_o, parts_o = P.gw_loglike(th, parts=True)
    logl_g, parts_g = nsgw.Handle(spec).gw_loglike_batch(dev(th), parts=True)
    _check_logl(logl_g.cpu().numpy(), parts_g.cpu().numpy(), logl_o, parts_o, 2)


def _two_free_dims(spec):
    kinds, lo, hi = list(spec["prior_kind"]), list(spec["prior_lo"]), list(spec["prior_hi"])
    for d in range(11):
        if d not in (4, 5):
            kinds[d] = W.FIXED
            lo[d] = hi[d] = W.INJ_C3[d]
    spec["prior_kind"], spec["prior_lo"], spec["prior_hi"] = kinds, lo, hi
    spec["periodic"] = [0] * 11
    return spec


def test_gw_2d_logz_against_quadrature(nsgw):
    """BJ pin 'brute-force quadrature of logZ in 2-D', on the CUDA path: GW likelihood with only (dL, theta_jn) free, the rest
    FIXED at the injection; 256^2 midpoint quadrature of exp(logL) over the unit square (evaluated by gw_loglike through
    ns_loglike_u_batch and cross-checked on a sub-grid against the oracle) vs full nested-sampling runs of the library."""
    spec = W.gw_spec(W.LIKE_TAYLORF2, ["H1", "L1"], 4.0, 96.0, (20.0, 40.0))
    spec = _two_free_dims(W.make_data(spec, W.INJ_C3, 8.0, wf))
    G = 256
    g = (np.arange(G) + 0.5) / G
    u = np.full((G * G, 11), 0.5)
    u[:, 4] = np.repeat(g, G)
    u[:, 5] = np.tile(g, G)
    hq = nsgw.Handle(spec)
    ll = hq.loglike_u_batch(dev(u)).cpu().numpy()
    sub = np.arange(0, G * G, 97)
    lo = O.OracleProblem(spec).loglike_u(u[sub])
    assert np.max(np.abs(ll[sub] - lo)) < 1e-9
    m = ll.max()
    logz_quad = m + math.log(np.mean(np.exp(ll - m)))
    smp = dict(n_live=200, n_delete=100, naccept=20, maxmcmc=5000, walks0=100.0, delay=-1.0)
    pulls = []
    for seed in range(1, 7):
        h = nsgw.Handle(spec, smp, seed=seed)
        h.run(0, 0.01, 400)
        logz, err, _ = h.finalize_evidence()
        pulls.append((logz - logz_quad) / err)
    assert np.all(np.abs(pulls) < 4.0) and abs(np.mean(pulls)) < 2.0, (pulls, logz_quad)


def test_gw_full_run_vs_oracle_run_statistics(nsgw):
    """Full runs are chaotic chains, so GPU and oracle agree statistically only (BJ): logZ within the combined error bars, and
    one-dimensional two-sample KS tests on equal-weight posterior resamples of every sampled parameter.  Problem sized so that
    the chains mix (two oracle runs with different seeds pass the same KS bar; with all 11 dimensions free and a short maxmcmc
    they do not, which says nothing about parity): PhenomD-form, H1+L1, 20-128 Hz = 433 bins, SNR 10, free Mc, q, dL, tc (the
    rest FIXED at the injection), n_live 400, k 200, naccept 20; the oracle run takes about half a minute."""
    from scipy import stats
    free = (0, 1, 4, 8)
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 128.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 10.0, wf)
    kinds, lo_, hi_ = list(spec["prior_kind"]), list(spec["prior_lo"]), list(spec["prior_hi"])
    for d in range(11):
        if d not in free:
            kinds[d] = W.FIXED
            lo_[d] = hi_[d] = W.INJ_C3[d]
    spec["prior_kind"], spec["prior_lo"], spec["prior_hi"] = kinds, lo_, hi_
    spec["periodic"] = [0] * 11
    smp = dict(n_live=400, n_delete=200, naccept=20, maxmcmc=2000, walks0=50.0, delay=-1.0)
    P = O.OracleProblem(spec)

    def posterior(dead, live_u, live_l, logx_end, rng, n=1000):
        # dead rows: u.., logL, logw, n_i; remaining live points share the final volume equally
        u = np.concatenate([dead[:, :11], live_u])
        lw = np.concatenate([dead[:, 11] + dead[:, 12], live_l + logx_end - math.log(len(live_l))])
        w = np.exp(lw - lw.max())
        return u[rng.choice(len(u), n, p=w / w.sum())]

    max_it = 80
    # GPU run
    h = nsgw.Handle(spec, smp, seed=5)
    dead_g = torch.zeros(max_it * smp["n_delete"], 14, dtype=torch.float64, device="cuda")
    n_g, st_g = h.run(0, 0.1, max_it, dead=dead_g)
    zg, eg, _ = h.finalize_evidence()
    lu, ll = h.get_live()
    rng = np.random.default_rng(1)
    post_g = posterior(dead_g.cpu().numpy()[: n_g * smp["n_delete"]], lu.cpu().numpy(), ll.cpu().numpy(), st_g["logx"], rng)
    # oracle run (different seed: independent chains)
    S = O.OracleSampler(P, smp["n_live"], smp["n_delete"], smp["naccept"], smp["maxmcmc"], smp["walks0"], smp["delay"], seed=6)
    n_o, st_o, dead_o = S.run(0, 0.1, max_it, want_dead=True)
    zo, eo, _ = S.finalize()
    uo, lo = S.live()
    post_o = posterior(dead_o, uo, lo, st_o["logx"], rng)
    assert abs(zg - zo) < 3.0 * math.hypot(eg, eo), (zg, eg, zo, eo)
    assert abs(n_g - n_o) <= 4
    assert abs(st_g["walk_len"] - st_o["walk_len"]) < 0.5 * st_o["walk_len"]      # both adapt to the same walk length
    pvals = [stats.ks_2samp(post_g[:, d], post_o[:, d]).pvalue for d in free]
    # resamples of weighted chains are not independent draws: the bar is BJ's p > 0.01 / n_dim on every sampled parameter
    assert min(pvals) > 0.01 / len(free), pvals


def test_run_many_equals_single_runs(nsgw):
    """ns_run_many steps several samplers concurrently on streams of their own; every run must be bit-identical to the same
    handle driven alone by ns_run (toy and GW problems mixed in one call, different lengths)."""
    spec1, smp1, _ = W.config1()
    specg = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 128.0, (20.0, 40.0))
    specg = W.make_data(specg, W.INJ_C3, 10.0, wf)
    smpg = dict(n_live=300, n_delete=150, naccept=10, maxmcmc=200, walks0=20.0, delay=-1.0)
    jobs = [(spec1, smp1, 3), (specg, smpg, 4), (spec1, smp1, 5), (specg, smpg, 6)]
    max_it = 90
    single = []
    for spec, smp, seed in jobs:
        h = nsgw.Handle(spec, smp, seed=seed)
        n, st = h.run(0, 0.5, max_it)
        single.append((n, st, h.finalize_evidence(), h.get_live()[0].cpu().numpy()))
    hs = [nsgw.Handle(spec, smp, seed=seed) for spec, smp, seed in jobs]
    dead = [torch.zeros(max_it * smp["n_delete"], spec["ndim"] + 3, dtype=torch.float64, device="cuda") for spec, smp, _ in jobs]
    its, sts = nsgw.run_many(hs, 0, 0.5, max_it, dead=dead)
    assert len(set(its)) > 1                                          # runs of different lengths in one call
    for h, n_m, st_m, (n_s, st_s, fin_s, live_s), d, (spec, smp, _) in zip(hs, its, sts, single, dead, jobs):
        assert n_m == n_s and st_m == st_s
        assert h.finalize_evidence() == fin_s
        assert np.array_equal(h.get_live()[0].cpu().numpy(), live_s)
        rows = d.cpu().numpy()[: n_m * smp["n_delete"]]
        assert np.all(np.diff(rows[:, spec["ndim"]]) >= 0)            # dead points come out in ascending logL


# ------------------------------------------------------------------------------------------------------
# Relative binning (R:L24): set-up (edges: integers, bit-exact; summary data) and evaluation against the oracle's
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind,dets,f_max,T", [(W.LIKE_TAYLORF2, ["H1", "L1"], 1024.0, 4.0),       # config-2 shape
                                               (W.LIKE_PHENOMD, ["H1", "L1"], 1024.0, 4.0),        # config-3 shape
                                               (W.LIKE_PHENOMD, ["H1", "L1", "V1"], 512.0, 8.0),   # three detectors
                                               (W.LIKE_TAYLORF2, ["L1"], 128.0, 2.0)])             # one detector, short grid
def test_relbin_parity(nsgw, kind, dets, f_max, T):
    spec = W.gw_spec(kind, dets, T, f_max, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 15.0, wf)
    P = O.OracleProblem(spec)
    nd = len(dets)
    h = nsgw.Handle(spec)
    for eps in (0.5, 0.11):
        rb = P.relbin(W.INJ_C3, eps=eps)
        nb = h.relbin_setup(W.INJ_C3, eps=eps)
        ed, A0, A1, B0, B1 = h.relbin_get()
        assert nb == rb.n_bins and np.array_equal(ed, rb.edges())          # integer work: bit-exact
        oA0, oA1, oB0, oB1 = rb.summary()
        sc = np.abs(oA0).max()
        np.testing.assert_allclose(A0, oA0, rtol=0, atol=1e-10 * sc)
        np.testing.assert_allclose(A1, oA1, rtol=0, atol=1e-10 * np.abs(oA1).max())
        np.testing.assert_allclose(B0, oB0, rtol=1e-11, atol=0)
        np.testing.assert_allclose(B1, oB1, rtol=0, atol=1e-11 * np.abs(oB1).max())
        # rows: prior draws (far from the fiducial point: large, but identical, approximation errors), posterior-like scatter,
        # the fiducial point itself and an unphysical row
        rng = np.random.default_rng(8)
        u0 = np.array([0.4, 0.771, 0.652, 0.399, 0.0041, 0.0395, 0.8467, 0.2069, 0.5, 0.2196, 0.0317])
        u = np.concatenate([W.uniforms(200, 11, 55), u0[None, :] + rng.normal(0, 1, (330, 11)) * np.array(W.C5_SIGMA) * 0.1])
        per = np.array(spec["periodic"], bool)
        u[:, per] -= np.floor(u[:, per])
        u[:, ~per] = np.clip(u[:, ~per], 1e-6, 1 - 1e-6)
        th = P.prior_transform(u)
        th[0] = W.INJ_C3
        th[1, 1] = 1.5
        lo, po = rb.loglike(th, parts=True)
        lg, pg = h.gw_loglike_relbin_batch(dev(th), parts=True)
        lg, pg = lg.cpu().numpy(), pg.cpu().numpy()
        assert np.isneginf(lg[1]) and np.isneginf(lo[1])
        ok = np.isfinite(lo)
        scale = np.maximum(1.0, np.abs(po[ok, 0::2]).sum(1) + 0.5 * np.abs(po[ok, 1::2]).sum(1))
        assert np.max(np.abs(lg[ok] - lo[ok]) / scale) < 1e-10
        np.testing.assert_allclose(pg[ok], po[ok], rtol=0, atol=1e-10 * scale.max())
        # and the approximation itself: equal to the exact kernel at the fiducial point
        exact = h.gw_loglike_batch(dev(th[:1])).cpu().numpy()[0]
        assert abs(lg[0] - exact) < 1e-9 * max(1.0, abs(exact))


def test_ns_step_parity_gw_relbin(nsgw):
    # the sampler on the relative-binning likelihood: step-for-step against the oracle's sampler on its relative-binning likelihood
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 256.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 12.0, wf)
    smp = dict(n_live=120, n_delete=60, naccept=8, maxmcmc=60, walks0=12.0, delay=-1.0)
    _step_parity(nsgw, spec, smp, 4, 8, 1e-8, relbin_theta0=W.INJ_C3)


@pytest.mark.parametrize("kind,dets", [(W.LIKE_TAYLORF2, ["H1", "L1"]), (W.LIKE_PHENOMD, ["H1", "L1", "V1"])])
def test_walk_relbin_decision_parity(nsgw, kind, dets):
    spec = W.gw_spec(kind, dets, 4.0, 256.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 12.0, wf)
    P = O.OracleProblem(spec)
    P.use_relbin(P.relbin(W.INJ_C3, eps=0.3))
    h = nsgw.Handle(spec)
    h.relbin_setup(W.INJ_C3, eps=0.3)
    h.set_option(2, 1)
    rng = np.random.default_rng(14)
    m, B, Wlen = 250, 300, 9
    u_inj = np.array([0.4, 0.771, 0.652, 0.399, 0.0041, 0.0395, 0.8467, 0.2069, 0.5, 0.2196, 0.0317])
    donors = u_inj[None, :] + rng.normal(0, 1, (m, 11)) * np.array(W.C5_SIGMA) * 0.5
    per = np.array(spec["periodic"], bool)
    donors[:, per] -= np.floor(donors[:, per])
    donors[:, ~per] = np.clip(donors[:, ~per], 1e-6, 1 - 1e-6)
    ld = P.loglike_u(donors)
    np.testing.assert_allclose(h.loglike_u_batch(dev(donors)).cpu().numpy(), ld, rtol=0, atol=1e-9 * np.abs(ld).max())
    lstar = float(np.median(ld))
    start = rng.integers(0, m, B)
    u0, l0 = donors[start].copy(), ld[start].copy()
    res_o = P.walk(donors, u0, l0, lstar, Wlen, 4242, (5 << 24) | 2, slot0=0, trace=True)
    ug, lg_ = dev(u0), dev(l0)
    res_g = h.walk_batch(dev(donors), ug, lg_, lstar, Wlen, 4242, (5 << 24) | 2, slot0=0, trace=True)
    clean, n_exc, n_steps = _compare_traces(res_g, res_o, lstar, Wlen, replay=(spec, P, donors, u0, 4242, (5 << 24) | 2, 0))
    assert n_exc <= 2
    for key in ("n_accept", "n_eval", "n_oob"):
        assert np.array_equal(res_g[key].cpu().numpy()[clean], res_o[key][clean])
    np.testing.assert_allclose(ug.cpu().numpy()[clean], res_o["u"][clean], rtol=0, atol=1e-13)
    fl = res_o["flags"]
    assert (fl & 1).any() and (fl & 2).any()


def test_relbin_run_agrees_with_exact_run(nsgw):
    """A full run on the relative-binning likelihood against the same run on the exact one (same seed, same live points): the
    evidence agrees within the nested-sampling error (the approximation error in the bulk is < 0.05, pinned on the oracle)."""
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 512.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 12.0, wf)
    free = (0, 1, 4, 8)
    kinds, lo_, hi_ = list(spec["prior_kind"]), list(spec["prior_lo"]), list(spec["prior_hi"])
    for d in range(11):
        if d not in free:
            kinds[d] = W.FIXED
            lo_[d] = hi_[d] = W.INJ_C3[d]
    spec["prior_kind"], spec["prior_lo"], spec["prior_hi"] = kinds, lo_, hi_
    spec["periodic"] = [0] * 11
    smp = dict(n_live=400, n_delete=200, naccept=20, maxmcmc=2000, walks0=50.0, delay=-1.0)
    he = nsgw.Handle(spec, smp, seed=9)
    ne, _ = he.run(0, 0.1, 200)
    ze, ee, _ = he.finalize_evidence()
    hr = nsgw.Handle(spec, smp, seed=9)
    hr.relbin_setup(W.INJ_C3)
    hr.set_option(2, 1)
    nr, _ = hr.run(0, 0.1, 200)
    zr, er, _ = hr.finalize_evidence()
    assert abs(nr - ne) <= 3
    assert abs(zr - ze) < 3.0 * math.hypot(ee, er) + 0.05, (zr, er, ze, ee)


def test_relbin_given_edges_and_errors(nsgw, c2):
    h = nsgw.Handle(c2)
    P = O.OracleProblem(c2)
    with pytest.raises(nsgw.NsgwError):
        h.gw_loglike_relbin_batch(dev(np.array([W.INJ_C3])))              # no set-up yet
    nf = c2["n_freq"]
    edges = [0, 5, 6, 40, 400, 2000, nf - 1]
    assert h.relbin_setup(W.INJ_C3, edges=edges) == len(edges) - 1
    ed, A0, A1, B0, B1 = h.relbin_get()
    assert list(ed) == edges
    _, parts = P.gw_loglike(np.array([W.INJ_C3]), parts=True)
    assert abs(B0[0].sum() - parts[0, 1]) < 1e-10 * parts[0, 1]           # the bins partition <h0, h0>
    for bad in ([1, 5, nf - 1], [0, 5, 5, nf - 1], [0, 7, nf - 2], [0]):
        with pytest.raises(nsgw.NsgwError):
            h.relbin_setup(W.INJ_C3, edges=bad)
    bad_th = list(W.INJ_C3)
    bad_th[1] = 2.0
    with pytest.raises(nsgw.NsgwError):
        h.relbin_setup(bad_th)
    with pytest.raises(nsgw.NsgwError):
        h.relbin_setup(W.INJ_C3, eps=-1.0)
    with pytest.raises(nsgw.NsgwError):
        h.relbin_setup(W.INJ_C3, eps=1e-9)                                # more bins than grid points
    spec1, smp1, _ = W.config1()
    with pytest.raises(nsgw.NsgwError):
        nsgw.Handle(spec1, smp1).relbin_setup(W.INJ_C3)                   # not a GW handle


def test_ns_step_parity_slice_kernel(nsgw):
    # the sampler with the slice kernel inside (covariance factor computed on the device every iteration), step for step
    spec, smp, _ = W.config1()
    _step_parity(nsgw, spec, smp, 8, 13, 1e-10, slice_steps=9)
    _step_parity(nsgw, W.shell_spec(5, [0, 1, 0, 0, 0]), dict(n_live=150, n_delete=50, naccept=10, maxmcmc=200, walks0=20.0, delay=-1.0),
                 6, 14, 1e-12, slice_steps=7)
    gspec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 128.0, (20.0, 40.0))
    gspec = W.make_data(gspec, W.INJ_C3, 10.0, wf)
    _step_parity(nsgw, gspec, dict(n_live=100, n_delete=50, naccept=8, maxmcmc=60, walks0=12.0, delay=-1.0), 3, 15, 1e-8, slice_steps=5)


def test_slice_and_walk_kernels_agree_on_gw_evidence(nsgw):
    """Two different inner kernels, one evidence: PhenomD-form, H1+L1, 20-512 Hz, SNR 12, free Mc, q, dL, tc (a problem on which
    both chains mix: the walk reaches its naccept, the slice kernel moves at every step); three seeds each."""
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 512.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 12.0, wf)
    free = (0, 1, 4, 8)
    kinds, lo_, hi_ = list(spec["prior_kind"]), list(spec["prior_lo"]), list(spec["prior_hi"])
    for d in range(11):
        if d not in free:
            kinds[d] = W.FIXED
            lo_[d] = hi_[d] = W.INJ_C3[d]
    spec["prior_kind"], spec["prior_lo"], spec["prior_hi"] = kinds, lo_, hi_
    spec["periodic"] = [0] * 11
    smp = dict(n_live=600, n_delete=300, naccept=30, maxmcmc=3000, walks0=60.0, delay=-1.0)
    out = {}
    for name, opts in (("walk", []), ("slice", [(4, 24), (3, 1)])):
        zs, es = [], []
        for seed in (1, 2, 3):
            h = nsgw.Handle(spec, smp, seed=seed)
            for k_, v_ in opts:
                h.set_option(k_, v_)
            h.run(0, 0.1, 2000)
            z, e, _ = h.finalize_evidence()
            zs.append(z)
            es.append(e)
        out[name] = (np.mean(zs), np.mean(es) / math.sqrt(3))
    (zw, ew), (zs_, es_) = out["walk"], out["slice"]
    assert abs(zw - zs_) < 3.5 * math.hypot(ew, es_), out


def test_slice_sampler_config1_closed_form_logz(nsgw):
    spec, smp, ref = W.config1()
    pulls = []
    for seed in range(1, 9):
        h = nsgw.Handle(spec, smp, seed=seed)
        h.set_option(4, 20)
        h.set_option(3, 1)
        nit, st = h.run(smp["term_kind"], smp["term_tol"], 500)
        assert st["walk_len"] == 20 and st["accept_min"] >= 19 and st["dlogz"] < smp["term_tol"]
        logz, err, _ = h.finalize_evidence()
        pulls.append((logz - ref["logz_exact"]) / err)
    pulls = np.array(pulls)
    assert np.all(np.abs(pulls) < 3.5) and abs(pulls.mean()) < 1.3, pulls


# ------------------------------------------------------------------------------------------------------
# Hit-and-run slice sampling (R:L25): the same chains as the oracle on shared Philox streams
# ------------------------------------------------------------------------------------------------------
def _slice_compare(res_g, ug, lg, res_o, lstar):
    """Walkers whose per-step evaluation counts all agree made the same decisions: identical counters, end points to rounding.
    A walker may differ only where a candidate's logL sits within 1e-8 of L* (or a coordinate within 1e-12 of a bound)."""
    te_g, te_o = res_g["trace_evals"].cpu().numpy(), res_o["trace_evals"]
    clean = np.all(te_g == te_o, axis=1)
    assert clean.mean() > 0.98, clean.mean()
    for key in ("n_eval", "n_oob", "n_expand", "n_shrink", "n_stuck"):
        assert np.array_equal(res_g[key].cpu().numpy()[clean], res_o[key][clean]), key
    np.testing.assert_allclose(ug.cpu().numpy()[clean], res_o["u"][clean], rtol=0, atol=1e-11)
    np.testing.assert_allclose(lg.cpu().numpy()[clean], res_o["logl"][clean], rtol=0, atol=1e-9 * max(1.0, abs(lstar)))
    np.testing.assert_allclose(res_g["trace_logl"].cpu().numpy()[clean], res_o["trace_logl"][clean], rtol=0,
                               atol=1e-9 * max(1.0, abs(lstar)))
    return clean


def test_slice_toy_and_shell_parity(nsgw):
    for spec, lc_scale in ((W.config1()[0], 0.05), (W.shell_spec(6, [0, 1, 0, 0, 1, 0]), 0.2)):
        P = O.OracleProblem(spec)
        D = spec["ndim"]
        h = nsgw.Handle(spec)
        pts = O.draw_live(D, 300, 5)
        ld = P.loglike_u(pts)
        lstar = float(np.quantile(ld, 0.5))
        keep = np.where(ld > lstar)[0][:97]
        u0, l0 = pts[keep].copy(), ld[keep].copy()
        rng = np.random.default_rng(3)
        A = rng.normal(size=(D, D)) * lc_scale
        Lc = np.linalg.cholesky(A @ A.T + 1e-4 * np.eye(D))
        res_o = P.slice_walk(Lc, u0, l0, lstar, 12, 31337, (6 << 24) | 4, slot0=2, trace=True)
        ug, lg = dev(u0), dev(l0)
        res_g = h.slice_batch(dev(Lc), ug, lg, lstar, 12, 31337, (6 << 24) | 4, slot0=2, trace=True)
        clean = _slice_compare(res_g, ug, lg, res_o, lstar)
        assert clean.all()                                    # no transcendental in these likelihoods near a threshold
        assert res_o["n_expand"].sum() > 0 and res_o["n_shrink"].sum() > 0


@pytest.mark.parametrize("kind,dets", [(W.LIKE_TAYLORF2, ["H1", "L1"]), (W.LIKE_PHENOMD, ["H1", "L1", "V1"]), (W.LIKE_PHENOMD, ["L1"])])
def test_slice_gw_parity(nsgw, kind, dets):
    spec = W.gw_spec(kind, dets, 4.0, 256.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 12.0, wf)
    P = O.OracleProblem(spec)
    h = nsgw.Handle(spec)
    rng = np.random.default_rng(17)
    m, B, S = 250, 120, 6
    u_inj = np.array([0.4, 0.771, 0.652, 0.399, 0.0041, 0.0395, 0.8467, 0.2069, 0.5, 0.2196, 0.0317])
    pts = u_inj[None, :] + rng.normal(0, 1, (m, 11)) * np.array(W.C5_SIGMA) * 0.5
    per = np.array(spec["periodic"], bool)
    pts[:, per] -= np.floor(pts[:, per])
    pts[:, ~per] = np.clip(pts[:, ~per], 1e-6, 1 - 1e-6)
    ld = P.loglike_u(pts)
    lstar = float(np.median(ld))
    surv = pts[ld > lstar]
    Lc = np.linalg.cholesky(np.cov(surv.T) + 1e-12 * np.eye(11))      # the live points' covariance, as a sampler would use it
    start = rng.integers(0, len(surv), B)
    u0, l0 = surv[start].copy(), ld[ld > lstar][start].copy()
    res_o = P.slice_walk(Lc, u0, l0, lstar, S, 2024, (6 << 24) | 9, slot0=0, trace=True)
    ug, lg = dev(u0), dev(l0)
    res_g = h.slice_batch(dev(Lc), ug, lg, lstar, S, 2024, (6 << 24) | 9, slot0=0, trace=True)
    _slice_compare(res_g, ug, lg, res_o, lstar)
    te = res_o["trace_evals"]
    assert te.min() >= 1 and te.max() > te.min() + 2           # the per-step cost really varies from walker to walker
    assert np.all(res_o["logl"] > lstar)


def test_error_codes(nsgw, c2):
    import ctypes as C
    h = nsgw.Handle(c2)
    with pytest.raises(nsgw.NsgwError):
        h.step()                                    # no live set in a likelihood-only handle
    bad = dict(c2)
    bad["psd"] = np.array(c2["psd"]); bad["psd"][1, 5] = 0.0
    with pytest.raises(nsgw.NsgwError):
        nsgw.Handle(bad)
    u = dev(W.uniforms(4, 11, 1))
    rc = nsgw.lib().ns_walk_batch(h._h, C.c_void_p(u.data_ptr()), C.c_int32(1), C.c_void_p(u.data_ptr()), C.c_void_p(u.data_ptr()),
                                  C.c_int64(4), C.c_double(0.0), C.c_int32(5), C.c_uint64(1), C.c_uint32(0), C.c_int64(0),
                                  None, None, None, None, None, None)
    assert rc == -1


def test_fp64_peak_probe(nsgw):
    tf = nsgw.measure_fp64_peak(1 << 16)
    assert 10.0 < tf < 60.0, tf


# ---- posterior weights (ns_posterior; reading R:L26) --------------------------------------------------------------------------
def _posterior_parity(nsgw, spec, smp, seed, max_iter, ref, term=(0, 0.01)):
    h = nsgw.Handle(spec, smp, seed=seed)
    k, D = smp["n_delete"], spec["ndim"]
    dead, nit, logx = None, 0, 0.0
    if max_iter:
        buf = torch.full((max_iter * k, D + 3), float("nan"), dtype=torch.float64, device="cuda")
        nit, st = h.run(term[0], term[1], max_iter, dead=buf)
        dead, logx = buf[: nit * k].contiguous(), st["logx"]
    out = h.posterior(dead, theta_ref=ref)
    lu, ll = h.get_live()
    want = O.posterior(O.OracleProblem(spec), None if dead is None else dead.cpu().numpy(), lu.cpu().numpy(), ll.cpu().numpy(), logx,
                       theta_ref=ref)
    N = nit * k + smp["n_live"]
    assert out["theta"].shape == (N, D) and out["logp"].shape == (N,)
    np.testing.assert_allclose(out["theta"].cpu().numpy(), want["theta"], rtol=4e-15, atol=4e-15)
    np.testing.assert_allclose(out["logp"].cpu().numpy(), want["logp"], rtol=0, atol=1e-10)
    assert abs(out["logz"] - want["logz"]) < 1e-10
    assert abs(out["ess"] / want["ess"] - 1.0) < 1e-10
    np.testing.assert_allclose(out["cl"], want["cl"], rtol=0, atol=1e-12)
    assert abs(out["logz"] - h.finalize_evidence()[0]) < 1e-9          # same terms as the sequential scan, other summation order
    assert abs(float(torch.exp(out["logp"]).sum()) - 1.0) < 1e-12
    # the sampler's state is untouched and the call is bit-reproducible (fixed-order reductions)
    again = h.posterior(dead, theta_ref=ref)
    assert torch.equal(again["logp"], out["logp"]) and again["ess"] == out["ess"] and np.array_equal(again["cl"], out["cl"])
    lu2, ll2 = h.get_live()
    assert torch.equal(lu2, lu) and torch.equal(ll2, ll)
    return out, want


def test_posterior_parity_config1(nsgw):
    spec, smp, _ = W.config1()
    ref = [0.1, -0.3, 0.4, 0.2]
    out, _ = _posterior_parity(nsgw, spec, smp, 5, 500, ref)        # to termination: 50+ iterations, several thousand rows
    assert 300 < out["ess"] < 3000
    _posterior_parity(nsgw, spec, smp, 6, 28, ref)                  # stopped early: the live points' rows carry the mass
    out0, _ = _posterior_parity(nsgw, spec, smp, 7, 0, ref)         # no dead points at all: live rows only, logX = 0
    assert out0["theta"].shape[0] == smp["n_live"]
    # without a reference point: NaN levels, same weights
    h = nsgw.Handle(spec, smp, seed=7)
    o2 = h.posterior(None)
    assert np.all(np.isnan(o2["cl"])) and torch.equal(o2["logp"], out0["logp"])
    o3 = h.posterior(None, want_theta=False)
    assert o3["theta"] is None and torch.equal(o3["logp"], out0["logp"])


def test_posterior_parity_gw_priors(nsgw):
    # PhenomD-form problem with the full 11-parameter prior box (power-law distance, sine / cosine angles, periodic dims)
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 200.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 10.0, wf)
    smp = dict(n_live=90, n_delete=45, naccept=8, maxmcmc=40, walks0=10.0, delay=-1.0)
    _posterior_parity(nsgw, spec, smp, 8, 7, list(W.INJ_C3), term=(0, 1e-9))


def test_posterior_argument_errors(nsgw):
    import ctypes as C
    spec, smp, _ = W.config1()
    h = nsgw.Handle(spec, smp, seed=1)
    L = nsgw.lib()
    logp = torch.empty(smp["n_live"] + 5, dtype=torch.float64, device="cuda")
    ref = (C.c_double * 4)(0.0, 0.0, 0.0, 0.0)
    null = C.c_void_p(0)
    assert L.ns_posterior(h._h, null, C.c_int64(5), null, C.c_void_p(logp.data_ptr()), None, None, null) == -1     # rows without a buffer
    assert L.ns_posterior(h._h, null, C.c_int64(0), null, null, None, None, null) == -1                          # no output
    assert L.ns_posterior(h._h, null, C.c_int64(0), null, C.c_void_p(logp.data_ptr()), ref, None, null) == -1      # levels need theta
    assert L.ns_posterior(h._h, null, C.c_int64(-1), null, C.c_void_p(logp.data_ptr()), None, None, null) == -1
    assert L.ns_posterior(None, null, C.c_int64(0), null, C.c_void_p(logp.data_ptr()), None, None, null) == -3
    hb = nsgw.Handle(W.config2(wf))                                                                              # no live set
    assert L.ns_posterior(hb._h, null, C.c_int64(0), null, C.c_void_p(logp.data_ptr()), None, None, null) == -3


def test_posterior_config1_moments_from_device_runs(nsgw):
    # end to end on the device: weighted second moments and marginal CDFs of the analytic Gaussian over 24 runs
    spec, smp, _ = W.config1()
    cov, _ = W.givens_cov()
    ref = np.array([0.1, -0.3, 0.4, 0.2])
    k, D = smp["n_delete"], 4
    second, cls, esss = [], [], []
    for seed in range(101, 125):
        h = nsgw.Handle(spec, smp, seed=seed)
        buf = torch.empty((500 * k, D + 3), dtype=torch.float64, device="cuda")
        nit, st = h.run(smp["term_kind"], smp["term_tol"], 500, dead=buf)
        out = h.posterior(buf[: nit * k].contiguous(), theta_ref=ref)
        pw = torch.exp(out["logp"])
        second.append(((out["theta"] * pw[:, None]).T @ out["theta"]).cpu().numpy())
        cls.append(out["cl"])
        esss.append(out["ess"])
    sig = np.sqrt(np.diag(cov))
    assert np.allclose(np.mean(second, axis=0), cov, atol=0.06 * float(np.max(sig)) ** 2, rtol=0.08)
    cdf = np.array([0.5 * (1 + math.erf(r / s / math.sqrt(2))) for r, s in zip(ref, sig)])
    assert np.all(np.abs(np.mean(cls, axis=0) - cdf) < 4.5 * 0.5 / np.sqrt(np.mean(esss) * len(cls)))


# ---- PP harness (pp.credible_levels: ns_run_many + ns_posterior) -----------------------------------------
def test_pp_levels_uniform_gaussian_toy(nsgw):
    from scipy import stats
    from paper_2509_04336_b200 import pp
    from test_oracle_posterior import _toy_pp_specs
    specs, th, smp = _toy_pp_specs(120, 43)
    res = pp.credible_levels(specs, th, smp, smp["term_kind"], smp["term_tol"], 500, seed0=2000, group=8)
    cl = res["cl"]
    assert np.all((cl >= 0) & (cl <= 1)) and np.all(res["iters"] > 30)
    pv = [stats.kstest(cl[:, d], "uniform").pvalue for d in range(4)]
    assert min(pv) > 0.01 / 4, pv
    assert np.all(np.abs(cl.var(axis=0) - 1 / 12) < 0.035)
    # the harness's own KS routine agrees with scipy's
    for d in range(4):
        D_, p_ = pp.ks_uniform(cl[:, d])
        r = stats.kstest(cl[:, d], "uniform")
        assert abs(D_ - r.statistic) < 1e-12 and abs(p_ - r.pvalue) < 0.03
    # one injection checked against the oracle's posterior of the same dead / live points is covered by test_posterior_parity_*


def test_pp_levels_uniform_gw_four_parameters(nsgw):
    """48 injections from the prior (Mc, q, dL in [400, 1600] Mpc, tc free; PhenomD-form, H1+L1, 433 bins; PSD scaled so that the
    config-3 injection at 800 Mpc has SNR 10), each in its own noise: credible levels of the injected values uniform."""
    from scipy import stats
    from paper_2509_04336_b200 import pp
    free = (0, 1, 4, 8)
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 128.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 10.0, wf)
    spec = W.fix_dims(spec, free, W.INJ_C3)
    spec["prior_lo"][4], spec["prior_hi"][4] = 400.0, 1600.0
    specs, th = W.pp_problem_set(spec, 48, 77, wf, lambda s, u: O.OracleProblem(s).prior_transform(u))
    smp = dict(n_live=400, n_delete=200, naccept=20, maxmcmc=2000, walks0=50.0, delay=-1.0)
    res = pp.credible_levels(specs, th, smp, 0, 0.1, 120, seed0=300, group=8)
    cl = res["cl"][:, free]
    assert np.all(res["cl"][:, [d for d in range(11) if d not in free]] == 0.0)      # FIXED parameters sit at the injected value
    pv = [stats.kstest(cl[:, j], "uniform").pvalue for j in range(len(free))]
    assert min(pv) > 0.01 / len(free), (pv, cl.mean(axis=0))
    assert np.all(res["ess"] > 100)


def test_ns_step_parity_gw_single_deletion(nsgw):
    # k = 1 (the sequential limit): one walker per iteration, adaptation after every replacement
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 200.0, (20.0, 40.0))
    spec = W.make_data(spec, W.INJ_C3, 10.0, wf)
    smp = dict(n_live=40, n_delete=1, naccept=6, maxmcmc=60, walks0=12.0, delay=-1.0)
    _step_parity(nsgw, spec, smp, 12, 3, 1e-8)


def test_posterior_resample_parity(nsgw):
    # systematic resampling of a run's weighted rows (R:L27): same rows as the oracle except where a comb position falls within
    # rounding of a cumulative weight (the two sides sum p in different orders), and there by one row at most
    spec, smp, _ = W.config1()
    h = nsgw.Handle(spec, smp, seed=9)
    k, D = smp["n_delete"], 4
    buf = torch.empty((500 * k, D + 3), dtype=torch.float64, device="cuda")
    nit, st = h.run(smp["term_kind"], smp["term_tol"], 500, dead=buf)
    out = h.posterior(buf[: nit * k].contiguous())
    logp = out["logp"].cpu().numpy()
    cum = np.cumsum(np.exp(logp))
    for n_out, seed in ((4000, 1), (333, 2 ** 33 + 7), (1, 3), (20000, 4)):
        idx_g, th_g = h.posterior_resample(out["logp"], n_out, seed, theta=out["theta"])
        idx_o, U = O.posterior_resample(logp, n_out, seed)
        ig = idx_g.cpu().numpy()
        bad = np.nonzero(ig != idx_o)[0]
        t = (bad + U) / n_out * cum[-1]
        assert np.all(np.abs(ig[bad] - idx_o[bad]) <= 1)
        assert np.all(np.minimum(np.abs(cum[ig[bad]] - t), np.abs(cum[idx_o[bad]] - t)) < 1e-12 * cum[-1])
        assert bad.size <= max(1, n_out // 1000)
        assert torch.equal(th_g, out["theta"][idx_g])
        cnt = np.bincount(ig, minlength=logp.size)
        p = np.exp(logp)
        assert np.all(cnt >= np.floor(n_out * p - 1e-6)) and np.all(cnt <= np.ceil(n_out * p + 1e-6))
        again, _ = h.posterior_resample(out["logp"], n_out, seed, theta=out["theta"])
        assert torch.equal(again, idx_g)
    # equal-weight sample reproduces the weighted second moments (n_out >> ESS: resampling noise 1/n_out per weight)
    cov, _ = W.givens_cov()
    pw = torch.exp(out["logp"])
    m2w = ((out["theta"] * pw[:, None]).T @ out["theta"]).cpu().numpy()
    m2s = (th_g.T @ th_g / th_g.shape[0]).cpu().numpy()
    assert np.allclose(m2s, m2w, atol=8e-3)
    # argument errors
    import ctypes as C
    L, null = nsgw.lib(), C.c_void_p(0)
    lp, cm = C.c_void_p(out["logp"].data_ptr()), C.c_void_p(torch.empty(logp.size, dtype=torch.float64, device="cuda").data_ptr())
    assert L.ns_posterior_resample(h._h, lp, null, C.c_int64(logp.size), C.c_int64(10), C.c_uint64(1), cm, null, null, null) == -1   # no output
    assert L.ns_posterior_resample(h._h, lp, null, C.c_int64(0), C.c_int64(10), C.c_uint64(1), cm, cm, null, null) == -1             # no rows
    assert L.ns_posterior_resample(h._h, lp, null, C.c_int64(logp.size), C.c_int64(10), C.c_uint64(1), cm, null, cm, null) == -1     # gather needs theta
