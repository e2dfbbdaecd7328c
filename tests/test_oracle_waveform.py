"""Pins for the oracle's waveform + likelihood (DESIGN.md section 3 / appendix A): closed forms, textbook chirp rate,
invariants and special cases -- none of them re-calls the oracle's own formula except the labelled mpmath precision twin."""
import math

import mpmath as mp
import numpy as np
import pytest

from oracle import oracle as O
from paper_2509_04336_b200 import workloads as W

# CODATA / IAU values typed independently of oracle.cpp
G_SI, C_SI, MSUN_KG, PC_M = 6.67430e-11, 299792458.0, 1.988409870698051e30, 3.0856775814913673e16
GM_S = G_SI * MSUN_KG / C_SI ** 3


def wf(spec, th):
    return O.OracleProblem(spec).waveform(th)


def small_spec(kind=W.LIKE_TAYLORF2, dets=("H1", "L1"), T=4.0, fmax=128.0, mc=(20.0, 40.0)):
    return W.gw_spec(kind, list(dets), T, fmax, mc)


# --------------------------------------------------------------------------------------------------------
# TaylorF2
# --------------------------------------------------------------------------------------------------------
def fdot_series(f, m1, m2, chi1, chi2):
    """Textbook chirp rate df/dt through 1.5PN (+ non-spinning 2PN): quadrupole formula, 1PN term
    (743/336 + 11 eta/4), tail 4 pi, spin-orbit beta (Cutler & Flanagan 1994; Blanchet et al. 1995)."""
    M = (m1 + m2) * GM_S
    eta = m1 * m2 / (m1 + m2) ** 2
    Mc = M * eta ** 0.6
    v = (math.pi * M * f) ** (1 / 3)
    beta = sum((113 / 12 * (m / (m1 + m2)) ** 2 + 25 / 4 * eta) * c for m, c in ((m1, chi1), (m2, chi2)))
    a2 = 743 / 336 + 11 * eta / 4
    a4 = 34103 / 18144 + 13661 * eta / 2016 + 59 * eta ** 2 / 18
    return 96 / 5 * math.pi ** (8 / 3) * Mc ** (5 / 3) * f ** (11 / 3) * (1 - a2 * v ** 2 + (4 * math.pi - beta) * v ** 3 + a4 * v ** 4)


@pytest.mark.parametrize("chi1,chi2,tol", [(0.0, 0.0, 1.5e-4), (0.6, -0.3, 4e-4), (-0.5, 0.5, 4e-4)])
def test_taylorf2_stationary_phase_matches_textbook_chirp(chi1, chi2, tol):
    # stationary phase: Psi''(f) = 2 pi / (df/dt).  Light system so that v << 1 at 20-40 Hz.
    m1, m2 = 0.6, 0.45
    q = m2 / m1
    Mc = (m1 * m2) ** 0.6 / (m1 + m2) ** 0.2
    P = O.OracleProblem(small_spec())
    th = [Mc, q, chi1, chi2, 100.0, 0.3, 0.2, 0.7, 0.0, 1.0, 0.1]
    for f0 in (20.0, 30.0, 40.0):
        h = 0.02
        _, psi = P.amp_phase(th, [f0 - h, f0, f0 + h])
        d2 = (psi[0] - 2 * psi[1] + psi[2]) / h ** 2
        assert abs(d2 * fdot_series(f0, m1, m2, chi1, chi2) / (2 * math.pi) - 1) < tol


def test_taylorf2_newtonian_chirp_time():
    # (1/2pi) dPsi0/df -> -tau(f) = -(5/256) Mc^-5/3 (pi f)^-8/3 (time to coalescence), leading order
    P = O.OracleProblem(small_spec())
    Mc = 0.3
    th = [Mc, 1.0, 0, 0, 100.0, 0, 0, 0, 0, 0, 0]
    f0, h = 20.0, 0.01
    _, psi = P.amp_phase(th, [f0 - h, f0 + h])
    tau = 5 / 256 * (Mc * GM_S) ** (-5 / 3) * (math.pi * f0) ** (-8 / 3)
    got = (psi[1] - psi[0]) / (2 * h) / (2 * math.pi)
    assert abs(got / (-tau) - 1) < 0.02          # 1PN correction is ~1 % here
    assert got < 0


def test_taylorf2_phase_constant_terms():
    # Psi0 holds -2*phase - pi/4 and no tc (R:L3): shifting phase by a moves Psi0 by -2a; tc does not enter.
    P = O.OracleProblem(small_spec())
    th = np.array(W.INJ_C3)
    f = np.linspace(20, 128, 7)
    _, p0 = P.amp_phase(th, f)
    th2 = th.copy(); th2[7] += 0.4; th2[8] = 0.05
    _, p1 = P.amp_phase(th2, f)
    np.testing.assert_allclose(p1 - p0, -0.8, atol=1e-10)


def test_taylorf2_phase_fp64_vs_mpmath_precision_twin():
    # PRECISION twin only (same printed formula, 40 digits): bounds the fp64 evaluation error, not the formula.
    mp.mp.dps = 40
    P = O.OracleProblem(small_spec())
    th = W.INJ_C3
    Mc, q, c1, c2 = [mp.mpf(x) for x in th[:4]]
    eta = q / (1 + q) ** 2
    M = Mc * mp.mpf("4.925490947641267e-6") * eta ** (mp.mpf(-3) / 5)
    d = (1 - q) / (1 + q)
    xs, xa = (c1 + c2) / 2, (c1 - c2) / 2
    pi = mp.pi
    ph = [mp.mpf(1), mp.mpf(0), mp.mpf(3715) / 756 + 55 * eta / 9,
          -16 * pi + mp.mpf(113) / 3 * d * xa + (mp.mpf(113) / 3 - 76 * eta / 3) * xs,
          mp.mpf(15293365) / 508032 + 27145 * eta / 504 + 3085 * eta ** 2 / 72 + (mp.mpf(-405) / 8 + 200 * eta) * xa ** 2
          - mp.mpf(405) / 4 * d * xa * xs + (mp.mpf(-405) / 8 + 5 * eta / 2) * xs ** 2]
    c5 = 38645 * pi / 756 - 65 * pi * eta / 9 + d * (mp.mpf(-732985) / 2268 - 140 * eta / 9) * xa + \
        (mp.mpf(-732985) / 2268 + 24260 * eta / 81 + 340 * eta ** 2 / 9) * xs
    p6 = mp.mpf(11583231236531) / 4694215680 - 6848 * mp.euler / 21 - 640 * pi ** 2 / 3 + \
        (mp.mpf(-15737765635) / 3048192 + 2255 * pi ** 2 / 12) * eta + 76055 * eta ** 2 / 1728 - 127825 * eta ** 3 / 1296 - \
        mp.mpf(6848) / 63 * mp.log(64) + 2270 * pi / 3 * d * xa + (2270 * pi / 3 - 520 * pi * eta) * xs
    p7 = 77096675 * pi / 254016 + 378515 * pi * eta / 1512 - 74045 * pi * eta ** 2 / 756 + \
        d * (mp.mpf(-25150083775) / 3048192 + 26804935 * eta / 6048 - 1985 * eta ** 2 / 48) * xa + \
        (mp.mpf(-25150083775) / 3048192 + 10566655595 * eta / 762048 - 1042165 * eta ** 2 / 3024 + 5345 * eta ** 3 / 36) * xs
    for f in (20.0, 77.25, 511.5, 1024.0):
        v = (pi * M * mp.mpf(f)) ** (mp.mpf(1) / 3)
        lv = mp.log(v)
        s = sum(ph[k] * v ** k for k in range(5)) + (c5 + 3 * c5 * lv) * v ** 5 + (p6 - mp.mpf(6848) / 21 * lv) * v ** 6 + p7 * v ** 7
        ref = -pi / 4 + 3 / (128 * eta) * v ** -5 * s - 2 * mp.mpf(th[7])
        _, got = P.amp_phase(th, [f])
        assert abs(got[0] - float(ref)) < 2e-12 * max(1.0, abs(float(ref)))


def test_amplitude_normalisation_textbook():
    # |h+| face-on = sqrt(5/24) pi^-2/3 (G Mc/c^3)^(5/6) (c/dL) f^-7/6 with independently typed SI constants
    P = O.OracleProblem(small_spec())
    th = [30.0, 0.5, 0, 0, 410.0, 0, 0, 0, 0, 0, 0]
    f = np.array([20.0, 100.0])
    amp, _ = P.amp_phase(th, f)
    ref = math.sqrt(5 / 24) * math.pi ** (-2 / 3) * (30.0 * GM_S) ** (5 / 6) / (410.0 * 1e6 * PC_M / C_SI) * f ** (-7 / 6)
    np.testing.assert_allclose(amp, ref, rtol=2e-6)     # limited by the 5-6 digit CODATA G*Msun used here


def _cdet2(P, det, th):
    fp, fx, _ = P.detector_response(det, th[9], th[10], th[6])
    ci = math.cos(th[5])
    return (fp * (1 + ci * ci) / 2) ** 2 + (fx * ci) ** 2


def test_hh_closed_form_power_law():
    # BJ: analytic <h,h> for a pure power-law inspiral amplitude: <h,h>_det = |C_det|^2 A0^2 * 4 df sum_k f_k^-7/3 / S_k
    spec = W.config2(wf, with_noise=True)
    P = O.OracleProblem(spec)
    f = spec["f_min"] + spec["df"] * np.arange(spec["n_freq"])
    rng = np.random.default_rng(5)
    for _ in range(3):
        th = P.prior_transform(rng.uniform(0.05, 0.95, 11))[0]
        _, parts = P.gw_loglike(th[None, :], parts=True)
        A0 = math.sqrt(5 / 24) * math.pi ** (-2 / 3) * (th[0] * 4.925490947641267e-6) ** (5 / 6) / (th[4] * 3.0856775814913673e22 / C_SI)
        for det in range(2):
            I73 = 4 * spec["df"] * math.fsum(f ** (-7 / 3) / spec["psd"][det])
            assert abs(parts[0, 2 * det + 1] / (_cdet2(P, det, th) * A0 ** 2 * I73) - 1) < 1e-12


def test_hh_flat_psd_integral():
    # flat PSD: df * sum_k f_k^-7/3 = (3/4)(f_lo^-4/3 - f_hi^-4/3) + (df/2)(f_lo^-7/3 + f_hi^-7/3) + O(df^2)  (Euler-Maclaurin);
    # pins the inclusive bin range and the 4 df normalisation
    spec = small_spec(T=16.0, fmax=512.0)
    n = spec["n_freq"]
    spec["psd"] = np.full((2, n), 3e-47)
    spec["strain"] = np.zeros((2, n, 2))
    P = O.OracleProblem(spec)
    th = np.array(W.INJ_C3)
    _, parts = P.gw_loglike(th[None, :], parts=True)
    A0 = math.sqrt(5 / 24) * math.pi ** (-2 / 3) * (th[0] * 4.925490947641267e-6) ** (5 / 6) / (th[4] * 3.0856775814913673e22 / C_SI)
    flo, fhi, df = 20.0, 512.0, 1 / 16.0
    integral = 0.75 * (flo ** (-4 / 3) - fhi ** (-4 / 3)) + df / 2 * (flo ** (-7 / 3) + fhi ** (-7 / 3)) \
        + df ** 2 / 12 * (7 / 3) * (flo ** (-10 / 3) - fhi ** (-10 / 3))
    for det in range(2):
        ref = _cdet2(P, det, th) * A0 ** 2 * 4 * integral / 3e-47
        assert abs(parts[0, 2 * det + 1] / ref - 1) < 1e-9
    assert parts[0, 0] == 0.0 and parts[0, 2] == 0.0      # zero data -> <d,h> = 0


@pytest.mark.parametrize("kind", [W.LIKE_TAYLORF2, W.LIKE_PHENOMD])
def test_noise_free_maximum_and_symmetries(kind):
    spec = small_spec(kind, fmax=256.0)
    spec = W.make_data(spec, W.INJ_C3, 20.0, wf, with_noise=False)
    P = O.OracleProblem(spec)
    th0 = np.array(W.INJ_C3)
    l0, parts = P.gw_loglike(th0[None, :], parts=True)
    # d = h(theta0): logL(theta0) = <h,h>/2 = SNR^2/2, and <d,h> = <h,h> per detector
    assert abs(l0[0] - 200.0) < 1e-9
    np.testing.assert_allclose(parts[0, 0::2], parts[0, 1::2], rtol=1e-13)
    # global maximum: any perturbation lowers logL (Cauchy-Schwarz)
    rng = np.random.default_rng(2)
    for _ in range(30):
        th = th0 + rng.normal(0, 1, 11) * np.array([0.05, 0.02, 0.05, 0.05, 20, 0.05, 0.05, 0.05, 1e-4, 0.02, 0.02])
        th[1] = min(th[1], 1.0)
        assert P.gw_loglike(th[None, :])[0] < l0[0]
    # exact symmetries of h: (psi, phase) -> (psi + pi/2, phase + pi/2); phase -> phase + pi
    a = th0.copy(); a[6] += math.pi / 2; a[7] += math.pi / 2
    b = th0.copy(); b[7] += math.pi
    la, lb = P.gw_loglike(np.stack([a, b]))
    assert abs(la - l0[0]) < 1e-9 and abs(lb - l0[0]) < 1e-9
    # phase -> phase + pi/2 flips the sign of h: <d,h> -> -<d,h>
    c = th0.copy(); c[7] += math.pi / 2
    _, pc = P.gw_loglike(c[None, :], parts=True)
    np.testing.assert_allclose(pc[0, 0::2], -parts[0, 0::2], rtol=1e-10)
    # distance scaling: <d,h> ~ 1/dL, <h,h> ~ 1/dL^2
    d = th0.copy(); d[4] *= 2
    _, pd = P.gw_loglike(d[None, :], parts=True)
    np.testing.assert_allclose(pd[0, 0::2], parts[0, 0::2] / 2, rtol=1e-13)
    np.testing.assert_allclose(pd[0, 1::2], parts[0, 1::2] / 4, rtol=1e-13)


def test_time_shift_covariance():
    # d_k -> d_k e^{-2 pi i f_k tau} and tc -> tc + tau leaves <d,h> unchanged
    spec = W.config2(wf)
    f = spec["f_min"] + spec["df"] * np.arange(spec["n_freq"])
    P = O.OracleProblem(spec)
    th = P.prior_transform(np.full(11, 0.37))[0]
    _, p0 = P.gw_loglike(th[None, :], parts=True)
    tau = 0.0123
    d = spec["strain"][..., 0] + 1j * spec["strain"][..., 1]
    d2 = d * np.exp(-2j * np.pi * f * tau)[None, :]
    P.set_data(np.stack([d2.real, d2.imag], -1), spec["psd"])
    th2 = th.copy(); th2[8] += tau
    _, p1 = P.gw_loglike(th2[None, :], parts=True)
    np.testing.assert_allclose(p1, p0, rtol=0, atol=2e-9)


def test_noise_normalisation():
    # E[4 df |n_k|^2 / S_k] = 2 per bin
    spec = W.config2(wf)
    n = W.noise(spec, spec["psd"])
    x = 4 * spec["df"] * (n[..., 0] ** 2 + n[..., 1] ** 2) / spec["psd"]
    assert abs(x.mean() / 2 - 1) < 3 / math.sqrt(x.size)


def test_unphysical_theta_is_minus_inf():
    spec = W.config2(wf)
    P = O.OracleProblem(spec)
    base = np.array(W.INJ_C3)
    bad = []
    for i, v in [(1, 1.2), (1, 0.0), (2, 1.01), (3, -1.5), (4, 0.0), (0, -3.0), (8, float("nan"))]:
        t = base.copy(); t[i] = v; bad.append(t)
    assert np.all(np.isneginf(P.gw_loglike(np.stack(bad))))


# --------------------------------------------------------------------------------------------------------
# PhenomD-form (structure only; fidelity to the published fit is unpinned -- see oracle.cpp header)
# --------------------------------------------------------------------------------------------------------
def _pd(table=None):
    spec = small_spec(W.LIKE_PHENOMD)
    if table is not None:
        spec["phenom_table"] = table
    return O.OracleProblem(spec)


THETAS = [W.INJ_C3, W.INJ_C4, [35.0, 0.2, 0.9, -0.9, 300.0, 1.0, 0.1, 0.2, 0.01, 3.0, 0.5], [9.0, 1.0, -0.8, 0.7, 900.0, 2.0, 1.1, 4.2, -0.03, 5.0, -0.5]]


def test_phenomd_qnm_hand_values():
    info = _pd().phenomd_info([30.0, 1.0, 0.0, 0.0, 500.0, 0, 0, 0, 0, 0, 0])
    assert abs(info["eta"] - 0.25) < 1e-15
    assert abs(info["Frd"] - 0.08854) < 5e-5      # hand-evaluated from the Berti-type fit at a_f = 0.6868
    assert abs(info["Fdamp"] - 0.013697) < 1e-5
    assert abs(info["M"] - 30.0 * 0.25 ** -0.6 * 4.925490947641267e-6) < 1e-18


@pytest.mark.parametrize("th", THETAS)
def test_phenomd_phase_and_amplitude_are_C1(th):
    P = _pd()
    info = P.phenomd_info(th)
    M = info["M"]
    for Fj, what in [(0.018, "phase"), (0.5 * info["Frd"], "phase"), (0.014, "amp"), (info["Fpeak"], "amp")]:
        fj = Fj / M
        e = fj * 1e-9
        h = fj * 1e-5
        a, p = P.amp_phase(th, [fj - e - h, fj - e, fj + e, fj + e + h])
        y = p if what == "phase" else a
        scale = max(abs(y[1]), 1e-300)
        assert abs(y[2] - y[1]) < 1e-7 * scale + 1e-9 * (what == "phase"), (Fj, what)      # C0
        dl, dr = (y[1] - y[0]) / h, (y[3] - y[2]) / h
        assert abs(dl - dr) < 2e-4 * max(abs(dl), abs(dr), scale / fj), (Fj, what)            # C1 (one-sided differences)


@pytest.mark.parametrize("th", THETAS)
def test_phenomd_alignment_and_midpoint(th):
    P = _pd()
    info = P.phenomd_info(th)
    M = info["M"]
    fpk = info["Fpeak"] / M
    h = fpk * 1e-6
    _, p = P.amp_phase(th, [fpk - h, fpk + h])
    slope = (p[1] - p[0]) / (2 * h)                        # dPsi0/df at the amplitude peak is zero (time alignment)
    assert abs(slope) < 1e-6 * info["t0"] * M
    # MR amplitude ansatz peaks at Fpeak: numerical argmax over a fine grid
    F = np.linspace(info["Fpeak"], info["Fpeak"] * 1.3, 4001)
    a, _ = P.amp_phase(th, F / M)
    ahat = a * (F / M) ** (7 / 6)
    assert np.argmax(ahat) == 0 or abs(F[np.argmax(ahat)] - info["Fpeak"]) < 2 * (F[1] - F[0])
    # Hermite + bubble quartic takes the tabulated value v2 at the midpoint of [0.014, Fpeak]
    Fm = 0.5 * (0.014 + info["Fpeak"])
    a, _ = P.amp_phase(th, [Fm / M])
    A0 = math.sqrt(5 / 24) * math.pi ** (-2 / 3) * (th[0] * 4.925490947641267e-6) ** (5 / 6) / (th[4] * 3.0856775814913673e22 / C_SI)
    assert abs(a[0] / (A0 * (Fm / M) ** (-7 / 6)) / info["Lambda"][3] - 1) < 1e-10


def test_phenomd_peak_formula_gamma2_below_one_and_lorentzian():
    tab = W.surrogate_table()
    tab[5, :] = 0; tab[5, 0] = 0.6                  # gamma2 < 1 branch
    P = _pd(tab)
    th = W.INJ_C3
    info = P.phenomd_info(th)
    M = info["M"]
    F = np.linspace(info["Fpeak"] * 0.98, info["Fpeak"] * 1.02, 4001)
    # evaluate the MR ansatz on both sides of Fpeak via a table whose intermediate region is pushed away: compare shape only above Fpeak
    a, _ = P.amp_phase(th, F[F >= info["Fpeak"]] / M)
    ahat = a * (F[F >= info["Fpeak"]] / M) ** (7 / 6)
    assert np.argmax(ahat) <= 2
    # gamma2 = 0: pure Lorentzian, value gamma1/w at F_RD and half of it at F_RD + w, w = gamma3 * Fdamp
    tab[5, 0] = 1e-9   # (gamma2 = 0 exactly is the 0/0 limit of the Fpeak formula)
    P = _pd(tab)
    info = P.phenomd_info(th)
    g1, g3 = info["Lambda"][4], info["Lambda"][6]
    w = g3 * info["Fdamp"]
    assert abs(info["Fpeak"] - info["Frd"]) < 1e-12
    A0 = math.sqrt(5 / 24) * math.pi ** (-2 / 3) * (th[0] * 4.925490947641267e-6) ** (5 / 6) / (th[4] * 3.0856775814913673e22 / C_SI)
    Fs = np.array([info["Frd"] + w, info["Frd"] + 2 * w])
    a, _ = P.amp_phase(th, Fs / M)
    ahat = a / (A0 * (Fs / M) ** (-7 / 6))
    np.testing.assert_allclose(ahat, [g1 / w / 2, g1 / w / 5], rtol=1e-8)


def test_phenomd_reduces_to_taylorf2_in_inspiral():
    tab = W.surrogate_table()
    tab[7:11, :] = 0.0                               # sigma_i = 0
    spec = small_spec(W.LIKE_PHENOMD)
    spec["phenom_table"] = tab
    Pd = O.OracleProblem(spec)
    Pt = O.OracleProblem(small_spec(W.LIKE_TAYLORF2))
    th = W.INJ_C3
    info = Pd.phenomd_info(th)
    f = np.linspace(20.0, 0.0179 / info["M"], 9)
    _, pd_ = Pd.amp_phase(th, f)
    _, pt = Pt.amp_phase(th, f)
    np.testing.assert_allclose(pd_ - pt, -info["t0"] * info["M"] * f, rtol=1e-9, atol=1e-8)
    # and the inspiral amplitude tends to the restricted Newtonian one as F -> 0 (A_0 = 1 leading term)
    th_light = [1.0, 1.0, 0, 0, 100.0, 0, 0, 0, 0, 0, 0]
    a_pd, _ = Pd.amp_phase(th_light, [20.0])
    a_t, _ = Pt.amp_phase(th_light, [20.0])
    v2 = (math.pi * 2 ** 1.2 * 4.925490947641267e-6 * 20.0) ** (2 / 3)      # M = Mc * eta^-3/5 = 2^1.2 Msun
    assert abs(a_pd[0] / a_t[0] - 1 - (-323 / 224 + 451 * 0.25 / 168) * v2) < 5e-4   # textbook 1PN amplitude term


def test_phenomd_spin_columns_of_table():
    # Lambda = l00 + l10 eta + xi (l01 + l11 eta + l21 eta^2) + xi^2 (...) + xi^3 (...), xi = chi_PN - 1
    tab = np.zeros((19, 11))
    tab[0, :] = [1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11]
    P = _pd(tab)
    th = [30.0, 0.5, 0.4, -0.1, 500.0, 0, 0, 0, 0, 0, 0]
    q = 0.5
    eta = q / (1 + q) ** 2
    m1, m2 = 1 / (1 + q), q / (1 + q)
    xi = (m1 * 0.4 + m2 * -0.1) - 38 * eta / 113 * (0.4 - 0.1) - 1
    ref = 1 + 2 * eta + xi * (3 + 4 * eta + 5 * eta ** 2) + xi ** 2 * (6 + 7 * eta + 8 * eta ** 2) + xi ** 3 * (9 + 10 * eta + 11 * eta ** 2)
    got = P.phenomd_info(th)["Lambda"][0]
    assert abs(got - ref) < 1e-12 * abs(ref)
