"""Pins the oracle's TaylorF2 phase coefficients (oracle.cpp: taylorf2_coeffs; DESIGN.md A.1; the model BASELINE.json config 2 names,
and the inspiral part of the PhenomD-form model P:174 names) by DERIVING them instead of retyping them.

The stationary-phase phase of a quasi-circular inspiral follows from the orbital energy E(v) and the gravitational-wave flux F(v)
alone: dt/dv = -E'(v)/F(v), d(phi_orb)/dv = -v^3 E'(v)/F(v) (G = c = M = 1, v = (pi M f)^(1/3)), and
Psi(f) = 2 pi f t(f) - 2 phi_orb(f) - pi/4 up to a constant and a term linear in f (absorbed by phase and tc).  Below, E and F are typed
from the post-Newtonian literature in THEIR OWN form (series in v with the spin variables S_l, Sigma_l; Blanchet's Living Review
for the non-spinning terms, Kidder 1995 / Poisson 1998 for spin-spin at 2PN, Bohe-Marsat-Blanchet 2013 for spin-orbit up to 3.5PN),
the ratio is expanded with sympy in exact arithmetic, integrated term by term, and the resulting coefficients of
(3 / 128 eta) v^-5 sum_k (psi_k + psi_k^(l) ln v) v^k are compared with the oracle's numbers.  None of the phase coefficients of the
formula sheet is typed here.  The typed E and F are themselves pinned in their test-mass limit by closed forms that do not come
from a PN expansion: the energy of circular equatorial Kerr geodesics (exact) and the black-hole-perturbation flux of
Tagoshi-Shibata-Tanaka-Sasaki 1996 (spin terms 11/4, 33/16, 59/16, 65 pi/6, 162035/3888).

Spin orders compared (the sheet is the PhenomD inspiral, linear in spin beyond 2PN): spin-independent terms at every order;
terms linear in the spins at 1.5, 2.5 (with its logarithm), 3 and 3.5PN; quadratic terms at 2PN.
"""
import ctypes as C
import math

import numpy as np
import pytest
import sympy as sp
from sympy import Rational as R, pi, EulerGamma, log

from oracle import oracle as O

v, Lv, d, c1, c2 = sp.symbols("v Lv delta chi1 chi2")        # Lv stands for ln v
ETA = (1 - d ** 2) / 4                                          # eta = m1 m2 / M^2 with m1,2 = (1 +- delta)/2
M1, M2 = (1 + d) / 2, (1 - d) / 2
S_L = M1 ** 2 * c1 + M2 ** 2 * c2                               # (S1 + S2) . l / M^2
SIG_L = M2 * c2 - M1 * c1                                       # M (S2/m2 - S1/m1) . l / M^2


def energy_coeffs():
    """E(v) = -(eta v^2 / 2) sum_k e_k v^k.  Spin-spin at 2PN from the leading-order Hamiltonian of two aligned spinning black holes,
    H_SS = [-S1 S2 - (m2/2m1) S1^2 - (m1/2m2) S2^2] / r^3 (spin-spin attraction of parallel spins side by side; the oblate
    spin-induced quadrupole, kappa = 1), which for circular orbits at fixed frequency gives e4_SS = 2 H_SS r^3 / (mu M^3)."""
    eta = ETA
    e = [0] * 8
    e[0] = 1
    e[2] = -R(3, 4) - eta / 12
    e[3] = R(14, 3) * S_L + 2 * d * SIG_L
    e[4] = -R(27, 8) + R(19, 8) * eta - eta ** 2 / 24 + (-2 * eta * c1 * c2 - M1 ** 2 * c1 ** 2 - M2 ** 2 * c2 ** 2)
    e[5] = (11 - R(61, 9) * eta) * S_L + d * (3 - R(10, 3) * eta) * SIG_L
    e[6] = -R(675, 64) + (R(34445, 576) - R(205, 96) * pi ** 2) * eta - R(155, 96) * eta ** 2 - R(35, 5184) * eta ** 3
    e[7] = (R(135, 4) - R(367, 4) * eta + R(29, 12) * eta ** 2) * S_L + d * (R(27, 4) - 39 * eta + R(5, 4) * eta ** 2) * SIG_L
    return e


def flux_coeffs():
    """F(v) = (32/5) eta^2 v^10 sum_k f_k v^k (f_6 holds ln v).  Spin-spin at 2PN: Kidder's (eta/48)(289 (l.chi1)(l.chi2) - 103 chi1.chi2)
    plus quadrupole-monopole and self-spin terms (2 + 1/16) (m_i/M)^2 chi_i^2."""
    eta = ETA
    f = [0] * 8
    f[0] = 1
    f[2] = -R(1247, 336) - R(35, 12) * eta
    f[3] = 4 * pi - 4 * S_L - R(5, 4) * d * SIG_L
    f[4] = (-R(44711, 9072) + R(9271, 504) * eta + R(65, 18) * eta ** 2
            + R(289 - 103, 48) * eta * c1 * c2 + R(33, 16) * (M1 ** 2 * c1 ** 2 + M2 ** 2 * c2 ** 2))
    f[5] = (-R(8191, 672) - R(583, 24) * eta) * pi + (-R(9, 2) + R(272, 9) * eta) * S_L + (-R(13, 16) + R(43, 4) * eta) * d * SIG_L
    f[6] = (R(6643739519, 69854400) + R(16, 3) * pi ** 2 - R(1712, 105) * EulerGamma - R(856, 105) * (4 * log(2) + 2 * Lv)
            + (-R(134543, 7776) + R(41, 48) * pi ** 2) * eta - R(94403, 3024) * eta ** 2 - R(775, 324) * eta ** 3
            - 16 * pi * S_L - R(31, 6) * pi * d * SIG_L)
    f[7] = ((-R(16285, 504) + R(214745, 1728) * eta + R(193385, 3024) * eta ** 2) * pi
            + (R(476645, 6804) + R(6172, 189) * eta - R(2810, 27) * eta ** 2) * S_L
            + (R(9535, 336) + R(1849, 126) * eta - R(1501, 36) * eta ** 2) * d * SIG_L)
    return f


def spin_truncate(expr, max_deg):
    """Keeps the terms of total degree <= max_deg in (chi1, chi2)."""
    poly = sp.Poly(sp.expand(expr), c1, c2)
    return sp.Integer(0) + sum(co * c1 ** i * c2 ** j for (i, j), co in poly.terms() if i + j <= max_deg)


@pytest.fixture(scope="module")
def derived():
    """psi_k, psi_k^(l) for k = 0..7 as sympy expressions in (delta, chi1, chi2), from E and F only."""
    e, f = energy_coeffs(), flux_coeffs()
    # -E'(v) = eta v sum_k ((k + 2)/2) e_k v^k;  Q = that series divided by the flux series, to v^7
    N = [R(k + 2, 2) * e[k] for k in range(8)]
    Q = [0] * 8
    for k in range(8):
        Q[k] = sp.expand(N[k] - sum(Q[j] * f[k - j] for j in range(k)))
    # dt/dv = (5 / 32 eta) v^-9 Q(v), dphi/dv = v^3 dt/dv.  Psi = 2 v^3 T(v) - 2 Phi(v) with T, Phi the term-by-term
    # antiderivatives; normalised by (3 / 128 eta) v^-5 this is (20/3) (2 T_k - 2 Phi_k) per power k.
    psi, psil = [0] * 8, [0] * 8
    for k in range(8):
        a, b = Q[k].coeff(Lv, 0), Q[k].coeff(Lv, 1)

        def integ(n):                      # int (a + b ln v) v^n dv = v^(n+1) (c0 + c1 ln v), constants of integration dropped
            if n == -1:
                assert b == 0
                return 0, a                # a ln v
            return a / (n + 1) - b / (n + 1) ** 2, b / (n + 1)

        T0, T1 = integ(k - 9)
        P0, P1 = integ(k - 6)
        psi[k] = sp.expand(R(20, 3) * (2 * T0 - 2 * P0))
        psil[k] = sp.expand(R(20, 3) * (2 * T1 - 2 * P1))
    return psi, psil


def oracle_coeffs(q, x1, x2):
    lib = O._lib
    phi, phil = (C.c_double * 8)(), (C.c_double * 8)()
    lib.orc_taylorf2_coeffs(C.c_double(q), C.c_double(x1), C.c_double(x2), phi, phil)
    return np.array(phi), np.array(phil)


POINTS = [(1.0, 0.0, 0.0), (0.8, 0.3, -0.2), (0.125, -0.99, 0.99), (0.5, 0.7, 0.65), (0.31, -0.45, 0.1), (0.97, 0.9, -0.9)]
# highest spin degree the formula sheet keeps at each order (DESIGN.md A.1: quadratic at 2PN, linear beyond)
SPIN_DEG = {0: 0, 1: 0, 2: 0, 3: 1, 4: 2, 5: 1, 6: 1, 7: 1}


@pytest.mark.parametrize("k", range(8))
def test_phase_coefficient_from_energy_and_flux(derived, k):
    psi, psil = derived
    pk, pl = spin_truncate(psi[k], SPIN_DEG[k]), spin_truncate(psil[k], SPIN_DEG[k])
    for q, x1, x2 in POINTS:
        dl = (1.0 - q) / (1.0 + q)
        sub = {d: sp.Float(dl, 40), c1: sp.Float(x1, 40), c2: sp.Float(x2, 40)}
        want, want_l = float(pk.evalf(30, subs=sub)), float(pl.evalf(30, subs=sub))
        phi, phil = oracle_coeffs(q, x1, x2)
        scale = max(1.0, abs(want))
        if k != 5:     # the non-logarithmic 2.5PN term is a constant phase (conventional); its logarithm is not
            assert abs(phi[k] - want) <= 2e-13 * scale, (k, q, x1, x2, phi[k], want)
        assert abs(phil[k] - want_l) <= 2e-13 * max(1.0, abs(want_l)), (k, q, x1, x2, phil[k], want_l)


def test_2p5pn_constant_follows_the_usual_convention(derived):
    """phi_5 = phi_5^(l) / 3 (the sheet's c5 [1 + 3 ln v]): with the constants of integration dropped, the derivation gives exactly that."""
    psi, psil = derived
    assert sp.expand(spin_truncate(psi[5], 1) - spin_truncate(psil[5], 1) / 3) == 0
    for q, x1, x2 in POINTS:
        phi, phil = oracle_coeffs(q, x1, x2)
        assert abs(phi[5] - phil[5] / 3.0) <= 1e-13 * abs(phi[5])


def test_typed_energy_matches_kerr_geodesics():
    """Test-mass limit (delta -> 1, the heavy body carries chi1): E(v)/mu of a circular equatorial Kerr geodesic is exact,
    E = (1 - 2u^2 + chi u^3) / sqrt(1 - 3u^2 + 2 chi u^3) - 1 with u^2 = M/r and M Omega = u^3 / (1 + chi u^3).  Its expansion in
    v = (M Omega)^(1/3) must reproduce every typed e_k (spin-orbit at 1.5, 2.5, 3.5PN and the chi^2 term at 2PN) at eta -> 0."""
    u, x = sp.symbols("u chi")
    E = (1 - 2 * u ** 2 + x * u ** 3) / sp.sqrt(1 - 3 * u ** 2 + 2 * x * u ** 3) - 1
    # invert v^3 = u^3 / (1 + chi u^3):  u^3 = v^3 / (1 - chi v^3)
    Ev = sp.series(E.subs(u, v * (1 - x * v ** 3) ** R(-1, 3)), v, 0, 10).removeO()
    ser = sp.expand(Ev / (-v ** 2 / 2))
    e = energy_coeffs()
    for k in range(8):
        typed = sp.expand(sp.limit(sp.expand(e[k]).subs({c1: x, c2: 0}), d, 1)) if e[k] != 0 else 0
        kerr = ser.coeff(v, k)
        if k <= 5 or k == 7:
            keep = 2 if k == 4 else 1          # the sheet's spin orders: higher powers of chi at 3PN+ are not typed
            assert sp.expand(spin_trunc1(kerr, x, keep) - typed) == 0, (k, kerr, typed)
        else:                                  # 3PN: no linear-in-spin term in the energy; spin-independent part -675/64
            assert sp.expand(spin_trunc1(kerr, x, 1) - typed) == 0, (k, kerr, typed)


def spin_trunc1(expr, x, max_deg):
    poly = sp.Poly(sp.expand(expr), x)
    return sum(co * x ** i for (i,), co in poly.terms() if i <= max_deg)


def test_typed_flux_matches_black_hole_perturbation_theory():
    """Test-mass limit of the typed flux against Tagoshi, Shibata, Tanaka & Sasaki 1996 (a particle on a circular equatorial
    Kerr orbit): spin terms -11 q/4 v^3, +33 q^2/16 v^4, -59 q/16 v^5, -65 pi q/6 v^6, +162035 q/3888 v^7; and the
    Schwarzschild terms of Tagoshi & Sasaki 1994."""
    x = sp.Symbol("chi")
    f = flux_coeffs()
    lim = [sp.expand(sp.limit(sp.expand(fk).subs({c1: x, c2: 0}), d, 1)) if fk != 0 else 0 for fk in f]
    assert lim[2] == -R(1247, 336)
    assert sp.expand(lim[3] - (4 * pi - R(11, 4) * x)) == 0
    assert sp.expand(lim[4] - (-R(44711, 9072) + R(33, 16) * x ** 2)) == 0
    assert sp.expand(lim[5] - (-R(8191, 672) * pi - R(59, 16) * x)) == 0
    assert sp.expand(lim[6].coeff(x, 1) + R(65, 6) * pi) == 0
    assert sp.expand(lim[6].coeff(Lv, 1) + R(1712, 105)) == 0
    assert sp.expand(lim[7] - (-R(16285, 504) * pi + R(162035, 3888) * x)) == 0


def test_a_perturbed_digit_would_fail(derived):
    """The pin has teeth: the derived 3PN and 3.5PN numbers differ from the sheet's with one digit changed by far more than the tolerance."""
    psi, _ = derived
    sub = {d: sp.Float(1.0 / 9.0, 40), c1: sp.Float(0.3, 40), c2: sp.Float(-0.2, 40)}
    w6 = float(spin_truncate(psi[6], 1).evalf(30, subs=sub))
    w7 = float(spin_truncate(psi[7], 1).evalf(30, subs=sub))
    phi, _ = oracle_coeffs(0.8, 0.3, -0.2)
    eta = 0.8 / 1.8 ** 2
    assert abs((phi[6] + (76056.0 - 76055.0) * eta * eta / 1728.0) - w6) > 1e-8 * abs(w6)
    assert abs((phi[7] + math.pi * eta * (378516.0 - 378515.0) / 1512.0) - w7) > 1e-8 * abs(w7)


# ---- inspiral amplitude of the PhenomD-form model (DESIGN.md A.2: A_hat = sum_i A_i (pi F)^(i/3) + ...) -------------------------
def h22_coeffs():
    """Modulus of the (2,2) mode's PN amplitude series H_22(v) (Blanchet et al. 2008 / Kidder 2008; spin-orbit term of Arun et al.
    2009), typed in its own form; imaginary parts enter the modulus beyond 3PN only.  Spin terms beyond 1.5PN are NOT typed."""
    eta = ETA
    xs, xa = (c1 + c2) / 2, (c1 - c2) / 2
    H = [0] * 7
    H[0] = 1
    H[2] = -R(107, 42) + R(55, 42) * eta
    H[3] = 2 * pi - R(4, 3) * (d * xa + (1 - eta) * xs)
    H[4] = -R(2173, 1512) - R(1069, 216) * eta + R(2047, 1512) * eta ** 2
    H[5] = -(R(107, 21) - R(34, 21) * eta) * pi
    H[6] = (R(27027409, 646800) - R(856, 105) * EulerGamma + R(2, 3) * pi ** 2 + (-R(278185, 33264) + R(41, 96) * pi ** 2) * eta
            - R(20261, 2772) * eta ** 2 + R(114635, 99792) * eta ** 3 - R(428, 105) * (4 * log(2) + 2 * Lv))
    return H


def test_inspiral_amplitude_coefficients_from_mode_amplitude_and_chirp_rate():
    """Stationary phase: |h(f)| is proportional to v^2 |H_22(v)| / sqrt(df/dt), df/dt proportional to v^11 F / (-E'), so relative to the Newtonian f^-7/6
    amplitude A_hat(v) = |H_22| sqrt(-E'(v) / (eta v F_hat(v))).  Pins the spin-independent part of A_2..A_6 (the logarithms of H_22 and of
    the flux cancel) and the full A_3.  The spin parts of A_4..A_6 stay this build's constants (oracle header, DESIGN.md A.2)."""
    e, f, H = energy_coeffs(), flux_coeffs(), h22_coeffs()
    N = [R(k + 2, 2) * e[k] for k in range(8)]
    Q = [0] * 7
    for k in range(7):
        Q[k] = sp.expand(N[k] - sum(Q[j] * f[k - j] for j in range(k)))
    s = [1] + [0] * 6                                           # sqrt(Q) as a series
    for k in range(1, 7):
        s[k] = sp.expand((Q[k] - sum(s[j] * s[k - j] for j in range(1, k))) / 2)
    A = [sp.expand(sum(H[j] * s[k - j] for j in range(k + 1))) for k in range(7)]
    assert all(sp.expand(A[k]).diff(Lv) == 0 for k in range(7))  # no logarithm survives
    spec = dict(like_kind=2, ndim=11, prior_kind=[0] * 11, prior_lo=[0.0] * 11, prior_hi=[1.0] * 11, periodic=[0] * 11, n_det=0, n_freq=0,
                phenom_table=np.zeros((19, 11)))
    P = O.OracleProblem(spec)
    for q, x1, x2 in POINTS:
        dl = (1.0 - q) / (1.0 + q)
        got = (C.c_double * 7)()
        th = np.array([30.0, q, x1, x2, 500.0, 0.3, 0.1, 0.2, 0.0, 1.0, 0.5])
        O._lib.orc_phenomd_amp_coeffs(C.byref(P.p), th.ctypes.data_as(O.c_d_p), got)
        got0 = (C.c_double * 7)()
        th0 = th.copy(); th0[2] = th0[3] = 0.0
        O._lib.orc_phenomd_amp_coeffs(C.byref(P.p), th0.ctypes.data_as(O.c_d_p), got0)
        for k in range(7):
            want0 = float(spin_truncate(A[k], 0).evalf(30, subs={d: sp.Float(dl, 40)}))
            assert abs(got0[k] - want0) <= 2e-13 * max(1.0, abs(want0)), (k, q, got0[k], want0)
        want3 = float(spin_truncate(A[3], 1).evalf(30, subs={d: sp.Float(dl, 40), c1: sp.Float(x1, 40), c2: sp.Float(x2, 40)}))
        assert abs(got[3] - want3) <= 2e-13 * max(1.0, abs(want3)), (q, x1, x2, got[3], want3)
