"""Pins for prior transforms (CDF inversion identities) and detector geometry (invariants of DESIGN.md A.3)."""
import math

import numpy as np

from oracle import oracle as O
from paper_2509_04336_b200 import workloads as W

C = 299792458.0


def _prob():
    return O.OracleProblem(W.gw_spec(W.LIKE_TAYLORF2, ["H1", "L1", "V1"], 4.0, 64.0, (20.0, 40.0)))


def test_prior_cdf_inversion():
    P = _prob()
    u = W.uniforms(2000, 11, 3)
    th = P.prior_transform(u)
    spec = W.gw_spec(W.LIKE_TAYLORF2, ["H1"], 4.0, 64.0, (20.0, 40.0))
    lo, hi, kind = np.array(spec["prior_lo"]), np.array(spec["prior_hi"]), spec["prior_kind"]
    for d in range(11):
        x = th[:, d]
        assert np.all(x >= lo[d]) and np.all(x <= hi[d])
        if kind[d] == W.UNIFORM:
            F = (x - lo[d]) / (hi[d] - lo[d])
        elif kind[d] == W.POWERLAW2:   # P:182 p(dL) ~ dL^2
            F = (x ** 3 - lo[d] ** 3) / (hi[d] ** 3 - lo[d] ** 3)
        elif kind[d] == W.SINE:        # Table 1, theta_jn
            F = (1 - np.cos(x)) / 2
        elif kind[d] == W.COSINE:      # Table 1, dec
            F = (1 + np.sin(x)) / 2
        np.testing.assert_allclose(F, u[:, d], rtol=0, atol=2e-13)


def test_config5_injection_image():
    spec = W.gw_spec(W.LIKE_PHENOMD, ["H1"], 4.0, 64.0, (8.0, 20.0))
    th = O.OracleProblem(spec).prior_transform(np.array([W.U_INJ_C4]))[0]
    np.testing.assert_allclose(th, W.INJ_C4, rtol=2e-5, atol=2e-5)


def test_arms_and_light_travel_times():
    for name, (r, x, y) in W.DETECTORS.items():
        r, x, y = map(np.array, (r, x, y))
        assert abs(np.linalg.norm(x) - 1) < 1e-10 and abs(np.linalg.norm(y) - 1) < 1e-10
        assert abs(x @ y) < 2e-7
        assert 6.36e6 < np.linalg.norm(r) < 6.38e6
    d = lambda a, b: np.linalg.norm(np.array(W.DETECTORS[a][0]) - np.array(W.DETECTORS[b][0])) / C
    assert abs(d("H1", "L1") - 10.0128e-3) < 2e-6
    assert abs(d("H1", "V1") - 27.288e-3) < 2e-6
    assert abs(d("L1", "V1") - 26.448e-3) < 2e-6


def test_time_delay_bounded_by_light_travel_and_zenith():
    P = _prob()
    rng = np.random.default_rng(0)
    for _ in range(200):
        ra, dec, psi = rng.uniform(0, 2 * math.pi), math.asin(rng.uniform(-1, 1)), rng.uniform(0, math.pi)
        dts = [P.detector_response(i, ra, dec, psi)[2] for i in range(3)]
        for i in range(3):
            assert abs(dts[i]) <= 6.38e6 / C
        assert abs(dts[0] - dts[1]) <= 10.0128e-3 + 1e-6
    # source at the H1 zenith: the wave reaches H1 before the geocentre by |r|/c = 21.238 ms and F+^2+Fx^2 ~ 1
    r = np.array(W.DETECTORS["H1"][0])
    n = r / np.linalg.norm(r)
    dec = math.asin(n[2])
    g = math.atan2(-n[1], n[0])          # n = (cos d cos g, -cos d sin g, sin d)
    ra = W.GMST - g
    fp, fx, dt = P.detector_response(0, ra, dec, 0.3)
    assert abs(dt + 21.238e-3) < 2e-6
    assert abs(fp * fp + fx * fx - 1.0) < 1e-4


def test_antenna_pattern_invariants():
    P = _prob()
    rng = np.random.default_rng(1)
    acc = []
    for _ in range(3000):
        ra, dec, psi = rng.uniform(0, 2 * math.pi), math.asin(rng.uniform(-1, 1)), rng.uniform(0, math.pi)
        fp, fx, _ = P.detector_response(1, ra, dec, psi)
        fp2, fx2, _ = P.detector_response(1, ra, dec, psi + math.pi / 2)
        fp3, fx3, _ = P.detector_response(1, ra, dec, psi + 0.7)
        assert abs(fp + fp2) < 1e-12 and abs(fx + fx2) < 1e-12         # spin-2: psi + pi/2 flips the sign
        assert abs(fp * fp + fx * fx - fp3 * fp3 - fx3 * fx3) < 1e-12   # power independent of psi
        # rotation by psi: (F+, Fx)(psi+a) = (F+ cos2a + Fx sin2a, -F+ sin2a + Fx cos2a) up to the convention's sign
        c, s = math.cos(1.4), math.sin(1.4)
        assert min(abs(fp3 - (fp * c + fx * s)) + abs(fx3 - (-fp * s + fx * c)),
                   abs(fp3 - (fp * c - fx * s)) + abs(fx3 - (fp * s + fx * c))) < 1e-12
        assert abs(fp) <= 1 + 1e-12 and abs(fx) <= 1 + 1e-12
        acc.append(fp * fp + fx * fx)
    assert abs(np.mean(acc) - 0.4) < 0.015     # sky average of F+^2 + Fx^2 = 2/5 for a 90-degree interferometer
