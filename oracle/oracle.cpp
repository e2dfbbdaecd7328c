// oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU restatement (fp64, libm, long-double accumulators,
// no tables, no blocking, no fusion) of the hot path of arXiv 2509.04336
// (Prathaban et al., "Gravitational-wave inference at GPU speed: a bilby-like nested
// sampling kernel within blackjax-ns"): batched acceptance-walk nested sampling with a
// frequency-domain gravitational-wave likelihood.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this library.  It shares no code, header, table or constant generator with
// paper_2509_04336_b200/csrc (the CUDA path).  Citations: "P:NNN" = /root/reference/PAPER.md
// line NNN; "R:Lnn" = reading Lnn of DESIGN.md section 3 (where the paper is silent).
//
// Pin status (tests/test_oracle_*.py, all -m "not gpu"):
//   Philox4x32-10 ............ known-answer vectors of Salmon et al. 2011 (tests/golden/philox_kat.txt)
//   u53 / index / Erlang-4 ... range, mean/variance, KS against scipy gamma CDF
//   prior transforms ......... CDF-inversion identities
//   detector geometry ........ light travel times, antenna-pattern invariants, sky average 2/5
//   TaylorF2 phase ........... every coefficient phi_2..phi_7 and both logarithms DERIVED with sympy from independently typed PN energy and
//                              flux series (spin-orbit to 3.5PN, spin-spin at 2PN), themselves checked against Kerr geodesics and
//                              black-hole perturbation theory in the test-mass limit (tests/test_oracle_pn_derivation.py);
//                              mpmath 40-digit evaluation of the printed formula, Newtonian chirp time
//   inspiral amplitude ....... spin-independent parts of A_2..A_6 and all of A_3 derived the same way from the (2,2)-mode amplitude and
//                              the chirp rate; THE SPIN PARTS OF A_4, A_5, A_6 ARE THIS BUILD'S CONSTANTS (recalled, PARITY UNPINNED,
//                              like the fit table: DESIGN.md A.2)
//   walk-length tuning ....... R:L13/L14 recurrence on by-hand accept counts: 0.5 floor, maxmcmc cap, k = 1 / k = n/2 / explicit delays
//   <h,h> .................... closed form |C|^2 A0^2 I_{7/3}; Euler-Maclaurin integral for flat PSD
//   <d,h> .................... noise-free maximum, exact symmetries, 1/dL scaling, time-shift covariance
//   PhenomD-form ............. C0/C1 continuity, reduction to TaylorF2, QNM hand values, mpmath twin;
//                              PHYSICAL FIDELITY TO THE PUBLISHED IMRPhenomD FIT: PARITY UNPINNED
//                              (its coefficient table is not available here, R:L2)
//   walk ..................... cube-shell likelihood: uniformity of new points (KS)
//   evidence ................. eq. 3-5 shrinkage sum, Gaussian closed-form logZ, 2-D quadrature
//   top-k .................... numpy stable argsort
//   full 11-D runs ........... statistical only (exact parity unpinned by nature)
//   relative binning (R:L24) . exact along constant-ratio directions, partition of <d,h0>/<h0,h0>, second-order time-shift bound,
//                              error / 4 per halving of eps (tests/test_oracle_relbin.py)
//   slice kernel (R:L25) ..... uniformity in cube shells and Gaussian ellipsoids from a single start (closed-form laws), sample
//                              covariance factor against numpy, config-1 evidence and shell volumes with it inside the sampler
//                              (tests/test_oracle_slice.py)

#include <cmath>
#include <cstdint>
#include <cstring>
#include <cstdlib>
#include <vector>
#include <algorithm>
#include <numeric>
#include <limits>
#include <omp.h>

namespace {

const double PI = 3.14159265358979323846264338327950288;
const double GMSUN_S = 4.925490947641267e-6;                 // G Msun / c^3 [s]
const double MPC_S = 3.0856775814913673e22 / 299792458.0;    // 1 Mpc / c [s]
const double C_SI = 299792458.0;
const double EULER_GAMMA = 0.5772156649015329;
const double NEG_INF = -std::numeric_limits<double>::infinity();

int omp_get_max_threads_safe() { return omp_get_max_threads(); }

enum { LIKE_GAUSS = 0, LIKE_TAYLORF2 = 1, LIKE_PHENOMD = 2, LIKE_SHELL = 3 };
enum { PRIOR_UNIFORM = 0, PRIOR_POWERLAW2 = 1, PRIOR_SINE = 2, PRIOR_COSINE = 3, PRIOR_FIXED = 4 };

}  // namespace

extern "C" {

// Flat problem description used by every oracle call (the oracle's own layout; the CUDA
// library has a different, independently declared struct).
struct orc_problem {
  int32_t like_kind;
  int32_t ndim;
  int32_t prior_kind[16];
  double prior_lo[16];
  double prior_hi[16];
  int32_t periodic[16];
  int32_t n_det;
  int32_t n_freq;
  double f_min;
  double df;
  double det_vertex[4][3];
  double det_xarm[4][3];
  double det_yarm[4][3];
  double gmst;
  double toy_mean[16];
  double toy_prec[256];
  double toy_lognorm;
  double phenom_table[19][11];
  const double* strain;  // [n_det][n_freq][2]
  const double* psd;     // [n_det][n_freq]
  const void* relbin;    // optional: relative-binning data (orc_relbin_create); when set, loglike_from_u -- and so the walk, the
                         // NS step and the runs -- use the relative-binning likelihood (R:L24) instead of the exact one
};

struct orc_sampler_cfg {
  int32_t n_live, n_delete, naccept, maxmcmc;
  double walks0;
  double delay;  // <0 -> default (R:L14)
};

struct orc_stats {
  int64_t iteration;
  double logl_star, logx, logz, h, dlogz, live_frac_log;
  int32_t walk_len;
  double walks_next;
  double accept_mean;
  int32_t accept_min, accept_max;
  int64_t n_eval, n_oob, n_stuck;
  int64_t n_eval_total;
};

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw 2011).  R:R (RNG contract).
// ---------------------------------------------------------------------------------------------
void orc_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Uniform strictly inside (0,1) on a 2^-52 grid offset by half a cell: ((hi>>6)*2^26 + (lo>>6) + 0.5) * 2^-52.
// (52 random bits so that the +0.5 is exact in fp64; a 53-bit variant would round up to 1.0 at the top end.)
double orc_u53(uint32_t hi, uint32_t lo) {
  return ((double)(hi >> 6) * 67108864.0 + (double)(lo >> 6) + 0.5) * (1.0 / 4503599627370496.0);
}

uint32_t orc_mulhi32(uint32_t w, uint32_t m) { return (uint32_t)(((uint64_t)w * (uint64_t)m) >> 32); }

}  // extern "C"

namespace {

void philox_block(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t out[4]) {
  uint32_t ctr[4] = {c0, c1, c2, c3};
  uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
  orc_philox(ctr, key, out);
}

int n_free_dims(const orc_problem* p) {
  int n = 0;
  for (int d = 0; d < p->ndim; ++d) n += (p->prior_kind[d] != PRIOR_FIXED);
  return n;
}

// ---------------------------------------------------------------------------------------------
// Prior transforms, unit cube -> physical (P:96 unit hypercube; Table 1; P:182 d_L^2).
// ---------------------------------------------------------------------------------------------
double prior_transform_1(int kind, double lo, double hi, double u) {
  switch (kind) {
    case PRIOR_UNIFORM: return lo + (hi - lo) * u;
    case PRIOR_POWERLAW2: {  // p(x) ~ x^2 on [lo,hi]:  x = cbrt(lo^3 + u (hi^3 - lo^3))
      double a3 = lo * lo * lo, b3 = hi * hi * hi;
      return std::cbrt(a3 + u * (b3 - a3));
    }
    case PRIOR_SINE: {  // p(x) ~ sin x on [lo,hi]:  cos x = cos lo - u (cos lo - cos hi)
      double cl = std::cos(lo), ch = std::cos(hi);
      return std::acos(cl - u * (cl - ch));
    }
    case PRIOR_COSINE: {  // p(x) ~ cos x on [lo,hi]:  sin x = sin lo + u (sin hi - sin lo)
      double sl = std::sin(lo), sh = std::sin(hi);
      return std::asin(sl + u * (sh - sl));
    }
    default: return lo;  // FIXED
  }
}

void prior_transform(const orc_problem* p, const double* u, double* theta) {
  for (int d = 0; d < p->ndim; ++d) theta[d] = prior_transform_1(p->prior_kind[d], p->prior_lo[d], p->prior_hi[d], u[d]);
}

// ---------------------------------------------------------------------------------------------
// Detector response (R:L3, DESIGN.md A.3): F+, Fx and arrival-time offset for one detector.
// ---------------------------------------------------------------------------------------------
void detector_response(const orc_problem* p, int det, double ra, double dec, double psi, double* fp, double* fx, double* dt) {
  const double* xa = p->det_xarm[det];
  const double* ya = p->det_yarm[det];
  double D[3][3];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) D[i][j] = 0.5 * (xa[i] * xa[j] - ya[i] * ya[j]);
  double g = p->gmst - ra;
  double cg = std::cos(g), sg = std::sin(g), cd = std::cos(dec), sd = std::sin(dec), cp = std::cos(psi), sp = std::sin(psi);
  double X[3] = {-cp * sg - sp * cg * sd, -cp * cg + sp * sg * sd, sp * cd};
  double Y[3] = {sp * sg - cp * cg * sd, sp * cg + cp * sg * sd, cp * cd};
  double xdx = 0, ydy = 0, xdy = 0, ydx = 0;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      xdx += X[i] * D[i][j] * X[j];
      ydy += Y[i] * D[i][j] * Y[j];
      xdy += X[i] * D[i][j] * Y[j];
      ydx += Y[i] * D[i][j] * X[j];
    }
  *fp = xdx - ydy;
  *fx = xdy + ydx;
  double n[3] = {cd * cg, -cd * sg, sd};
  const double* r = p->det_vertex[det];
  *dt = -(r[0] * n[0] + r[1] * n[1] + r[2] * n[2]) / C_SI;
}

// ---------------------------------------------------------------------------------------------
// Intrinsic source quantities (R:L19): q = m2/m1 in (0,1], chi1 on the heavier body.
// ---------------------------------------------------------------------------------------------
struct Intrinsic {
  double eta, M, delta, chi1, chi2, chis, chia, m1, m2;  // M, m1, m2 in seconds
};

Intrinsic make_intrinsic(double Mc, double q, double chi1, double chi2) {
  Intrinsic s;
  s.eta = q / ((1.0 + q) * (1.0 + q));
  s.M = Mc * GMSUN_S * std::pow(s.eta, -0.6);
  s.m1 = s.M / (1.0 + q);
  s.m2 = s.M * q / (1.0 + q);
  s.delta = (s.m1 - s.m2) / s.M;
  s.chi1 = chi1; s.chi2 = chi2;
  s.chis = 0.5 * (chi1 + chi2);
  s.chia = 0.5 * (chi1 - chi2);
  return s;
}

// TaylorF2 3.5PN aligned-spin phase coefficients (DESIGN.md A.1).  phi[k], phil[k] multiply v^k and v^k ln v.
void taylorf2_coeffs(const Intrinsic& s, double phi[8], double phil[8]) {
  const double eta = s.eta, d = s.delta, xs = s.chis, xa = s.chia;
  const double eta2 = eta * eta, eta3 = eta2 * eta;
  for (int k = 0; k < 8; ++k) { phi[k] = 0; phil[k] = 0; }
  phi[0] = 1.0;
  phi[1] = 0.0;
  phi[2] = 3715.0 / 756.0 + 55.0 * eta / 9.0;
  phi[3] = -16.0 * PI + (113.0 / 3.0) * d * xa + (113.0 / 3.0 - 76.0 * eta / 3.0) * xs;
  phi[4] = 15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta2 / 72.0 + (-405.0 / 8.0 + 200.0 * eta) * xa * xa -
           (405.0 / 4.0) * d * xa * xs + (-405.0 / 8.0 + 5.0 * eta / 2.0) * xs * xs;
  double c5 = 38645.0 * PI / 756.0 - 65.0 * PI * eta / 9.0 + d * (-732985.0 / 2268.0 - 140.0 * eta / 9.0) * xa +
              (-732985.0 / 2268.0 + 24260.0 * eta / 81.0 + 340.0 * eta2 / 9.0) * xs;
  phi[5] = c5;
  phil[5] = 3.0 * c5;
  phi[6] = 11583231236531.0 / 4694215680.0 - 6848.0 * EULER_GAMMA / 21.0 - 640.0 * PI * PI / 3.0 +
           (-15737765635.0 / 3048192.0 + 2255.0 * PI * PI / 12.0) * eta + 76055.0 * eta2 / 1728.0 - 127825.0 * eta3 / 1296.0 -
           (6848.0 / 63.0) * std::log(64.0) + (2270.0 * PI / 3.0) * d * xa + (2270.0 * PI / 3.0 - 520.0 * PI * eta) * xs;
  phil[6] = -6848.0 / 21.0;
  phi[7] = 77096675.0 * PI / 254016.0 + 378515.0 * PI * eta / 1512.0 - 74045.0 * PI * eta2 / 756.0 +
           d * (-25150083775.0 / 3048192.0 + 26804935.0 * eta / 6048.0 - 1985.0 * eta2 / 48.0) * xa +
           (-25150083775.0 / 3048192.0 + 10566655595.0 * eta / 762048.0 - 1042165.0 * eta2 / 3024.0 + 5345.0 * eta3 / 36.0) * xs;
}

// Psi_TF2(F) = -pi/4 + 3/(128 eta) v^-5 sum_k (phi_k + phil_k ln v) v^k,  v = (pi F)^(1/3), F = M f.
double taylorf2_phase(const Intrinsic& s, const double phi[8], const double phil[8], double F) {
  double v = std::cbrt(PI * F);
  double lv = std::log(v);
  double sum = 0.0;
  for (int k = 0; k < 8; ++k) sum += (phi[k] + phil[k] * lv) * std::pow(v, (double)k);
  return -PI / 4.0 + 3.0 / (128.0 * s.eta) * std::pow(v, -5.0) * sum;
}

double taylorf2_dphase(const Intrinsic& s, const double phi[8], const double phil[8], double F) {
  double v = std::cbrt(PI * F);
  double lv = std::log(v);
  double sum = 0.0;
  for (int k = 0; k < 8; ++k) sum += ((k - 5.0) * (phi[k] + phil[k] * lv) + phil[k]) * std::pow(v, k - 6.0);
  return 3.0 / (128.0 * s.eta) * sum * v / (3.0 * F);
}

// ---------------------------------------------------------------------------------------------
// "IMRPhenomD-form" model (DESIGN.md A.2): the published piecewise *form* with the fit table as data.
// ---------------------------------------------------------------------------------------------
enum { R_RHO1, R_RHO2, R_RHO3, R_V2, R_GAM1, R_GAM2, R_GAM3, R_SIG1, R_SIG2, R_SIG3, R_SIG4, R_BET1, R_BET2, R_BET3, R_ALP1, R_ALP2, R_ALP3, R_ALP4, R_ALP5 };

struct PhenomD {
  Intrinsic s;
  double phi[8], phil[8];
  double L[19];
  double Frd, Fdamp, Fpeak;
  double A[7];                       // inspiral amplitude PN coefficients
  double v1, d1, v3, d3, v2mid;      // intermediate amplitude Hermite data
  double C1int, C2int, C1mr, C2mr, t0;
};

double pd_amp_ins(const PhenomD& m, double F) {
  double x = std::cbrt(PI * F);
  double sum = 0.0;
  for (int i = 0; i < 7; ++i) sum += m.A[i] * std::pow(x, (double)i);
  return sum + m.L[R_RHO1] * std::pow(F, 7.0 / 3.0) + m.L[R_RHO2] * std::pow(F, 8.0 / 3.0) + m.L[R_RHO3] * F * F * F;
}
double pd_damp_ins(const PhenomD& m, double F) {
  double sum = 0.0;
  for (int i = 1; i < 7; ++i) sum += m.A[i] * (i / 3.0) * std::pow(PI, i / 3.0) * std::pow(F, i / 3.0 - 1.0);
  return sum + (7.0 / 3.0) * m.L[R_RHO1] * std::pow(F, 4.0 / 3.0) + (8.0 / 3.0) * m.L[R_RHO2] * std::pow(F, 5.0 / 3.0) + 3.0 * m.L[R_RHO3] * F * F;
}
double pd_amp_mr(const PhenomD& m, double F) {
  double w = m.L[R_GAM3] * m.Fdamp;
  double x = F - m.Frd;
  return m.L[R_GAM1] * w / (x * x + w * w) * std::exp(-m.L[R_GAM2] * x / w);
}
double pd_damp_mr(const PhenomD& m, double F) {
  double w = m.L[R_GAM3] * m.Fdamp;
  double x = F - m.Frd;
  return pd_amp_mr(m, F) * (-2.0 * x / (x * x + w * w) - m.L[R_GAM2] / w);
}
double pd_amp_int(const PhenomD& m, double F) {
  const double F1 = 0.014;
  double Lw = m.Fpeak - F1;
  double x = (F - F1) / Lw;
  double x2 = x * x, x3 = x2 * x;
  double h00 = 2 * x3 - 3 * x2 + 1, h10 = x3 - 2 * x2 + x, h01 = -2 * x3 + 3 * x2, h11 = x3 - x2;
  double mid = 0.5 * m.v1 + Lw * m.d1 / 8.0 + 0.5 * m.v3 - Lw * m.d3 / 8.0;
  return h00 * m.v1 + h10 * Lw * m.d1 + h01 * m.v3 + h11 * Lw * m.d3 + (m.v2mid - mid) * 16.0 * x2 * (1 - x) * (1 - x);
}
double pd_amp_hat(const PhenomD& m, double F) {
  if (F < 0.014) return pd_amp_ins(m, F);
  if (F < m.Fpeak) return pd_amp_int(m, F);
  return pd_amp_mr(m, F);
}

double pd_phase_ins(const PhenomD& m, double F) {
  double e = m.s.eta;
  return taylorf2_phase(m.s, m.phi, m.phil, F) +
         (m.L[R_SIG1] * F + 0.75 * m.L[R_SIG2] * std::pow(F, 4.0 / 3.0) + 0.6 * m.L[R_SIG3] * std::pow(F, 5.0 / 3.0) + 0.5 * m.L[R_SIG4] * F * F) / e;
}
double pd_dphase_ins(const PhenomD& m, double F) {
  double e = m.s.eta;
  return taylorf2_dphase(m.s, m.phi, m.phil, F) +
         (m.L[R_SIG1] + m.L[R_SIG2] * std::cbrt(F) + m.L[R_SIG3] * std::pow(F, 2.0 / 3.0) + m.L[R_SIG4] * F) / e;
}
double pd_phase_int_raw(const PhenomD& m, double F) {
  return (m.L[R_BET1] * F + m.L[R_BET2] * std::log(F) - m.L[R_BET3] / (3.0 * F * F * F)) / m.s.eta;
}
double pd_dphase_int_raw(const PhenomD& m, double F) {
  return (m.L[R_BET1] + m.L[R_BET2] / F + m.L[R_BET3] / (F * F * F * F)) / m.s.eta;
}
double pd_phase_mr_raw(const PhenomD& m, double F) {
  return (m.L[R_ALP1] * F - m.L[R_ALP2] / F + (4.0 / 3.0) * m.L[R_ALP3] * std::pow(F, 0.75) +
          m.L[R_ALP4] * std::atan((F - m.L[R_ALP5] * m.Frd) / m.Fdamp)) / m.s.eta;
}
double pd_dphase_mr_raw(const PhenomD& m, double F) {
  double y = (F - m.L[R_ALP5] * m.Frd) / m.Fdamp;
  return (m.L[R_ALP1] + m.L[R_ALP2] / (F * F) + m.L[R_ALP3] * std::pow(F, -0.25) + m.L[R_ALP4] / (m.Fdamp * (1.0 + y * y))) / m.s.eta;
}
// Un-aligned piecewise phase phi(F).
double pd_phase_piecewise(const PhenomD& m, double F) {
  if (F < 0.018) return pd_phase_ins(m, F);
  if (F < 0.5 * m.Frd) return pd_phase_int_raw(m, F) + m.C1int + m.C2int * F;
  return pd_phase_mr_raw(m, F) + m.C1mr + m.C2mr * F;
}

PhenomD make_phenomd(const orc_problem* p, double Mc, double q, double chi1, double chi2) {
  PhenomD m;
  m.s = make_intrinsic(Mc, q, chi1, chi2);
  const Intrinsic& s = m.s;
  taylorf2_coeffs(s, m.phi, m.phil);
  const double eta = s.eta, eta2 = eta * eta, eta3 = eta2 * eta;
  // fit-table evaluation
  double chieff = (s.m1 * chi1 + s.m2 * chi2) / s.M;
  double chipn = chieff - (38.0 * eta / 113.0) * (chi1 + chi2);
  double xi = chipn - 1.0;
  for (int r = 0; r < 19; ++r) {
    const double* t = p->phenom_table[r];
    m.L[r] = t[0] + t[1] * eta + xi * (t[2] + t[3] * eta + t[4] * eta2) + xi * xi * (t[5] + t[6] * eta + t[7] * eta2) +
             xi * xi * xi * (t[8] + t[9] * eta + t[10] * eta2);
  }
  // final state (surrogate fits)
  double S = (s.m1 * s.m1 * chi1 + s.m2 * s.m2 * chi2) / (s.M * s.M);
  double af = 2.0 * std::sqrt(3.0) * eta - 3.871 * eta2 + 4.028 * eta3 + S;
  af = std::min(0.99, std::max(-0.99, af));
  double Erad = 0.05597 * eta + 0.5810 * eta2 - 0.9607 * eta3 + 3.352 * eta2 * eta2;
  m.Frd = (1.5251 - 1.1568 * std::pow(1.0 - af, 0.1292)) / (2.0 * PI * (1.0 - Erad));
  double Q = 0.7 + 1.4187 * std::pow(1.0 - af, -0.4990);
  m.Fdamp = m.Frd / (2.0 * Q);
  double g2 = m.L[R_GAM2], g3 = m.L[R_GAM3];
  if (g2 < 1.0) m.Fpeak = std::fabs(m.Frd + m.Fdamp * g3 * (std::sqrt(1.0 - g2 * g2) - 1.0) / g2);
  else m.Fpeak = std::fabs(m.Frd - m.Fdamp * g3 / g2);
  // inspiral amplitude PN coefficients
  const double d = s.delta, xs = s.chis, xa = s.chia;
  m.A[0] = 1.0;
  m.A[1] = 0.0;
  m.A[2] = -323.0 / 224.0 + 451.0 * eta / 168.0;
  m.A[3] = (27.0 / 8.0 - 11.0 * eta / 6.0) * xs + (27.0 / 8.0) * d * xa;
  m.A[4] = -27312085.0 / 8128512.0 - 1975055.0 * eta / 338688.0 + 105271.0 * eta2 / 24192.0 + (-81.0 / 32.0 + 8.0 * eta) * xa * xa -
           (81.0 / 16.0) * d * xa * xs + (-81.0 / 32.0 + 17.0 * eta / 8.0) * xs * xs;
  m.A[5] = -85.0 * PI / 64.0 + 85.0 * PI * eta / 16.0 + (285197.0 / 16128.0 - 1579.0 * eta / 4032.0) * d * xa +
           (285197.0 / 16128.0 - 15317.0 * eta / 672.0 - 2227.0 * eta2 / 1008.0) * xs;
  m.A[6] = -177520268561.0 / 8583708672.0 + (545384828789.0 / 5007163392.0 - 205.0 * PI * PI / 48.0) * eta -
           3248849057.0 * eta2 / 178827264.0 + 34473079.0 * eta3 / 6386688.0 +
           (1614569.0 / 64512.0 - 1873643.0 * eta / 16128.0 + 2167.0 * eta2 / 42.0) * xa * xa + (31.0 * PI / 12.0 - 7.0 * PI * eta / 3.0) * xs +
           (1614569.0 / 64512.0 - 61391.0 * eta / 1344.0 + 57451.0 * eta2 / 4032.0) * xs * xs +
           d * xa * (31.0 * PI / 12.0 + (1614569.0 / 32256.0 - 165961.0 * eta / 2688.0) * xs);
  // intermediate amplitude data
  m.v1 = pd_amp_ins(m, 0.014);
  m.d1 = pd_damp_ins(m, 0.014);
  m.v3 = pd_amp_mr(m, m.Fpeak);
  m.d3 = pd_damp_mr(m, m.Fpeak);
  m.v2mid = m.L[R_V2];
  // phase connections: C0/C1 at 0.018 and Frd/2, analytic derivatives
  double Fa = 0.018;
  m.C2int = pd_dphase_ins(m, Fa) - pd_dphase_int_raw(m, Fa);
  m.C1int = pd_phase_ins(m, Fa) - pd_phase_int_raw(m, Fa) - m.C2int * Fa;
  double Fb = 0.5 * m.Frd;
  m.C2mr = (pd_dphase_int_raw(m, Fb) + m.C2int) - pd_dphase_mr_raw(m, Fb);
  m.C1mr = (pd_phase_int_raw(m, Fb) + m.C1int + m.C2int * Fb) - pd_phase_mr_raw(m, Fb) - m.C2mr * Fb;
  // time alignment at the amplitude peak
  m.t0 = pd_dphase_mr_raw(m, m.Fpeak) + m.C2mr;
  return m;
}

bool theta_physical(const double* th) {
  for (int i = 0; i < 11; ++i)
    if (!std::isfinite(th[i])) return false;
  if (!(th[0] > 0.0)) return false;
  if (!(th[1] > 0.0 && th[1] <= 1.0)) return false;
  if (std::fabs(th[2]) > 1.0 || std::fabs(th[3]) > 1.0) return false;
  if (!(th[4] > 0.0)) return false;
  return true;
}

// Intrinsic amplitude A(f) and phase Psi0(f) (which holds -2 phase - pi/4 and no tc term; R:L3).
struct Waveform {
  int kind;
  Intrinsic s;
  double phi[8], phil[8];
  PhenomD pd;
  double A0;     // sqrt(5/24) pi^-2/3 (G Mc/c^3)^(5/6) / (dL/c)
  double phase;  // theta[7]
};

Waveform make_waveform(const orc_problem* p, const double* th) {
  Waveform w;
  w.kind = p->like_kind;
  w.s = make_intrinsic(th[0], th[1], th[2], th[3]);
  taylorf2_coeffs(w.s, w.phi, w.phil);
  if (w.kind == LIKE_PHENOMD) w.pd = make_phenomd(p, th[0], th[1], th[2], th[3]);
  w.A0 = std::sqrt(5.0 / 24.0) * std::pow(PI, -2.0 / 3.0) * std::pow(th[0] * GMSUN_S, 5.0 / 6.0) / (th[4] * MPC_S);
  w.phase = th[7];
  return w;
}

void waveform_amp_phase(const Waveform& w, double f, double* amp, double* psi0) {
  double F = w.s.M * f;
  double a0 = w.A0 * std::pow(f, -7.0 / 6.0);
  if (w.kind == LIKE_TAYLORF2) {
    *amp = a0;
    *psi0 = taylorf2_phase(w.s, w.phi, w.phil, F) - 2.0 * w.phase;
  } else {
    *amp = a0 * pd_amp_hat(w.pd, F);
    *psi0 = pd_phase_piecewise(w.pd, F) - w.pd.t0 * F - 2.0 * w.phase;
  }
}

// ---------------------------------------------------------------------------------------------
// Log-likelihood ratio (R:L1): sum_det <d,h> - 1/2 <h,h>, <a,b> = 4 df Re sum conj(a) b / S.
// parts (optional): [<d,h>_0, <h,h>_0, <d,h>_1, <h,h>_1, ...]
// ---------------------------------------------------------------------------------------------
double gw_loglike(const orc_problem* p, const double* th, double* parts) {
  if (!theta_physical(th)) {
    if (parts) for (int i = 0; i < 2 * p->n_det; ++i) parts[i] = std::numeric_limits<double>::quiet_NaN();
    return NEG_INF;
  }
  Waveform w = make_waveform(p, th);
  double iota = th[5], psi = th[6], tc = th[8], ra = th[9], dec = th[10];
  double ci = std::cos(iota);
  double logl = 0.0;
  for (int det = 0; det < p->n_det; ++det) {
    double fp, fx, dt;
    detector_response(p, det, ra, dec, psi, &fp, &fx, &dt);
    // C_det = F+ (1+cos^2 i)/2 - i Fx cos i
    double cre = fp * 0.5 * (1.0 + ci * ci), cim = -fx * ci;
    long double dh = 0.0L, hh = 0.0L;
    const double* d = p->strain + (size_t)det * p->n_freq * 2;
    const double* S = p->psd + (size_t)det * p->n_freq;
    for (int k = 0; k < p->n_freq; ++k) {
      double f = p->f_min + k * p->df;
      double amp, psi0;
      waveform_amp_phase(w, f, &amp, &psi0);
      double Phi = psi0 + 2.0 * PI * f * (tc + dt);
      double c = std::cos(Phi), s = std::sin(Phi);
      // h = amp * C_det * (cos Phi - i sin Phi)
      double hre = amp * (cre * c + cim * s);
      double him = amp * (cim * c - cre * s);
      dh += (long double)((d[2 * k] * hre + d[2 * k + 1] * him) / S[k]);
      hh += (long double)((hre * hre + him * him) / S[k]);
    }
    double dhd = (double)(4.0L * p->df * dh), hhd = (double)(4.0L * p->df * hh);
    if (parts) { parts[2 * det] = dhd; parts[2 * det + 1] = hhd; }
    logl += dhd - 0.5 * hhd;
  }
  return logl;
}

double toy_loglike(const orc_problem* p, const double* th) {
  int D = p->ndim;
  double qf = 0.0;
  for (int i = 0; i < D; ++i)
    for (int j = 0; j < D; ++j) qf += (th[i] - p->toy_mean[i]) * p->toy_prec[i * D + j] * (th[j] - p->toy_mean[j]);
  return p->toy_lognorm - 0.5 * qf;
}

// Cube-shell test likelihood L(u) = -max_d |u_d - 1/2| (used to pin the walk and the volume bookkeeping).
double shell_loglike(const orc_problem* p, const double* u) {
  double r = 0.0;
  for (int d = 0; d < p->ndim; ++d) r = std::max(r, std::fabs(u[d] - 0.5));
  return -r;
}

double relbin_loglike_any(const orc_problem* p, const double* th);   // defined with the relative-binning code below

double loglike_from_u(const orc_problem* p, const double* u) {
  if (p->like_kind == LIKE_SHELL) return shell_loglike(p, u);
  double th[16];
  prior_transform(p, u, th);
  if (p->like_kind == LIKE_GAUSS) return toy_loglike(p, th);
  if (p->relbin) return relbin_loglike_any(p, th);
  return gw_loglike(p, th, nullptr);
}

double logaddexp(double a, double b) {
  if (a == NEG_INF) return b;
  if (b == NEG_INF) return a;
  double m = std::max(a, b);
  return m + std::log1p(std::exp(-std::fabs(a - b)));
}

}  // namespace

extern "C" {

void orc_prior_transform(const orc_problem* p, const double* u, int64_t B, double* theta) {
  for (int64_t i = 0; i < B; ++i) prior_transform(p, u + i * p->ndim, theta + i * p->ndim);
}

void orc_detector_response(const orc_problem* p, int det, double ra, double dec, double psi, double out[3]) {
  detector_response(p, det, ra, dec, psi, &out[0], &out[1], &out[2]);
}

// Intrinsic amplitude and phase on an arbitrary frequency list (for continuity / closed-form pins).
void orc_amp_phase(const orc_problem* p, const double* theta, const double* f, int64_t n, double* amp, double* psi0) {
  Waveform w = make_waveform(p, theta);
  for (int64_t i = 0; i < n; ++i) waveform_amp_phase(w, f[i], &amp[i], &psi0[i]);
}

// PhenomD-form derived quantities: [Frd, Fdamp, Fpeak, t0, C1int, C2int, C1mr, C2mr, M_seconds, eta, 19 Lambda values]
// TaylorF2 phase coefficients phi_k, phi_k^(l) (DESIGN.md A.1) for mass ratio q and aligned spins: accessor for the pin that
// derives them from the PN energy and flux (tests/test_oracle_pn_derivation.py).  They do not depend on the chirp mass.
void orc_taylorf2_coeffs(double q, double chi1, double chi2, double* phi, double* phil) {
  Intrinsic s = make_intrinsic(30.0, q, chi1, chi2);
  taylorf2_coeffs(s, phi, phil);
}

void orc_phenomd_info(const orc_problem* p, const double* theta, double* out) {
  PhenomD m = make_phenomd(p, theta[0], theta[1], theta[2], theta[3]);
  out[0] = m.Frd; out[1] = m.Fdamp; out[2] = m.Fpeak; out[3] = m.t0;
  out[4] = m.C1int; out[5] = m.C2int; out[6] = m.C1mr; out[7] = m.C2mr; out[8] = m.s.M; out[9] = m.s.eta;
  for (int r = 0; r < 19; ++r) out[10 + r] = m.L[r];
}

// Inspiral amplitude PN coefficients A_0..A_6 of the PhenomD-form model (DESIGN.md A.2): accessor for the pin that derives their
// spin-independent parts and A_3 from the PN energy, flux and (2,2)-mode amplitude (tests/test_oracle_pn_derivation.py).
void orc_phenomd_amp_coeffs(const orc_problem* p, const double* theta, double* A) {
  PhenomD m = make_phenomd(p, theta[0], theta[1], theta[2], theta[3]);
  for (int i = 0; i < 7; ++i) A[i] = m.A[i];
}

// Detector-frame waveform h_det(f_k) on the problem's grid: out[n_det][n_freq][2].  Used by tests to inject signals.
void orc_waveform(const orc_problem* p, const double* th, double* out) {
  Waveform w = make_waveform(p, th);
  double ci = std::cos(th[5]);
  for (int det = 0; det < p->n_det; ++det) {
    double fp, fx, dt;
    detector_response(p, det, th[9], th[10], th[6], &fp, &fx, &dt);
    double cre = fp * 0.5 * (1.0 + ci * ci), cim = -fx * ci;
    for (int k = 0; k < p->n_freq; ++k) {
      double f = p->f_min + k * p->df, amp, psi0;
      waveform_amp_phase(w, f, &amp, &psi0);
      double Phi = psi0 + 2.0 * PI * f * (th[8] + dt);
      double c = std::cos(Phi), s = std::sin(Phi);
      out[((size_t)det * p->n_freq + k) * 2] = amp * (cre * c + cim * s);
      out[((size_t)det * p->n_freq + k) * 2 + 1] = amp * (cim * c - cre * s);
    }
  }
}

// Batched GW log-likelihood on physical theta[B,11]; OpenMP over rows (threads<=0 -> all cores).
void orc_gw_loglike(const orc_problem* p, const double* theta, int64_t B, double* logl, double* parts, int threads) {
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 0 ? threads : omp_get_max_threads_safe())
  for (int64_t i = 0; i < B; ++i) logl[i] = gw_loglike(p, theta + i * 11, parts ? parts + i * 2 * p->n_det : nullptr);
}

// Log-likelihood of unit-cube points for whatever like_kind the problem names.
void orc_loglike_u(const orc_problem* p, const double* u, int64_t B, double* logl, int threads) {
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 0 ? threads : omp_get_max_threads_safe())
  for (int64_t i = 0; i < B; ++i) logl[i] = loglike_from_u(p, u + i * p->ndim);
}

// ---------------------------------------------------------------------------------------------
// Acceptance walk (P:96 DE proposal; P:100 fixed walk length; R:L8-L12, R:R RNG contract).
// For each walker slot j = slot0 + row: W proposals, each
//   block0 = Philox(ctr=(0,t,j,stream_id)) -> a, b (distinct survivors), coin
//   block1, block2 -> U1..U4 -> gamma = 2.38/sqrt(2 n_free) * (-0.25 ln(U1 U2 U3 U4))   (P:120 footnote)
//   u' = fma(gamma, U[a]-U[b], u); wrap periodic dims; reject if outside (0,1); else evaluate, accept iff logL' > L*.
// trace (optional): flags[B,W] bit0 oob, bit1 accepted, bit2 evaluated; tlogl[B,W] (NaN when not evaluated).
// ---------------------------------------------------------------------------------------------
void orc_walk(const orc_problem* p, const double* surv_u, int32_t m, double* u, double* logl, int64_t B, double logl_star,
              int32_t W, uint64_t seed, uint32_t stream_id, int64_t slot0, int32_t* n_accept, int32_t* n_eval, int32_t* n_oob,
              uint8_t* tflags, double* tlogl, int threads) {
  const int D = p->ndim;
  const double gscale = 2.38 / std::sqrt(2.0 * n_free_dims(p));
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 0 ? threads : omp_get_max_threads_safe())
  for (int64_t row = 0; row < B; ++row) {
    uint32_t j = (uint32_t)(slot0 + row);
    double cur[16], prop[16];
    for (int d = 0; d < D; ++d) cur[d] = u[row * D + d];
    double curl = logl[row];
    int na = 0, ne = 0, no = 0;
    for (int t = 0; t < W; ++t) {
      uint32_t b0[4], b1[4], b2[4];
      philox_block(seed, 0u, (uint32_t)t, j, stream_id, b0);
      philox_block(seed, 1u, (uint32_t)t, j, stream_id, b1);
      philox_block(seed, 2u, (uint32_t)t, j, stream_id, b2);
      uint32_t a = orc_mulhi32(b0[0], (uint32_t)m);
      uint32_t bp = orc_mulhi32(b0[1], (uint32_t)(m - 1));
      uint32_t b = bp + (bp >= a ? 1u : 0u);
      double gamma;
      if (b0[2] < 0x80000000u) gamma = 1.0;
      else {
        double U1 = orc_u53(b1[0], b1[1]), U2 = orc_u53(b1[2], b1[3]), U3 = orc_u53(b2[0], b2[1]), U4 = orc_u53(b2[2], b2[3]);
        double prod = ((U1 * U2) * U3) * U4;
        gamma = gscale * (-0.25 * std::log(prod));
      }
      bool oob = false;
      for (int d = 0; d < D; ++d) {
        if (p->prior_kind[d] == PRIOR_FIXED) { prop[d] = cur[d]; continue; }
        double diff = surv_u[(size_t)a * D + d] - surv_u[(size_t)b * D + d];
        double x = std::fma(gamma, diff, cur[d]);
        if (p->periodic[d]) x = x - std::floor(x);
        else if (!(x > 0.0 && x < 1.0)) oob = true;
        prop[d] = x;
      }
      uint8_t fl = 0;
      double pl = std::numeric_limits<double>::quiet_NaN();
      if (oob) { ++no; fl |= 1; }
      else {
        pl = loglike_from_u(p, prop);
        ++ne; fl |= 4;
        if (pl > logl_star) {
          for (int d = 0; d < D; ++d) cur[d] = prop[d];
          curl = pl; ++na; fl |= 2;
        }
      }
      if (tflags) tflags[row * W + t] = fl;
      if (tlogl) tlogl[row * W + t] = pl;
    }
    for (int d = 0; d < D; ++d) u[row * D + d] = cur[d];
    logl[row] = curl;
    if (n_accept) n_accept[row] = na;
    if (n_eval) n_eval[row] = ne;
    if (n_oob) n_oob[row] = no;
  }
}

// ---------------------------------------------------------------------------------------------
// Hit-and-run slice sampling inner kernel (the blackjax-ns default the paper builds on, and names as future
// comparison; no formula in the paper: DESIGN.md reading R:L25).  One slice step from x under the constraint
// "inside the unit cube (periodic dims wrap) and logL > L*":
//   direction: z ~ N(0, I) over the free dims (Box-Muller on Philox blocks 0..7: z_2i = sqrt(-2 ln U1) cos(2 pi U2), z_2i+1 = .. sin),
//              dir = Lc z / |z| with Lc a lower-triangular factor given by the caller (Cholesky of the live points' covariance);
//   bracket:   l = -U0, r = l + 1 (U0 from block 8); stepping out: while inside(l) l -= 1 (at most 32 times), same for r;
//   shrinkage: t = l + U_k (r - l) (U_k from block 9 + k/2, first or second pair of words); inside(t) -> move there; else the
//              bracket end on t's side becomes t; at most 64 candidates, then the point stays.
// Every inside() test of an in-cube point is one likelihood evaluation.  trace (optional): per step the number of evaluations
// and the logL after the step.
// ---------------------------------------------------------------------------------------------
void orc_slice_walk(const orc_problem* p, const double* Lc /*[D][D] lower, row-major, free dims only used*/, double* u, double* logl,
                    int64_t B, double logl_star, int32_t S, uint64_t seed, uint32_t stream_id, int64_t slot0, int32_t* n_eval,
                    int32_t* n_oob, int32_t* n_expand, int32_t* n_shrink, int32_t* n_stuck, int32_t* t_evals, double* t_logl,
                    int threads) {
  const int D = p->ndim;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 0 ? threads : omp_get_max_threads_safe())
  for (int64_t row = 0; row < B; ++row) {
    const uint32_t j = (uint32_t)(slot0 + row);
    double x[16], y[16], dir[16], z[16];
    for (int d = 0; d < D; ++d) x[d] = u[row * D + d];
    double xl = logl[row];
    int ne = 0, no = 0, nx = 0, ns = 0, nk = 0;
    int fr[16], nfree = 0;
    for (int d = 0; d < D; ++d)
      if (p->prior_kind[d] != PRIOR_FIXED) fr[nfree++] = d;
    for (int s = 0; s < S; ++s) {
      const int ne0 = ne;
      // direction
      double z2 = 0.0;
      for (int i = 0; 2 * i < nfree; ++i) {
        uint32_t w[4];
        philox_block(seed, (uint32_t)i, (uint32_t)s, j, stream_id, w);
        const double U1 = orc_u53(w[0], w[1]), U2 = orc_u53(w[2], w[3]);
        const double rad = std::sqrt(-2.0 * std::log(U1));
        z[2 * i] = rad * std::cos(2.0 * PI * U2);
        if (2 * i + 1 < nfree) z[2 * i + 1] = rad * std::sin(2.0 * PI * U2);
      }
      for (int a = 0; a < nfree; ++a) z2 += z[a] * z[a];
      const double inv = 1.0 / std::sqrt(z2);
      for (int d = 0; d < D; ++d) dir[d] = 0.0;
      for (int a = 0; a < nfree; ++a) {
        double acc = 0.0;
        for (int b = 0; b <= a; ++b) acc += Lc[(size_t)fr[a] * D + fr[b]] * z[b];
        dir[fr[a]] = acc * inv;
      }
      auto inside = [&](double t, double* lout) -> bool {
        bool oob = false;
        for (int d = 0; d < D; ++d) {
          if (p->prior_kind[d] == PRIOR_FIXED) { y[d] = x[d]; continue; }
          double v = std::fma(t, dir[d], x[d]);
          if (p->periodic[d]) v = v - std::floor(v);
          else if (!(v > 0.0 && v < 1.0)) oob = true;
          y[d] = v;
        }
        if (oob) { ++no; return false; }
        const double l = loglike_from_u(p, y);
        ++ne;
        *lout = l;
        return l > logl_star;
      };
      uint32_t w8[4];
      philox_block(seed, 8u, (uint32_t)s, j, stream_id, w8);
      double l = -orc_u53(w8[0], w8[1]), r = l + 1.0, tmp;
      for (int k = 0; k < 32 && inside(l, &tmp); ++k) { l -= 1.0; ++nx; }
      for (int k = 0; k < 32 && inside(r, &tmp); ++k) { r += 1.0; ++nx; }
      bool moved = false;
      for (int k = 0; k < 64; ++k) {
        uint32_t w[4];
        philox_block(seed, 9u + (uint32_t)(k / 2), (uint32_t)s, j, stream_id, w);
        const double U = (k % 2 == 0) ? orc_u53(w[0], w[1]) : orc_u53(w[2], w[3]);
        const double t = l + U * (r - l);
        double lt;
        if (inside(t, &lt)) {
          for (int d = 0; d < D; ++d) x[d] = y[d];
          xl = lt; moved = true;
          break;
        }
        ++ns;
        if (t < 0.0) l = t; else r = t;
      }
      if (!moved) ++nk;
      if (t_evals) t_evals[row * S + s] = ne - ne0;
      if (t_logl) t_logl[row * S + s] = xl;
    }
    for (int d = 0; d < D; ++d) u[row * D + d] = x[d];
    logl[row] = xl;
    if (n_eval) n_eval[row] = ne;
    if (n_oob) n_oob[row] = no;
    if (n_expand) n_expand[row] = nx;
    if (n_shrink) n_shrink[row] = ns;
    if (n_stuck) n_stuck[row] = nk;
  }
}

// Proposal scale draw exposed for distribution pins: gamma for (seed, t, j, stream_id); returns coin via *is_one.
double orc_gamma_draw(int n_free, uint64_t seed, uint32_t t, uint32_t j, uint32_t stream_id, int32_t m, int32_t* a_out, int32_t* b_out, int32_t* is_one) {
  uint32_t b0[4], b1[4], b2[4];
  philox_block(seed, 0u, t, j, stream_id, b0);
  philox_block(seed, 1u, t, j, stream_id, b1);
  philox_block(seed, 2u, t, j, stream_id, b2);
  uint32_t a = orc_mulhi32(b0[0], (uint32_t)m);
  uint32_t bp = orc_mulhi32(b0[1], (uint32_t)(m - 1));
  *a_out = (int32_t)a;
  *b_out = (int32_t)(bp + (bp >= a ? 1u : 0u));
  *is_one = b0[2] < 0x80000000u;
  double U1 = orc_u53(b1[0], b1[1]), U2 = orc_u53(b1[2], b1[3]), U3 = orc_u53(b2[0], b2[1]), U4 = orc_u53(b2[2], b2[3]);
  double g = 2.38 / std::sqrt(2.0 * n_free) * (-0.25 * std::log(((U1 * U2) * U3) * U4));
  return *is_one ? 1.0 : g;
}

// Initial live points drawn by the library when the caller passes none (tag 2): dim d of point i uses
// Philox(ctr=(d/2, 0, i, 2<<24)) words (0,1) for even d and (2,3) for odd d.
void orc_draw_live(int32_t ndim, int64_t n, uint64_t seed, double* u) {
  for (int64_t i = 0; i < n; ++i)
    for (int d = 0; d < ndim; ++d) {
      uint32_t w[4];
      philox_block(seed, (uint32_t)(d / 2), 0u, (uint32_t)i, 2u << 24, w);
      u[i * ndim + d] = (d & 1) ? orc_u53(w[2], w[3]) : orc_u53(w[0], w[1]);
    }
}

// ---------------------------------------------------------------------------------------------
// Outer nested-sampling state and step (P:74-80 batch deletion; eq. 3-5 saw-tooth volume;
// R:L6, L7, L13-L18).
// ---------------------------------------------------------------------------------------------
struct orc_state {
  orc_problem prob;
  orc_sampler_cfg cfg;
  uint64_t seed;
  int D;
  std::vector<double> u, logl;
  double logx, logz, h, walks, delay;
  int64_t iter, n_eval_total;
  int threads;
  int inner_kind = 0;   // 0 acceptance walk, 1 hit-and-run slice sampling (R:L25)
  int n_slice = 0;      // slice steps per replacement
};

// Lower-triangular factor of the covariance of m points (unit-cube coordinates, free dims; FIXED dims get zero rows), the
// direction factor of the slice kernel inside the sampler (R:L25): mean and covariance by sequential sums over the points in the
// order given, 1/(m-1) normalisation, diagonal times (1 + 1e-12), textbook row-by-row Cholesky.  Lc [D][D] row-major.
void orc_live_cholesky(const orc_problem* p, const double* pts, int32_t m, double* Lc) {
  const int D = p->ndim;
  double mean[16], C[16][16];
  for (int a = 0; a < D; ++a) {
    double acc = 0.0;
    for (int i = 0; i < m; ++i) acc += pts[(size_t)i * D + a];
    mean[a] = acc / m;
  }
  for (int a = 0; a < D; ++a)
    for (int b = 0; b <= a; ++b) {
      double acc = 0.0;
      for (int i = 0; i < m; ++i) acc += (pts[(size_t)i * D + a] - mean[a]) * (pts[(size_t)i * D + b] - mean[b]);
      C[a][b] = acc / (m - 1);
    }
  for (int a = 0; a < D * D; ++a) Lc[a] = 0.0;
  for (int a = 0; a < D; ++a) {
    if (p->prior_kind[a] == PRIOR_FIXED) continue;
    for (int b = 0; b <= a; ++b) {
      if (p->prior_kind[b] == PRIOR_FIXED) continue;
      double sum = (a == b) ? C[a][a] * (1.0 + 1e-12) : C[a][b];
      for (int c = 0; c < b; ++c) sum -= Lc[a * D + c] * Lc[b * D + c];
      Lc[a * D + b] = (a == b) ? std::sqrt(sum) : sum / Lc[b * D + b];
    }
  }
}

void orc_state_set_inner(struct orc_state* s, int32_t kind, int32_t n_slice);

orc_state* orc_state_create(const orc_problem* p, const orc_sampler_cfg* c, const double* live_u, uint64_t seed, int threads) {
  orc_state* s = new orc_state();
  s->prob = *p; s->cfg = *c; s->seed = seed; s->D = p->ndim; s->threads = threads;
  s->u.resize((size_t)c->n_live * s->D);
  s->logl.resize(c->n_live);
  if (live_u) std::memcpy(s->u.data(), live_u, sizeof(double) * s->u.size());
  else orc_draw_live(s->D, c->n_live, seed, s->u.data());
  orc_loglike_u(&s->prob, s->u.data(), c->n_live, s->logl.data(), threads);
  s->logx = 0.0; s->logz = NEG_INF; s->h = 0.0;
  s->walks = c->walks0;
  s->delay = c->delay >= 0.0 ? c->delay : std::max((double)c->n_live / (10.0 * c->n_delete) - 1.0, 0.0);
  s->iter = 0; s->n_eval_total = c->n_live;
  return s;
}

void orc_state_free(orc_state* s) { delete s; }
void orc_state_set_inner(orc_state* s, int32_t kind, int32_t n_slice) { s->inner_kind = kind; s->n_slice = n_slice; }

void orc_state_get_live(const orc_state* s, double* u, double* logl) {
  std::memcpy(u, s->u.data(), sizeof(double) * s->u.size());
  std::memcpy(logl, s->logl.data(), sizeof(double) * s->logl.size());
}

// Stable ascending argsort of logL (ties by lower index, R:L6).
void orc_argsort(const double* x, int64_t n, int32_t* idx) {
  std::vector<int32_t> v(n);
  std::iota(v.begin(), v.end(), 0);
  std::stable_sort(v.begin(), v.end(), [&](int32_t a, int32_t b) { return x[a] < x[b]; });
  std::memcpy(idx, v.data(), sizeof(int32_t) * n);
}

// One dead point through the evidence accumulator (R:L16, L17): n_i live points at the moment of deletion.
void orc_evidence_update(double logl_i, double n_i, double* logx, double* logz, double* h, double* logw_out) {
  double logw = *logx + std::log(-std::expm1(-1.0 / n_i));
  double lw = logl_i + logw;
  double logz_new = logaddexp(*logz, lw);
  double hn = std::exp(lw - logz_new) * logl_i;
  if (*logz != NEG_INF) hn += std::exp(*logz - logz_new) * (*h + *logz);
  hn -= logz_new;
  *h = hn;
  *logz = logz_new;
  *logx -= 1.0 / n_i;
  if (logw_out) *logw_out = logw;
}

// dead (optional): [k, D+3] rows (u.., logL, logw, n_i).
void orc_step(orc_state* s, orc_stats* st, double* dead) {
  const int n = s->cfg.n_live, k = s->cfg.n_delete, D = s->D, m = n - k;
  std::vector<int32_t> order(n);
  orc_argsort(s->logl.data(), n, order.data());
  double lstar = s->logl[order[k - 1]];
  // (2) evidence scan over the k dead points in ascending logL, live count n - i (saw-tooth)
  for (int i = 0; i < k; ++i) {
    int32_t id = order[i];
    double logw;
    orc_evidence_update(s->logl[id], (double)(n - i), &s->logx, &s->logz, &s->h, &logw);
    if (dead) {
      double* row = dead + (size_t)i * (D + 3);
      for (int d = 0; d < D; ++d) row[d] = s->u[(size_t)id * D + d];
      row[D] = s->logl[id]; row[D + 1] = logw; row[D + 2] = (double)(n - i);
    }
  }
  // survivor array in ascending-logL order (the order is part of the contract: a, b index into it)
  std::vector<double> surv((size_t)m * D), survl(m);
  for (int i = 0; i < m; ++i) {
    int32_t id = order[k + i];
    for (int d = 0; d < D; ++d) surv[(size_t)i * D + d] = s->u[(size_t)id * D + d];
    survl[i] = s->logl[id];
  }
  // (3) walk length (R:L12)
  int W = (int)std::floor(s->walks);
  W = std::max(1, std::min(W, s->cfg.maxmcmc));
  // (4) start points (R:L7): uniformly chosen survivor, Philox tag 1
  uint32_t it24 = (uint32_t)(s->iter & 0xFFFFFF);
  std::vector<double> cu((size_t)k * D), cl(k);
  for (int j = 0; j < k; ++j) {
    uint32_t w[4];
    philox_block(s->seed, 0u, 0u, (uint32_t)j, (1u << 24) | it24, w);
    uint32_t sj = orc_mulhi32(w[0], (uint32_t)m);
    for (int d = 0; d < D; ++d) cu[(size_t)j * D + d] = surv[(size_t)sj * D + d];
    cl[j] = survl[sj];
  }
  std::vector<int32_t> na(k), ne(k), no(k);
  const bool slice = s->inner_kind == 1;
  if (slice) {
    // R:L25 inside the sampler: directions from the survivors' covariance, n_slice steps per replacement, no walk-length adaptation
    std::vector<double> Lc((size_t)D * D);
    orc_live_cholesky(&s->prob, surv.data(), m, Lc.data());
    std::vector<int32_t> nk(k);
    W = s->n_slice;
    orc_slice_walk(&s->prob, Lc.data(), cu.data(), cl.data(), k, lstar, W, s->seed, (0u << 24) | it24, 0, ne.data(), no.data(), nullptr,
                   nullptr, nk.data(), nullptr, nullptr, s->threads);
    for (int j = 0; j < k; ++j) na[j] = W - nk[j];      // steps that moved the point
  } else
  orc_walk(&s->prob, surv.data(), m, cu.data(), cl.data(), k, lstar, W, s->seed, (0u << 24) | it24, 0, na.data(), ne.data(), no.data(),
           nullptr, nullptr, s->threads);
  // (5) write back into the dead slots
  for (int j = 0; j < k; ++j) {
    int32_t id = order[j];
    for (int d = 0; d < D; ++d) s->u[(size_t)id * D + d] = cu[(size_t)j * D + d];
    s->logl[id] = cl[j];
  }
  // (6) batch-level walk-length adaptation (R:L13, L14)
  int64_t sa = 0, se = 0, so = 0, stuck = 0;
  int amin = na[0], amax = na[0];
  for (int j = 0; j < k; ++j) {
    sa += na[j]; se += ne[j]; so += no[j]; stuck += (na[j] == 0);
    amin = std::min(amin, na[j]); amax = std::max(amax, na[j]);
  }
  double amean = (double)sa / k;
  double r = std::max(0.5, amean) / W;
  if (!slice) s->walks = std::min((s->walks * s->delay + s->cfg.naccept / r) / (s->delay + 1.0), (double)s->cfg.maxmcmc);
  s->n_eval_total += se;
  // (7) termination quantities (R:L18)
  double lmax = NEG_INF, lse = NEG_INF;
  for (int i = 0; i < n; ++i) { lmax = std::max(lmax, s->logl[i]); }
  {
    long double acc = 0.0L;
    for (int i = 0; i < n; ++i) acc += std::exp((long double)(s->logl[i] - lmax));
    lse = lmax + (double)std::log(acc);
  }
  if (st) {
    st->iteration = s->iter;
    st->logl_star = lstar; st->logx = s->logx; st->logz = s->logz; st->h = s->h;
    st->dlogz = logaddexp(s->logz, lmax + s->logx) - s->logz;
    st->live_frac_log = lse - std::log((double)n) + s->logx - s->logz;
    st->walk_len = W; st->walks_next = s->walks;
    st->accept_mean = amean; st->accept_min = amin; st->accept_max = amax;
    st->n_eval = se; st->n_oob = so; st->n_stuck = stuck; st->n_eval_total = s->n_eval_total;
  }
  s->iter += 1;
}

// Adds the remaining live points (n_i = n, n-1, ..., 1) to a COPY of the accumulators (R:L17).
void orc_finalize(const orc_state* s, double* logz, double* logz_err, double* h) {
  const int n = s->cfg.n_live, k = s->cfg.n_delete;
  std::vector<int32_t> order(n);
  orc_argsort(s->logl.data(), n, order.data());
  double lx = s->logx, lz = s->logz, hh = s->h;
  for (int i = 0; i < n; ++i) orc_evidence_update(s->logl[order[i]], (double)(n - i), &lx, &lz, &hh, nullptr);
  double neff = k / std::log((double)n / (double)(n - k));
  *logz = lz; *h = hh; *logz_err = std::sqrt(std::max(hh, 0.0) / neff);
}

// Runs steps until the termination rule fires (kind 0: dlogz < tol; kind 1: live fraction < tol) or max_iter.
// dead_sink (optional): [max_iter*k, D+3]. Returns the number of steps done.
int64_t orc_run(orc_state* s, int32_t term_kind, double tol, int64_t max_iter, orc_stats* last, double* dead_sink) {
  const int k = s->cfg.n_delete, D = s->D;
  int64_t it = 0;
  orc_stats st;
  std::memset(&st, 0, sizeof(st));
  while (it < max_iter) {
    orc_step(s, &st, dead_sink ? dead_sink + (size_t)it * k * (D + 3) : nullptr);
    ++it;
    if (term_kind == 0 && st.dlogz < tol) break;
    if (term_kind == 1 && st.live_frac_log < std::log(tol)) break;
  }
  if (last) *last = st;
  return it;
}

double orc_neff(int32_t n, int32_t k) { return k / std::log((double)n / (double)(n - k)); }

}  // extern "C"

// =============================================================================================
// Relative binning ("heterodyned likelihood"; P:155 says the paper does NOT use it, P:172, P:338 and P:503 name it as the remedy
// for the bins x samples cost).  The paper gives no formula: DESIGN.md reading R:L24 restates the published scheme
// (Zackay, Dai & Venumadhav 2018, as in bilby's relative-binning likelihood) and this is that reading, step by step:
//  1. fiducial theta0 -> h0_d(f_k) on the full grid;
//  2. bin edges: Delta(f) = 2 pi chi sum_gamma sgn(gamma) (f / f*_gamma)^gamma, gamma in {-5/3, -2/3, 1, 5/3, 7/3}, f*_gamma = f_min
//     for gamma < 0 and f_max for gamma > 0 (monotone increasing); N_b = max(1, floor((Delta(f_max) - Delta(f_min)) / eps)) bins
//     equally spaced in Delta; edge i = first grid index with Delta(f_k) - Delta(f_0) >= i (Delta_tot / N_b); edge N_b = N_f - 1;
//     duplicates removed;
//  3. summary data per detector and bin b (grid indices [e_b, e_b+1), the last bin also holds e_Nb), f_m = (f_lo + f_hi)/2:
//     A0 = 4 df sum d conj(h0)/S, A1 = 4 df sum d conj(h0)/S (f - f_m), B0 = 4 df sum |h0|^2/S, B1 = 4 df sum |h0|^2/S (f - f_m);
//  4. for theta: r = h(f_e; theta)/h0(f_e) at the edges, per bin r0 = (r_lo + r_hi)/2, r1 = (r_hi - r_lo)/(f_hi - f_lo);
//     <d,h> ~ Re sum_b [A0 conj(r0) + A1 conj(r1)],  <h,h> ~ sum_b [B0 |r0|^2 + 2 B1 Re(r0 conj(r1))].
// It is an approximation: exact when r is constant (same waveform up to amplitude/phase: the d_L and phase directions) and second
// order in the bin width otherwise.  Pins: tests/test_oracle_relbin.py.
// =============================================================================================
namespace {

struct RelBin {
  int n_det = 0, n_bins = 0;
  std::vector<int> edge;            // [n_bins + 1] grid indices
  std::vector<double> fe;           // [n_bins + 1]
  std::vector<double> h0;           // [n_det][n_bins + 1][2]
  std::vector<double> A0, A1;       // [n_det][n_bins][2]
  std::vector<double> B0, B1;       // [n_det][n_bins]
};

double relbin_delta(double f, double f_lo, double f_hi, double chi) {
  const double g[5] = {-5.0 / 3.0, -2.0 / 3.0, 1.0, 5.0 / 3.0, 7.0 / 3.0};
  double s = 0.0;
  for (int i = 0; i < 5; ++i) s += (g[i] < 0.0) ? -std::pow(f / f_lo, g[i]) : std::pow(f / f_hi, g[i]);
  return 2.0 * PI * chi * s;
}

// detector-frame waveform of theta at one frequency for every detector: out[n_det][2]
void waveform_at(const orc_problem* p, const Waveform& w, const double* th, const double* fp, const double* fx, const double* dt,
                 double f, double* out) {
  double amp, psi0;
  waveform_amp_phase(w, f, &amp, &psi0);
  const double ci = std::cos(th[5]);
  for (int det = 0; det < p->n_det; ++det) {
    double cre = fp[det] * 0.5 * (1.0 + ci * ci), cim = -fx[det] * ci;
    double Phi = psi0 + 2.0 * PI * f * (th[8] + dt[det]);
    double c = std::cos(Phi), s_ = std::sin(Phi);
    out[2 * det] = amp * (cre * c + cim * s_);
    out[2 * det + 1] = amp * (cim * c - cre * s_);
  }
}

}  // namespace

extern "C" {

void* orc_relbin_create(const orc_problem* p, const double* theta0, double chi, double eps) {
  if (!theta_physical(theta0) || !(eps > 0.0) || !(chi > 0.0) || p->n_freq < 2) return nullptr;
  RelBin* rb = new RelBin();
  const int nf = p->n_freq, nd = p->n_det;
  rb->n_det = nd;
  const double f_lo = p->f_min, f_hi = p->f_min + (nf - 1) * p->df;
  const double d0 = relbin_delta(f_lo, f_lo, f_hi, chi), dtot = relbin_delta(f_hi, f_lo, f_hi, chi) - d0;
  const int nb_req = std::max(1, (int)std::floor(dtot / eps));
  // step 2: edges
  std::vector<int> e;
  e.push_back(0);
  int k = 0;
  for (int i = 1; i < nb_req; ++i) {
    const double target = i * (dtot / nb_req);
    while (k < nf - 1 && relbin_delta(p->f_min + k * p->df, f_lo, f_hi, chi) - d0 < target) ++k;
    if (k > e.back() && k < nf - 1) e.push_back(k);
  }
  e.push_back(nf - 1);
  rb->edge = e;
  rb->n_bins = (int)e.size() - 1;
  const int nb = rb->n_bins;
  rb->fe.resize(nb + 1);
  for (int i = 0; i <= nb; ++i) rb->fe[i] = p->f_min + e[i] * p->df;
  // step 1: fiducial waveform on the grid
  Waveform w0 = make_waveform(p, theta0);
  std::vector<double> fp(nd), fx(nd), dt(nd);
  for (int det = 0; det < nd; ++det) detector_response(p, det, theta0[9], theta0[10], theta0[6], &fp[det], &fx[det], &dt[det]);
  std::vector<double> hk(2 * nd);
  rb->h0.assign((size_t)nd * (nb + 1) * 2, 0.0);
  for (int i = 0; i <= nb; ++i) {
    waveform_at(p, w0, theta0, fp.data(), fx.data(), dt.data(), rb->fe[i], hk.data());
    for (int det = 0; det < nd; ++det) {
      rb->h0[((size_t)det * (nb + 1) + i) * 2] = hk[2 * det];
      rb->h0[((size_t)det * (nb + 1) + i) * 2 + 1] = hk[2 * det + 1];
    }
  }
  // step 3: summary data
  rb->A0.assign((size_t)nd * nb * 2, 0.0); rb->A1.assign((size_t)nd * nb * 2, 0.0);
  rb->B0.assign((size_t)nd * nb, 0.0); rb->B1.assign((size_t)nd * nb, 0.0);
  for (int b = 0; b < nb; ++b) {
    const int k_lo = e[b], k_hi = (b == nb - 1) ? e[b + 1] + 1 : e[b + 1];
    const double fm = 0.5 * (rb->fe[b] + rb->fe[b + 1]);
    std::vector<long double> a0r(nd, 0.0L), a0i(nd, 0.0L), a1r(nd, 0.0L), a1i(nd, 0.0L), b0(nd, 0.0L), b1(nd, 0.0L);
    for (int kk = k_lo; kk < k_hi; ++kk) {
      const double f = p->f_min + kk * p->df;
      waveform_at(p, w0, theta0, fp.data(), fx.data(), dt.data(), f, hk.data());
      for (int det = 0; det < nd; ++det) {
        const double dr = p->strain[((size_t)det * nf + kk) * 2], di = p->strain[((size_t)det * nf + kk) * 2 + 1];
        const double S = p->psd[(size_t)det * nf + kk];
        const double hr = hk[2 * det], hi = hk[2 * det + 1];
        // d conj(h0) / S
        const double zr = (dr * hr + di * hi) / S, zi = (di * hr - dr * hi) / S;
        const double h2 = (hr * hr + hi * hi) / S;
        a0r[det] += zr; a0i[det] += zi; a1r[det] += zr * (f - fm); a1i[det] += zi * (f - fm);
        b0[det] += h2; b1[det] += h2 * (f - fm);
      }
    }
    for (int det = 0; det < nd; ++det) {
      const size_t ib = (size_t)det * nb + b;
      rb->A0[2 * ib] = (double)(4.0L * p->df * a0r[det]); rb->A0[2 * ib + 1] = (double)(4.0L * p->df * a0i[det]);
      rb->A1[2 * ib] = (double)(4.0L * p->df * a1r[det]); rb->A1[2 * ib + 1] = (double)(4.0L * p->df * a1i[det]);
      rb->B0[ib] = (double)(4.0L * p->df * b0[det]); rb->B1[ib] = (double)(4.0L * p->df * b1[det]);
    }
  }
  return rb;
}

void orc_relbin_free(void* h) { delete static_cast<RelBin*>(h); }
int32_t orc_relbin_nbins(const void* h) { return static_cast<const RelBin*>(h)->n_bins; }
void orc_relbin_edges(const void* h, int32_t* out) {
  const RelBin* rb = static_cast<const RelBin*>(h);
  for (int i = 0; i <= rb->n_bins; ++i) out[i] = rb->edge[i];
}
// summary data: A0, A1 [n_det][n_bins][2]; B0, B1 [n_det][n_bins]
void orc_relbin_summary(const void* h, double* A0, double* A1, double* B0, double* B1) {
  const RelBin* rb = static_cast<const RelBin*>(h);
  std::copy(rb->A0.begin(), rb->A0.end(), A0); std::copy(rb->A1.begin(), rb->A1.end(), A1);
  std::copy(rb->B0.begin(), rb->B0.end(), B0); std::copy(rb->B1.begin(), rb->B1.end(), B1);
}

static double relbin_loglike_one(const orc_problem* p, const RelBin* rb, const double* th, double* parts) {
  const int nd = p->n_det, nb = rb->n_bins;
  if (!theta_physical(th)) {
    if (parts) for (int i = 0; i < 2 * nd; ++i) parts[i] = std::numeric_limits<double>::quiet_NaN();
    return NEG_INF;
  }
  Waveform w = make_waveform(p, th);
  std::vector<double> fp(nd), fx(nd), dt(nd);
  for (int det = 0; det < nd; ++det) detector_response(p, det, th[9], th[10], th[6], &fp[det], &fx[det], &dt[det]);
  // step 4: ratios at the edges
  std::vector<double> r((size_t)nd * (nb + 1) * 2), hk(2 * nd);
  for (int i = 0; i <= nb; ++i) {
    waveform_at(p, w, th, fp.data(), fx.data(), dt.data(), rb->fe[i], hk.data());
    for (int det = 0; det < nd; ++det) {
      const double ar = hk[2 * det], ai = hk[2 * det + 1];
      const double br = rb->h0[((size_t)det * (nb + 1) + i) * 2], bi = rb->h0[((size_t)det * (nb + 1) + i) * 2 + 1];
      const double den = br * br + bi * bi;
      r[((size_t)det * (nb + 1) + i) * 2] = (ar * br + ai * bi) / den;
      r[((size_t)det * (nb + 1) + i) * 2 + 1] = (ai * br - ar * bi) / den;
    }
  }
  double logl = 0.0;
  for (int det = 0; det < nd; ++det) {
    long double dh = 0.0L, hh = 0.0L;
    for (int b = 0; b < nb; ++b) {
      const double* rl = &r[((size_t)det * (nb + 1) + b) * 2];
      const double* rh = rl + 2;
      const double w_ = rb->fe[b + 1] - rb->fe[b];
      const double r0r = 0.5 * (rl[0] + rh[0]), r0i = 0.5 * (rl[1] + rh[1]);
      const double r1r = (rh[0] - rl[0]) / w_, r1i = (rh[1] - rl[1]) / w_;
      const size_t ib = (size_t)det * nb + b;
      // Re(A conj(r)) = Ar rr + Ai ri
      dh += (long double)(rb->A0[2 * ib] * r0r + rb->A0[2 * ib + 1] * r0i + rb->A1[2 * ib] * r1r + rb->A1[2 * ib + 1] * r1i);
      hh += (long double)(rb->B0[ib] * (r0r * r0r + r0i * r0i) + 2.0 * rb->B1[ib] * (r0r * r1r + r0i * r1i));
    }
    if (parts) { parts[2 * det] = (double)dh; parts[2 * det + 1] = (double)hh; }
    logl += (double)dh - 0.5 * (double)hh;
  }
  return logl;
}

}  // extern "C"
namespace {
double relbin_loglike_any(const orc_problem* p, const double* th) {
  return relbin_loglike_one(p, static_cast<const RelBin*>(p->relbin), th, nullptr);
}
}  // namespace
extern "C" {

void orc_relbin_loglike(const orc_problem* p, const void* h, const double* theta, int64_t B, double* logl, double* parts, int threads) {
  const RelBin* rb = static_cast<const RelBin*>(h);
#pragma omp parallel for schedule(dynamic, 4) num_threads(threads > 0 ? threads : omp_get_max_threads_safe())
  for (int64_t i = 0; i < B; ++i) logl[i] = relbin_loglike_one(p, rb, theta + i * 11, parts ? parts + i * 2 * p->n_det : nullptr);
}

}  // extern "C"
