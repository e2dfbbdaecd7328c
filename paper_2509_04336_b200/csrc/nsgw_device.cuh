// nsgw_device.cuh -- device-side building blocks of libnsgw (sm_100a, fp64 ALU path; no tensor cores: the
// per-(particle, bin) work is a transcendental-heavy map + reduction, not a dense contraction).
//
// Contents: Philox4x32-10 and the uniform/index draws of the RNG contract, prior transforms
// (Table 1), quarter-turn sincos, detector response (DESIGN.md A.3), per-particle waveform set-up
// (DESIGN.md A.1/A.2) and the per-bin evaluation used by both the likelihood kernel and the walk kernel.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace nsgw {

constexpr double kPi = 3.14159265358979323846;
constexpr double kGMsunS = 4.925490947641267e-6;                     // G Msun / c^3 [s]
constexpr double kMpcS = 3.0856775814913673e22 / 299792458.0;        // 1 Mpc / c [s]
constexpr double kC = 299792458.0;
constexpr double kEulerGamma = 0.5772156649015329;
constexpr double kQT = 2.0 / kPi;                                    // radians -> quarter turns

constexpr int kMaxDim = 16;
constexpr int kMaxDet = 4;

// Device copy of the problem description (lives in global memory, one per handle).
struct DevCfg {
  int like_kind, ndim, n_free, n_det, n_freq;
  int prior_kind[kMaxDim];
  int periodic[kMaxDim];
  double prior_lo[kMaxDim], prior_hi[kMaxDim];
  double f_min, df, gmst;
  double det_vertex[kMaxDet][3];
  double det_D[kMaxDet][6];  // detector tensor (xx, xy, xz, yy, yz, zz) of D = (x x^T - y y^T)/2
  double toy_mean[kMaxDim];
  double toy_prec[kMaxDim * kMaxDim];
  double toy_lognorm;
  double table[19][11];
  double i73[kMaxDet];       // 4 df sum_k f_k^-7/3 / S_k  (parameter-independent part of <h,h> for a power-law amplitude)
};

// Per-frequency tables built once by ns_init (length n_freq).  The ten basis functions of the PN phase are stored as
// double2 pairs so that a thread fetches them with coalesced 128-bit loads and the bin loop has no pow/log/cbrt and no
// per-bin products.
struct Tables {
  const double2* t01;   // (f^-5/3, f^-1)
  const double2* t23;   // (f^-2/3, f^-1/3)
  const double2* t45;   // (ln f, f^1/3)
  const double2* t67;   // (f^1/3 ln f, f^2/3)
  const double* f;      // f_k
  const double* f34;    // f^3/4
  const double2* wd[kMaxDet];  // 4 df d_k f_k^-7/6 / S_k   (complex)
  const double* ws[kMaxDet];   // 4 df f_k^-7/3 / S_k
  const struct MathTables* mt; // sin/cos, 2^(j/64), atan(j/32) tables (built once per handle; CTAs copy them to shared memory)
  const double2* sc9;          // exp(2 pi i k / 512), the lane-per-row kernels' sin/cos table (sincos_lut9)
  const double2* sc11;         // exp(2 pi i k / 2048) (sincos_lut11)
};

// ------------------------------------------------------------------------------------------------------
// Philox4x32-10, counter (c0 block, c1 step, c2 slot, c3 stream id), key = seed.
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                                              uint32_t (&out)[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Uniform on the half-offset 2^-52 grid, strictly inside (0,1).
__device__ __forceinline__ double u01(uint32_t hi, uint32_t lo) {
  return ((double)(hi >> 6) * 67108864.0 + (double)(lo >> 6) + 0.5) * (1.0 / 4503599627370496.0);
}

// ------------------------------------------------------------------------------------------------------
// sin/cos of an angle given in quarter turns (q = angle * 2/pi).  Exact reduction: k = rint(q), r = q - k in
// [-1/2, 1/2]; polynomials in r^2 fitted to sin(pi r/2)/r and cos(pi r/2) (max error 5e-18 / 3e-20).  The coefficients
// live in constant memory so that every DFMA takes its constant as a c[bank][offset] operand (a literal would cost two
// UMOVs per use), and the quadrant fix-up is integer work on the sign/high words (no FP64 pipe slots).
// ------------------------------------------------------------------------------------------------------
__constant__ double kSinQ[7] = {1.5707963267948966143, -0.64596409750624431654, 0.079692626246043040805, -0.0046817541323416188617,
                                0.00016044115074714990863, -3.5986433706134925899e-6, 5.633936132273839028e-8};
__constant__ double kCosQ[8] = {1.0, -1.2337005501361698118, 0.25366950790104670948, -0.020863480763311218307,
                                0.00091926027418326090632, -0.000025202036771077321298, 4.710609744708126973e-7,
                                -6.3212589210323875261e-9};

__device__ __forceinline__ void sincos_qt(double q, double& s, double& c) {
  const double magic = 6755399441055744.0;  // 1.5 * 2^52
  double kk = q + magic;
  const int ki = __double2loint(kk);
  kk -= magic;
  const double r = q - kk;
  const double z = r * r;
  double ps = kSinQ[6];
  double pc = kCosQ[7];
  pc = fma(pc, z, kCosQ[6]);
  ps = fma(ps, z, kSinQ[5]);
  pc = fma(pc, z, kCosQ[5]);
  ps = fma(ps, z, kSinQ[4]);
  pc = fma(pc, z, kCosQ[4]);
  ps = fma(ps, z, kSinQ[3]);
  pc = fma(pc, z, kCosQ[3]);
  ps = fma(ps, z, kSinQ[2]);
  pc = fma(pc, z, kCosQ[2]);
  ps = fma(ps, z, kSinQ[1]);
  pc = fma(pc, z, kCosQ[1]);
  ps = fma(ps, z, kSinQ[0]);
  pc = fma(pc, z, kCosQ[0]);
  ps *= r;
  // quadrant: k odd swaps; sin is negated for k = 2, 3 (mod 4), cos for k = 1, 2
  const int slo = __double2loint(ps), shi = __double2hiint(ps), clo = __double2loint(pc), chi = __double2hiint(pc);
  const bool sw = (ki & 1) != 0;
  const int s_lo = sw ? clo : slo, c_lo = sw ? slo : clo;
  int s_hi = sw ? chi : shi, c_hi = sw ? shi : chi;
  s_hi ^= (ki & 2) << 30;
  c_hi ^= ((ki + 1) & 2) << 30;
  s = __hiloint2double(s_hi, s_lo);
  c = __hiloint2double(c_hi, c_lo);
}

// Table-driven variant for the hot loops (sincos_lut): the angle is given in units of 1/256 turn (u = 64 q), k = rint(u) selects
// exp(2 pi i k / 256) from a 256-entry table in shared memory (MathTables::sc, built with sincos_qt on exact arguments) and the remainder
// |r| <= 1/2 unit (|alpha| <= pi/256) needs three-term polynomials (truncation 8e-18 / 1e-20).  Compared with sincos_qt it
// trades the quadrant selects (10 ALU instructions) and 8 FMAs for one LDS.128 and a complex product: 14 FP64 instructions
// instead of 18, 3 integer instructions instead of 10.
// ------------------------------------------------------------------------------------------------------
// Polynomial / reduction constants of the table-driven functions, in constant memory for the same reason as kSinQ/kCosQ.
// kLutC: sin (h, -h^3/6, h^5/120) and cos (-h^2/2, h^4/24, -h^6/720) Taylor coefficients for h = 2 pi / 256.
// kExpC: 64/ln2, ln2/64 (hi, lo), 1/120, 1/24, 1/6.   kAtanC: 1/9, -1/7, 1/5, -1/3.
__constant__ double kLutC[6] = {0.02454369260617026, -2.464157476448998e-06, 7.421954185344934e-11,
                                -0.0003011964233730883, 1.511988090879011e-08, -3.0360360343697477e-13};
__constant__ double kExpC[6] = {92.33248261689366, -0.010830424696905538, 6.563929801064195e-13, 1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0};
__constant__ double kAtanC[4] = {1.0 / 9.0, -1.0 / 7.0, 0.2, -1.0 / 3.0};

// Shared-memory tables of the hot loops (4.9 KB per CTA), built once per CTA.
struct MathTables {
  double2 sc[256];   // exp(2 pi i k / 256) = (cos, sin)
  double e2[64];     // 2^(j/64)
  double at[34];     // atan(j/32), j = 0..32 (+ pad)
};

__device__ __forceinline__ void build_math_tables(MathTables* mt, int tid, int nthreads) {
  for (int i = tid; i < 256; i += nthreads) {
    double s, c;
    sincos_qt(i * (1.0 / 64.0), s, c);
    mt->sc[i] = make_double2(c, s);
  }
  for (int i = tid; i < 64; i += nthreads) mt->e2[i] = exp2(i * (1.0 / 64.0));
  for (int i = tid; i < 34; i += nthreads) mt->at[i] = atan(i * (1.0 / 32.0));
}

// The exp / atan part alone (784 bytes), for kernels that take their sin/cos from the 512-entry table (k_pd_lp).
struct MathTablesEA {
  double e2[64];
  double at[34];
};
__device__ __forceinline__ void load_math_tables_ea(MathTablesEA* dst, const MathTables* __restrict__ src, int tid, int nthreads) {
  for (int i = tid; i < 64; i += nthreads) dst->e2[i] = __ldg(src->e2 + i);
  for (int i = tid; i < 34; i += nthreads) dst->at[i] = __ldg(src->at + i);
}

// CTA-wide copy of the handle's tables into shared memory (617 doubles).
__device__ __forceinline__ void load_math_tables(MathTables* dst, const MathTables* __restrict__ src, int tid, int nthreads) {
  static_assert(sizeof(MathTables) % sizeof(double) == 0, "MathTables is an array of doubles");
  double* d = reinterpret_cast<double*>(dst);
  const double* g = reinterpret_cast<const double*>(src);
  for (int i = tid; i < (int)(sizeof(MathTables) / sizeof(double)); i += nthreads) d[i] = __ldg(g + i);
}

// CVT = true reduces with F2I / I2F (conversion pipe, off the FP64 pipe: measured +3 % in k_bins_lp, whose loop has no other
// conversion-pipe work) instead of the three-add magic-number form (better where MUFU reciprocals already load that pipe).
template <bool CVT = false>
__device__ __forceinline__ void sincos_lut(double u, const MathTables* mt, double& s, double& c) {
  int ki;
  double r;
  if (CVT) {
    ki = __double2int_rn(u);
    r = u - (double)ki;                        // exact: |u - k| <= 1/2 and |u| < 2^31
  } else {
    const double magic = 6755399441055744.0;  // 1.5 * 2^52
    double kk = u + magic;
    ki = __double2loint(kk);
    kk -= magic;
    r = u - kk;
  }
  const double z = r * r;
  const double2 T = mt->sc[ki & 255];
  double ps = fma(z, kLutC[2], kLutC[1]);
  double pc = fma(z, kLutC[5], kLutC[4]);
  ps = fma(ps, z, kLutC[0]);
  pc = fma(pc, z, kLutC[3]);
  ps *= r;
  pc = fma(pc, z, 1.0);
  c = fma(T.x, pc, -(T.y * ps));
  s = fma(T.y, pc, T.x * ps);
}

// sincos_lut with a 512-entry table and the angle in units of 1/512 turn (u = 128 q): the remainder |r| <= 1/2 unit is |alpha| <= pi/512,
// where sin alpha = alpha - alpha^3/6 (truncation 7e-14) and cos alpha = 1 - alpha^2/2 + alpha^4/24 (7e-17): 10 FP64 instructions
// against sincos_lut's 12, for 8 KB of shared memory instead of 4.  Used by the lane-per-row kernels (k_bins_lp, k_pd_lp).
constexpr int kSc9N = 512;
__constant__ double kLut9C[4] = {0.012271846303085129838, -3.0801968455612480815e-7, -0.000075299105843272084189, 9.4499255679938202216e-10};
__device__ __forceinline__ void build_sc9(double2* sc9, int tid, int nthreads) {
  for (int i = tid; i < kSc9N; i += nthreads) {
    double s, c;
    sincos_qt(i * (1.0 / 128.0), s, c);
    sc9[i] = make_double2(c, s);
  }
}
__device__ __forceinline__ void load_sc9(double2* dst, const double2* __restrict__ src, int tid, int nthreads) {
  const double* g = reinterpret_cast<const double*>(src);
  double* d = reinterpret_cast<double*>(dst);
  for (int i = tid; i < 2 * kSc9N; i += nthreads) d[i] = __ldg(g + i);
}
__device__ __forceinline__ void sincos_lut9(double u, const double2* sc9, double& s, double& c) {
  const int ki = __double2int_rn(u);
  const double r = u - (double)ki;             // exact: |u - k| <= 1/2 and |u| < 2^31
  const double z = r * r;
  const double2 T = sc9[ki & (kSc9N - 1)];
  double ps = fma(z, kLut9C[1], kLut9C[0]);
  double pc = fma(z, kLut9C[3], kLut9C[2]);
  ps *= r;
  pc = fma(pc, z, 1.0);
  c = fma(T.x, pc, -(T.y * ps));
  s = fma(T.y, pc, T.x * ps);
}

// The same with 2048 entries and the angle in units of 1/2048 turn (u = 512 q): |alpha| <= pi/2048, sin alpha = alpha - alpha^3/6
// (7e-17), cos alpha = 1 - alpha^2/2 (2.3e-13): 8 FP64 instructions, 32 KB of shared memory.
constexpr int kSc11N = 2048;
__constant__ double kLut11C[3] = {0.0030679615757712824594, -4.8128075711894501273e-9, -4.7061941152045052618e-6};
__device__ __forceinline__ void build_sc11(double2* sc, int tid, int nthreads) {
  for (int i = tid; i < kSc11N; i += nthreads) {
    double s, c;
    sincos_qt(i * (1.0 / 512.0), s, c);
    sc[i] = make_double2(c, s);
  }
}
__device__ __forceinline__ void sincos_lut11(double u, const double2* sc, double& s, double& c) {
  const int ki = __double2int_rn(u);
  const double r = u - (double)ki;
  const double z = r * r;
  const double2 T = sc[ki & (kSc11N - 1)];
  const double ps = fma(z, kLut11C[1], kLut11C[0]) * r;
  const double pc = fma(z, kLut11C[2], 1.0);
  c = fma(T.x, pc, -(T.y * ps));
  s = fma(T.y, pc, T.x * ps);
}

// Programmatic dependent launch (a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may start while the
// kernel before it on the stream still runs): pdl_wait() returns once that kernel has completed and its writes are visible -- everything
// it produced is read after this (a no-op in a kernel launched the ordinary way).  The kernels here never signal early
// (griddepcontrol.launch_dependents): the next kernel's CTAs then become resident as this one's exit, which hides the launch latency;
// signalling at the start of k_wl_head and k_pd_lp, or after k_wl_head's proposals, made the config-3 run 25 % and 4 % SLOWER (the early
// CTAs of the persistent sweep land where there is room and wait there).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// 1/d for finite normal d well inside the exponent range (no special cases): MUFU.RCP64H seed (>= 20 bits) and two Newton
// steps (relative error 2^-20 -> 2^-40 -> 2^-80, i.e. rounding-limited).  The hot loops only divide by sums of squares of
// O(1..1e6) magnitude.
__device__ __forceinline__ double rcp_nr(double d) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
  double e = fma(-d, y, 1.0);
  y = fma(y, e, y);
  e = fma(-d, y, 1.0);
  y = fma(y, e, y);
  return y;
}

// One Newton step only: relative error <= (seed error)^2 ~ 2^-40 -- for quantities that enter logL through a smooth factor
// (a 1e-12 relative error of the amplitude or of the small remainder t of atan_tab is 1e-12 of that bin's term).
__device__ __forceinline__ double rcp_nr1(double d) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
  const double e = fma(-d, y, 1.0);
  return fma(y, e, y);
}

// exp(x) for |x| <= 700: n = rint(64 x / ln 2), r = x - n ln2/64 (two-term Cody-Waite, |r| <= 0.0055), degree-5 Taylor
// (truncation 3.4e-17 relative), 2^(n/64) from the table and an exponent-field add.
template <class MT /* has e2[64] */>
__device__ __forceinline__ double exp_tab(double x, const MT* mt) {
  const double magic = 6755399441055744.0;
  double t = fma(x, kExpC[0], magic);
  const int n = __double2loint(t);
  t -= magic;
  double r = fma(t, kExpC[1], x);
  r = fma(t, kExpC[2], r);
  double p = fma(r, kExpC[3], kExpC[4]);
  p = fma(p, r, kExpC[5]);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);
  const double v = mt->e2[n & 63] * p;
  return __hiloint2double(__double2hiint(v) + ((n >> 6) << 20), __double2loint(v));
}

// atan(y), any finite y: |y| >= 1 goes through atan(y) = sgn(y) pi/2 + atan(-1/y) written as the fraction n/d = -1/y (no
// division); a 20-bit estimate of n/d picks the table point c = j/32, and atan(n/d) = atan(c) + atan((n - c d)/(d + c n))
// with |t| <= 1/64 + 2^-19, so five odd Taylor terms suffice (t^11/11 < 1.3e-21).  One full reciprocal (d + c n >= 1 in
// magnitude by construction).
template <class MT /* has at[34] */>
__device__ __forceinline__ double atan_tab(double y, const MT* mt) {
  const int hi = __double2hiint(y);
  const bool big = (hi & 0x7fffffff) >= 0x3ff00000;      // |y| >= 1
  const double n = big ? -1.0 : y;
  const double d = big ? y : 1.0;
  const double base = big ? __hiloint2double((hi & 0x80000000) | 0x3ff921fb, 0x54442d18) : 0.0;   // sgn(y) pi/2
  double r0;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r0) : "d"(d));
  const double magic = 6755399441055744.0;
  double jq = fma(n * r0, 32.0, magic);                   // j = rint(32 n/d), |j| <= 32
  const int j = __double2loint(jq);
  jq -= magic;
  const double c = jq * (1.0 / 32.0);
  const double num = fma(-c, d, n), den = fma(c, n, d);
  const double t = num * rcp_nr1(den);
  const double z = t * t;
  double p = fma(z, kAtanC[0], kAtanC[1]);
  p = fma(p, z, kAtanC[2]);
  p = fma(p, z, kAtanC[3]);
  const double at = fma(t * z, p, t);
  const int ja = j < 0 ? -j : j;
  const double tj = mt->at[ja];
  return base + ((j < 0 ? -tj : tj) + at);
}

// ------------------------------------------------------------------------------------------------------
// Prior transform of one coordinate (Table 1; d_L^2 power law P:182).
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double prior_transform_dim(int kind, double lo, double hi, double u) {
  if (kind == 0) return lo + (hi - lo) * u;
  if (kind == 1) { double a3 = lo * lo * lo, b3 = hi * hi * hi; return cbrt(a3 + u * (b3 - a3)); }
  if (kind == 2) { double cl = cos(lo), ch = cos(hi); return acos(cl - u * (cl - ch)); }
  if (kind == 3) { double sl = sin(lo), sh = sin(hi); return asin(sl + u * (sh - sl)); }
  return lo;
}

// ------------------------------------------------------------------------------------------------------
// Coefficient block of one particle (doubles).  Written by setup_particle, read by the bin loop.
// ------------------------------------------------------------------------------------------------------
enum {
  CB_VALID = 0,
  CB_DET = 1,        // per detector, stride 4: Cr, Ci (A0 * C_det), dtq (-4 (dt_det - dt_0): quarter turns per Hz relative to
                     // detector 0, whose delay is folded into the f coefficient of the common phase), c2 (|A0 C_det|^2)
  CB_PH = 17,        // TaylorF2 / inspiral phase: y5 y3 y2 y 1 L x xL x2 f | fx fx2 ff   (13)
  CB_PB = 30,        // intermediate phase: 1 L f f^-3                                   (4)
  CB_PM = 34,        // merger-ringdown phase: 1 f 1/f f^3/4 | atan coefficient, f0, 1/fd  (7)
  CB_FP1 = 41, CB_FP2 = 42, CB_FA1 = 43, CB_FA2 = 44,   // region boundaries [Hz]
  CB_AI = 45,        // inspiral amplitude: degree-9 polynomial in x = f^1/3              (10)
  CB_AH = 55,        // intermediate amplitude: f1, 1/(f3-f1), quartic h0..h4             (7)
  CB_AM = 62,        // merger-ringdown amplitude: f_rd, g1, wh^2, -gamma2/wh             (4)
  CB_FMR = 66,       // PhenomD-form: max(CB_FP2, CB_FA2) [Hz]: from here up both phase and amplitude are merger-ringdown
  CB_SIZE = 68
};

// First bin of the branch-free merger-ringdown loops for a region boundary fs [Hz]: every bin k >= k_mr has f_k >= fs (two bins of
// margin against the rounding of f_k); the bins below go through the general (piecewise) evaluation.
__device__ __forceinline__ int mr_first_bin(double fs, double f_min, double df, int nf) {
  const double ks = (fs - f_min) / df + 2.0;
  if (!(ks < (double)nf)) return nf;
  return (int)fmax(ks, 0.0) + 1;
}

struct DetResp { double fp, fx, dt; };

__device__ __forceinline__ DetResp detector_response(const DevCfg& cfg, int det, double sg, double cg, double sd, double cd,
                                                     double sp, double cp) {
  // polarisation basis X, Y and propagation direction n (DESIGN.md A.3), g = gmst - ra
  double X0 = -cp * sg - sp * cg * sd, X1 = -cp * cg + sp * sg * sd, X2 = sp * cd;
  double Y0 = sp * sg - cp * cg * sd, Y1 = sp * cg + cp * sg * sd, Y2 = cp * cd;
  const double* D = cfg.det_D[det];
  // D X and D Y with the symmetric tensor (xx xy xz yy yz zz)
  double DX0 = D[0] * X0 + D[1] * X1 + D[2] * X2, DX1 = D[1] * X0 + D[3] * X1 + D[4] * X2, DX2 = D[2] * X0 + D[4] * X1 + D[5] * X2;
  double DY0 = D[0] * Y0 + D[1] * Y1 + D[2] * Y2, DY1 = D[1] * Y0 + D[3] * Y1 + D[4] * Y2, DY2 = D[2] * Y0 + D[4] * Y1 + D[5] * Y2;
  DetResp r;
  r.fp = (X0 * DX0 + X1 * DX1 + X2 * DX2) - (Y0 * DY0 + Y1 * DY1 + Y2 * DY2);
  r.fx = 2.0 * (X0 * DY0 + X1 * DY1 + X2 * DY2);
  const double* v = cfg.det_vertex[det];
  r.dt = -(v[0] * cd * cg - v[1] * cd * sg + v[2] * sd) / kC;
  return r;
}

// 3.5PN aligned-spin TaylorF2 phase coefficients phi_k, phi_k^(l) (DESIGN.md A.1).
__device__ __forceinline__ void pn_phase_coeffs(double eta, double delta, double chis, double chia, double (&ph)[8], double& c5,
                                                double& p6l) {
  const double pi = kPi, e2 = eta * eta, e3 = e2 * eta;
  ph[0] = 1.0; ph[1] = 0.0;
  ph[2] = 3715.0 / 756.0 + 55.0 / 9.0 * eta;
  ph[3] = -16.0 * pi + 113.0 / 3.0 * delta * chia + (113.0 / 3.0 - 76.0 / 3.0 * eta) * chis;
  ph[4] = 15293365.0 / 508032.0 + 27145.0 / 504.0 * eta + 3085.0 / 72.0 * e2 + (-405.0 / 8.0 + 200.0 * eta) * chia * chia -
          405.0 / 4.0 * delta * chia * chis + (-405.0 / 8.0 + 2.5 * eta) * chis * chis;
  c5 = 38645.0 / 756.0 * pi - 65.0 / 9.0 * pi * eta + delta * (-732985.0 / 2268.0 - 140.0 / 9.0 * eta) * chia +
       (-732985.0 / 2268.0 + 24260.0 / 81.0 * eta + 340.0 / 9.0 * e2) * chis;
  ph[5] = c5;
  ph[6] = 11583231236531.0 / 4694215680.0 - 6848.0 / 21.0 * kEulerGamma - 640.0 / 3.0 * pi * pi +
          (-15737765635.0 / 3048192.0 + 2255.0 / 12.0 * pi * pi) * eta + 76055.0 / 1728.0 * e2 - 127825.0 / 1296.0 * e3 -
          6848.0 / 63.0 * 4.1588830833596715 /* ln 64 */ + 2270.0 / 3.0 * pi * delta * chia + (2270.0 / 3.0 * pi - 520.0 * pi * eta) * chis;
  p6l = -6848.0 / 21.0;
  ph[7] = 77096675.0 / 254016.0 * pi + 378515.0 / 1512.0 * pi * eta - 74045.0 / 756.0 * pi * e2 +
          delta * (-25150083775.0 / 3048192.0 + 26804935.0 / 6048.0 * eta - 1985.0 / 48.0 * e2) * chia +
          (-25150083775.0 / 3048192.0 + 10566655595.0 / 762048.0 * eta - 1042165.0 / 3024.0 * e2 + 5345.0 / 36.0 * e3) * chis;
}

// Per-particle set-up: theta[11] -> coefficient block cb[CB_SIZE] (generic pointer: shared or global).
// Returns false (and sets cb[CB_VALID] = 0) for unphysical theta (logL = -inf).
template <int MODEL>
__device__ bool setup_particle(const DevCfg& cfg, const double* th, double* cb) {
  const double Mc = th[0], q = th[1], chi1 = th[2], chi2 = th[3], dL = th[4], iota = th[5], psi = th[6], phic = th[7], tc = th[8],
               ra = th[9], dec = th[10];
  bool ok = true;
#pragma unroll
  for (int i = 0; i < 11; ++i) ok = ok && isfinite(th[i]);
  ok = ok && (Mc > 0.0) && (q > 0.0) && (q <= 1.0) && (fabs(chi1) <= 1.0) && (fabs(chi2) <= 1.0) && (dL > 0.0);
  if (!ok) { cb[CB_VALID] = 0.0; return false; }
  cb[CB_VALID] = 1.0;

  const double eta = q / ((1.0 + q) * (1.0 + q));
  // (powers as exp(c log x): half the dependent instructions of pow(), a few ulp -- this set-up is the serial latency of a walk chunk)
  const double M = Mc * kGMsunS * exp(-0.6 * log(eta));
  const double m1 = M / (1.0 + q), m2 = M * q / (1.0 + q);
  const double delta = (m1 - m2) / M;
  const double chis = 0.5 * (chi1 + chi2), chia = 0.5 * (chi1 - chi2);

  // ---- extrinsic: detector projections -------------------------------------------------------------
  double sg, cg, sd, cd, sp, cp;
  sincos(cfg.gmst - ra, &sg, &cg);
  sincos(dec, &sd, &cd);
  sincos(psi, &sp, &cp);
  const double ci = cos(iota);
  const double A0 = 0.2127875101396634 /* sqrt(5/24) pi^-2/3 */ * exp((5.0 / 6.0) * log(Mc * kGMsunS)) / (dL * kMpcS);
  double tc0 = tc, dt0 = 0.0;   // tc0 = tc + dt of detector 0: the common phase carries detector 0's arrival time
  for (int d = 0; d < cfg.n_det; ++d) {
    DetResp r = detector_response(cfg, d, sg, cg, sd, cd, sp, cp);
    double cr = A0 * r.fp * 0.5 * (1.0 + ci * ci), cim = -A0 * r.fx * ci;
    if (d == 0) { dt0 = r.dt; tc0 = tc + dt0; }
    cb[CB_DET + 4 * d + 0] = cr;
    cb[CB_DET + 4 * d + 1] = cim;
    cb[CB_DET + 4 * d + 2] = -4.0 * (r.dt - dt0);
    cb[CB_DET + 4 * d + 3] = cr * cr + cim * cim;
  }

  // ---- intrinsic phase: PN part in the basis y5 y3 y2 y 1 L x xL x2 f ---------------------------------
  double ph[8], c5, p6l;
  pn_phase_coeffs(eta, delta, chis, chia, ph, c5, p6l);
  const double cv = cbrt(kPi * M), lncv = log(cv);
  const double K = 3.0 / (128.0 * eta);
  const double cv2 = cv * cv;
  const double e5 = K, e4 = K / cv, e3 = K / cv2, e2 = e3 / cv, e0 = e2 / cv2, e6 = K * cv, e7 = K * cv2;
  double a[13];
  a[0] = e0 * ph[0];
  a[1] = e2 * ph[2];
  a[2] = e3 * ph[3];
  a[3] = e4 * ph[4];
  a[4] = -0.25 * kPi - 2.0 * phic + e5 * (c5 + 3.0 * c5 * lncv);
  a[5] = e5 * c5;                       // phi5^(l)/3 = c5
  a[6] = e6 * (ph[6] + p6l * lncv);
  a[7] = e6 * p6l / 3.0;
  a[8] = e7 * ph[7];
  a[9] = 2.0 * kPi * tc0;
  a[10] = a[11] = a[12] = 0.0;

  if (MODEL == 1) {
#pragma unroll
    for (int i = 0; i < 13; ++i) cb[CB_PH + i] = a[i] * kQT;
    return true;
  }

  // ---- PhenomD-form (DESIGN.md A.2) ------------------------------------------------------------------
  double Lm[19];
  {
    const double chieff = (m1 * chi1 + m2 * chi2) / M;
    const double xi = chieff - 38.0 / 113.0 * eta * (chi1 + chi2) - 1.0;
    const double e2_ = eta * eta, xi2 = xi * xi, xi3 = xi2 * xi;
    for (int r = 0; r < 19; ++r) {
      const double* t = cfg.table[r];
      Lm[r] = t[0] + t[1] * eta + xi * (t[2] + t[3] * eta + t[4] * e2_) + xi2 * (t[5] + t[6] * eta + t[7] * e2_) +
              xi3 * (t[8] + t[9] * eta + t[10] * e2_);
    }
  }
  const double rho1 = Lm[0], rho2 = Lm[1], rho3 = Lm[2], v2 = Lm[3], gam1 = Lm[4], gam2 = Lm[5], gam3 = Lm[6];
  const double sig1 = Lm[7], sig2 = Lm[8], sig3 = Lm[9], sig4 = Lm[10], bet1 = Lm[11], bet2 = Lm[12], bet3 = Lm[13];
  const double alp1 = Lm[14], alp2 = Lm[15], alp3 = Lm[16], alp4 = Lm[17], alp5 = Lm[18];
  // final state and ringdown frequencies (surrogate fits)
  const double eta2 = eta * eta, eta3 = eta2 * eta;
  const double S = (m1 * m1 * chi1 + m2 * m2 * chi2) / (M * M);
  double af = 2.0 * sqrt(3.0) * eta - 3.871 * eta2 + 4.028 * eta3 + S;
  af = fmin(0.99, fmax(-0.99, af));
  const double Erad = 0.05597 * eta + 0.5810 * eta2 - 0.9607 * eta3 + 3.352 * eta2 * eta2;
  const double lg1af = log(1.0 - af);
  const double Frd = (1.5251 - 1.1568 * exp(0.1292 * lg1af)) / (2.0 * kPi * (1.0 - Erad));
  const double Qf = 0.7 + 1.4187 * exp(-0.4990 * lg1af);
  const double Fdamp = Frd / (2.0 * Qf);
  const double wF = gam3 * Fdamp;
  double Fpeak;
  if (gam2 < 1.0) Fpeak = fabs(Frd + wF * (sqrt(1.0 - gam2 * gam2) - 1.0) / gam2);
  else Fpeak = fabs(Frd - wF / gam2);

  // -- phase pieces in F = M f and their connection (C0/C1 at 0.018 and Frd/2, analytic derivatives) --
  const double ieta = 1.0 / eta;
  auto pn_phase = [&](double F, double& val, double& der) {   // only ever called at F = 0.018
    const double v = 0.3838316585355026 /* cbrt(pi 0.018) */, lv = -0.957551211745524 /* ln of it */;
    double vk[8];
    vk[0] = 1.0;
#pragma unroll
    for (int k = 1; k < 8; ++k) vk[k] = vk[k - 1] * v;
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      double pl = (k == 5) ? 3.0 * c5 : ((k == 6) ? p6l : 0.0);
      double t = ph[k] + pl * lv;
      s0 += t * vk[k];
      s1 += ((k - 5.0) * t + pl) * vk[k];
    }
    double v5 = vk[5];
    val = -0.25 * kPi + K * s0 / v5;
    der = K * s1 / (v5 * v) * v / (3.0 * F);
  };
  auto ins_phase = [&](double F, double& val, double& der) {
    pn_phase(F, val, der);
    const double F13 = 0.26207413942088964 /* cbrt(0.018) */, F23 = F13 * F13;
    val += ieta * (sig1 * F + 0.75 * sig2 * F * F13 + 0.6 * sig3 * F * F23 + 0.5 * sig4 * F * F);
    der += ieta * (sig1 + sig2 * F13 + sig3 * F23 + sig4 * F);
  };
  auto int_phase = [&](double F, double& val, double& der) {
    double iF = 1.0 / F, iF3 = iF * iF * iF;
    val = ieta * (bet1 * F + bet2 * log(F) - bet3 * iF3 / 3.0);
    der = ieta * (bet1 + bet2 * iF + bet3 * iF3 * iF);
  };
  auto mr_phase = [&](double F, double& val, double& der) {
    double yy = (F - alp5 * Frd) / Fdamp;
    double F14 = sqrt(sqrt(F));
    val = ieta * (alp1 * F - alp2 / F + 4.0 / 3.0 * alp3 * F14 * F14 * F14 + alp4 * atan(yy));
    der = ieta * (alp1 + alp2 / (F * F) + alp3 / F14 + alp4 / (Fdamp * (1.0 + yy * yy)));
  };
  double vi, di, vb, db, vm, dm;
  const double Fa = 0.018, Fb = 0.5 * Frd;
  ins_phase(Fa, vi, di);
  int_phase(Fa, vb, db);
  const double C2i = di - db, C1i = vi - vb - C2i * Fa;
  int_phase(Fb, vb, db);
  mr_phase(Fb, vm, dm);
  const double C2m = (db + C2i) - dm, C1m = (vb + C1i + C2i * Fb) - vm - C2m * Fb;
  mr_phase(Fpeak, vm, dm);
  const double t0 = dm + C2m;

  const double M13 = cv * 0.6827840632552957 /* pi^-1/3 */, M23 = M13 * M13;
  a[4] = -0.25 * kPi - 2.0 * phic + e5 * (c5 + 3.0 * c5 * lncv);
  a[9] = 2.0 * kPi * tc0 + (sig1 * ieta - t0) * M;
  a[10] = 0.75 * sig2 * ieta * M * M13;
  a[11] = 0.6 * sig3 * ieta * M * M23;
  a[12] = 0.5 * sig4 * ieta * M * M;
#pragma unroll
  for (int i = 0; i < 13; ++i) cb[CB_PH + i] = a[i] * kQT;
  cb[CB_PB + 0] = (bet2 * ieta * (3.0 * lncv - 1.1447298858494002 /* ln pi */) + C1i - 2.0 * phic) * kQT;
  cb[CB_PB + 1] = bet2 * ieta * kQT;
  cb[CB_PB + 2] = ((bet1 * ieta + C2i - t0) * M + 2.0 * kPi * tc0) * kQT;
  cb[CB_PB + 3] = -bet3 * ieta / (3.0 * M * M * M) * kQT;
  const double M34 = sqrt(sqrt(M * M * M));
  cb[CB_PM + 0] = (C1m - 2.0 * phic) * kQT;
  cb[CB_PM + 1] = ((alp1 * ieta + C2m - t0) * M + 2.0 * kPi * tc0) * kQT;
  cb[CB_PM + 2] = -alp2 * ieta / M * kQT;
  cb[CB_PM + 3] = 4.0 / 3.0 * alp3 * ieta * M34 * kQT;
  cb[CB_PM + 4] = alp4 * ieta * kQT;
  cb[CB_PM + 5] = alp5 * Frd / M;
  cb[CB_PM + 6] = M / Fdamp;
  cb[CB_FP1] = Fa / M;
  cb[CB_FP2] = Fb / M;
  cb[CB_FA1] = 0.014 / M;
  cb[CB_FA2] = Fpeak / M;
  cb[CB_FMR] = fmax(Fb, Fpeak) / M;

  // -- amplitude --------------------------------------------------------------------------------------
  double A[7];
  A[0] = 1.0; A[1] = 0.0;
  A[2] = -323.0 / 224.0 + 451.0 / 168.0 * eta;
  A[3] = (27.0 / 8.0 - 11.0 / 6.0 * eta) * chis + 27.0 / 8.0 * delta * chia;
  A[4] = -27312085.0 / 8128512.0 - 1975055.0 / 338688.0 * eta + 105271.0 / 24192.0 * eta2 + (-81.0 / 32.0 + 8.0 * eta) * chia * chia -
         81.0 / 16.0 * delta * chia * chis + (-81.0 / 32.0 + 17.0 / 8.0 * eta) * chis * chis;
  A[5] = -85.0 / 64.0 * kPi + 85.0 / 16.0 * kPi * eta + (285197.0 / 16128.0 - 1579.0 / 4032.0 * eta) * delta * chia +
         (285197.0 / 16128.0 - 15317.0 / 672.0 * eta - 2227.0 / 1008.0 * eta2) * chis;
  A[6] = -177520268561.0 / 8583708672.0 + (545384828789.0 / 5007163392.0 - 205.0 / 48.0 * kPi * kPi) * eta -
         3248849057.0 / 178827264.0 * eta2 + 34473079.0 / 6386688.0 * eta3 +
         (1614569.0 / 64512.0 - 1873643.0 / 16128.0 * eta + 2167.0 / 42.0 * eta2) * chia * chia +
         (31.0 / 12.0 * kPi - 7.0 / 3.0 * kPi * eta) * chis + (1614569.0 / 64512.0 - 61391.0 / 1344.0 * eta + 57451.0 / 4032.0 * eta2) * chis * chis +
         delta * chia * (31.0 / 12.0 * kPi + (1614569.0 / 32256.0 - 165961.0 / 2688.0 * eta) * chis);
  // inspiral amplitude as a degree-9 polynomial in x = f^1/3: (pi F)^(i/3) = (cv x)^i, F^(7/3) = M^(7/3) x^7, ...
  double ai[10];
  {
    double cvp = 1.0;
#pragma unroll
    for (int i = 0; i < 7; ++i) { ai[i] = A[i] * cvp; cvp *= cv; }
    const double M2 = M * M;
    ai[7] = rho1 * M2 * M13;
    ai[8] = rho2 * M2 * M23;
    ai[9] = rho3 * M2 * M;
#pragma unroll
    for (int i = 0; i < 10; ++i) cb[CB_AI + i] = ai[i];
  }
  // value and slope (per unit F) of the inspiral amplitude at F1 = 0.014
  const double F1 = 0.014;
  double v1, d1;
  {
    double x1 = 0.241014226417523 /* cbrt(0.014) */ / M13;  // x at the junction: f^1/3
    double p = 0.0, dp = 0.0;
#pragma unroll
    for (int i = 9; i >= 0; --i) { dp = dp * x1 + p; p = p * x1 + ai[i]; }
    v1 = p;
    d1 = dp * x1 / (3.0 * F1);   // dA/dF = dA/dx * x/(3 f) / M, with f = F1/M
  }
  // merger-ringdown amplitude at its peak
  double v3, d3;
  {
    double xx = Fpeak - Frd;
    double lor = gam1 * wF / (xx * xx + wF * wF);
    v3 = lor * exp(-gam2 * xx / wF);
    d3 = v3 * (-2.0 * xx / (xx * xx + wF * wF) - gam2 / wF);
  }
  {
    const double Lw = Fpeak - F1;
    const double t1 = Lw * d1, t3 = Lw * d3;
    const double Bb = v2 - (0.5 * v1 + 0.125 * t1 + 0.5 * v3 - 0.125 * t3);
    cb[CB_AH + 0] = F1 / M;
    cb[CB_AH + 1] = M / Lw;
    cb[CB_AH + 2] = v1;
    cb[CB_AH + 3] = t1;
    cb[CB_AH + 4] = -3.0 * v1 - 2.0 * t1 + 3.0 * v3 - t3 + 16.0 * Bb;
    cb[CB_AH + 5] = 2.0 * v1 + t1 - 2.0 * v3 + t3 - 32.0 * Bb;
    cb[CB_AH + 6] = 16.0 * Bb;
  }
  {
    const double wh = wF / M;
    cb[CB_AM + 0] = Frd / M;
    cb[CB_AM + 1] = gam1 * wh / M;
    cb[CB_AM + 2] = wh * wh;
    cb[CB_AM + 3] = -gam2 / wh;
  }
  return true;
}

// ------------------------------------------------------------------------------------------------------
// Per-bin evaluation: common phase (quarter turns) and amplitude factor relative to A0 f^-7/6.
// ------------------------------------------------------------------------------------------------------
struct BinBasis {
  double f, y, L, x, f34;
  double y2, y3, y5, xL, x2;
};

// Asynchronous global -> shared copies of 8 / 16 bytes (LDGSTS) and the wait for this thread's own copies.  Used where a thread
// stages the table values of ITS next bin in a shared-memory slot only it reads: no barrier is involved.
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __forceinline__ BinBasis make_basis(const Tables& tb, int k, bool phenom) {
  BinBasis b;
  const double2 a = __ldg(tb.t01 + k), c = __ldg(tb.t23 + k), e = __ldg(tb.t45 + k), g = __ldg(tb.t67 + k);
  b.y5 = a.x; b.y3 = a.y; b.y2 = c.x; b.y = c.y; b.L = e.x; b.x = e.y; b.xL = g.x; b.x2 = g.y;
  b.f = __ldg(tb.f + k);
  b.f34 = phenom ? __ldg(tb.f34 + k) : 0.0;
  return b;
}

// PN phase in the tabulated basis: nine FMAs (independent particles held by the same thread supply the ILP).
__device__ __forceinline__ double phase_pn_qt(const double* a, const BinBasis& b) {
  double q = fma(a[0], b.y5, a[4]);
  q = fma(a[1], b.y3, q);
  q = fma(a[2], b.y2, q);
  q = fma(a[3], b.y, q);
  q = fma(a[5], b.L, q);
  q = fma(a[6], b.x, q);
  q = fma(a[7], b.xL, q);
  q = fma(a[8], b.x2, q);
  q = fma(a[9], b.f, q);
  return q;
}

// Accessors of a coefficient block: contiguous (shared or global memory, one particle) or strided (block transposed in shared
// memory so that each lane of a warp reads its own particle without bank conflicts).
struct CbPtr {
  const double* p;
  __device__ __forceinline__ double operator()(int i) const { return p[i]; }
};
struct CbStrided {
  const double* p;
  int stride;
  __device__ __forceinline__ double operator()(int i) const { return p[i * stride]; }
};

// PhenomD-form: phase [quarter turns] and amplitude factor for one bin.
// `ex` = exp(-gamma2 (f - f_RD)/w) of this bin, supplied by the caller (the bin loops carry it as a geometric sequence along a
// thread's bins; k_waveform and the relative-binning kernels evaluate it directly).
template <class CB>
__device__ __forceinline__ void phenom_bin_t(const CB& cb, const BinBasis& b, const MathTables* mt, double ex, double& q, double& amp) {
  const double f = b.f;
  if (f < cb(CB_FP1)) {
    q = fma(cb(CB_PH + 0), b.y5, cb(CB_PH + 4));
    q = fma(cb(CB_PH + 1), b.y3, q);
    q = fma(cb(CB_PH + 2), b.y2, q);
    q = fma(cb(CB_PH + 3), b.y, q);
    q = fma(cb(CB_PH + 5), b.L, q);
    q = fma(cb(CB_PH + 6), b.x, q);
    q = fma(cb(CB_PH + 7), b.xL, q);
    q = fma(cb(CB_PH + 8), b.x2, q);
    q = fma(cb(CB_PH + 9), b.f, q);
    double fx = f * b.x;
    q = fma(cb(CB_PH + 10), fx, q);
    q = fma(cb(CB_PH + 11), fx * b.x, q);
    q = fma(cb(CB_PH + 12), f * f, q);
  } else if (f < cb(CB_FP2)) {
    double if3 = b.y3 * b.y3 * b.y3;
    q = fma(cb(CB_PB + 1), b.L, cb(CB_PB + 0));
    q = fma(cb(CB_PB + 2), f, q);
    q = fma(cb(CB_PB + 3), if3, q);
  } else {
    q = fma(cb(CB_PM + 1), f, cb(CB_PM + 0));
    q = fma(cb(CB_PM + 2), b.y3, q);
    q = fma(cb(CB_PM + 3), b.f34, q);
    q = fma(cb(CB_PM + 4), atan_tab((f - cb(CB_PM + 5)) * cb(CB_PM + 6), mt), q);
  }
  if (f < cb(CB_FA1)) {
    double p = cb(CB_AI + 9);
#pragma unroll
    for (int i = 8; i >= 0; --i) p = fma(p, b.x, cb(CB_AI + i));
    amp = p;
  } else if (f < cb(CB_FA2)) {
    double xh = (f - cb(CB_AH + 0)) * cb(CB_AH + 1);
    double p = cb(CB_AH + 6);
    p = fma(p, xh, cb(CB_AH + 5));
    p = fma(p, xh, cb(CB_AH + 4));
    p = fma(p, xh, cb(CB_AH + 3));
    p = fma(p, xh, cb(CB_AH + 2));
    amp = p;
  } else {
    double fx = f - cb(CB_AM + 0);
    amp = cb(CB_AM + 1) * rcp_nr1(fma(fx, fx, cb(CB_AM + 2))) * ex;
  }
}

__device__ __forceinline__ void phenom_bin(const double* cb, const BinBasis& b, const MathTables* mt, double ex, double& q, double& amp) {
  phenom_bin_t(CbPtr{cb}, b, mt, ex, q, amp);
}

}  // namespace nsgw
