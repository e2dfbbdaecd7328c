// nsgw.cu -- kernels and C-ABI of libnsgw.so (see include/nsgw.h for the contract, DESIGN.md for the design).
//
// Kernels
//   k_tables          ns_init: per-bin tables and noise-weighted data (parameter independent)
//   k_setup           theta[B,11] -> per-particle coefficient blocks (one thread per particle)
//   k_bins            K1: CTA per P particles, bins strided over threads, shuffle + smem reduction
//   k_walk_gw         K2: persistent lock-step acceptance walk, CTA per P walkers, W steps in-kernel
//   k_walk_simple     K2 for bin-less likelihoods (Gaussian toy, cube shell): one thread per walker
//   k_rank / k_evidence / k_gather_start / k_writeback / k_adapt   K3: select, evidence scan, replacement, adaptation
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <string>
#include <atomic>
#include <vector>
#include <algorithm>
#include <climits>

#include "../../include/nsgw.h"
#include "nsgw_device.cuh"

using namespace nsgw;

namespace {

std::atomic<long long> g_launches{0};
thread_local std::string g_init_error;

// CTA width of the CTA-per-particle sweep kernel (k_bins); the walk kernel chooses 128 / 96 / 64 by batch size.
constexpr int kBinsThreads = 256;

// ======================================================================================================
// Device state of the sampler
// ======================================================================================================
struct DevState {
  double logx, logz, h, walks, delay, lstar;
  long long iter, n_eval_total;
  int W, naccept, maxmcmc, pad;
  ns_stats stats;
};

// ======================================================================================================
// ns_init kernels
// ======================================================================================================
__global__ void k_tables(DevCfg* cfg, const double* __restrict__ strain, const double* __restrict__ psd, double2* t01, double2* t23,
                         double2* t45, double2* t67, double* tf, double* tf34, double2* wd, double* ws) {
  const int nf = cfg->n_freq, nd = cfg->n_det;
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < nf; k += gridDim.x * blockDim.x) {
    double f = cfg->f_min + k * cfg->df;
    double x = cbrt(f), y = 1.0 / x, L = log(f);
    double y2 = y * y, y3 = y2 * y;
    t01[k] = make_double2(y3 * y2, y3);
    t23[k] = make_double2(y2, y);
    t45[k] = make_double2(L, x);
    t67[k] = make_double2(x * L, x * x);
    tf[k] = f; tf34[k] = sqrt(sqrt(f * f * f));
    double a76 = 1.0 / (f * sqrt(x));      // f^-7/6
    for (int d = 0; d < nd; ++d) {
      double S = psd[(size_t)d * nf + k];
      double w = 4.0 * cfg->df / S;
      wd[(size_t)d * nf + k] = make_double2(w * a76 * strain[((size_t)d * nf + k) * 2], w * a76 * strain[((size_t)d * nf + k) * 2 + 1]);
      ws[(size_t)d * nf + k] = w * a76 * a76;
    }
  }
}

__global__ void k_math_tables(MathTables* mt) { build_math_tables(mt, threadIdx.x, blockDim.x); }

// I_{7/3} per detector: deterministic single-CTA tree sum.
__global__ void k_i73(DevCfg* cfg, const double* __restrict__ ws) {
  __shared__ double sh[256];
  const int nf = cfg->n_freq;
  for (int d = 0; d < cfg->n_det; ++d) {
    double acc = 0.0;
    for (int k = threadIdx.x; k < nf; k += 256) acc += ws[(size_t)d * nf + k];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
      if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
      __syncthreads();
    }
    if (threadIdx.x == 0) cfg->i73[d] = sh[0];
    __syncthreads();
  }
}

__global__ void k_draw_live(int ndim, long long n, uint32_t k0, uint32_t k1, double* u) {
  long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  for (int d = 0; d < ndim; d += 2) {
    uint32_t w[4];
    philox4x32_10((uint32_t)(d / 2), 0u, (uint32_t)i, 2u << 24, k0, k1, w);
    u[i * ndim + d] = u01(w[0], w[1]);
    if (d + 1 < ndim) u[i * ndim + d + 1] = u01(w[2], w[3]);
  }
}

__global__ void k_prior_transform(const DevCfg* __restrict__ cfg, const double* __restrict__ u, long long B, double* theta) {
  long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  const int D = cfg->ndim;
  if (i >= B * D) return;
  int d = (int)(i % D);
  theta[i] = prior_transform_dim(cfg->prior_kind[d], cfg->prior_lo[d], cfg->prior_hi[d], u[i]);
}

// ======================================================================================================
// K1: set-up + bin loop
// ======================================================================================================
template <int MODEL>
__global__ void k_setup(const DevCfg* __restrict__ cfg, const double* __restrict__ theta, long long B, double* cbs) {
  long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= B) return;
  double th[11];
#pragma unroll
  for (int d = 0; d < 11; ++d) th[d] = theta[i * 11 + d];
  setup_particle<MODEL>(*cfg, th, cbs + i * CB_SIZE);
}

// Number of per-thread partial sums of one particle: X0 = sum conj(wd_0) amp E (complex; detector 0 carries no phasor, its
// C_0 is applied once after the reduction), dh_d for d >= 1, and for PhenomD-form hh_d = sum amp^2 ws_d for every detector.
template <int MODEL, int NDET>
struct AccLayout {
  static constexpr int ND1 = NDET - 1;
  static constexpr int kDh = 2;                          // dh_d at kDh + d - 1 (d >= 1)
  static constexpr int kHh = 2 + ND1;                    // hh_d at kHh + d (PhenomD-form only)
  static constexpr int N = 2 + ND1 + (MODEL == 2 ? NDET : 0);
};

// Start phasors of the detectors d >= 1: for particle p, thread t (bin t of the first sweep)
//   R = (Cr + i Ci) * exp(i * dtq * f_t)  [dtq: quarter turns per Hz relative to detector 0],
// built as lane-table x warp-table to keep it to one sincos per entry.
// tabL[(p*ND1+d-1)*32 + lane] = exp(i dtq df lane); tabW[(p*ND1+d-1)*NW + w] = C * exp(i dtq (f_min + 32 w df)).
template <int NDET, int NT>
__device__ __forceinline__ void build_phasor_tables(const DevCfg& cfg, const double* cbs /*smem [np][CB_SIZE]*/, int np, double2* tabL,
                                                    double2* tabW, double2* step) {
  constexpr int NW = NT / 32, ND1 = NDET - 1, ND1s = NDET > 1 ? NDET - 1 : 1;
  const int NE = np * ND1 * (32 + NW + 1);
  for (int e = threadIdx.x; e < NE; e += NT) {
    int pd = e / (32 + NW + 1), j = e % (32 + NW + 1);
    int p = pd / ND1s, d = pd % ND1s + 1;
    const double* cb = cbs + p * CB_SIZE;
    double dtq = cb[CB_DET + 4 * d + 2];
    double s, c;
    if (j < 32) {
      sincos_qt(dtq * (cfg.df * j), s, c);
      tabL[pd * 32 + j] = make_double2(c, s);
    } else if (j < 32 + NW) {
      int w = j - 32;
      sincos_qt(dtq * (cfg.f_min + cfg.df * (32 * w)), s, c);
      double cr = cb[CB_DET + 4 * d], ci = cb[CB_DET + 4 * d + 1];
      tabW[pd * NW + w] = make_double2(cr * c - ci * s, cr * s + ci * c);
    } else {
      sincos_qt(dtq * (cfg.df * NT), s, c);
      step[pd] = make_double2(c, s);
    }
  }
}

// Bin loop for P particles held by this CTA: thread t handles bins t, t + NT, ...; the table values of a bin are loaded once
// and used for the P particles.  Per (particle, bin): common phase (9 FMA), one sincos, 4 FMA for detector 0, and for each
// further detector a complex product with its phasor, 2 FMA and the phasor advance.
template <int MODEL, int NDET, int P, int NT>
__device__ __forceinline__ void bin_loop(const DevCfg& cfg, const Tables& tb, const double* cbs, const double2* tabL,
                                         const double2* tabW, const double2* step, const MathTables* mt, const bool* active,
                                         const int* slot /*smem [P]: coefficient-block / phasor-table slot of particle p*/,
                                         double (&acc)[P][AccLayout<MODEL, NDET>::N]) {
  using AL = AccLayout<MODEL, NDET>;
  constexpr int NW = NT / 32, ND1 = NDET - 1;
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  double2 R[P][ND1 > 0 ? ND1 : 1], St[P][ND1 > 0 ? ND1 : 1];
  double a[P][MODEL == 1 ? 10 : 1];
  const double* cbp[P];
  bool any = false;
#pragma unroll
  for (int p = 0; p < P; ++p) {
    const int sl = slot[p];
    cbp[p] = cbs + sl * CB_SIZE;
    any = any || active[p];
#pragma unroll
    for (int i = 0; i < AL::N; ++i) acc[p][i] = 0.0;
#pragma unroll
    for (int d = 0; d < ND1; ++d) {
      double2 u = tabL[(sl * ND1 + d) * 32 + lane], v = tabW[(sl * ND1 + d) * NW + wrp];
      R[p][d] = make_double2(u.x * v.x - u.y * v.y, u.x * v.y + u.y * v.x);
      St[p][d] = step[sl * ND1 + d];
    }
    if (MODEL == 1) {
#pragma unroll
      for (int i = 0; i < 10; ++i) a[p][i] = 64.0 * cbp[p][CB_PH + i];   // quarter turns -> 1/256 turn (exact)
    }
  }
  if (!any) return;   // block-uniform: nothing to evaluate (all proposals of this CTA were out of bounds)
  const int nf = cfg.n_freq;
  // shared tail of a (particle, bin): E = amp exp(-i Phi) and the accumulations
  auto tail = [&](int p, double q, double amp, const double2 (&w)[NDET], const double (&wsv)[NDET]) {
    double sn, cs;
    sincos_lut(q, mt, sn, cs);
    if (MODEL == 2) { sn *= amp; cs *= amp; }
    // E = cs - i sn;  X0 += conj(wd_0) E
    acc[p][0] = fma(w[0].x, cs, acc[p][0]);
    acc[p][1] = fma(-w[0].x, sn, acc[p][1]);
    acc[p][0] = fma(-w[0].y, sn, acc[p][0]);
    acc[p][1] = fma(-w[0].y, cs, acc[p][1]);
    if (MODEL == 2) {
      const double a2 = amp * amp;
#pragma unroll
      for (int d = 0; d < NDET; ++d) acc[p][AL::kHh + d] = fma(a2, wsv[d], acc[p][AL::kHh + d]);
    }
#pragma unroll
    for (int d = 0; d < ND1; ++d) {
      const double rx = R[p][d].x, ry = R[p][d].y;
      // G = E R_d;  dh_d += Re(conj(wd_d) G)
      const double gr = fma(cs, rx, sn * ry);
      const double gi = fma(cs, ry, -(sn * rx));
      acc[p][AL::kDh + d] = fma(w[d + 1].x, gr, acc[p][AL::kDh + d]);
      acc[p][AL::kDh + d] = fma(w[d + 1].y, gi, acc[p][AL::kDh + d]);
      // advance the detector phasor by one sweep
      R[p][d].x = fma(rx, St[p][d].x, -(ry * St[p][d].y));
      R[p][d].y = fma(rx, St[p][d].y, ry * St[p][d].x);
    }
  };
  // PhenomD-form: from the first sweep whose bins all lie in the merger-ringdown region of BOTH phase and amplitude for every
  // particle of this group (about 80 % of the band), a branch-free loop with that region's 11 coefficients in registers.
  int k_mr = nf;   // first bin of the specialised loop (multiple of NT)
  if (MODEL == 2) {
    double fs = 0.0;
#pragma unroll
    for (int p = 0; p < P; ++p) fs = fmax(fs, fmax(cbp[p][CB_FP2], cbp[p][CB_FA2]));
    const double ks = (fs - cfg.f_min) / cfg.df + 2.0;          // two bins of margin against rounding of f_k
    if (ks < (double)nf) k_mr = ((int)fmax(ks, 0.0) + NT - 1) / NT * NT;
  }
  const int k_gen = (MODEL == 2) ? min(nf, k_mr) : nf;
  // PhenomD-form: exp(-gamma2 (f - f_RD)/w) along a thread's bins is a geometric sequence (ratio exp(c3 NT df)): one exp_tab per
  // thread and particle here, one multiplication per bin in both loops below (<= 32 ulp of accumulated rounding).  The sequence
  // starts at the thread's first bin whatever the loop split, so a particle's logL does not depend on its group partner.
  double ex[P], exr[P];
#pragma unroll
  for (int p = 0; p < P; ++p) {
    ex[p] = (MODEL == 2) ? exp_tab(cbp[p][CB_AM + 3] * (cfg.f_min + cfg.df * tid - cbp[p][CB_AM]), mt) : 1.0;
    exr[p] = (MODEL == 2) ? exp_tab(cbp[p][CB_AM + 3] * (cfg.df * NT), mt) : 1.0;
  }
  for (int k = tid; k < k_gen; k += NT) {
    const BinBasis b = make_basis(tb, k, MODEL == 2);
    double2 w[NDET];
    double wsv[NDET];
#pragma unroll
    for (int d = 0; d < NDET; ++d) {
      w[d] = __ldg(tb.wd[d] + k);
      wsv[d] = (MODEL == 2) ? __ldg(tb.ws[d] + k) : 0.0;
    }
#pragma unroll
    for (int p = 0; p < P; ++p) {
      double q, amp = 1.0;
      if (MODEL == 1) q = phase_pn_qt(a[p], b);
      else { phenom_bin(cbp[p], b, mt, ex[p], q, amp); q *= 64.0; ex[p] *= exr[p]; }
      tail(p, q, amp, w, wsv);
    }
  }
  if (MODEL == 2 && k_mr < nf) {
    double pm[P][7], am[P][4];
#pragma unroll
    for (int p = 0; p < P; ++p) {
#pragma unroll
      for (int i = 0; i < 5; ++i) pm[p][i] = 64.0 * cbp[p][CB_PM + i];     // phase in 1/256 turn (exact scaling)
      pm[p][5] = cbp[p][CB_PM + 5]; pm[p][6] = cbp[p][CB_PM + 6];
#pragma unroll
      for (int i = 0; i < 4; ++i) am[p][i] = cbp[p][CB_AM + i];
    }
#pragma unroll 2
    for (int k = k_mr + tid; k < nf; k += NT) {
      const double f = __ldg(tb.f + k), f34 = __ldg(tb.f34 + k);
      const double y3 = __ldg(tb.t01 + k).y;       // 1/f
      double2 w[NDET];
      double wsv[NDET];
#pragma unroll
      for (int d = 0; d < NDET; ++d) { w[d] = __ldg(tb.wd[d] + k); wsv[d] = __ldg(tb.ws[d] + k); }
#pragma unroll
      for (int p = 0; p < P; ++p) {
        double q = fma(pm[p][1], f, pm[p][0]);
        q = fma(pm[p][2], y3, q);
        q = fma(pm[p][3], f34, q);
        q = fma(pm[p][4], atan_tab((f - pm[p][5]) * pm[p][6], mt), q);
        const double fx = f - am[p][0];
        const double amp = am[p][1] * rcp_nr(fma(fx, fx, am[p][2])) * ex[p];
        ex[p] *= exr[p];
        tail(p, q, amp, w, wsv);
      }
    }
  }
}

// Deterministic block reduction of NV values per thread: warp shuffle tree, then fixed-order sum over warps by thread 0..NV-1.
template <int NV, int NT>
__device__ __forceinline__ void block_reduce(double (&v)[NV], double* red /*smem [NT/32][NV]*/, double* out /*smem [NV]*/) {
  constexpr int NW = NT / 32;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    double x = v[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    v[i] = x;
  }
  if ((threadIdx.x & 31) == 0) {
#pragma unroll
    for (int i = 0; i < NV; ++i) red[(threadIdx.x >> 5) * NV + i] = v[i];
  }
  __syncthreads();
  if (threadIdx.x < NV) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < NW; ++w) s += red[w * NV + threadIdx.x];
    out[threadIdx.x] = s;
  }
  __syncthreads();
}

// Finishes logL of one particle from its reduced sums (AccLayout order).
template <int MODEL, int NDET>
__device__ __forceinline__ double finish_logl(const DevCfg& cfg, const double* cb, const double* sums, double* parts) {
  using AL = AccLayout<MODEL, NDET>;
  if (cb[CB_VALID] == 0.0) {
    if (parts) for (int d = 0; d < 2 * NDET; ++d) parts[d] = nan("");
    return -INFINITY;
  }
  double logl = 0.0;
#pragma unroll
  for (int d = 0; d < NDET; ++d) {
    double dh = (d == 0) ? fma(cb[CB_DET], sums[0], -(cb[CB_DET + 1] * sums[1])) : sums[AL::kDh + d - 1];
    double hh = (MODEL == 1) ? cb[CB_DET + 4 * d + 3] * cfg.i73[d] : cb[CB_DET + 4 * d + 3] * sums[AL::kHh + d];
    if (parts) { parts[2 * d] = dh; parts[2 * d + 1] = hh; }
    logl += dh - 0.5 * hh;
  }
  return logl;
}

template <int MODEL, int NDET, int P>
__global__ void __launch_bounds__(kBinsThreads, 2) k_bins(const DevCfg* __restrict__ cfgp, Tables tb, const double* __restrict__ cbs_g,
                                                           long long B, double* logl, double* parts) {
  using AL = AccLayout<MODEL, NDET>;
  constexpr int NT = kBinsThreads, NW = NT / 32, NV = P * AL::N, ND1 = NDET > 1 ? NDET - 1 : 1;
  __shared__ __align__(16) double cbs[P * CB_SIZE];
  __shared__ double2 tabL[P * ND1 * 32], tabW[P * ND1 * NW], step[P * ND1];
  __shared__ double red[NW * NV], out[NV];
  __shared__ MathTables mtab;
  __shared__ bool active[P];
  __shared__ int slot[P];
  const DevCfg& cfg = *cfgp;
  const long long p0 = (long long)blockIdx.x * P;
  load_math_tables(&mtab, tb.mt, threadIdx.x, NT);
  if (threadIdx.x < P) slot[threadIdx.x] = threadIdx.x;
  for (int e = threadIdx.x; e < P * CB_SIZE; e += NT) {
    long long p = p0 + e / CB_SIZE;
    cbs[e] = (p < B) ? cbs_g[p * CB_SIZE + e % CB_SIZE] : 0.0;
  }
  __syncthreads();
  if (threadIdx.x < P) active[threadIdx.x] = cbs[threadIdx.x * CB_SIZE + CB_VALID] != 0.0;
  build_phasor_tables<NDET, NT>(cfg, cbs, P, tabL, tabW, step);
  __syncthreads();
  double acc[P][AL::N];
  bin_loop<MODEL, NDET, P, NT>(cfg, tb, cbs, tabL, tabW, step, &mtab, active, slot, acc);
  double v[NV];
#pragma unroll
  for (int p = 0; p < P; ++p)
#pragma unroll
    for (int i = 0; i < AL::N; ++i) v[p * AL::N + i] = acc[p][i];
  block_reduce<NV, NT>(v, red, out);
  if (threadIdx.x < P && p0 + threadIdx.x < B) {
    int p = threadIdx.x;
    logl[p0 + p] = finish_logl<MODEL, NDET>(cfg, cbs + p * CB_SIZE, out + p * AL::N, parts ? parts + (p0 + p) * 2 * NDET : nullptr);
  }
}

// ------------------------------------------------------------------------------------------------------
// K1 for large batches, lane = particle: every thread owns ONE particle (phase coefficients, detector phasors and partial
// sums in registers for the whole task), and the CTA walks a range of KR bins whose table values are staged once in shared
// memory and read with warp-uniform (broadcast) LDS.  No per-bin global traffic, no cross-thread reduction, no phasor
// tables: a task costs each thread 2 sincos per extra detector plus KR x (the same per-bin arithmetic as bin_loop).
// Task = (group of NT PP particles, range of kr bins); partial[n_ranges][N][B] is summed in range order by k_finish.
// Built for TaylorF2 (no per-particle branches in the bin loop; PhenomD-form's piecewise regions would diverge across lanes).
// ------------------------------------------------------------------------------------------------------
template <int NDET, int KR>
struct LpSmem {
  double2 t01[KR], t23[KR], t45[KR], t67[KR];
  double2 wd[NDET][KR];
  double f[KR];
};

template <int NDET, int NT, int KR, int PP, int UNR, int OCC>
__global__ void __launch_bounds__(NT, OCC) k_bins_lp(const DevCfg* __restrict__ cfgp, Tables tb, const double* __restrict__ cbs_g,
                                                     long long B, int kr /*bins per range, <= KR, multiple of UNR*/, int nranges,
                                                     long long ntasks, double* __restrict__ partial) {
  using AL = AccLayout<1, NDET>;
  constexpr int ND1 = NDET - 1, ND1s = NDET > 1 ? NDET - 1 : 1;
  __shared__ __align__(16) LpSmem<NDET, KR> sm;
  __shared__ MathTables mtab;
  const DevCfg& cfg = *cfgp;
  const int tid = threadIdx.x;
  const int nf = cfg.n_freq;
  load_math_tables(&mtab, tb.mt, tid, NT);
  for (long long task = blockIdx.x; task < ntasks; task += gridDim.x) {
    const long long grp = task / nranges;
    const int rng = (int)(task % nranges);
    const int k0 = rng * kr;
    const int nk = min(kr, nf - k0);
    const int nk2 = (nk + UNR - 1) / UNR * UNR;   // padded with zero-weight bins
    __syncthreads();   // readers of the previous tile are done
    for (int i = tid; i < nk2; i += NT) {
      const bool ok = i < nk;
      const int k = k0 + (ok ? i : nk - 1);
      sm.t01[i] = __ldg(tb.t01 + k); sm.t23[i] = __ldg(tb.t23 + k); sm.t45[i] = __ldg(tb.t45 + k); sm.t67[i] = __ldg(tb.t67 + k);
      sm.f[i] = __ldg(tb.f + k);
#pragma unroll
      for (int d = 0; d < NDET; ++d) sm.wd[d][i] = ok ? __ldg(tb.wd[d] + k) : make_double2(0.0, 0.0);
    }
    // ---- this thread's PP particles (a warp-wide load of the table values of a bin then serves 32 PP particle-bins)
    double a[PP][10];
    double2 R[PP][ND1s], St[PP][ND1s];
    double acc[PP][AL::N];
#pragma unroll
    for (int j = 0; j < PP; ++j) {
      const long long p = (grp * PP + j) * NT + tid;
      const bool have = p < B;
      const double* cb = cbs_g + (have ? p : 0) * CB_SIZE;
#pragma unroll
      for (int i = 0; i < 10; ++i) a[j][i] = have ? 64.0 * __ldg(cb + CB_PH + i) : 0.0;   // quarter turns -> 1/256 turn (exact)
#pragma unroll
      for (int d = 0; d < ND1; ++d) {
        const double cr = have ? __ldg(cb + CB_DET + 4 * (d + 1)) : 0.0, ci = have ? __ldg(cb + CB_DET + 4 * (d + 1) + 1) : 0.0;
        const double dtq = have ? __ldg(cb + CB_DET + 4 * (d + 1) + 2) : 0.0;
        double sn, cs;
        sincos_qt(dtq * (cfg.f_min + cfg.df * k0), sn, cs);
        R[j][d] = make_double2(cr * cs - ci * sn, cr * sn + ci * cs);
        sincos_qt(dtq * cfg.df, sn, cs);
        St[j][d] = make_double2(cs, sn);
      }
#pragma unroll
      for (int i = 0; i < AL::N; ++i) acc[j][i] = 0.0;
    }
    __syncthreads();
    // Detectors d >= 1: sum_k conj(wd_k) E_k R_k with R_k = R_0 rho^k is evaluated as R_0 * Horner(rho) over the tile's bins in
    // DESCENDING order, S <- S rho + conj(wd_k) E_k (8 FP64 instructions per bin instead of 10 for product + accumulate + phasor
    // advance).  The zero-weight padding bins come first and leave S = 0.
    double2 S[PP][ND1s];
#pragma unroll
    for (int j = 0; j < PP; ++j)
#pragma unroll
      for (int d = 0; d < ND1s; ++d) S[j][d] = make_double2(0.0, 0.0);
#pragma unroll UNR
    for (int kk = nk2 - 1; kk >= 0; --kk) {
      BinBasis b;
      { const double2 v = sm.t01[kk]; b.y5 = v.x; b.y3 = v.y; }
      { const double2 v = sm.t23[kk]; b.y2 = v.x; b.y = v.y; }
      { const double2 v = sm.t45[kk]; b.L = v.x; b.x = v.y; }
      { const double2 v = sm.t67[kk]; b.xL = v.x; b.x2 = v.y; }
      b.f = sm.f[kk]; b.f34 = 0.0;
      double2 w[NDET];
#pragma unroll
      for (int d = 0; d < NDET; ++d) w[d] = sm.wd[d][kk];
#pragma unroll
      for (int j = 0; j < PP; ++j) {
        const double q = phase_pn_qt(a[j], b);
        double sn, cs;
        sincos_lut(q, &mtab, sn, cs);
        acc[j][0] = fma(w[0].x, cs, acc[j][0]);
        acc[j][1] = fma(-w[0].x, sn, acc[j][1]);
        acc[j][0] = fma(-w[0].y, sn, acc[j][0]);
        acc[j][1] = fma(-w[0].y, cs, acc[j][1]);
#pragma unroll
        for (int d = 0; d < ND1; ++d) {
          const double ax = fma(w[d + 1].x, cs, -(w[d + 1].y * sn));      // conj(wd) E, E = cs - i sn
          const double ay = -fma(w[d + 1].x, sn, w[d + 1].y * cs);
          const double sx = S[j][d].x, sy = S[j][d].y;
          S[j][d].x = fma(sx, St[j][d].x, fma(-sy, St[j][d].y, ax));
          S[j][d].y = fma(sx, St[j][d].y, fma(sy, St[j][d].x, ay));
        }
      }
    }
#pragma unroll
    for (int j = 0; j < PP; ++j)
#pragma unroll
      for (int d = 0; d < ND1; ++d) acc[j][AL::kDh + d] = fma(R[j][d].x, S[j][d].x, -(R[j][d].y * S[j][d].y));   // Re(R_0 S)
#pragma unroll
    for (int j = 0; j < PP; ++j) {
      const long long p = (grp * PP + j) * NT + tid;
      if (p < B) {
#pragma unroll
        for (int i = 0; i < AL::N; ++i) partial[((long long)rng * AL::N + i) * B + p] = acc[j][i];   // [range][N][B]: coalesced
      }
    }
  }
}

// Adds the per-range partial sums in range order and finishes logL.
template <int MODEL, int NDET>
__global__ void k_finish(const DevCfg* __restrict__ cfgp, const double* __restrict__ cbs_g, const double* __restrict__ partial, int nchunks,
                         long long B, double* logl, double* parts) {
  using AL = AccLayout<MODEL, NDET>;
  long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (p >= B) return;
  double sums[AL::N];
#pragma unroll
  for (int i = 0; i < AL::N; ++i) sums[i] = 0.0;
  for (int c = 0; c < nchunks; ++c)
#pragma unroll
    for (int i = 0; i < AL::N; ++i) sums[i] += partial[((long long)c * AL::N + i) * B + p];
  logl[p] = finish_logl<MODEL, NDET>(*cfgp, cbs_g + p * CB_SIZE, sums, parts ? parts + p * 2 * NDET : nullptr);
}

// Detector-frame waveform of one theta on the grid (for injections): out[n_det][n_freq][2].
template <int MODEL>
__global__ void k_waveform(const DevCfg* __restrict__ cfgp, Tables tb, const double* __restrict__ theta, double* out) {
  __shared__ double cb[CB_SIZE];
  __shared__ MathTables mtab;
  const DevCfg& cfg = *cfgp;
  load_math_tables(&mtab, tb.mt, threadIdx.x, blockDim.x);
  if (threadIdx.x == 0) {
    double th[11];
    for (int d = 0; d < 11; ++d) th[d] = theta[d];
    setup_particle<MODEL>(cfg, th, cb);
  }
  __syncthreads();
  const int nf = cfg.n_freq;
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < nf; k += gridDim.x * blockDim.x) {
    BinBasis b = make_basis(tb, k, MODEL == 2);
    double q, amp = 1.0;
    if (MODEL == 1) q = phase_pn_qt(cb + CB_PH, b);
    else phenom_bin(cb, b, &mtab, exp_tab(cb[CB_AM + 3] * (b.f - cb[CB_AM]), &mtab), q, amp);
    double a76 = b.y3 * sqrt(b.y);   // f^-7/6
    for (int d = 0; d < cfg.n_det; ++d) {
      double s, c;
      sincos_qt(q - cb[CB_DET + 4 * d + 2] * b.f, s, c);   // Phi_det = Phi_c + 2 pi f dt
      double cr = cb[CB_DET + 4 * d] * amp * a76, ci = cb[CB_DET + 4 * d + 1] * amp * a76;
      bool ok = cb[CB_VALID] != 0.0;
      out[((size_t)d * nf + k) * 2] = ok ? cr * c + ci * s : nan("");
      out[((size_t)d * nf + k) * 2 + 1] = ok ? ci * c - cr * s : nan("");
    }
  }
}

// ======================================================================================================
// Relative binning (heterodyned likelihood; DESIGN.md R:L24): summary data about a fiducial theta0 on N_b
// coarse bins, then per evaluation the waveform at the N_b + 1 bin edges only.
// ======================================================================================================
struct RbDev {
  const int* edge;        // [nb + 1] grid indices of the bin edges
  const double2* A0;      // [n_det][nb]  sum wd conj(g0)              (g = h f^{7/6}: the f^{-7/6} of the amplitude lives in wd, ws)
  const double2* A1;      // [n_det][nb]  sum wd conj(g0) (f - f_m)
  const double* B0;       // [n_det][nb]  sum ws |g0|^2
  const double* B1;       // [n_det][nb]  sum ws |g0|^2 (f - f_m)
  const double2* ig0;     // [n_det][nb + 1]  1 / g0 at the edges
  const double* inv_w;    // [nb]  1 / (f_hi - f_lo)
  int nb;
};

// g_d(f_k) = amp C_d exp(-i Phi_d) for every detector at grid bin k (Phi_d = common phase - relative delay; the same pieces as
// the bin loops, with a direct sincos per detector because the edges are not equally spaced).
template <int MODEL, int NDET, class CB>
__device__ __forceinline__ void gw_g_at(const CB& cb, const Tables& tb, int k, const MathTables* mt, double2 (&g)[NDET]) {
  const BinBasis b = make_basis(tb, k, MODEL == 2);
  double q, amp = 1.0;
  if (MODEL == 1) {
    q = fma(cb(CB_PH + 0), b.y5, cb(CB_PH + 4));
    q = fma(cb(CB_PH + 1), b.y3, q);
    q = fma(cb(CB_PH + 2), b.y2, q);
    q = fma(cb(CB_PH + 3), b.y, q);
    q = fma(cb(CB_PH + 5), b.L, q);
    q = fma(cb(CB_PH + 6), b.x, q);
    q = fma(cb(CB_PH + 7), b.xL, q);
    q = fma(cb(CB_PH + 8), b.x2, q);
    q = fma(cb(CB_PH + 9), b.f, q);
  } else {
    phenom_bin_t(cb, b, mt, exp_tab(cb(CB_AM + 3) * (b.f - cb(CB_AM + 0)), mt), q, amp);
  }
#pragma unroll
  for (int d = 0; d < NDET; ++d) {
    double sn, cs;
    sincos_lut(64.0 * fma(-cb(CB_DET + 4 * d + 2), b.f, q), mt, sn, cs);
    const double cr = cb(CB_DET + 4 * d), ci = cb(CB_DET + 4 * d + 1);
    g[d] = make_double2(amp * fma(cr, cs, ci * sn), amp * fma(ci, cs, -(cr * sn)));
  }
}

// Delta(f_k) of reading L24, one thread per grid bin.
__global__ void k_rb_delta(const DevCfg* __restrict__ cfg, double chi, double* delta) {
  const int nf = cfg->n_freq;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= nf) return;
  const double f = cfg->f_min + k * cfg->df, f_lo = cfg->f_min, f_hi = cfg->f_min + (nf - 1) * cfg->df;
  const double g[5] = {-5.0 / 3.0, -2.0 / 3.0, 1.0, 5.0 / 3.0, 7.0 / 3.0};
  double s = 0.0;
  for (int i = 0; i < 5; ++i) s += (g[i] < 0.0) ? -pow(f / f_lo, g[i]) : pow(f / f_hi, g[i]);
  delta[k] = 2.0 * kPi * chi * s;
}

// Bin edges equally spaced in Delta (sequential, as the reading states it; N_f steps in total).  out[0] = number of bins.
__global__ void k_rb_select(const DevCfg* __restrict__ cfg, const double* __restrict__ delta, double eps, int cap, int* nb_out, int* edge) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const int nf = cfg->n_freq;
  const double d0 = delta[0], dtot = delta[nf - 1] - d0;
  const double want = floor(dtot / eps);
  if (!(want <= 4.0 * nf)) { *nb_out = -1; return; }     // eps far below what the grid resolves
  const int nb_req = max(1, (int)want);
  int n = 0, k = 0;
  edge[n++] = 0;
  for (int i = 1; i < nb_req && n < cap - 1; ++i) {
    const double target = i * (dtot / nb_req);
    while (k < nf - 1 && delta[k] - d0 < target) ++k;
    if (k > edge[n - 1] && k < nf - 1) edge[n++] = k;
  }
  edge[n++] = nf - 1;
  *nb_out = n - 1;
}

// Summary data: CTA b sums grid bins [e_b, e_b+1) (the last one up to and including e_nb) for every detector; fixed-order
// reduction.  Also 1/g0 at the edges and 1/(bin width).
template <int MODEL, int NDET>
__global__ void __launch_bounds__(128) k_rb_summary(const DevCfg* __restrict__ cfgp, Tables tb, const double* __restrict__ cb0_g,
                                                    const int* __restrict__ edge, int nb, double2* A0, double2* A1, double* B0, double* B1,
                                                    double2* ig0, double* inv_w) {
  constexpr int NT = 128, NW = NT / 32, NV = 6 * NDET;
  __shared__ MathTables mtab;
  __shared__ double cb0[CB_SIZE];
  __shared__ double red[NW * NV], out[NV];
  const int tid = threadIdx.x, b = blockIdx.x;
  load_math_tables(&mtab, tb.mt, tid, NT);
  for (int i = tid; i < CB_SIZE; i += NT) cb0[i] = cb0_g[i];
  __syncthreads();
  const CbPtr cb{cb0};
  const int k_lo = edge[b], k_hi = (b == nb - 1) ? edge[b + 1] + 1 : edge[b + 1];
  const double f_lo = __ldg(tb.f + edge[b]), f_hi = __ldg(tb.f + edge[b + 1]);
  const double fm = 0.5 * (f_lo + f_hi);
  double v[NV];
#pragma unroll
  for (int i = 0; i < NV; ++i) v[i] = 0.0;
  for (int k = k_lo + tid; k < k_hi; k += NT) {
    double2 g[NDET];
    gw_g_at<MODEL, NDET>(cb, tb, k, &mtab, g);
    const double df_ = __ldg(tb.f + k) - fm;
#pragma unroll
    for (int d = 0; d < NDET; ++d) {
      const double2 w = __ldg(tb.wd[d] + k);
      // wd conj(g0)
      const double zr = fma(w.x, g[d].x, w.y * g[d].y), zi = fma(w.y, g[d].x, -(w.x * g[d].y));
      const double h2 = __ldg(tb.ws[d] + k) * fma(g[d].x, g[d].x, g[d].y * g[d].y);
      v[6 * d + 0] += zr; v[6 * d + 1] += zi;
      v[6 * d + 2] = fma(zr, df_, v[6 * d + 2]); v[6 * d + 3] = fma(zi, df_, v[6 * d + 3]);
      v[6 * d + 4] += h2; v[6 * d + 5] = fma(h2, df_, v[6 * d + 5]);
    }
  }
  block_reduce<NV, NT>(v, red, out);
  if (tid < NDET) {
    const int d = tid;
    A0[(size_t)d * nb + b] = make_double2(out[6 * d + 0], out[6 * d + 1]);
    A1[(size_t)d * nb + b] = make_double2(out[6 * d + 2], out[6 * d + 3]);
    B0[(size_t)d * nb + b] = out[6 * d + 4];
    B1[(size_t)d * nb + b] = out[6 * d + 5];
  }
  if (tid == 32) inv_w[b] = 1.0 / (f_hi - f_lo);
  if (tid == 64 || (tid == 96 && b == nb - 1)) {
    const int i = (tid == 64) ? b : nb;
    double2 g[NDET];
    gw_g_at<MODEL, NDET>(cb, tb, edge[i], &mtab, g);
#pragma unroll
    for (int d = 0; d < NDET; ++d) {
      const double den = 1.0 / fma(g[d].x, g[d].x, g[d].y * g[d].y);
      ig0[(size_t)d * (nb + 1) + i] = make_double2(g[d].x * den, -g[d].y * den);
    }
  }
}

// Evaluation: one thread per particle, loop over the N_b + 1 edges (all lanes at the same edge).  The per-edge data -- the ten
// basis values, f^3/4, 1/g0 per detector -- and the per-bin summary data are staged once per CTA in shared memory (18 + 8 n_det
// and 1 + 6 n_det doubles per edge / bin) and read with warp-uniform LDS; ratio r = g/g0 at the edge, then the bin between the
// previous edge and this one.
constexpr int kRbThreads = 128;

template <int NDET>
struct RbEdge {           // one edge (and the bin that ends at it)
  double y5, y3, y2, y, L, x, xL, x2, f, f34;
  double2 ig0[NDET];      // 1 / g0 at the edge
  double2 A0[NDET], A1[NDET];
  double B0[NDET], B1[NDET];
  double inv_w;
  double pad;
};

template <int MODEL, int NDET, class CB>
__device__ __forceinline__ void gw_g_edge(const CB& cb, const RbEdge<NDET>& e, const MathTables* mt, double2 (&g)[NDET]) {
  BinBasis b;
  b.y5 = e.y5; b.y3 = e.y3; b.y2 = e.y2; b.y = e.y; b.L = e.L; b.x = e.x; b.xL = e.xL; b.x2 = e.x2; b.f = e.f; b.f34 = e.f34;
  double q, amp = 1.0;
  if (MODEL == 1) {
    q = fma(cb(CB_PH + 0), b.y5, cb(CB_PH + 4));
    q = fma(cb(CB_PH + 1), b.y3, q);
    q = fma(cb(CB_PH + 2), b.y2, q);
    q = fma(cb(CB_PH + 3), b.y, q);
    q = fma(cb(CB_PH + 5), b.L, q);
    q = fma(cb(CB_PH + 6), b.x, q);
    q = fma(cb(CB_PH + 7), b.xL, q);
    q = fma(cb(CB_PH + 8), b.x2, q);
    q = fma(cb(CB_PH + 9), b.f, q);
  } else {
    phenom_bin_t(cb, b, mt, exp_tab(cb(CB_AM + 3) * (b.f - cb(CB_AM + 0)), mt), q, amp);
  }
#pragma unroll
  for (int d = 0; d < NDET; ++d) {
    double sn, cs;
    sincos_lut(64.0 * fma(-cb(CB_DET + 4 * d + 2), b.f, q), mt, sn, cs);
    const double cr = cb(CB_DET + 4 * d), ci = cb(CB_DET + 4 * d + 1);
    g[d] = make_double2(amp * fma(cr, cs, ci * sn), amp * fma(ci, cs, -(cr * sn)));
  }
}

template <int MODEL, int NDET>
__global__ void __launch_bounds__(kRbThreads) k_relbin(const DevCfg* __restrict__ cfgp, Tables tb, RbDev rb, const double* __restrict__ cbs_g,
                                                        long long B, double* logl, double* parts) {
  constexpr int NT = kRbThreads;
  __shared__ MathTables mtab;
  extern __shared__ __align__(16) unsigned char rb_smem[];
  const int nb = rb.nb;
  RbEdge<NDET>* ed = reinterpret_cast<RbEdge<NDET>*>(rb_smem);                    // [nb + 1]
  double* rb_cbT = reinterpret_cast<double*>(ed + (nb + 1));                       // PhenomD-form: [CB_SIZE][NT], transposed
  const int tid = threadIdx.x;
  const long long p0 = (long long)blockIdx.x * NT, p = p0 + tid;
  const bool have = p < B;
  load_math_tables(&mtab, tb.mt, tid, NT);
  for (int i = tid; i <= nb; i += NT) {
    const int k = __ldg(rb.edge + i);
    const BinBasis b = make_basis(tb, k, MODEL == 2);
    RbEdge<NDET> e;
    e.y5 = b.y5; e.y3 = b.y3; e.y2 = b.y2; e.y = b.y; e.L = b.L; e.x = b.x; e.xL = b.xL; e.x2 = b.x2; e.f = b.f; e.f34 = b.f34;
    e.inv_w = (i > 0) ? __ldg(rb.inv_w + (i - 1)) : 0.0;
    e.pad = 0.0;
#pragma unroll
    for (int d = 0; d < NDET; ++d) {
      e.ig0[d] = __ldg(rb.ig0 + (size_t)d * (nb + 1) + i);
      const size_t ib = (size_t)d * nb + (i > 0 ? i - 1 : 0);
      e.A0[d] = __ldg(rb.A0 + ib); e.A1[d] = __ldg(rb.A1 + ib); e.B0[d] = __ldg(rb.B0 + ib); e.B1[d] = __ldg(rb.B1 + ib);
    }
    ed[i] = e;
  }
  // coefficient block of this thread's particle: TaylorF2 -> registers; PhenomD-form -> shared memory, transposed
  double cbl[MODEL == 1 ? 30 : 1];
  if (MODEL == 1) {
#pragma unroll
    for (int i = 0; i < 30; ++i) cbl[i] = have ? __ldg(cbs_g + p * CB_SIZE + i) : 0.0;
  } else {
    for (int e = tid; e < NT * CB_SIZE; e += NT) {
      const int part = e % NT, i = e / NT;
      rb_cbT[i * NT + part] = (p0 + part < B) ? __ldg(cbs_g + (p0 + part) * CB_SIZE + i) : 0.0;
    }
  }
  __syncthreads();
  double2 prev[NDET];
  double dh[NDET], hh[NDET];
#pragma unroll
  for (int d = 0; d < NDET; ++d) { dh[d] = 0.0; hh[d] = 0.0; prev[d] = make_double2(0.0, 0.0); }
#pragma unroll 2
  for (int i = 0; i <= nb; ++i) {
    const RbEdge<NDET>& e = ed[i];
    double2 g[NDET];
    if (MODEL == 1) gw_g_edge<MODEL, NDET>(CbPtr{cbl}, e, &mtab, g);
    else gw_g_edge<MODEL, NDET>(CbStrided{rb_cbT + tid, NT}, e, &mtab, g);
#pragma unroll
    for (int d = 0; d < NDET; ++d) {
      const double2 ig = e.ig0[d];
      const double2 r = make_double2(fma(g[d].x, ig.x, -(g[d].y * ig.y)), fma(g[d].x, ig.y, g[d].y * ig.x));
      if (i > 0) {
        const double iw = e.inv_w;
        const double r0r = 0.5 * (prev[d].x + r.x), r0i = 0.5 * (prev[d].y + r.y);
        const double r1r = (r.x - prev[d].x) * iw, r1i = (r.y - prev[d].y) * iw;
        const double2 a0 = e.A0[d], a1 = e.A1[d];
        dh[d] += fma(a0.x, r0r, a0.y * r0i) + fma(a1.x, r1r, a1.y * r1i);
        hh[d] += fma(e.B0[d], fma(r0r, r0r, r0i * r0i), 2.0 * e.B1[d] * fma(r0r, r1r, r0i * r1i));
      }
      prev[d] = r;
    }
  }
  if (!have) return;
  const bool valid = ((MODEL == 1) ? cbl[CB_VALID] : rb_cbT[CB_VALID * NT + tid]) != 0.0;
  double l = 0.0;
#pragma unroll
  for (int d = 0; d < NDET; ++d) {
    if (parts) { parts[p * 2 * NDET + 2 * d] = valid ? dh[d] : nan(""); parts[p * 2 * NDET + 2 * d + 1] = valid ? hh[d] : nan(""); }
    l += dh[d] - 0.5 * hh[d];
  }
  logl[p] = valid ? l : -INFINITY;
}

// shared memory of k_relbin: the staged edges (+ the transposed coefficient blocks for PhenomD-form)
template <int MODEL, int NDET>
size_t relbin_smem_bytes(int nb) {
  return sizeof(RbEdge<NDET>) * ((size_t)nb + 1) + (MODEL == 2 ? sizeof(double) * CB_SIZE * kRbThreads : 0);
}

// ======================================================================================================
// K2: acceptance walk
// ======================================================================================================
struct WalkArgs {
  const double* donors;  // [m, D]
  int m;
  double* u;             // [B, D]
  double* logl;          // [B]
  long long B;
  double lstar;
  const double* lstar_dev;  // if non-null overrides lstar
  int W;
  const int* W_dev;         // if non-null overrides W
  uint32_t k0, k1, stream_id;
  const long long* iter_dev;  // if non-null: stream_id |= (*iter & 0xFFFFFF)
  long long slot0;
  int* n_accept; int* n_eval; int* n_oob;
  uint8_t* tflags; double* tlogl;
  int trace_stride;
  int spec;                 // speculative steps per chunk: cap (1..kWalkDMax) of the per-walker adaptive length ...
  int spec_fixed;           // ... or, if non-zero, the fixed length
  int spec_cap;             // chunk buffers in shared memory hold this many steps (>= spec)
};

// DE proposal for one walker (footnote P:120; R:L8-L10).  Returns false if out of bounds.
__device__ __forceinline__ bool de_propose(const DevCfg& cfg, const WalkArgs& a, uint32_t sid, uint32_t t, uint32_t slot,
                                           const double* cur, double* prop) {
  uint32_t b0[4];
  philox4x32_10(0u, t, slot, sid, a.k0, a.k1, b0);
  uint32_t ia = __umulhi(b0[0], (uint32_t)a.m);
  uint32_t ib = __umulhi(b0[1], (uint32_t)(a.m - 1));
  ib += (ib >= ia) ? 1u : 0u;
  double gamma = 1.0;
  if (b0[2] >= 0x80000000u) {
    uint32_t b1[4], b2[4];
    philox4x32_10(1u, t, slot, sid, a.k0, a.k1, b1);
    philox4x32_10(2u, t, slot, sid, a.k0, a.k1, b2);
    double prod = ((u01(b1[0], b1[1]) * u01(b1[2], b1[3])) * u01(b2[0], b2[1])) * u01(b2[2], b2[3]);
    gamma = (2.38 / sqrt(2.0 * cfg.n_free)) * (-0.25 * log(prod));
  }
  const int D = cfg.ndim;
  bool inb = true;
  for (int d = 0; d < D; ++d) {
    if (cfg.prior_kind[d] == 4) { prop[d] = cur[d]; continue; }
    double diff = a.donors[(size_t)ia * D + d] - a.donors[(size_t)ib * D + d];
    double x = fma(gamma, diff, cur[d]);
    if (cfg.periodic[d]) x = x - floor(x);
    else if (!(x > 0.0 && x < 1.0)) inb = false;
    prop[d] = x;
  }
  return inb;
}

__device__ __forceinline__ double simple_loglike(const DevCfg& cfg, const double* u) {
  const int D = cfg.ndim;
  if (cfg.like_kind == 3) {
    double r = 0.0;
    for (int d = 0; d < D; ++d) r = fmax(r, fabs(u[d] - 0.5));
    return -r;
  }
  double th[kMaxDim];
  for (int d = 0; d < D; ++d) th[d] = prior_transform_dim(cfg.prior_kind[d], cfg.prior_lo[d], cfg.prior_hi[d], u[d]) - cfg.toy_mean[d];
  double qf = 0.0;
  for (int i = 0; i < D; ++i)
    for (int j = 0; j < D; ++j) qf += th[i] * cfg.toy_prec[i * D + j] * th[j];
  return cfg.toy_lognorm - 0.5 * qf;
}

__global__ void k_loglike_simple(const DevCfg* __restrict__ cfgp, const double* __restrict__ u, long long B, double* logl) {
  long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= B) return;
  double uu[kMaxDim];
  for (int d = 0; d < cfgp->ndim; ++d) uu[d] = u[i * cfgp->ndim + d];
  logl[i] = simple_loglike(*cfgp, uu);
}

__global__ void k_walk_simple(const DevCfg* __restrict__ cfgp, WalkArgs a) {
  long long row = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (row >= a.B) return;
  const DevCfg& cfg = *cfgp;
  const int D = cfg.ndim;
  const int W = a.W_dev ? *a.W_dev : a.W;
  const double lstar = a.lstar_dev ? *a.lstar_dev : a.lstar;
  const uint32_t sid = a.stream_id | (a.iter_dev ? (uint32_t)(*a.iter_dev & 0xFFFFFF) : 0u);
  const uint32_t slot = (uint32_t)(a.slot0 + row);
  double cur[kMaxDim], prop[kMaxDim];
  for (int d = 0; d < D; ++d) cur[d] = a.u[row * D + d];
  double curl = a.logl[row];
  int na = 0, ne = 0, no = 0;
  for (int t = 0; t < W; ++t) {
    bool inb = de_propose(cfg, a, sid, (uint32_t)t, slot, cur, prop);
    uint8_t fl = 0;
    double pl = nan("");
    if (!inb) { ++no; fl = 1; }
    else {
      pl = simple_loglike(cfg, prop);
      ++ne; fl = 4;
      if (pl > lstar) {
        for (int d = 0; d < D; ++d) cur[d] = prop[d];
        curl = pl; ++na; fl |= 2;
      }
    }
    if (a.tflags) a.tflags[row * a.trace_stride + t] = fl;
    if (a.tlogl) a.tlogl[row * a.trace_stride + t] = pl;
  }
  for (int d = 0; d < D; ++d) a.u[row * D + d] = cur[d];
  a.logl[row] = curl;
  if (a.n_accept) a.n_accept[row] = na;
  if (a.n_eval) a.n_eval[row] = ne;
  if (a.n_oob) a.n_oob[row] = no;
}

// GW walk: one CTA per walker, all W steps in one launch, speculative chunks of up to DMAX steps.
//
// A walker's chain is serial (proposal t+1 starts from the point accepted at t), and one step is: propose + transform + ~3 kflop
// of serial waveform set-up by ONE thread, then a bin sweep.  With acceptance rates of 0.1-10 % per step the outcome "rejected" is
// almost certain, so the kernel works on a CHUNK of future steps at once, all proposed from the current point: warp 0 draws the
// proposals of steps t0, t0+1, ... 32 at a time (Philox counters are per step) until E of them are in bounds, builds the E
// coefficient blocks side by side (SIMT: E set-ups for the latency of one), the physical ones are swept PG at a time (shared
// table loads, ILP), and thread 0 then walks through the chunk's steps in order: out-of-bounds -> counted; logL' > L* -> accepted,
// and the steps after it are DISCARDED (they started from a stale point) and redone in the next chunk from t0 + j + 1.  The
// decisions, counters and trace are exactly those of the sequential algorithm (oracle_walk); only work is wasted, never semantics
// changed.  Each walker adapts its own E (start 2; halved after a chunk with an acceptance, doubled up to the slot cap after one
// without), or E is fixed by option.
constexpr int kWalkDMax = 32;   // evaluations per chunk (cap): one warp sets them up side by side
constexpr int kWalkPG = 2;     // particles per bin sweep
constexpr int kWalkSteps = 128;   // steps per chunk (cap): proposals are drawn 32 at a time until enough are in bounds

template <int MODEL, int NDET, int PG, int NT>
__device__ __forceinline__ void sweep_group(const DevCfg& cfg, const Tables& tb, const double* cbs, const double2* tabL,
                                            const double2* tabW, const double2* step, const MathTables* mt, const bool* active,
                                            const int* slot, double* red, double* out /*smem [PG][N]*/) {
  using AL = AccLayout<MODEL, NDET>;
  constexpr int NV = PG * AL::N;
  double acc[PG][AL::N];
  bin_loop<MODEL, NDET, PG, NT>(cfg, tb, cbs, tabL, tabW, step, mt, active, slot, acc);
  double v[NV];
#pragma unroll
  for (int p = 0; p < PG; ++p)
#pragma unroll
    for (int i = 0; i < AL::N; ++i) v[p * AL::N + i] = acc[p][i];
  block_reduce<NV, NT>(v, red, out);
}

// dynamic shared memory of k_walk_gw for a chunk cap of dm steps
template <int NDET, int NT>
constexpr size_t walk_smem_bytes(int dm) {
  return sizeof(double2) * dm * (NDET > 1 ? NDET - 1 : 1) * (32 + NT / 32 + 1) + sizeof(double) * dm * (CB_SIZE + kMaxDim);
}

// NT threads per walker: 128 when all walkers of the batch are resident at 4 CTAs per SM, 96 (5 per SM) or 64 (8 per SM) when
// that keeps a larger batch in one wave (config 4: k = 700 on 148 SMs).
// RB: the likelihood of a proposal is the relative-binning one (edges instead of a full bin sweep).
template <int MODEL, int NDET, int NT, bool RB>
__global__ void __launch_bounds__(NT, 512 / NT) k_walk_gw(const DevCfg* __restrict__ cfgp, Tables tb, WalkArgs a, RbDev rb) {
  using AL = AccLayout<MODEL, NDET>;
  constexpr int NW = NT / 32, PG = kWalkPG, ND1 = NDET > 1 ? NDET - 1 : 1;
  constexpr int DMX = kWalkDMax;
  const int DM = max(1, min(DMX, a.spec_cap));   // buffers are carved for this many steps per chunk
  // per-chunk buffers in dynamic shared memory (WalkSmem<NDET>::kBytes): coefficient blocks, phasor tables, proposals
  extern __shared__ __align__(16) unsigned char walk_smem[];
  double2* tabL = reinterpret_cast<double2*>(walk_smem);          // [DM][ND1][32]
  double2* tabW = tabL + DM * ND1 * 32;                            // [DM][ND1][NW]
  double2* step = tabW + DM * ND1 * NW;                            // [DM][ND1]
  double* cbs = reinterpret_cast<double*>(step + DM * ND1);        // [DM][CB_SIZE]
  double (*s_prop)[kMaxDim] = reinterpret_cast<double (*)[kMaxDim]>(cbs + DM * CB_SIZE);   // [DM][kMaxDim]
  double2* rbuf = reinterpret_cast<double2*>(cbs + DM * (CB_SIZE + kMaxDim));              // RB: partial sums [32][NT/32][2 NDET]
  __shared__ double red[NW * PG * AL::N], out[PG * AL::N], s_logl[DMX];
  __shared__ MathTables mtab;
  __shared__ bool active[PG];
  __shared__ int slot[PG];
  __shared__ double s_cur[kMaxDim], s_curl;
  __shared__ double s_stage[32][kMaxDim];       // phase A1: one proposal per lane of warp 0
  __shared__ int s_flag[DMX];                   // per slot: 1 in bounds but unphysical theta (logL = -inf), 2 to be swept
  __shared__ unsigned char s_step[kWalkSteps];  // per step of the chunk: 0 out of bounds, else slot + 1
  __shared__ int s_t0, s_d, s_nsteps, s_nslots;
  const DevCfg& cfg = *cfgp;
  const int D = cfg.ndim;
  const int W = a.W_dev ? *a.W_dev : a.W;
  const int spec = max(1, min(DM, a.spec));   // cap of the evaluations per chunk
  const bool spec_fixed = a.spec_fixed != 0;
  const double lstar = a.lstar_dev ? *a.lstar_dev : a.lstar;
  const uint32_t sid = a.stream_id | (a.iter_dev ? (uint32_t)(*a.iter_dev & 0xFFFFFF) : 0u);
  const int tid = threadIdx.x, lane = tid & 31;
  const long long row = blockIdx.x;
  int na = 0, ne = 0, no = 0;   // thread 0's counters
  load_math_tables(&mtab, tb.mt, tid, NT);
  if (tid == 0) {
    for (int d = 0; d < D; ++d) s_cur[d] = a.u[row * D + d];
    s_curl = a.logl[row];
    s_t0 = 0;
    s_d = spec_fixed ? spec : min(spec, 2);
  }
  __syncthreads();
  while (true) {
    const int t0 = s_t0;
    if (t0 >= W) break;
    // ---- phase A (warp 0).  A1: propose steps t0, t0+1, ... 32 at a time from the current point until s_d of them are in
    // bounds (out-of-bounds steps cost a Philox block and 11 FMAs, nothing else) or the step cap is reached; the chunk ends with
    // the step of the last collected in-bounds proposal.  A2: the expensive part -- prior transform and waveform set-up -- for the
    // collected proposals, one per lane, all lanes busy.
    if (tid < 32) {
      const int emax = s_d;
      int nslots = 0, nsteps = 0;
      while (nslots < emax && nsteps < kWalkSteps && t0 + nsteps < W) {
        const int j = nsteps + lane;
        const bool live = j < kWalkSteps && t0 + j < W;
        const bool inb = live && de_propose(cfg, a, sid, (uint32_t)(t0 + j), (uint32_t)(a.slot0 + row), s_cur, s_stage[lane]);
        const unsigned bal = __ballot_sync(0xffffffffu, inb);
        const int rank = __popc(bal & ((1u << lane) - 1u));
        const int room = emax - nslots, cnt = __popc(bal);
        int consumed = min(32, min(kWalkSteps - nsteps, W - t0 - nsteps));
        if (cnt > room) {   // more in-bounds proposals than slots left: stop right after the room-th one
          const unsigned m2 = __ballot_sync(0xffffffffu, inb && rank == room - 1);
          consumed = __ffs(m2);
        }
        if (lane < consumed) {
          s_step[j] = inb ? (unsigned char)(nslots + rank + 1) : 0;
          if (inb)
            for (int d = 0; d < D; ++d) s_prop[nslots + rank][d] = s_stage[lane][d];
        }
        nslots += min(cnt, room);
        nsteps += consumed;
        __syncwarp();
      }
      if (lane == 0) { s_nsteps = nsteps; s_nslots = nslots; }
      if (lane < nslots) {
        double th[11];
#pragma unroll
        for (int d = 0; d < 11; ++d) th[d] = prior_transform_dim(cfg.prior_kind[d], cfg.prior_lo[d], cfg.prior_hi[d], s_prop[lane][d]);
        s_flag[lane] = setup_particle<MODEL>(cfg, th, cbs + lane * CB_SIZE) ? 2 : 1;
      }
    }
    __syncthreads();
    const int nd = s_nslots, nsteps = s_nsteps;
    // the proposals that need a sweep, in order (every thread counts them the same way)
    int n_in = 0;
#pragma unroll
    for (int j = 0; j < DMX; ++j) n_in += (j < nd && s_flag[j] == 2) ? 1 : 0;
    if (RB && n_in > 0) {
      // ---- phase B, relative binning: NT/32 threads per proposal, each walks a contiguous run of bins edge by edge (ratio r = g/g0
      // at the edge, then the bin between the previous edge and this one; the first edge of a run is recomputed by its owner), no
      // barrier until the partial sums meet in shared memory
      constexpr int T = NT / 32;
      const int nbn = rb.nb;
      const int sl = tid / T, part = tid % T;
      double v[2 * NDET];
#pragma unroll
      for (int i = 0; i < 2 * NDET; ++i) v[i] = 0.0;
      if (sl < nd && s_flag[sl] == 2) {
        const CbPtr cb{cbs + sl * CB_SIZE};
        const int per = (nbn + T - 1) / T, b0 = part * per, b1 = min(nbn, b0 + per);
        double2 prev[NDET];
        for (int i = b0; i <= b1 && b0 < b1; ++i) {
          double2 g[NDET];
          gw_g_at<MODEL, NDET>(cb, tb, __ldg(rb.edge + i), &mtab, g);
#pragma unroll
          for (int d = 0; d < NDET; ++d) {
            const double2 ig = __ldg(rb.ig0 + (size_t)d * (nbn + 1) + i);
            const double2 r = make_double2(fma(g[d].x, ig.x, -(g[d].y * ig.y)), fma(g[d].x, ig.y, g[d].y * ig.x));
            if (i > b0) {
              const size_t ib = (size_t)d * nbn + (i - 1);
              const double iw = __ldg(rb.inv_w + (i - 1));
              const double r0r = 0.5 * (prev[d].x + r.x), r0i = 0.5 * (prev[d].y + r.y);
              const double r1r = (r.x - prev[d].x) * iw, r1i = (r.y - prev[d].y) * iw;
              const double2 a0 = __ldg(rb.A0 + ib), a1 = __ldg(rb.A1 + ib);
              v[2 * d] += fma(a0.x, r0r, a0.y * r0i) + fma(a1.x, r1r, a1.y * r1i);
              v[2 * d + 1] += fma(__ldg(rb.B0 + ib), fma(r0r, r0r, r0i * r0i), 2.0 * __ldg(rb.B1 + ib) * fma(r0r, r1r, r0i * r1i));
            }
            prev[d] = r;
          }
        }
      }
      double* rpart = reinterpret_cast<double*>(rbuf);      // [32 slots][T][2 NDET]
#pragma unroll
      for (int i = 0; i < 2 * NDET; ++i) rpart[(sl * T + part) * 2 * NDET + i] = v[i];
      __syncthreads();
      if (part == 0 && sl < nd && s_flag[sl] == 2) {
        double l = 0.0;
#pragma unroll
        for (int d = 0; d < NDET; ++d) {
          double dh = 0.0, hh = 0.0;
#pragma unroll
          for (int t = 0; t < T; ++t) { dh += rpart[(sl * T + t) * 2 * NDET + 2 * d]; hh += rpart[(sl * T + t) * 2 * NDET + 2 * d + 1]; }
          l += dh - 0.5 * hh;
        }
        s_logl[sl] = l;
      }
      __syncthreads();
    }
    if (!RB && n_in > 0) {
      build_phasor_tables<NDET, NT>(cfg, cbs, nd, tabL, tabW, step);
      __syncthreads();
      // ---- phase B: sweeps, PG particles at a time (a single left-over goes through the one-particle loop)
      for (int g = 0; g < n_in; g += PG) {
        const int ng = min(PG, n_in - g);
        if (tid < PG) {
          int cnt = 0, mine = -1, first = 0;
#pragma unroll
          for (int j = 0; j < DMX; ++j) {
            if (j < nd && s_flag[j] == 2) {
              if (cnt == g) first = j;
              if (cnt == g + tid) mine = j;
              ++cnt;
            }
          }
          slot[tid] = (mine >= 0) ? mine : first;
          active[tid] = mine >= 0;
        }
        __syncthreads();
        if (ng == PG) sweep_group<MODEL, NDET, PG, NT>(cfg, tb, cbs, tabL, tabW, step, &mtab, active, slot, red, out);
        else sweep_group<MODEL, NDET, 1, NT>(cfg, tb, cbs, tabL, tabW, step, &mtab, active, slot, red, out);
        if (tid < ng) s_logl[slot[tid]] = finish_logl<MODEL, NDET>(cfg, cbs + slot[tid] * CB_SIZE, out + tid * AL::N, nullptr);
        __syncthreads();
      }
    }
    // ---- phase C: the chunk's steps in order; the first acceptance invalidates the rest of the chunk
    if (tid == 0) {
      int used = nsteps;
      bool hit = false;
      for (int j = 0; j < nsteps; ++j) {
        const int t = t0 + j;
        const int sl = (int)s_step[j] - 1;
        if (sl < 0) {
          ++no;
          if (a.tflags) a.tflags[row * a.trace_stride + t] = 1;
          if (a.tlogl) a.tlogl[row * a.trace_stride + t] = nan("");
          continue;
        }
        ++ne;
        const double pl = (s_flag[sl] == 2) ? s_logl[sl] : -INFINITY;
        uint8_t tf = 4;
        const bool acc_ = pl > lstar;
        if (acc_) {
          for (int d = 0; d < D; ++d) s_cur[d] = s_prop[sl][d];
          s_curl = pl; ++na; tf |= 2;
        }
        if (a.tflags) a.tflags[row * a.trace_stride + t] = tf;
        if (a.tlogl) a.tlogl[row * a.trace_stride + t] = pl;
        if (acc_) { used = j + 1; hit = true; break; }
      }
      s_t0 = t0 + used;
      // per-walker chunk size (evaluations): halve after a chunk that ended in an acceptance (the rest of it was wasted), double
      // after one that did not; a function of the walker's own chain only, so still deterministic
      if (!spec_fixed) s_d = hit ? max(1, s_d >> 1) : min(spec, s_d << 1);
    }
    __syncthreads();
  }
  if (tid == 0) {
    for (int d = 0; d < D; ++d) a.u[row * D + d] = s_cur[d];
    a.logl[row] = s_curl;
    if (a.n_accept) a.n_accept[row] = na;
    if (a.n_eval) a.n_eval[row] = ne;
    if (a.n_oob) a.n_oob[row] = no;
  }
}

// ======================================================================================================
// K3: selection, evidence, replacement, adaptation
// ======================================================================================================
// Stable rank by counting: order[rank(i)] = i with rank(i) = #{j : l_j < l_i or (l_j == l_i and j < i)}  (R:L6).
__global__ void k_rank(const double* __restrict__ logl, int n, int* order) {
  __shared__ double tile[256];
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  double li = (i < n) ? logl[i] : 0.0;
  int rank = 0;
  for (int base = 0; base < n; base += 256) {
    int j = base + threadIdx.x;
    tile[threadIdx.x] = (j < n) ? logl[j] : INFINITY;
    __syncthreads();
    int lim = min(256, n - base);
    for (int jj = 0; jj < lim; ++jj) {
      double lj = tile[jj];
      rank += (lj < li) || (lj == li && (base + jj) < i);
    }
    __syncthreads();
  }
  if (i < n) order[rank] = i;
}

__device__ __forceinline__ double logaddexp_d(double a, double b) {
  if (a == -INFINITY) return b;
  if (b == -INFINITY) return a;
  double m = fmax(a, b);
  return m + log1p(exp(-fabs(a - b)));
}

__device__ __forceinline__ void evidence_update(double li, double ni, double& logx, double& logz, double& h, double& logw) {
  logw = logx + log(-expm1(-1.0 / ni));
  double lw = li + logw;
  double zn = logaddexp_d(logz, lw);
  double hn = exp(lw - zn) * li;
  if (logz != -INFINITY) hn += exp(logz - zn) * (h + logz);
  hn -= zn;
  h = hn; logz = zn; logx -= 1.0 / ni;
}

// Sequential evidence scan over the k dead points in ascending logL (eq. 3-5 with the saw-tooth live count; R:L16, L17).
__global__ void k_evidence(DevState* st, const double* __restrict__ logl, const double* __restrict__ u, const int* __restrict__ order,
                           int n, int k, int D, double* dead) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double logx = st->logx, logz = st->logz, h = st->h;
  for (int i = 0; i < k; ++i) {
    int id = order[i];
    double logw;
    evidence_update(logl[id], (double)(n - i), logx, logz, h, logw);
    if (dead) {
      double* row = dead + (size_t)i * (D + 3);
      for (int d = 0; d < D; ++d) row[d] = u[(size_t)id * D + d];
      row[D] = logl[id]; row[D + 1] = logw; row[D + 2] = (double)(n - i);
    }
  }
  st->logx = logx; st->logz = logz; st->h = h;
  st->lstar = logl[order[k - 1]];
  int W = (int)floor(st->walks);
  st->W = max(1, min(W, st->maxmcmc));
}

// Survivor array in ascending-logL order + start points (uniform survivor, Philox tag 1; R:L7).
__global__ void k_gather_start(const DevState* __restrict__ st, const double* __restrict__ u, const double* __restrict__ logl,
                               const int* __restrict__ order, int n, int k, int D, uint32_t k0, uint32_t k1, double* surv, double* cur_u,
                               double* cur_l) {
  const int m = n - k;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < m) {
    int id = order[k + i];
    for (int d = 0; d < D; ++d) surv[(size_t)i * D + d] = u[(size_t)id * D + d];
  }
  if (i < k) {
    uint32_t w[4];
    philox4x32_10(0u, 0u, (uint32_t)i, (1u << 24) | (uint32_t)(st->iter & 0xFFFFFF), k0, k1, w);
    int id = order[k + __umulhi(w[0], (uint32_t)m)];
    for (int d = 0; d < D; ++d) cur_u[(size_t)i * D + d] = u[(size_t)id * D + d];
    cur_l[i] = logl[id];
  }
}

__global__ void k_writeback(const int* __restrict__ order, int k, int D, const double* __restrict__ cur_u, const double* __restrict__ cur_l,
                            double* u, double* logl) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= k) return;
  int id = order[j];
  for (int d = 0; d < D; ++d) u[(size_t)id * D + d] = cur_u[(size_t)j * D + d];
  logl[id] = cur_l[j];
}

// Batch-level adaptation (R:L13-L15) and termination quantities (R:L18).  Single CTA, fixed-order reductions.
__global__ void k_adapt(DevState* st, const int* __restrict__ na, const int* __restrict__ ne, const int* __restrict__ no, int k,
                        const double* __restrict__ logl, int n) {
  __shared__ long long s_a[256], s_e[256], s_o[256], s_s[256];
  __shared__ int s_min[256], s_max[256];
  __shared__ double s_d[256];
  const int t = threadIdx.x;
  long long a = 0, e = 0, o = 0, s = 0;
  int mn = INT_MAX, mx = INT_MIN;
  for (int j = t; j < k; j += 256) {
    a += na[j]; e += ne[j]; o += no[j]; s += (na[j] == 0);
    mn = min(mn, na[j]); mx = max(mx, na[j]);
  }
  s_a[t] = a; s_e[t] = e; s_o[t] = o; s_s[t] = s; s_min[t] = mn; s_max[t] = mx;
  double lm = -INFINITY;
  for (int i = t; i < n; i += 256) lm = fmax(lm, logl[i]);
  s_d[t] = lm;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (t < w) {
      s_a[t] += s_a[t + w]; s_e[t] += s_e[t + w]; s_o[t] += s_o[t + w]; s_s[t] += s_s[t + w];
      s_min[t] = min(s_min[t], s_min[t + w]); s_max[t] = max(s_max[t], s_max[t + w]);
      s_d[t] = fmax(s_d[t], s_d[t + w]);
    }
    __syncthreads();
  }
  const double lmax = s_d[0];
  __syncthreads();
  double acc = 0.0;
  for (int i = t; i < n; i += 256) acc += exp(logl[i] - lmax);
  s_d[t] = acc;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (t < w) s_d[t] += s_d[t + w];
    __syncthreads();
  }
  if (t == 0) {
    const int W = st->W;
    double amean = (double)s_a[0] / k;
    double r = fmax(0.5, amean) / W;
    double walks = fmin((st->walks * st->delay + st->naccept / r) / (st->delay + 1.0), (double)st->maxmcmc);
    st->walks = walks;
    st->n_eval_total += s_e[0];
    double lse = lmax + log(s_d[0]);
    ns_stats& o_ = st->stats;
    o_.iteration = st->iter;
    o_.logl_star = st->lstar; o_.logx = st->logx; o_.logz = st->logz; o_.h = st->h;
    o_.dlogz = logaddexp_d(st->logz, lmax + st->logx) - st->logz;
    o_.live_frac_log = lse - log((double)n) + st->logx - st->logz;
    o_.walk_len = W; o_.pad0 = 0; o_.walks_next = walks;
    o_.accept_mean = amean; o_.accept_min = s_min[0]; o_.accept_max = s_max[0];
    o_.n_eval = s_e[0]; o_.n_oob = s_o[0]; o_.n_stuck = s_s[0]; o_.n_eval_total = st->n_eval_total;
    st->iter += 1;
  }
}

// Final evidence: adds the live points with n_i = n..1 to a copy of the accumulators (R:L17).  out: logz, h.
__global__ void k_finalize(const DevState* __restrict__ st, const double* __restrict__ logl, const int* __restrict__ order, int n,
                           double* out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double logx = st->logx, logz = st->logz, h = st->h, lw;
  for (int i = 0; i < n; ++i) evidence_update(logl[order[i]], (double)(n - i), logx, logz, h, lw);
  out[0] = logz; out[1] = h;
}

// FP64 FMA throughput probe: 8 independent chains per thread.
__global__ void k_dfma_probe(long long iters, double* sink) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const double m = 0.999999, c = 1e-7;
  for (long long i = 0; i < iters; ++i) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) sink[0] = s;
}

}  // namespace

// ======================================================================================================
// Host side
// ======================================================================================================
struct ns_handle {
  ns_config cfg;
  DevCfg* d_cfg = nullptr;
  DevState* d_state = nullptr;
  Tables tb{};
  double* d_tab = nullptr;      // four double2 pair tables, f, f34 (10 * nf doubles)
  cudaStream_t s_own = nullptr; // ns_run_many: this run's stream
  // relative binning (ns_relbin_setup)
  int rb_nb = 0;
  int* d_rb_edge = nullptr;      // [rb_nb + 1]
  double* d_rb_buf = nullptr;    // A0, A1 (complex), B0, B1, ig0 (complex), inv_w, cb0, theta0
  RbDev rb{};
  MathTables* d_mtab = nullptr; // sin/cos, exp2, atan tables
  double2* d_wd = nullptr;      // [n_det][nf]
  double* d_ws = nullptr;       // [n_det][nf]
  double* d_live_u = nullptr;   // [n_live][D]
  double* d_live_l = nullptr;
  int* d_order = nullptr;
  double* d_surv = nullptr;     // [n_live - k][D]
  double* d_cur_u = nullptr;    // [k][D]
  double* d_cur_l = nullptr;
  int* d_cnt = nullptr;         // 3 * k
  double* d_cb = nullptr;       // coefficient blocks scratch
  double* d_partial = nullptr;  // k_bins_lp: per-range partial sums [n_ranges][N][B]
  size_t partial_cap = 0;
  int n_sm = 148;
  int opt_like = 0;             // 0 exact likelihood, 1 relative binning (sampler and ns_loglike_u_batch)
  int opt_walk_spec = 0;        // 0 auto (per-walker adaptive), 1..32 fixed speculative chunk length
  int opt_bins_kernel = 0;      // 0 auto, 1 CTA-per-particle (k_bins), 2 lane-per-particle (k_bins_lp; TaylorF2 only)
  long long cb_cap = 0;
  double* d_theta = nullptr;    // scratch theta
  long long theta_cap = 0;
  double* d_hio = nullptr;      // host-entry scratch: theta [B,11] + logl [B]
  long long hio_cap = 0;
  double* d_fin = nullptr;      // 2 doubles
  ns_stats* h_stats = nullptr;  // pinned
  double* h_fin = nullptr;      // pinned
  uint64_t seed = 0;
  std::string err;
  int n_free = 0;
  bool prof = false;                                   // nsgw_profile_enable
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_ev;  // event pairs around the dominant kernel
};

namespace {

int fail(ns_handle* h, int code, const std::string& msg) {
  if (h) h->err = msg; else g_init_error = msg;
  return code;
}

#define CU_CHECK(h, expr)                                                                         \
  do {                                                                                            \
    cudaError_t e_ = (expr);                                                                      \
    if (e_ != cudaSuccess)                                                                        \
      return fail(h, e_ == cudaErrorMemoryAllocation ? -4 : -2, std::string(#expr) + ": " + cudaGetErrorString(e_)); \
  } while (0)

#define LAUNCH_CHECK(h)                                                                           \
  do {                                                                                            \
    g_launches.fetch_add(1);                                                                      \
    cudaError_t e_ = cudaGetLastError();                                                          \
    if (e_ != cudaSuccess) return fail(h, -2, std::string("kernel launch: ") + cudaGetErrorString(e_)); \
  } while (0)

const double kSurrogate[19][2] = {
    {3931.9, -17395.8}, {-40105.5, 112253.0}, {83208.4, -191237.7}, {0.81498, 2.57476}, {0.0069274, 0.0302047},
    {1.010344, 0.000899}, {1.308162, -0.005538}, {2096.55, 1463.75}, {-10114.06, -44631.0}, {22933.66, 230960.0},
    {-14621.7, -377812.9}, {97.8975, -42.6597}, {-3.28270, -9.05138}, {-2.51564e-5, 1.97503e-5}, {43.3151, 638.633},
    {-0.0702021, -0.162698}, {9.59881, -397.054}, {-0.0298949, 1.40221}, {0.997441, -0.00788445}};

bool is_gw(int kind) { return kind == NSGW_LIKE_GW_TAYLORF2 || kind == NSGW_LIKE_GW_PHENOMD_FORM; }

int ensure_cb(ns_handle* h, long long B) {
  if (B > h->cb_cap) {
    if (h->d_cb) cudaFree(h->d_cb);
    h->d_cb = nullptr; h->cb_cap = 0;
    CU_CHECK(h, cudaMalloc(&h->d_cb, sizeof(double) * CB_SIZE * (size_t)B));
    h->cb_cap = B;
  }
  return 0;
}
int ensure_theta(ns_handle* h, long long B) {
  if (B > h->theta_cap) {
    if (h->d_theta) cudaFree(h->d_theta);
    h->d_theta = nullptr; h->theta_cap = 0;
    CU_CHECK(h, cudaMalloc(&h->d_theta, sizeof(double) * 16 * (size_t)B));
    h->theta_cap = B;
  }
  return 0;
}

// particles per CTA of the bin loop as a function of the batch (fill 148 SMs first, then reuse table loads)
int pick_p(long long B) { return B >= 4096 ? 2 : 1; }

// Lane-per-particle kernel (k_bins_lp): geometry and the batch size from which it is used (TaylorF2 only).
// (the four numbers can be overridden at compile time for tuning sweeps)
#ifndef NSGW_LP_NT
#define NSGW_LP_NT 128
#define NSGW_LP_PP 2
#define NSGW_LP_UNR 4
#define NSGW_LP_OCC 3
#endif
constexpr int kLpNT = NSGW_LP_NT, kLpKR = 256, kLpPP = NSGW_LP_PP, kLpUNR = NSGW_LP_UNR, kLpOCC = NSGW_LP_OCC;
constexpr long long kLpMinBatch = 2048;   // below this the CTA-per-particle kernel fills the machine better

int ensure_partial(ns_handle* h, size_t n) {
  if (n > h->partial_cap) {
    if (h->d_partial) cudaFree(h->d_partial);
    h->d_partial = nullptr; h->partial_cap = 0;
    CU_CHECK(h, cudaMalloc(&h->d_partial, sizeof(double) * n));
    h->partial_cap = n;
  }
  return 0;
}

template <int NDET>
int launch_bins_lp(ns_handle* h, long long B, double* logl, double* parts, cudaStream_t s) {
  using AL = AccLayout<1, NDET>;
  constexpr int NT = kLpNT, PP = kLpPP;
  const long long ngroups = (B + NT * PP - 1) / (NT * PP);
  const long long grid_max = (long long)h->n_sm * kLpOCC;
  // bins per task (multiple of the unroll, 32..256): the value that minimises rounds x (bins per task + per-task overhead),
  // rounds = ceil(tasks / resident CTAs) -- large tiles amortise the per-task set-up, small ones balance the last round
  int kr = kLpKR;
  {
    double best = 1e300;
    for (int c = 32; c <= kLpKR; c += kLpUNR) {
      const long long nt = ngroups * ((h->cfg.n_freq + c - 1) / c);
      const double cost = (double)((nt + grid_max - 1) / grid_max) * (c + 8);
      if (cost < best - 1e-9) { best = cost; kr = c; }
    }
  }
  const int nranges = (h->cfg.n_freq + kr - 1) / kr;
  const long long ntasks = ngroups * nranges;
  const long long grid = std::min<long long>(ntasks, grid_max);
  int rc = ensure_partial(h, (size_t)B * nranges * AL::N);
  if (rc) return rc;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (h->prof && h->prof_ev.size() < 4096) {
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0, s);
  }
  k_bins_lp<NDET, NT, kLpKR, PP, kLpUNR, kLpOCC><<<(unsigned)grid, NT, 0, s>>>(h->d_cfg, h->tb, h->d_cb, B, kr, nranges, ntasks,
                                                                              h->d_partial);
  if (e0) { cudaEventRecord(e1, s); h->prof_ev.emplace_back(e0, e1); }
  LAUNCH_CHECK(h);
  k_finish<1, NDET><<<(unsigned)((B + 127) / 128), 128, 0, s>>>(h->d_cfg, h->d_cb, h->d_partial, nranges, B, logl, parts);
  LAUNCH_CHECK(h);
  return 0;
}

template <int MODEL, int NDET>
int launch_bins_nd(ns_handle* h, long long B, double* logl, double* parts, cudaStream_t s) {
  if (MODEL == 1 && (h->opt_bins_kernel == 2 || (h->opt_bins_kernel == 0 && B >= kLpMinBatch)))
    return launch_bins_lp<NDET>(h, B, logl, parts, s);
  int P = pick_p(B);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (h->prof && h->prof_ev.size() < 4096) {
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0, s);
  }
  if (P == 2) {
    k_bins<MODEL, NDET, 2><<<(unsigned)((B + 1) / 2), kBinsThreads, 0, s>>>(h->d_cfg, h->tb, h->d_cb, B, logl, parts);
  } else {
    k_bins<MODEL, NDET, 1><<<(unsigned)B, kBinsThreads, 0, s>>>(h->d_cfg, h->tb, h->d_cb, B, logl, parts);
  }
  if (e0) { cudaEventRecord(e1, s); h->prof_ev.emplace_back(e0, e1); }
  LAUNCH_CHECK(h);
  return 0;
}
template <int MODEL>
int launch_bins(ns_handle* h, long long B, double* logl, double* parts, cudaStream_t s) {
  switch (h->cfg.n_det) {
    case 1: return launch_bins_nd<MODEL, 1>(h, B, logl, parts, s);
    case 2: return launch_bins_nd<MODEL, 2>(h, B, logl, parts, s);
    case 3: return launch_bins_nd<MODEL, 3>(h, B, logl, parts, s);
    default: return fail(h, -5, "n_det must be 1..3 for the GW kernels");
  }
}

int loglike_theta(ns_handle* h, const double* theta_dev, long long B, double* logl, double* parts, cudaStream_t s) {
  if (B == 0) return 0;
  int rc = ensure_cb(h, B);
  if (rc) return rc;
  unsigned g = (unsigned)((B + 127) / 128);
  if (h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2) {
    k_setup<1><<<g, 128, 0, s>>>(h->d_cfg, theta_dev, B, h->d_cb);
    LAUNCH_CHECK(h);
    return launch_bins<1>(h, B, logl, parts, s);
  }
  k_setup<2><<<g, 128, 0, s>>>(h->d_cfg, theta_dev, B, h->d_cb);
  LAUNCH_CHECK(h);
  return launch_bins<2>(h, B, logl, parts, s);
}

// theta[B,11] -> relative-binning logL (set-up kernel + edge evaluation).
int relbin_theta(ns_handle* h, const double* theta_dev, long long B, double* logl, double* parts, cudaStream_t s) {
  if (B == 0) return 0;
  int rc = ensure_cb(h, B);
  if (rc) return rc;
  const unsigned gs = (unsigned)((B + 127) / 128), gr = (unsigned)((B + kRbThreads - 1) / kRbThreads);
  const bool tf2 = h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2;
  const int nd = h->cfg.n_det;
  if (tf2) k_setup<1><<<gs, 128, 0, s>>>(h->d_cfg, theta_dev, B, h->d_cb);
  else k_setup<2><<<gs, 128, 0, s>>>(h->d_cfg, theta_dev, B, h->d_cb);
  LAUNCH_CHECK(h);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (h->prof && h->prof_ev.size() < 4096) {
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0, s);
  }
  const int nbn = h->rb_nb;
#define RB_EVAL(M, N)                                                                                                  \
  do {                                                                                                                 \
    const size_t sm_ = relbin_smem_bytes<M, N>(nbn);                                                                   \
    if (sm_ > 200 * 1024) return fail(h, -5, "too many relative-binning bins for one CTA's shared memory");            \
    if (sm_ > 48 * 1024) CU_CHECK(h, cudaFuncSetAttribute(k_relbin<M, N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_)); \
    k_relbin<M, N><<<gr, kRbThreads, sm_, s>>>(h->d_cfg, h->tb, h->rb, h->d_cb, B, logl, parts);                       \
  } while (0)
  if (tf2) { if (nd == 1) RB_EVAL(1, 1); else if (nd == 2) RB_EVAL(1, 2); else RB_EVAL(1, 3); }
  else { if (nd == 1) RB_EVAL(2, 1); else if (nd == 2) RB_EVAL(2, 2); else RB_EVAL(2, 3); }
#undef RB_EVAL
  if (e0) { cudaEventRecord(e1, s); h->prof_ev.emplace_back(e0, e1); }
  LAUNCH_CHECK(h);
  return 0;
}


int loglike_u(ns_handle* h, const double* u_dev, long long B, double* logl, cudaStream_t s) {
  if (B == 0) return 0;
  if (!is_gw(h->cfg.like_kind)) {
    k_loglike_simple<<<(unsigned)((B + 127) / 128), 128, 0, s>>>(h->d_cfg, u_dev, B, logl);
    LAUNCH_CHECK(h);
    return 0;
  }
  int rc = ensure_theta(h, B);
  if (rc) return rc;
  long long N = B * h->cfg.ndim;
  k_prior_transform<<<(unsigned)((N + 255) / 256), 256, 0, s>>>(h->d_cfg, u_dev, B, h->d_theta);
  LAUNCH_CHECK(h);
  if (h->opt_like == 1) return relbin_theta(h, h->d_theta, B, logl, nullptr, s);
  return loglike_theta(h, h->d_theta, B, logl, nullptr, s);
}

template <int MODEL, int NDET, int NT, bool RB>
int launch_walk_gw_k(ns_handle* h, WalkArgs a, int dm, cudaStream_t s) {
  auto kern = k_walk_gw<MODEL, NDET, NT, RB>;
  const size_t extra = RB ? sizeof(double) * NT * 2 * NDET : 0;   // partial sums of phase B
  static bool attr_set = false;
  if (!attr_set) {
    CU_CHECK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)(walk_smem_bytes<NDET, NT>(kWalkDMax) + extra)));
    attr_set = true;
  }
  a.spec_cap = dm;
  a.spec = std::min(a.spec, dm);
  kern<<<(unsigned)a.B, NT, walk_smem_bytes<NDET, NT>(dm) + extra, s>>>(h->d_cfg, h->tb, a, h->rb);
  LAUNCH_CHECK(h);
  return 0;
}

template <int MODEL, int NDET, int NT>
int launch_walk_gw_nt(ns_handle* h, const WalkArgs& a, int dm, cudaStream_t s) {
  return launch_walk_gw_k<MODEL, NDET, NT, false>(h, a, dm, s);
}

// Longest chunk buffers (32, 16 or 8 slots) with which `ctas` CTAs of the kernel still fit the SM's shared memory.
template <int NDET, int NT>
int walk_chunk_cap(const ns_handle* h, int ctas) {
  const size_t extra = h->opt_like == 1 ? sizeof(double) * NT * 2 * NDET : 0;
  for (int dm = kWalkDMax; dm > 8; dm /= 2)
    if ((size_t)ctas * (walk_smem_bytes<NDET, NT>(dm) + extra + 10496) <= (size_t)225 * 1024) return dm;
  return 8;
}

// Geometry by batch size: the widest CTA (and the longest chunk buffers) that still keeps every walker resident at once.
template <int MODEL, int NDET>
int launch_walk_gw(ns_handle* h, const WalkArgs& a, cudaStream_t s) {
  const long long sm = h->n_sm;
  // relative binning: the sweep is 62-odd edge evaluations, residency is not what limits it -- one geometry (128 threads)
  if (h->opt_like == 1) return launch_walk_gw_k<MODEL, NDET, 128, true>(h, a, walk_chunk_cap<NDET, 128>(h, 4), s);
  if (a.B <= 4 * sm || a.B > 8 * sm)   // <= 4 walkers per SM, or many waves anyway
    return launch_walk_gw_nt<MODEL, NDET, 128>(h, a, walk_chunk_cap<NDET, 128>(h, 4), s);
  if (a.B <= 5 * sm) return launch_walk_gw_nt<MODEL, NDET, 96>(h, a, walk_chunk_cap<NDET, 96>(h, 5), s);
  return launch_walk_gw_nt<MODEL, NDET, 64>(h, a, walk_chunk_cap<NDET, 64>(h, 8), s);
}

int launch_walk(ns_handle* h, const WalkArgs& a, cudaStream_t s) {
  if (a.B == 0) return 0;
  if (!is_gw(h->cfg.like_kind)) {
    k_walk_simple<<<(unsigned)((a.B + 63) / 64), 64, 0, s>>>(h->d_cfg, a);
    LAUNCH_CHECK(h);
    return 0;
  }
  const int nd = h->cfg.n_det;
  if (h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2) {
    if (nd == 1) return launch_walk_gw<1, 1>(h, a, s);
    if (nd == 2) return launch_walk_gw<1, 2>(h, a, s);
    if (nd == 3) return launch_walk_gw<1, 3>(h, a, s);
  } else {
    if (nd == 1) return launch_walk_gw<2, 1>(h, a, s);
    if (nd == 2) return launch_walk_gw<2, 2>(h, a, s);
    if (nd == 3) return launch_walk_gw<2, 3>(h, a, s);
  }
  return fail(h, -5, "n_det must be 1..3 for the GW kernels");
}

}  // namespace

extern "C" {

const char* ns_last_error(const ns_handle* h) { return h ? h->err.c_str() : g_init_error.c_str(); }

int64_t nsgw_launch_count(void) { return g_launches.load(); }

void ns_free(ns_handle* h) {
  if (!h) return;
  cudaFree(h->d_cfg); cudaFree(h->d_state); cudaFree(h->d_tab); cudaFree(h->d_mtab); cudaFree(h->d_wd); cudaFree(h->d_ws);
  cudaFree(h->d_live_u); cudaFree(h->d_live_l); cudaFree(h->d_order); cudaFree(h->d_surv); cudaFree(h->d_cur_u);
  cudaFree(h->d_cur_l); cudaFree(h->d_cnt); cudaFree(h->d_cb); cudaFree(h->d_partial); cudaFree(h->d_theta); cudaFree(h->d_fin); cudaFree(h->d_hio);
  if (h->s_own) cudaStreamDestroy(h->s_own);
  cudaFree(h->d_rb_edge); cudaFree(h->d_rb_buf);
  if (h->h_stats) cudaFreeHost(h->h_stats);
  if (h->h_fin) cudaFreeHost(h->h_fin);
  for (auto& pr : h->prof_ev) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
  delete h;
}

int ns_init(ns_handle** out, const ns_config* cfg, const double* live_u_dev, const double* strain_dev, const double* psd_dev,
            uint64_t seed, void* stream) {
  if (!out || !cfg) return fail(nullptr, -1, "null argument");
  *out = nullptr;
  if (cfg->struct_version != NSGW_STRUCT_VERSION) return fail(nullptr, -1, "struct_version mismatch");
  if (cfg->ndim < 1 || cfg->ndim > NSGW_MAX_DIM) return fail(nullptr, -1, "ndim out of range");
  if (cfg->like_kind < 0 || cfg->like_kind > 3) return fail(nullptr, -5, "unknown like_kind");
  const bool gw = is_gw(cfg->like_kind);
  if (gw && cfg->ndim != 11) return fail(nullptr, -5, "GW likelihoods need ndim = 11");
  if (gw && (cfg->n_det < 1 || cfg->n_det > 3)) return fail(nullptr, -5, "GW kernels are built for n_det = 1..3");
  if (gw && (cfg->n_freq < 1 || !(cfg->df > 0.0) || !(cfg->f_min > 0.0))) return fail(nullptr, -1, "bad frequency grid");
  if (gw && (!strain_dev || !psd_dev)) return fail(nullptr, -1, "GW likelihoods need strain and PSD");
  if (cfg->n_live < 0) return fail(nullptr, -1, "n_live < 0");
  if (cfg->n_live > 0) {
    if (cfg->n_delete < 1 || cfg->n_delete > cfg->n_live - 2) return fail(nullptr, -1, "need 1 <= n_delete <= n_live - 2");
    if (cfg->naccept < 1 || cfg->maxmcmc < 1 || !(cfg->walks0 >= 1.0)) return fail(nullptr, -1, "bad naccept/maxmcmc/walks0");
  }
  int n_free = 0;
  for (int d = 0; d < cfg->ndim; ++d) {
    if (cfg->prior_kind[d] < 0 || cfg->prior_kind[d] > 4) return fail(nullptr, -1, "bad prior kind");
    if (cfg->prior_kind[d] != NSGW_PRIOR_FIXED) {
      ++n_free;
      if (!(cfg->prior_hi[d] > cfg->prior_lo[d])) return fail(nullptr, -1, "prior hi must exceed lo");
    }
  }
  if (n_free == 0) return fail(nullptr, -1, "no free dimension");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(nullptr, -2, "no CUDA device (there is no CPU fallback)");

  cudaStream_t s = (cudaStream_t)stream;
  ns_handle* h = new ns_handle();
  {
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (h->n_sm < 1) h->n_sm = 148;
  }
  h->cfg = *cfg;
  h->cfg.phenom_table_host = nullptr;
  h->seed = seed;
  h->n_free = n_free;
  auto bail = [&](int rc) { g_init_error = h->err; ns_free(h); return rc; };

  // ---- device config
  DevCfg hc;
  memset(&hc, 0, sizeof(hc));
  hc.like_kind = cfg->like_kind; hc.ndim = cfg->ndim; hc.n_free = n_free; hc.n_det = gw ? cfg->n_det : 0; hc.n_freq = gw ? cfg->n_freq : 0;
  for (int d = 0; d < cfg->ndim; ++d) {
    hc.prior_kind[d] = cfg->prior_kind[d]; hc.periodic[d] = cfg->periodic[d];
    hc.prior_lo[d] = cfg->prior_lo[d]; hc.prior_hi[d] = cfg->prior_hi[d];
    hc.toy_mean[d] = cfg->toy_mean[d];
  }
  for (int i = 0; i < cfg->ndim * cfg->ndim; ++i) hc.toy_prec[i] = cfg->toy_prec[i];
  hc.toy_lognorm = cfg->toy_lognorm;
  hc.f_min = cfg->f_min; hc.df = cfg->df; hc.gmst = cfg->gmst;
  for (int d = 0; d < hc.n_det; ++d) {
    const double* x = cfg->det_xarm[d];
    const double* y = cfg->det_yarm[d];
    for (int j = 0; j < 3; ++j) hc.det_vertex[d][j] = cfg->det_vertex[d][j];
    int idx = 0;
    for (int i = 0; i < 3; ++i)
      for (int j = i; j < 3; ++j) hc.det_D[d][idx++] = 0.5 * (x[i] * x[j] - y[i] * y[j]);
  }
  for (int r = 0; r < 19; ++r)
    for (int c = 0; c < 11; ++c)
      hc.table[r][c] = cfg->phenom_table_host ? cfg->phenom_table_host[r * 11 + c] : (c < 2 ? kSurrogate[r][c] : 0.0);
  if (cudaMalloc(&h->d_cfg, sizeof(DevCfg)) != cudaSuccess) { h->err = "cudaMalloc cfg"; return bail(-4); }
  if (cudaMemcpyAsync(h->d_cfg, &hc, sizeof(DevCfg), cudaMemcpyHostToDevice, s) != cudaSuccess) { h->err = "H2D cfg"; return bail(-2); }

#define INIT_CHECK(expr, code)                                                        \
  do {                                                                                \
    cudaError_t e_ = (expr);                                                          \
    if (e_ != cudaSuccess) { h->err = std::string(#expr) + ": " + cudaGetErrorString(e_); return bail(e_ == cudaErrorMemoryAllocation ? -4 : code); } \
  } while (0)

  // ---- GW tables
  if (gw) {
    const size_t nf = cfg->n_freq, nd = cfg->n_det;
    // validate PSD on the host side of the boundary is impossible without a copy; do it on a host copy (init-time only)
    {
      std::vector<double> hp(nf * nd);
      INIT_CHECK(cudaMemcpyAsync(hp.data(), psd_dev, sizeof(double) * nf * nd, cudaMemcpyDeviceToHost, s), -2);
      INIT_CHECK(cudaStreamSynchronize(s), -2);
      for (double v : hp)
        if (!(v > 0.0) || !std::isfinite(v)) { h->err = "PSD values must be positive and finite"; return bail(-1); }
    }
    INIT_CHECK(cudaMalloc(&h->d_tab, sizeof(double) * 10 * nf), -2);
    INIT_CHECK(cudaMalloc(&h->d_wd, sizeof(double2) * nd * nf), -2);
    INIT_CHECK(cudaMalloc(&h->d_ws, sizeof(double) * nd * nf), -2);
    double2* t2 = reinterpret_cast<double2*>(h->d_tab);
    h->tb.t01 = t2; h->tb.t23 = t2 + nf; h->tb.t45 = t2 + 2 * nf; h->tb.t67 = t2 + 3 * nf;
    h->tb.f = h->d_tab + 8 * nf; h->tb.f34 = h->d_tab + 9 * nf;
    for (size_t d = 0; d < nd; ++d) { h->tb.wd[d] = h->d_wd + d * nf; h->tb.ws[d] = h->d_ws + d * nf; }
    k_tables<<<(unsigned)((nf + 255) / 256), 256, 0, s>>>(h->d_cfg, strain_dev, psd_dev, t2, t2 + nf, t2 + 2 * nf, t2 + 3 * nf,
                                                          h->d_tab + 8 * nf, h->d_tab + 9 * nf, h->d_wd, h->d_ws);
    g_launches.fetch_add(1);
    INIT_CHECK(cudaMalloc(&h->d_mtab, sizeof(MathTables)), -2);
    k_math_tables<<<1, 256, 0, s>>>(h->d_mtab);
    g_launches.fetch_add(1);
    h->tb.mt = h->d_mtab;
    k_i73<<<1, 256, 0, s>>>(h->d_cfg, h->d_ws);
    g_launches.fetch_add(1);
    INIT_CHECK(cudaGetLastError(), -2);
  }

  // ---- sampler state
  INIT_CHECK(cudaMalloc(&h->d_state, sizeof(DevState)), -2);
  INIT_CHECK(cudaMalloc(&h->d_fin, sizeof(double) * 2), -2);
  INIT_CHECK(cudaMallocHost(&h->h_stats, sizeof(ns_stats)), -2);
  INIT_CHECK(cudaMallocHost(&h->h_fin, sizeof(double) * 2), -2);
  const int n = cfg->n_live, k = cfg->n_delete, D = cfg->ndim;
  DevState hs;
  memset(&hs, 0, sizeof(hs));
  hs.logx = 0.0; hs.logz = -INFINITY; hs.h = 0.0; hs.walks = cfg->walks0;
  hs.delay = (n > 0) ? (cfg->delay >= 0.0 ? cfg->delay : std::max((double)n / (10.0 * k) - 1.0, 0.0)) : 0.0;
  hs.iter = 0; hs.n_eval_total = n; hs.W = 1; hs.naccept = cfg->naccept; hs.maxmcmc = cfg->maxmcmc;
  INIT_CHECK(cudaMemcpyAsync(h->d_state, &hs, sizeof(hs), cudaMemcpyHostToDevice, s), -2);
  if (n > 0) {
    INIT_CHECK(cudaMalloc(&h->d_live_u, sizeof(double) * (size_t)n * D), -2);
    INIT_CHECK(cudaMalloc(&h->d_live_l, sizeof(double) * (size_t)n), -2);
    INIT_CHECK(cudaMalloc(&h->d_order, sizeof(int) * (size_t)n), -2);
    INIT_CHECK(cudaMalloc(&h->d_surv, sizeof(double) * (size_t)(n - k) * D), -2);
    INIT_CHECK(cudaMalloc(&h->d_cur_u, sizeof(double) * (size_t)k * D), -2);
    INIT_CHECK(cudaMalloc(&h->d_cur_l, sizeof(double) * (size_t)k), -2);
    INIT_CHECK(cudaMalloc(&h->d_cnt, sizeof(int) * 3 * (size_t)k), -2);
    if (live_u_dev) {
      INIT_CHECK(cudaMemcpyAsync(h->d_live_u, live_u_dev, sizeof(double) * (size_t)n * D, cudaMemcpyDeviceToDevice, s), -2);
    } else {
      k_draw_live<<<(n + 127) / 128, 128, 0, s>>>(D, n, (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32), h->d_live_u);
      g_launches.fetch_add(1);
    }
    int rc = loglike_u(h, h->d_live_u, n, h->d_live_l, s);
    if (rc) return bail(rc);
  }
  INIT_CHECK(cudaStreamSynchronize(s), -2);
  INIT_CHECK(cudaGetLastError(), -2);
#undef INIT_CHECK
  *out = h;
  return 0;
}

int gw_loglike_batch(ns_handle* h, const double* theta_dev, int64_t B, double* logl_dev, double* parts_dev, void* stream) {
  if (!h) return -3;
  if (!is_gw(h->cfg.like_kind)) return fail(h, -3, "handle has no GW likelihood");
  if (B < 0 || (B > 0 && (!theta_dev || !logl_dev))) return fail(h, -1, "bad arguments");
  return loglike_theta(h, theta_dev, B, logl_dev, parts_dev, (cudaStream_t)stream);
}

int gw_loglike_batch_host(ns_handle* h, const double* theta_host, int64_t B, double* logl_host, void* stream) {
  if (!h) return -3;
  if (!is_gw(h->cfg.like_kind)) return fail(h, -3, "handle has no GW likelihood");
  if (B < 0 || (B > 0 && (!theta_host || !logl_host))) return fail(h, -1, "bad arguments");
  if (B == 0) return 0;
  cudaStream_t s = (cudaStream_t)stream;
  if (B > h->hio_cap) {
    if (h->d_hio) cudaFree(h->d_hio);
    h->d_hio = nullptr; h->hio_cap = 0;
    CU_CHECK(h, cudaMalloc(&h->d_hio, sizeof(double) * 12 * (size_t)B));
    h->hio_cap = B;
  }
  double* th = h->d_hio;
  double* lg = h->d_hio + 11 * (size_t)B;
  CU_CHECK(h, cudaMemcpyAsync(th, theta_host, sizeof(double) * 11 * (size_t)B, cudaMemcpyHostToDevice, s));
  int rc = loglike_theta(h, th, B, lg, nullptr, s);
  if (rc) return rc;
  CU_CHECK(h, cudaMemcpyAsync(logl_host, lg, sizeof(double) * (size_t)B, cudaMemcpyDeviceToHost, s));
  CU_CHECK(h, cudaStreamSynchronize(s));
  return 0;
}

int gw_waveform(ns_handle* h, const double* theta_dev, double* out_dev, void* stream) {
  if (!h) return -3;
  if (!is_gw(h->cfg.like_kind)) return fail(h, -3, "handle has no GW likelihood");
  if (!theta_dev || !out_dev) return fail(h, -1, "null argument");
  cudaStream_t s = (cudaStream_t)stream;
  unsigned g = (unsigned)((h->cfg.n_freq + 255) / 256);
  if (h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2) k_waveform<1><<<g, 256, 0, s>>>(h->d_cfg, h->tb, theta_dev, out_dev);
  else k_waveform<2><<<g, 256, 0, s>>>(h->d_cfg, h->tb, theta_dev, out_dev);
  LAUNCH_CHECK(h);
  return 0;
}

int ns_prior_transform_batch(ns_handle* h, const double* u_dev, int64_t B, double* theta_dev, void* stream) {
  if (!h) return -3;
  if (B < 0 || (B > 0 && (!u_dev || !theta_dev))) return fail(h, -1, "bad arguments");
  if (B == 0) return 0;
  long long N = B * h->cfg.ndim;
  k_prior_transform<<<(unsigned)((N + 255) / 256), 256, 0, (cudaStream_t)stream>>>(h->d_cfg, u_dev, B, theta_dev);
  LAUNCH_CHECK(h);
  return 0;
}

int ns_loglike_u_batch(ns_handle* h, const double* u_dev, int64_t B, double* logl_dev, void* stream) {
  if (!h) return -3;
  if (B < 0 || (B > 0 && (!u_dev || !logl_dev))) return fail(h, -1, "bad arguments");
  return loglike_u(h, u_dev, B, logl_dev, (cudaStream_t)stream);
}

int ns_walk_batch(ns_handle* h, const double* donors_u_dev, int32_t m, double* u_dev, double* logl_dev, int64_t B, double logl_star,
                  int32_t walk_len, uint64_t seed, uint32_t stream_id, int64_t slot0, int32_t* n_accept_dev, int32_t* n_eval_dev,
                  int32_t* n_oob_dev, uint8_t* trace_flags_dev, double* trace_logl_dev, void* stream) {
  if (!h) return -3;
  if (B < 0 || m < 2 || walk_len < 1 || !donors_u_dev || (B > 0 && (!u_dev || !logl_dev))) return fail(h, -1, "bad arguments");
  WalkArgs a;
  memset(&a, 0, sizeof(a));
  a.donors = donors_u_dev; a.m = m; a.u = u_dev; a.logl = logl_dev; a.B = B; a.lstar = logl_star; a.W = walk_len;
  a.k0 = (uint32_t)(seed & 0xFFFFFFFFull); a.k1 = (uint32_t)(seed >> 32); a.stream_id = stream_id; a.slot0 = slot0;
  a.n_accept = n_accept_dev; a.n_eval = n_eval_dev; a.n_oob = n_oob_dev; a.tflags = trace_flags_dev; a.tlogl = trace_logl_dev;
  a.trace_stride = walk_len;
  a.spec = h->opt_walk_spec > 0 ? h->opt_walk_spec : kWalkDMax;
  a.spec_fixed = h->opt_walk_spec > 0;
  return launch_walk(h, a, (cudaStream_t)stream);
}

}  // extern "C"

namespace {
// One nested-sampling iteration enqueued on stream s (no synchronisation, no host read-back).
int step_enqueue(ns_handle* h, double* dead_dev, cudaStream_t s) {
  const int n = h->cfg.n_live, k = h->cfg.n_delete, D = h->cfg.ndim, m = n - k;
  const uint32_t k0 = (uint32_t)(h->seed & 0xFFFFFFFFull), k1 = (uint32_t)(h->seed >> 32);
  k_rank<<<(n + 255) / 256, 256, 0, s>>>(h->d_live_l, n, h->d_order);
  LAUNCH_CHECK(h);
  k_evidence<<<1, 32, 0, s>>>(h->d_state, h->d_live_l, h->d_live_u, h->d_order, n, k, D, dead_dev);
  LAUNCH_CHECK(h);
  k_gather_start<<<(std::max(m, k) + 127) / 128, 128, 0, s>>>(h->d_state, h->d_live_u, h->d_live_l, h->d_order, n, k, D, k0, k1, h->d_surv,
                                                            h->d_cur_u, h->d_cur_l);
  LAUNCH_CHECK(h);
  WalkArgs a;
  memset(&a, 0, sizeof(a));
  a.donors = h->d_surv; a.m = m; a.u = h->d_cur_u; a.logl = h->d_cur_l; a.B = k;
  a.lstar_dev = &h->d_state->lstar; a.W_dev = &h->d_state->W; a.iter_dev = &h->d_state->iter;
  a.spec = h->opt_walk_spec > 0 ? h->opt_walk_spec : kWalkDMax;
  a.spec_fixed = h->opt_walk_spec > 0;
  a.k0 = k0; a.k1 = k1; a.stream_id = 0u; a.slot0 = 0;
  a.n_accept = h->d_cnt; a.n_eval = h->d_cnt + k; a.n_oob = h->d_cnt + 2 * k;
  int rc = launch_walk(h, a, s);
  if (rc) return rc;
  k_writeback<<<(k + 127) / 128, 128, 0, s>>>(h->d_order, k, D, h->d_cur_u, h->d_cur_l, h->d_live_u, h->d_live_l);
  LAUNCH_CHECK(h);
  k_adapt<<<1, 256, 0, s>>>(h->d_state, h->d_cnt, h->d_cnt + k, h->d_cnt + 2 * k, k, h->d_live_l, n);
  LAUNCH_CHECK(h);
  return 0;
}
}  // namespace

extern "C" {

int ns_step(ns_handle* h, ns_stats* stats_host, double* dead_dev, void* stream) {
  if (!h) return -3;
  if (h->cfg.n_live <= 0) return fail(h, -3, "handle has no live set");
  cudaStream_t s = (cudaStream_t)stream;
  int rc = step_enqueue(h, dead_dev, s);
  if (rc) return rc;
  if (stats_host) {
    CU_CHECK(h, cudaMemcpyAsync(h->h_stats, &h->d_state->stats, sizeof(ns_stats), cudaMemcpyDeviceToHost, s));
    CU_CHECK(h, cudaStreamSynchronize(s));
    *stats_host = *h->h_stats;
  }
  return 0;
}

int64_t ns_run(ns_handle* h, int32_t term_kind, double term_tol, int64_t max_iter, ns_stats* last_host, double* dead_dev, void* stream) {
  if (!h) return -3;
  if (term_kind < 0 || term_kind > 1 || max_iter < 0) return fail(h, -1, "bad arguments");
  const size_t stride = (size_t)h->cfg.n_delete * (h->cfg.ndim + 3);
  ns_stats st;
  memset(&st, 0, sizeof(st));
  int64_t it = 0;
  while (it < max_iter) {
    int rc = ns_step(h, &st, dead_dev ? dead_dev + it * stride : nullptr, stream);
    if (rc) return rc;
    ++it;
    if (term_kind == 0 && st.dlogz < term_tol) break;
    if (term_kind == 1 && st.live_frac_log < std::log(term_tol)) break;
  }
  if (last_host) *last_host = st;
  return it;
}

int64_t ns_run_many(ns_handle** hs, int32_t n_runs, int32_t term_kind, double term_tol, int64_t max_iter, ns_stats* last_host,
                    int64_t* iters_host, double** dead_dev) {
  if (!hs || n_runs < 1 || term_kind < 0 || term_kind > 1 || max_iter < 0) return -1;
  for (int r = 0; r < n_runs; ++r) {
    if (!hs[r]) return -3;
    if (hs[r]->cfg.n_live <= 0) return fail(hs[r], -3, "handle has no live set");
    if (!hs[r]->s_own && cudaStreamCreateWithFlags(&hs[r]->s_own, cudaStreamNonBlocking) != cudaSuccess)
      return fail(hs[r], -2, "cudaStreamCreate");
  }
  std::vector<char> active(n_runs, 1);
  std::vector<int64_t> it(n_runs, 0);
  std::vector<ns_stats> st(n_runs);
  memset(st.data(), 0, sizeof(ns_stats) * n_runs);
  int64_t total = 0;
  int n_active = max_iter > 0 ? n_runs : 0;
  while (n_active > 0) {
    // enqueue one iteration of every unfinished run on its own stream: the runs' kernels overlap on the device and fill the
    // SM slots a single run with k = n_live/2 walkers leaves empty (and one another's tails)
    for (int r = 0; r < n_runs; ++r) {
      if (!active[r]) continue;
      ns_handle* h = hs[r];
      const size_t stride = (size_t)h->cfg.n_delete * (h->cfg.ndim + 3);
      int rc = step_enqueue(h, (dead_dev && dead_dev[r]) ? dead_dev[r] + it[r] * stride : nullptr, h->s_own);
      if (rc) return rc;
      CU_CHECK(h, cudaMemcpyAsync(h->h_stats, &h->d_state->stats, sizeof(ns_stats), cudaMemcpyDeviceToHost, h->s_own));
    }
    for (int r = 0; r < n_runs; ++r) {
      if (!active[r]) continue;
      ns_handle* h = hs[r];
      CU_CHECK(h, cudaStreamSynchronize(h->s_own));
      st[r] = *h->h_stats;
      ++it[r]; ++total;
      const bool done = (term_kind == 0) ? (st[r].dlogz < term_tol) : (st[r].live_frac_log < std::log(term_tol));
      if (done || it[r] >= max_iter) { active[r] = 0; --n_active; }
    }
  }
  for (int r = 0; r < n_runs; ++r) {
    if (last_host) last_host[r] = st[r];
    if (iters_host) iters_host[r] = it[r];
  }
  return total;
}

int ns_relbin_setup(ns_handle* h, const double* theta0_host, double chi, double eps, const int32_t* edges_host, int32_t n_edges,
                    int32_t* n_bins_host, void* stream) {
  if (!h) return -3;
  if (!is_gw(h->cfg.like_kind)) return fail(h, -3, "handle has no GW likelihood");
  if (!theta0_host || !(chi > 0.0) || !(eps > 0.0) || h->cfg.n_freq < 2) return fail(h, -1, "bad arguments");
  cudaStream_t s = (cudaStream_t)stream;
  const int nf = h->cfg.n_freq, nd = h->cfg.n_det;
  cudaFree(h->d_rb_edge); cudaFree(h->d_rb_buf);
  h->d_rb_edge = nullptr; h->d_rb_buf = nullptr; h->rb_nb = 0;
  // ---- bin edges: given, or equally spaced in Delta(f) (reading L24)
  std::vector<int> edge;
  if (edges_host) {
    if (n_edges < 2 || edges_host[0] != 0 || edges_host[n_edges - 1] != nf - 1) return fail(h, -1, "edges must run from 0 to n_freq - 1");
    for (int i = 1; i < n_edges; ++i)
      if (edges_host[i] <= edges_host[i - 1]) return fail(h, -1, "edges must increase strictly");
    edge.assign(edges_host, edges_host + n_edges);
  } else {
    double* d_delta = nullptr;
    int* d_sel = nullptr;
    CU_CHECK(h, cudaMalloc(&d_delta, sizeof(double) * nf));
    if (cudaMalloc(&d_sel, sizeof(int) * ((size_t)nf + 2)) != cudaSuccess) { cudaFree(d_delta); return fail(h, -4, "cudaMalloc"); }
    k_rb_delta<<<(nf + 127) / 128, 128, 0, s>>>(h->d_cfg, chi, d_delta);
    k_rb_select<<<1, 1, 0, s>>>(h->d_cfg, d_delta, eps, nf + 1, d_sel, d_sel + 1);
    g_launches.fetch_add(2);
    std::vector<int> sel((size_t)nf + 2);
    cudaError_t e_ = cudaMemcpyAsync(sel.data(), d_sel, sizeof(int) * ((size_t)nf + 2), cudaMemcpyDeviceToHost, s);
    if (e_ == cudaSuccess) e_ = cudaStreamSynchronize(s);
    cudaFree(d_delta); cudaFree(d_sel);
    if (e_ != cudaSuccess) return fail(h, -2, std::string("relbin edges: ") + cudaGetErrorString(e_));
    if (sel[0] < 1) return fail(h, -1, "eps too small for this grid (more than 4 n_freq bins requested)");
    edge.assign(sel.begin() + 1, sel.begin() + 2 + sel[0]);
  }
  const int nb = (int)edge.size() - 1;
  // ---- device buffers: A0, A1 [nd][nb] complex, B0, B1 [nd][nb], ig0 [nd][nb+1] complex, inv_w [nb], cb0 [CB_SIZE], theta0 [16]
  const size_t n_buf = (size_t)nd * nb * 6 + (size_t)nd * (nb + 1) * 2 + nb + CB_SIZE + 16;
  CU_CHECK(h, cudaMalloc(&h->d_rb_edge, sizeof(int) * (nb + 1)));
  CU_CHECK(h, cudaMalloc(&h->d_rb_buf, sizeof(double) * n_buf));
  double* b = h->d_rb_buf;
  double2* A0 = reinterpret_cast<double2*>(b); b += (size_t)nd * nb * 2;
  double2* A1 = reinterpret_cast<double2*>(b); b += (size_t)nd * nb * 2;
  double2* ig0 = reinterpret_cast<double2*>(b); b += (size_t)nd * (nb + 1) * 2;
  double* B0 = b; b += (size_t)nd * nb;
  double* B1 = b; b += (size_t)nd * nb;
  double* inv_w = b; b += nb;
  double* cb0 = b; b += CB_SIZE;
  double* th0 = b;
  CU_CHECK(h, cudaMemcpyAsync(h->d_rb_edge, edge.data(), sizeof(int) * (nb + 1), cudaMemcpyHostToDevice, s));
  CU_CHECK(h, cudaMemcpyAsync(th0, theta0_host, sizeof(double) * 11, cudaMemcpyHostToDevice, s));
  const bool tf2 = h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2;
  if (tf2) k_setup<1><<<1, 32, 0, s>>>(h->d_cfg, th0, 1, cb0);
  else k_setup<2><<<1, 32, 0, s>>>(h->d_cfg, th0, 1, cb0);
  LAUNCH_CHECK(h);
#define RB_SUMMARY(M, N) k_rb_summary<M, N><<<nb, 128, 0, s>>>(h->d_cfg, h->tb, cb0, h->d_rb_edge, nb, A0, A1, B0, B1, ig0, inv_w)
  if (tf2) { if (nd == 1) RB_SUMMARY(1, 1); else if (nd == 2) RB_SUMMARY(1, 2); else RB_SUMMARY(1, 3); }
  else { if (nd == 1) RB_SUMMARY(2, 1); else if (nd == 2) RB_SUMMARY(2, 2); else RB_SUMMARY(2, 3); }
#undef RB_SUMMARY
  LAUNCH_CHECK(h);
  double valid = 0.0;
  CU_CHECK(h, cudaMemcpyAsync(&valid, cb0 + CB_VALID, sizeof(double), cudaMemcpyDeviceToHost, s));
  CU_CHECK(h, cudaStreamSynchronize(s));
  if (valid == 0.0) {
    cudaFree(h->d_rb_edge); cudaFree(h->d_rb_buf);
    h->d_rb_edge = nullptr; h->d_rb_buf = nullptr;
    return fail(h, -1, "fiducial theta0 is unphysical");
  }
  h->rb_nb = nb;
  h->rb.edge = h->d_rb_edge; h->rb.A0 = A0; h->rb.A1 = A1; h->rb.B0 = B0; h->rb.B1 = B1; h->rb.ig0 = ig0; h->rb.inv_w = inv_w; h->rb.nb = nb;
  if (n_bins_host) *n_bins_host = nb;
  return 0;
}

int ns_relbin_get(ns_handle* h, int32_t* edges_host, double* summary_host, void* stream) {
  if (!h) return -3;
  if (h->rb_nb <= 0) return fail(h, -3, "ns_relbin_setup has not been called");
  cudaStream_t s = (cudaStream_t)stream;
  const int nb = h->rb_nb, nd = h->cfg.n_det;
  if (edges_host) CU_CHECK(h, cudaMemcpyAsync(edges_host, h->d_rb_edge, sizeof(int) * (nb + 1), cudaMemcpyDeviceToHost, s));
  if (summary_host) {   // A0 [nd][nb][2], A1 [nd][nb][2], B0 [nd][nb], B1 [nd][nb]
    CU_CHECK(h, cudaMemcpyAsync(summary_host, h->rb.A0, sizeof(double) * (size_t)nd * nb * 4, cudaMemcpyDeviceToHost, s));
    CU_CHECK(h, cudaMemcpyAsync(summary_host + (size_t)nd * nb * 4, h->rb.B0, sizeof(double) * (size_t)nd * nb * 2, cudaMemcpyDeviceToHost, s));
  }
  CU_CHECK(h, cudaStreamSynchronize(s));
  return 0;
}

int gw_loglike_relbin_batch(ns_handle* h, const double* theta_dev, int64_t B, double* logl_dev, double* parts_dev, void* stream) {
  if (!h) return -3;
  if (!is_gw(h->cfg.like_kind)) return fail(h, -3, "handle has no GW likelihood");
  if (h->rb_nb <= 0) return fail(h, -3, "ns_relbin_setup has not been called");
  if (B < 0 || (B > 0 && (!theta_dev || !logl_dev))) return fail(h, -1, "bad arguments");
  return relbin_theta(h, theta_dev, B, logl_dev, parts_dev, (cudaStream_t)stream);
}

int ns_get_live(ns_handle* h, double* u_dev, double* logl_dev, void* stream) {
  if (!h) return -3;
  if (h->cfg.n_live <= 0) return fail(h, -3, "handle has no live set");
  cudaStream_t s = (cudaStream_t)stream;
  const size_t n = h->cfg.n_live, D = h->cfg.ndim;
  if (u_dev) CU_CHECK(h, cudaMemcpyAsync(u_dev, h->d_live_u, sizeof(double) * n * D, cudaMemcpyDeviceToDevice, s));
  if (logl_dev) CU_CHECK(h, cudaMemcpyAsync(logl_dev, h->d_live_l, sizeof(double) * n, cudaMemcpyDeviceToDevice, s));
  return 0;
}

int ns_finalize_evidence(ns_handle* h, double* logz_host, double* logz_err_host, double* h_host, void* stream) {
  if (!h) return -3;
  if (h->cfg.n_live <= 0) return fail(h, -3, "handle has no live set");
  cudaStream_t s = (cudaStream_t)stream;
  const int n = h->cfg.n_live, k = h->cfg.n_delete;
  k_rank<<<(n + 255) / 256, 256, 0, s>>>(h->d_live_l, n, h->d_order);
  LAUNCH_CHECK(h);
  k_finalize<<<1, 32, 0, s>>>(h->d_state, h->d_live_l, h->d_order, n, h->d_fin);
  LAUNCH_CHECK(h);
  CU_CHECK(h, cudaMemcpyAsync(h->h_fin, h->d_fin, sizeof(double) * 2, cudaMemcpyDeviceToHost, s));
  CU_CHECK(h, cudaStreamSynchronize(s));
  const double neff = k / std::log((double)n / (double)(n - k));
  if (logz_host) *logz_host = h->h_fin[0];
  if (h_host) *h_host = h->h_fin[1];
  if (logz_err_host) *logz_err_host = std::sqrt(std::max(h->h_fin[1], 0.0) / neff);
  return 0;
}

int nsgw_set_option(ns_handle* h, int32_t key, int32_t value) {
  if (!h) return -3;
  if (key == NSGW_OPT_BINS_KERNEL && value >= 0 && value <= 2) { h->opt_bins_kernel = value; return 0; }
  if (key == NSGW_OPT_WALK_SPEC && value >= 0 && value <= kWalkDMax) { h->opt_walk_spec = value; return 0; }
  if (key == NSGW_OPT_LIKELIHOOD && (value == 0 || value == 1)) {
    if (!is_gw(h->cfg.like_kind)) return fail(h, -3, "handle has no GW likelihood");
    if (value == 1 && h->rb_nb <= 0) return fail(h, -3, "ns_relbin_setup has not been called");
    h->opt_like = value;
    if (h->cfg.n_live > 0) {   // the live points' logL must come from the likelihood the sampler will compare against
      int rc = loglike_u(h, h->d_live_u, h->cfg.n_live, h->d_live_l, nullptr);
      if (rc) return rc;
      CU_CHECK(h, cudaStreamSynchronize(nullptr));
    }
    return 0;
  }
  return fail(h, -1, "unknown option or value");
}

int nsgw_profile_enable(ns_handle* h, int32_t on) {
  if (!h) return -3;
  h->prof = on != 0;
  return 0;
}

int nsgw_profile_read(ns_handle* h, double* total_ms_host, int64_t* launches_host) {
  if (!h || !total_ms_host || !launches_host) return -1;
  double tot = 0.0;
  for (auto& pr : h->prof_ev) {
    if (cudaEventSynchronize(pr.second) != cudaSuccess) return fail(h, -2, "event sync");
    float ms = 0.f;
    cudaEventElapsedTime(&ms, pr.first, pr.second);
    tot += ms;
    cudaEventDestroy(pr.first); cudaEventDestroy(pr.second);
  }
  *total_ms_host = tot;
  *launches_host = (int64_t)h->prof_ev.size();
  h->prof_ev.clear();
  return 0;
}

int nsgw_measure_fp64_peak(int64_t iters, double* tflops_host, void* stream) {
  if (iters < 1 || !tflops_host) return -1;
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -2;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  double* sink = nullptr;
  if (cudaMalloc(&sink, 8) != cudaSuccess) return -4;
  const int threads = 256, blocks = sms * 8;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  k_dfma_probe<<<blocks, threads, 0, s>>>(iters / 8 + 1, sink);   // warm-up
  cudaEventRecord(e0, s);
  k_dfma_probe<<<blocks, threads, 0, s>>>(iters, sink);
  cudaEventRecord(e1, s);
  g_launches.fetch_add(2);
  cudaError_t e = cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
  if (e != cudaSuccess) return -2;
  *tflops_host = 2.0 * 8.0 * (double)iters * threads * blocks / (ms * 1e-3) / 1e12;
  return 0;
}

}  // extern "C"
