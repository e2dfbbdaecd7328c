// kernels_k1.cuh -- ns_init kernels (tables, live draw, prior transform) and K1: per-particle set-up, the two bin-sweep kernels (k_bins, k_bins_lp), k_finish, k_waveform
// Part of libnsgw (one translation unit): included by nsgw.cu inside its anonymous namespace, after nsgw_device.cuh.
// See include/nsgw.h for the contract and DESIGN.md section 5 for the design of each kernel.
#pragma once

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

__global__ void k_math_tables(MathTables* mt, double2* sc9, double2* sc11) {
  build_math_tables(mt, threadIdx.x, blockDim.x);
  build_sc9(sc9, threadIdx.x, blockDim.x);
  build_sc11(sc11, threadIdx.x, blockDim.x);
}

// k_setup for theta in MAPPED HOST memory (gw_loglike_batch_host with pinned buffers): the CTA's rows are one contiguous block, fetched
// over the host link with coalesced loads into shared memory (a thread reading its own 11 doubles at an 88-byte stride would touch every
// 128-byte line eleven times), then set up one row per thread as k_setup does -- same arithmetic, same coefficient blocks.
template <int MODEL>
__global__ void __launch_bounds__(128) k_setup_staged(const DevCfg* __restrict__ cfg, const double* theta, long long B, double* cbs) {
  __shared__ double th_s[128 * 11];
  const long long r0 = blockIdx.x * 128LL;
  const int n = (int)min(128LL, B - r0);
  for (int i = threadIdx.x; i < n * 11; i += 128) th_s[i] = theta[r0 * 11 + i];
  __syncthreads();
  if ((int)threadIdx.x >= n) return;
  double th[11];
#pragma unroll
  for (int d = 0; d < 11; ++d) th[d] = th_s[threadIdx.x * 11 + d];
  setup_particle<MODEL>(*cfg, th, cbs + (r0 + threadIdx.x) * CB_SIZE);
}

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
                                         double (&acc)[P][AccLayout<MODEL, NDET>::N],
                                         double* stage = nullptr /*smem [NT (3 + 3 NDET)] or null: see the MR loop*/) {
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
    auto mr_bin = [&](int p, double f, double f34, double y3, const double2 (&w)[NDET], const double (&wsv)[NDET]) {
      double q = fma(pm[p][1], f, pm[p][0]);
      q = fma(pm[p][2], y3, q);
      q = fma(pm[p][3], f34, q);
      q = fma(pm[p][4], atan_tab((f - pm[p][5]) * pm[p][6], mt), q);
      const double fx = f - am[p][0];
      const double amp = am[p][1] * rcp_nr1(fma(fx, fx, am[p][2])) * ex[p];
      ex[p] *= exr[p];
      tail(p, q, amp, w, wsv);
    };
    if (stage) {
      // Walk / slice kernels: with 4 CTAs per SM shared memory leaves L1 some 20 KB, every table load comes from L2 (hit rate
      // 8 %) and at the 128-register cap the compiler issues the loads right before their use (25 % of the warp samples waited
      // there).  Each thread therefore stages the seven table values of ITS next bin in a shared-memory slot of its own with
      // LDGSTS while it works on the current bin: same values, same order of arithmetic, bit-identical sums.
      double* sf = stage; double* sf34 = stage + NT; double* sy3 = stage + 2 * NT; double* sws = stage + 3 * NT;
      double2* swd = reinterpret_cast<double2*>(stage + (3 + NDET) * NT);
      auto issue = [&](int k) {
        cp_async8(sf + tid, tb.f + k); cp_async8(sf34 + tid, tb.f34 + k); cp_async8(sy3 + tid, &tb.t01[k].y);
#pragma unroll
        for (int d = 0; d < NDET; ++d) { cp_async8(sws + d * NT + tid, tb.ws[d] + k); cp_async16(swd + d * NT + tid, tb.wd[d] + k); }
      };
      int k = k_mr + tid;
      if (k < nf) issue(k);
      for (; k < nf; k += NT) {
        cp_async_wait_all();
        const double f = sf[tid], f34 = sf34[tid], y3 = sy3[tid];
        double2 w[NDET];
        double wsv[NDET];
#pragma unroll
        for (int d = 0; d < NDET; ++d) { w[d] = swd[d * NT + tid]; wsv[d] = sws[d * NT + tid]; }
#pragma unroll
        for (int p = 0; p < P; ++p) {
          mr_bin(p, f, f34, y3, w, wsv);
          // the slot is free once its values have been consumed by the first particle: fetch the next bin behind the rest
          if (p == 0 && k + NT < nf) issue(k + NT);
        }
      }
    } else {
#pragma unroll 2
      for (int k = k_mr + tid; k < nf; k += NT) {
        const double f = __ldg(tb.f + k), f34 = __ldg(tb.f34 + k);
        const double y3 = __ldg(tb.t01 + k).y;       // 1/f
        double2 w[NDET];
        double wsv[NDET];
#pragma unroll
        for (int d = 0; d < NDET; ++d) { w[d] = __ldg(tb.wd[d] + k); wsv[d] = __ldg(tb.ws[d] + k); }
#pragma unroll
        for (int p = 0; p < P; ++p) mr_bin(p, f, f34, y3, w, wsv);
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
                                                           long long B_host, const int* __restrict__ B_dev /*overrides B_host*/,
                                                           double* logl, double* parts) {
  using AL = AccLayout<MODEL, NDET>;
  constexpr int NT = kBinsThreads, NW = NT / 32, NV = P * AL::N, ND1 = NDET > 1 ? NDET - 1 : 1;
  __shared__ __align__(16) double cbs[P * CB_SIZE];
  __shared__ double2 tabL[P * ND1 * 32], tabW[P * ND1 * NW], step[P * ND1];
  __shared__ double red[NW * NV], out[NV];
  __shared__ MathTables mtab;
  __shared__ bool active[P];
  __shared__ int slot[P];
  const DevCfg& cfg = *cfgp;
  // The coefficient blocks and the device-side row count are the output of the kernel before this one (see pdl_wait); the tables are the
  // handle's.  A batch copies them under that kernel's tail; a round of the worklist walk, whose grid is sized for the row capacity, first
  // lets the surplus CTAs go.
  if (B_dev) pdl_wait();
  const long long B = B_dev ? (long long)*B_dev : B_host;
  if ((long long)blockIdx.x * P >= B) return;
  load_math_tables(&mtab, tb.mt, threadIdx.x, NT);
  if (!B_dev) pdl_wait();
  const long long p0 = (long long)blockIdx.x * P;
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

constexpr double kLpLutScale = 512.0;                          // quarter turns -> 1/2048 turn
constexpr size_t kLpDynSmem = sizeof(double2) * kSc11N;        // the sin/cos table (32 KB)

template <int NDET, int NT, int KR, int PP, int UNR, int OCC>
__global__ void __launch_bounds__(NT, OCC) k_bins_lp(const DevCfg* __restrict__ cfgp, Tables tb, const double* __restrict__ cbs_g,
                                                     long long B_host, const int* __restrict__ B_dev /*overrides the row count; B_host
                                                     stays the stride of `partial`*/, int kr /*bins per range, <= KR, multiple of UNR*/,
                                                     int nranges, long long ntasks_host, double* __restrict__ partial) {
  using AL = AccLayout<1, NDET>;
  constexpr int ND1 = NDET - 1, ND1s = NDET > 1 ? NDET - 1 : 1;
  __shared__ __align__(16) LpSmem<NDET, KR> sm;
  extern __shared__ __align__(16) double2 sc11[];          // kSc11N entries (dynamic: with the tile it is past the 48 KB static limit)
  const DevCfg& cfg = *cfgp;
  const int tid = threadIdx.x;
  const int nf = cfg.n_freq;
  // the table is the handle's (ns_init): its copy runs under the tail of the kernel before this one (k_setup, k_wl_head) when the launch is a
  // programmatic dependent one; the coefficient blocks and the row count are that kernel's output
  for (int i = tid; i < 2 * kSc11N; i += NT) reinterpret_cast<double*>(sc11)[i] = __ldg(reinterpret_cast<const double*>(tb.sc11) + i);
  pdl_wait();
  const long long B = B_dev ? (long long)*B_dev : B_host;
  const long long ntasks = B_dev ? (B + NT * PP - 1) / (NT * PP) * nranges : ntasks_host;
  if (blockIdx.x >= ntasks) return;
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
      for (int i = 0; i < 10; ++i) a[j][i] = have ? kLpLutScale * __ldg(cb + CB_PH + i) : 0.0;   // quarter turns -> table units (exact)
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
        sincos_lut11(q, sc11, sn, cs);
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
        for (int i = 0; i < AL::N; ++i) partial[((long long)rng * AL::N + i) * B_host + p] = acc[j][i];   // [range][N][stride]: coalesced
      }
    }
  }
}

// Adds the per-range partial sums in range order and finishes logL.
template <int MODEL, int NDET>
__global__ void k_finish(const DevCfg* __restrict__ cfgp, const double* __restrict__ cbs_g, const double* __restrict__ partial, int nchunks,
                         long long B, double* logl, double* parts) {
  using AL = AccLayout<MODEL, NDET>;
  pdl_wait();   // (launched as a programmatic dependent of the sweep)
  long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (p >= B) return;
  double sums[AL::N];
#pragma unroll
  for (int i = 0; i < AL::N; ++i) sums[i] = 0.0;
  // range order is the summation order (fixed); loads of eight ranges are issued together (the sums themselves are short chains)
  int c = 0;
  for (; c + 8 <= nchunks; c += 8) {
    double v[8][AL::N];
#pragma unroll
    for (int j = 0; j < 8; ++j)
#pragma unroll
      for (int i = 0; i < AL::N; ++i) v[j][i] = __ldg(partial + ((long long)(c + j) * AL::N + i) * B + p);
#pragma unroll
    for (int j = 0; j < 8; ++j)
#pragma unroll
      for (int i = 0; i < AL::N; ++i) sums[i] += v[j][i];
  }
  for (; c < nchunks; ++c)
#pragma unroll
    for (int i = 0; i < AL::N; ++i) sums[i] += __ldg(partial + ((long long)c * AL::N + i) * B + p);
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

