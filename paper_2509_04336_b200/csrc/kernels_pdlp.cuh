// kernels_pdlp.cuh -- K1 for PhenomD-form at large batches and for the worklist walk: k_pd_lp (lane per particle over the
// merger-ringdown bins + warp per particle over the low-frequency bins) and k_finish_rows.
// Part of libnsgw (one translation unit): included by nsgw.cu inside its anonymous namespace, after kernels_k1.cuh.
//
// Why two mappings in one kernel.  About 80 % of a particle's bins (all above max(f_RD/2, f_peak), CB_FMR) use
// ONE formula -- phase = a + b f + c/f + d f^3/4 + e atan((f - f0)/fd), amplitude = Lorentzian x exponential -- and differ between
// particles only in the coefficients: that part runs lane = particle, coefficients in registers, the bins' table values broadcast
// from a shared-memory tile, no cross-lane reduction, no per-bin global traffic (the design that took TaylorF2 to 0.64 of the FP64
// peak).  Where that region starts depends on the particle (total mass, final spin), so the lanes of a warp disagree on the formula
// for the lowest 10-30 % of bins: those bins run warp = particle, lanes strided over bins, where the three phase and three amplitude
// regions are contiguous in the bin index and the branches are uniform but for one lane at each boundary.
//
// Two launches: k_pd_low (warp per row, many resident warps: that part is latency-bound) and k_pd_lp (nranges x ngroups tasks: group of
// NT x PP rows, range of `kr` bins on the fixed tile grid, persistent CTAs).  Every task writes its rows' partial sums to
// partial[slot][N][stride] (slot = range index, or nranges for the low part); k_finish_rows adds the slots in order.  A row's sums do not depend on which other rows share
// its warp, its task or the launch (masked bins contribute exact zeros; tiles sit on a grid fixed by `kr`), so the likelihood of a
// proposal is the same number whatever batch it is evaluated in -- the walk's chunking stays invisible.
#pragma once

#ifndef NSGW_PD_PP
#define NSGW_PD_PP 2
#define NSGW_PD_OCC 3
#define NSGW_PD_UNR 2
#endif
constexpr int kPdNT = 128;            // threads per CTA of the lane kernel
constexpr int kPdPP = NSGW_PD_PP;     // rows per thread
constexpr int kPdKT = 64;             // bins per shared-memory tile
constexpr int kPdOCC = NSGW_PD_OCC;   // CTAs per SM
constexpr int kPdUNR = NSGW_PD_UNR;   // bins per unrolled loop body
constexpr int kPdLowNT = 256;         // threads per CTA of the low kernel (warp = row)
constexpr int kPdLowOCC = 3;

template <int NDET>
struct PdTile {
  double f[kPdKT], f34[kPdKT], y3[kPdKT], lnf[kPdKT];
  double2 wd[NDET][kPdKT];
  double ws[NDET][kPdKT];
};

// Rows to evaluate: `n_rows_dev` (device, optional) overrides n_rows -- the worklist walk sizes its rounds on the device.
struct PdArgs {
  const double* cbs;          // [rows][CB_SIZE]
  long long n_rows;
  const int* n_rows_dev;
  long long stride;           // row stride of `partial` (>= rows)
  int kr;                     // bins per range (multiple of kPdKT)
  int nranges;
  double* partial;            // [nranges + 1][N][stride]
};

// Odd Taylor coefficients of atan beyond the linear term: -1/3, 1/5, -1/7, 1/9.
__constant__ double kAtanR[4] = {-1.0 / 3.0, 0.2, -1.0 / 7.0, 1.0 / 9.0};

// ---------------------------------------------------------------------------------------------------------------------
// low kernel: warp = row, lanes strided over the bins below the row's merger-ringdown start (general piecewise evaluation;
// the regions are contiguous in the bin index, so a warp diverges at one lane per boundary only).  Writes slot `nranges`.
// ---------------------------------------------------------------------------------------------------------------------
template <int NDET>
__global__ void __launch_bounds__(kPdLowNT, kPdLowOCC) k_pd_low(const DevCfg* __restrict__ cfgp, Tables tb, PdArgs a) {
  using AL = AccLayout<2, NDET>;
  constexpr int ND1 = NDET - 1, ND1s = NDET > 1 ? NDET - 1 : 1, NWARP = kPdLowNT / 32;
  __shared__ MathTables mtab;
  const DevCfg& cfg = *cfgp;
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const int nf = cfg.n_freq;
  const double f_min = cfg.f_min, df = cfg.df;
  const long long B = a.n_rows_dev ? (long long)*a.n_rows_dev : a.n_rows;
  if ((long long)blockIdx.x * NWARP >= B) return;
  load_math_tables(&mtab, tb.mt, tid, kPdLowNT);
  __syncthreads();
  for (long long p = (long long)blockIdx.x * NWARP + wrp; p < B; p += (long long)gridDim.x * NWARP) {
    const double* cb = a.cbs + p * CB_SIZE;
    const bool valid = __ldg(cb + CB_VALID) != 0.0;
    const int kmr = valid ? mr_first_bin(__ldg(cb + CB_FP1), f_min, df, nf) : 0;   // the lane kernel takes over from here
    double acc[AL::N];
#pragma unroll
    for (int j = 0; j < AL::N; ++j) acc[j] = 0.0;
    if (kmr > 0) {
      const CbPtr cbp{cb};
      // detector phasors R_d(f_k) = C_d exp(i dtq_d f_k) at this lane's first bin, advanced by 32 bins per iteration
      double2 R[ND1s], St[ND1s];
#pragma unroll
      for (int d = 0; d < ND1; ++d) {
        const double cr = __ldg(cb + CB_DET + 4 * (d + 1)), ci = __ldg(cb + CB_DET + 4 * (d + 1) + 1);
        const double dtq = __ldg(cb + CB_DET + 4 * (d + 1) + 2);
        double sn, cs;
        sincos_qt(dtq * (f_min + df * lane), sn, cs);
        R[d] = make_double2(cr * cs - ci * sn, cr * sn + ci * cs);
        sincos_qt(dtq * (df * 32), sn, cs);
        St[d] = make_double2(cs, sn);
      }
      const double c3 = __ldg(cb + CB_AM + 3), frd = __ldg(cb + CB_AM);
      double ex = exp_tab(c3 * (f_min + df * lane - frd), &mtab);
      const double exr = exp_tab(c3 * (df * 32), &mtab);
      for (int k = lane; k < kmr; k += 32) {
        const BinBasis b = make_basis(tb, k, true);
        double2 w[NDET];
        double wsv[NDET];
#pragma unroll
        for (int d = 0; d < NDET; ++d) { w[d] = __ldg(tb.wd[d] + k); wsv[d] = __ldg(tb.ws[d] + k); }
        double q, amp;
        phenom_bin_t(cbp, b, &mtab, ex, q, amp);
        ex *= exr;
        double sn, cs;
        sincos_lut(64.0 * q, &mtab, sn, cs);
        sn *= amp; cs *= amp;
        acc[0] = fma(w[0].x, cs, acc[0]);
        acc[1] = fma(-w[0].x, sn, acc[1]);
        acc[0] = fma(-w[0].y, sn, acc[0]);
        acc[1] = fma(-w[0].y, cs, acc[1]);
        const double a2 = amp * amp;
#pragma unroll
        for (int d = 0; d < NDET; ++d) acc[AL::kHh + d] = fma(a2, wsv[d], acc[AL::kHh + d]);
#pragma unroll
        for (int d = 0; d < ND1; ++d) {
          const double rx = R[d].x, ry = R[d].y;
          const double gr = fma(cs, rx, sn * ry);
          const double gi = fma(cs, ry, -(sn * rx));
          acc[AL::kDh + d] = fma(w[d + 1].x, gr, acc[AL::kDh + d]);
          acc[AL::kDh + d] = fma(w[d + 1].y, gi, acc[AL::kDh + d]);
          R[d].x = fma(rx, St[d].x, -(ry * St[d].y));
          R[d].y = fma(rx, St[d].y, ry * St[d].x);
        }
      }
#pragma unroll
      for (int j = 0; j < AL::N; ++j) {
        double x = acc[j];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        acc[j] = x;
      }
    }
    if (lane < AL::N) {
      double v = 0.0;
#pragma unroll
      for (int j = 0; j < AL::N; ++j) v = (lane == j) ? acc[j] : v;
      a.partial[((long long)a.nranges * AL::N + lane) * a.stride + p] = v;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------------
// lane kernel: lane = row (PP per thread) over the bins of a range from the row's intermediate-phase start (f >= 0.018/M, CB_FP1)
// upwards.  Task = (group of NT x PP rows, range); writes slot `range`.  Tiles wholly inside every row's merger-ringdown region
// (f >= CB_FMR, most of them) take the branch-free loop with that region's coefficients in registers; the tiles below evaluate,
// per row and bin, both candidate phases (intermediate / merger-ringdown) and both candidate amplitudes (intermediate quartic /
// Lorentzian) and select by the row's own boundaries, with the intermediate regions' coefficients read from a shared-memory
// block staged per task (conflict-free: consecutive lanes, consecutive words).
// ---------------------------------------------------------------------------------------------------------------------
constexpr int kPdMix = 13;   // per row: 64 PB0..3 (phase, 1/256 turn), AH0..6 (quartic), FP2, FA2 [Hz]

template <int NDET, int PP>
struct PdRow {
  static constexpr int ND1s = NDET > 1 ? NDET - 1 : 1;
  double pm[PP][5], yA[PP], yB[PP], am[PP][3], exd[PP];
  double2 St[PP][ND1s];
  int klo[PP];
  double acc[PP][AccLayout<2, NDET>::N];
  // per tile
  double ex[PP], yp[PP], At[PP];
  double2 S[PP][ND1s];
};

template <int NDET, int PP, bool MIXED>
__device__ __forceinline__ void pd_tile_loop(PdRow<NDET, PP>& r, const PdTile<NDET>& sm, const double* __restrict__ mix /*smem [kPdMix][NT PP]*/,
                                             const MathTables* mt, int t_lo, int n, int tid) {
  using AL = AccLayout<2, NDET>;
  constexpr int ND1 = NDET - 1, NR = kPdNT * PP;
#pragma unroll kPdUNR
  for (int kk = n - 1; kk >= 0; --kk) {
    const double f = sm.f[kk], f34 = sm.f34[kk], y3 = sm.y3[kk];
    double2 w[NDET];
    double wsv[NDET];
#pragma unroll
    for (int d = 0; d < NDET; ++d) { w[d] = sm.wd[d][kk]; wsv[d] = sm.ws[d][kk]; }
    double L = 0.0, if3 = 0.0;
    if (MIXED) { L = sm.lnf[kk]; if3 = y3 * y3 * y3; }
#pragma unroll
    for (int j = 0; j < PP; ++j) {
      // atan((f - f0)/fd) carried down from the bin above: atan(y') = atan(y) - atan((y - y') / (1 + y y'))
      const double y = fma(f, r.yA[j], r.yB[j]);
      const double t = (r.yp[j] - y) * rcp_nr1(fma(y, r.yp[j], 1.0));
      r.yp[j] = y;
      const double z = t * t;
      double pa = fma(z, kAtanR[2], kAtanR[1]);     // |t| <= df / fd < 0.03: t^9/9 < 1e-15
      pa = fma(pa, z, kAtanR[0]);
      r.At[j] -= fma(t * z, pa, t);
      double q = fma(r.pm[j][1], f, r.pm[j][0]);
      q = fma(r.pm[j][2], y3, q);
      q = fma(r.pm[j][3], f34, q);
      q = fma(r.pm[j][4], r.At[j], q);
      const double fx = f - r.am[j][0];
      double amp = rcp_nr1(fma(fx, fx, r.am[j][2])) * r.ex[j];       // ex carries the Lorentzian's numerator
      r.ex[j] *= r.exd[j];
      if (MIXED) {
        const double* m = mix + j * kPdNT + tid;
        double qi = fma(m[1 * NR], L, m[0 * NR]);
        qi = fma(m[2 * NR], f, qi);
        qi = fma(m[3 * NR], if3, qi);
        q = (f < m[11 * NR]) ? qi : q;
        const double xh = (f - m[4 * NR]) * m[5 * NR];
        double ph = m[10 * NR];
        ph = fma(ph, xh, m[9 * NR]);
        ph = fma(ph, xh, m[8 * NR]);
        ph = fma(ph, xh, m[7 * NR]);
        ph = fma(ph, xh, m[6 * NR]);
        amp = (f < m[12 * NR]) ? ph : amp;
        amp = (t_lo + kk >= r.klo[j]) ? amp : 0.0;      // bins below the row's intermediate-phase start belong to the low kernel
      }
      double sn, cs;
      sincos_lut<true>(q, mt, sn, cs);
      sn *= amp; cs *= amp;
      r.acc[j][0] = fma(w[0].x, cs, r.acc[j][0]);
      r.acc[j][1] = fma(-w[0].x, sn, r.acc[j][1]);
      r.acc[j][0] = fma(-w[0].y, sn, r.acc[j][0]);
      r.acc[j][1] = fma(-w[0].y, cs, r.acc[j][1]);
      const double a2 = amp * amp;
#pragma unroll
      for (int d = 0; d < NDET; ++d) r.acc[j][AL::kHh + d] = fma(a2, wsv[d], r.acc[j][AL::kHh + d]);
#pragma unroll
      for (int d = 0; d < ND1; ++d) {
        // Horner in the detector's per-bin phasor rho over the tile's bins in descending order: S <- S rho + conj(wd) E
        const double ax = fma(w[d + 1].x, cs, -(w[d + 1].y * sn));
        const double ay = -fma(w[d + 1].x, sn, w[d + 1].y * cs);
        const double sx = r.S[j][d].x, sy = r.S[j][d].y;
        r.S[j][d].x = fma(sx, r.St[j][d].x, fma(-sy, r.St[j][d].y, ax));
        r.S[j][d].y = fma(sx, r.St[j][d].y, fma(sy, r.St[j][d].x, ay));
      }
    }
  }
}

template <int NDET>
__global__ void __launch_bounds__(kPdNT, kPdOCC) k_pd_lp(const DevCfg* __restrict__ cfgp, Tables tb, PdArgs a) {
  using AL = AccLayout<2, NDET>;
  constexpr int NT = kPdNT, PP = kPdPP, KT = kPdKT, ND1 = NDET - 1, ND1s = NDET > 1 ? NDET - 1 : 1, NWARP = NT / 32;
  __shared__ __align__(16) PdTile<NDET> sm;
  __shared__ MathTables mtab;
  __shared__ double mix[kPdMix * NT * PP];
  __shared__ int s_kmin[NWARP], s_kmax[NWARP];
  const DevCfg& cfg = *cfgp;
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const int nf = cfg.n_freq;
  const double f_min = cfg.f_min, df = cfg.df;
  const long long B = a.n_rows_dev ? (long long)*a.n_rows_dev : a.n_rows;
  if (B <= 0) return;
  const long long ngroups = (B + NT * PP - 1) / (NT * PP);
  const long long ntasks = ngroups * a.nranges;
  if (blockIdx.x >= ntasks) return;
  load_math_tables(&mtab, tb.mt, tid, NT);
  __syncthreads();
  for (long long task = blockIdx.x; task < ntasks; task += gridDim.x) {
    const long long grp = task / a.nranges;
    const int rng = (int)(task % a.nranges);
    const int k0 = rng * a.kr, k1 = min(nf, k0 + a.kr);
    // per row: phase a + b f + c/f + d f^3/4 + e atan(yA f + yB) in 1/256 turn; amplitude g1 / ((f - f_RD)^2 + w^2) x ex(f)
    PdRow<NDET, PP> r;
    int kmr[PP];
    int kmin = nf, kmax = 0;            // over this thread's rows: lowest bin any row wants, highest merger-ringdown start
#pragma unroll
    for (int j = 0; j < PP; ++j) {
      const long long p = (grp * PP + j) * NT + tid;
      const bool have = p < B;
      const double* cb = a.cbs + (have ? p : 0) * CB_SIZE;
      const bool valid = have && __ldg(cb + CB_VALID) != 0.0;
      r.klo[j] = valid ? mr_first_bin(__ldg(cb + CB_FP1), f_min, df, nf) : nf;   // nf: every bin masked
      kmr[j] = valid ? mr_first_bin(__ldg(cb + CB_FMR), f_min, df, nf) : 0;
      kmin = min(kmin, r.klo[j]);
      kmax = max(kmax, kmr[j]);
#pragma unroll
      for (int i = 0; i < 5; ++i) r.pm[j][i] = 64.0 * __ldg(cb + CB_PM + i);     // quarter turns -> 1/256 turn (exact)
      r.yA[j] = __ldg(cb + CB_PM + 6);
      r.yB[j] = -__ldg(cb + CB_PM + 5) * r.yA[j];
      r.am[j][0] = __ldg(cb + CB_AM); r.am[j][1] = __ldg(cb + CB_AM + 1); r.am[j][2] = __ldg(cb + CB_AM + 2);
      r.exd[j] = exp_tab(-__ldg(cb + CB_AM + 3) * df, &mtab);                     // ex(f - df) = ex(f) exd
#pragma unroll
      for (int d = 0; d < ND1; ++d) {
        double sn, cs;
        sincos_qt(__ldg(cb + CB_DET + 4 * (d + 1) + 2) * df, sn, cs);
        r.St[j][d] = make_double2(cs, sn);
      }
#pragma unroll
      for (int i = 0; i < AL::N; ++i) r.acc[j][i] = 0.0;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      kmin = min(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
      kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
    }
    __syncthreads();                       // previous task's readers of sm / mix / s_k* are done
    if (lane == 0) { s_kmin[wrp] = kmin; s_kmax[wrp] = kmax; }
    __syncthreads();
    int kmin_cta = s_kmin[0], kmax_cta = s_kmax[0];
#pragma unroll
    for (int w = 1; w < NWARP; ++w) { kmin_cta = min(kmin_cta, s_kmin[w]); kmax_cta = max(kmax_cta, s_kmax[w]); }
    if (k0 < kmax_cta) {                   // CTA-uniform: some tile of this range needs the intermediate regions' coefficients
#pragma unroll
      for (int j = 0; j < PP; ++j) {
        const long long p = (grp * PP + j) * NT + tid;
        const double* cb = a.cbs + (p < B ? p : 0) * CB_SIZE;
        double* m = mix + j * NT + tid;
#pragma unroll
        for (int i = 0; i < 4; ++i) m[i * NT * PP] = 64.0 * __ldg(cb + CB_PB + i);
#pragma unroll
        for (int i = 0; i < 7; ++i) m[(4 + i) * NT * PP] = __ldg(cb + CB_AH + i);
        m[11 * NT * PP] = __ldg(cb + CB_FP2);
        m[12 * NT * PP] = __ldg(cb + CB_FA2);
      }
    }
    for (int t_lo = k0; t_lo < k1; t_lo += KT) {
      const int n = min(KT, k1 - t_lo);
      if (t_lo + n <= kmin_cta) continue;  // CTA-uniform: the whole tile lies below every row's start
      __syncthreads();
      for (int i = tid; i < n; i += NT) {
        const int k = t_lo + i;
        sm.f[i] = __ldg(tb.f + k); sm.f34[i] = __ldg(tb.f34 + k); sm.y3[i] = __ldg(tb.t01 + k).y; sm.lnf[i] = __ldg(tb.t45 + k).x;
#pragma unroll
        for (int d = 0; d < NDET; ++d) { sm.wd[d][i] = __ldg(tb.wd[d] + k); sm.ws[d][i] = __ldg(tb.ws[d] + k); }
      }
      __syncthreads();
      if (t_lo + n <= kmin) continue;      // warp-uniform (no barrier below)
      // tile start (top bin, the loop runs downwards): ex by exp_tab, the atan term by atan_tab one bin ABOVE the top, from where
      // it is carried down; the steps have one sign, so a relative error of 2^-40 in the reciprocal is 2^-40 of the tile's total
      // change (<= pi); the next tile starts afresh
      const double f_top = sm.f[n - 1];
#pragma unroll
      for (int j = 0; j < PP; ++j) {
        const long long p = (grp * PP + j) * NT + tid;
        const double c3 = __ldg(a.cbs + (p < B ? p : 0) * CB_SIZE + CB_AM + 3);
        r.ex[j] = r.am[j][1] * exp_tab(c3 * (f_top - r.am[j][0]), &mtab);
        r.yp[j] = fma(f_top + df, r.yA[j], r.yB[j]);
        r.At[j] = atan_tab(r.yp[j], &mtab);
#pragma unroll
        for (int d = 0; d < ND1s; ++d) r.S[j][d] = make_double2(0.0, 0.0);
      }
      if (t_lo >= kmax) pd_tile_loop<NDET, PP, false>(r, sm, mix, &mtab, t_lo, n, tid);   // warp-uniform: all merger-ringdown
      else pd_tile_loop<NDET, PP, true>(r, sm, mix, &mtab, t_lo, n, tid);
      // close the tile: dh_d += Re(R_d(f_tlo) S), R_d(f) = C_d exp(i dtq f)
      const double f_lo = sm.f[0];
#pragma unroll
      for (int j = 0; j < PP; ++j) {
        const long long p = (grp * PP + j) * NT + tid;
        const double* cb = a.cbs + (p < B ? p : 0) * CB_SIZE;
#pragma unroll
        for (int d = 0; d < ND1; ++d) {
          const double cr = __ldg(cb + CB_DET + 4 * (d + 1)), ci = __ldg(cb + CB_DET + 4 * (d + 1) + 1);
          double sn, cs;
          sincos_qt(__ldg(cb + CB_DET + 4 * (d + 1) + 2) * f_lo, sn, cs);
          const double rx = cr * cs - ci * sn, ry = cr * sn + ci * cs;
          r.acc[j][AL::kDh + d] += fma(rx, r.S[j][d].x, -(ry * r.S[j][d].y));
        }
      }
    }
#pragma unroll
    for (int j = 0; j < PP; ++j) {
      const long long p = (grp * PP + j) * NT + tid;
      if (p < B) {
#pragma unroll
        for (int i = 0; i < AL::N; ++i) a.partial[((long long)rng * AL::N + i) * a.stride + p] = r.acc[j][i];
      }
    }
  }
}

// Adds a row's partial sums in slot order and finishes logL (R:L1).  n_rows_dev / stride as in PdArgs.
template <int MODEL, int NDET>
__global__ void k_finish_rows(const DevCfg* __restrict__ cfgp, const double* __restrict__ cbs_g, const double* __restrict__ partial, int nslots,
                              long long n_rows, const int* __restrict__ n_rows_dev, long long stride, double* logl, double* parts) {
  using AL = AccLayout<MODEL, NDET>;
  const long long B = n_rows_dev ? (long long)*n_rows_dev : n_rows;
  for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < B; p += (long long)gridDim.x * blockDim.x) {
    double sums[AL::N];
#pragma unroll
    for (int i = 0; i < AL::N; ++i) sums[i] = 0.0;
    int c = 0;
    for (; c + 4 <= nslots; c += 4) {
      double v[4][AL::N];
#pragma unroll
      for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int i = 0; i < AL::N; ++i) v[j][i] = __ldg(partial + ((long long)(c + j) * AL::N + i) * stride + p);
#pragma unroll
      for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int i = 0; i < AL::N; ++i) sums[i] += v[j][i];
    }
    for (; c < nslots; ++c)
#pragma unroll
      for (int i = 0; i < AL::N; ++i) sums[i] += __ldg(partial + ((long long)c * AL::N + i) * stride + p);
    logl[p] = finish_logl<MODEL, NDET>(*cfgp, cbs_g + p * CB_SIZE, sums, parts ? parts + p * 2 * NDET : nullptr);
  }
}
