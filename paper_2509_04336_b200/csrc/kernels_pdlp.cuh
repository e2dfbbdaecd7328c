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
// Task list of a launch: nranges x ngroups lane tasks (group of NT x PP rows, range of `kr` bins on the fixed tile grid), then
// ceil(rows / (warps x kPdLowPer)) low tasks.  Every task writes its rows' partial sums to partial[slot][N][stride] (slot = range
// index, or nranges for the low part); k_finish_rows adds the slots in order.  A row's sums do not depend on which other rows share
// its warp, its task or the launch (masked bins contribute exact zeros; tiles sit on a grid fixed by `kr`), so the likelihood of a
// proposal is the same number whatever batch it is evaluated in -- the walk's chunking stays invisible.
#pragma once

constexpr int kPdNT = 128;      // threads per CTA
constexpr int kPdPP = 2;        // rows per thread in a lane task
constexpr int kPdKT = 64;       // bins per shared-memory tile
constexpr int kPdOCC = 3;       // CTAs per SM
constexpr int kPdLowPer = 8;    // rows per warp in a low task

template <int NDET>
struct PdTile {
  double f[kPdKT], f34[kPdKT], y3[kPdKT];
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

template <int NDET>
__global__ void __launch_bounds__(kPdNT, kPdOCC) k_pd_lp(const DevCfg* __restrict__ cfgp, Tables tb, PdArgs a) {
  using AL = AccLayout<2, NDET>;
  constexpr int NT = kPdNT, PP = kPdPP, KT = kPdKT, ND1 = NDET - 1, ND1s = NDET > 1 ? NDET - 1 : 1, NWARP = NT / 32;
  __shared__ __align__(16) PdTile<NDET> sm;
  __shared__ MathTables mtab;
  __shared__ int s_kmin[NWARP];
  const DevCfg& cfg = *cfgp;
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const int nf = cfg.n_freq;
  const double f_min = cfg.f_min, df = cfg.df;
  const long long B = a.n_rows_dev ? (long long)*a.n_rows_dev : a.n_rows;
  if (B <= 0) return;
  const long long ngroups = (B + NT * PP - 1) / (NT * PP);
  const long long n_lane_tasks = ngroups * a.nranges;
  const long long n_low_tasks = (B + NWARP * kPdLowPer - 1) / (NWARP * kPdLowPer);
  load_math_tables(&mtab, tb.mt, tid, NT);
  __syncthreads();
  for (long long task = blockIdx.x; task < n_lane_tasks + n_low_tasks; task += gridDim.x) {
    if (task >= n_lane_tasks) {
      // ---------------------------------------------------------------------------------------------------------------
      // low task: warp = particle, lanes strided over the bins below the row's merger-ringdown start (general evaluation)
      // ---------------------------------------------------------------------------------------------------------------
      const long long p0 = ((task - n_lane_tasks) * NWARP + wrp) * kPdLowPer;
      for (int i = 0; i < kPdLowPer; ++i) {
        const long long p = p0 + i;
        if (p >= B) break;                                   // warp-uniform
        const double* cb = a.cbs + p * CB_SIZE;
        const bool valid = __ldg(cb + CB_VALID) != 0.0;
        const int kmr = valid ? mr_first_bin(__ldg(cb + CB_FMR), f_min, df, nf) : 0;
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
            double q, amp;
            phenom_bin_t(cbp, b, &mtab, ex, q, amp);
            ex *= exr;
            double sn, cs;
            sincos_lut(64.0 * q, &mtab, sn, cs);
            sn *= amp; cs *= amp;
            const double2 w0 = __ldg(tb.wd[0] + k);
            acc[0] = fma(w0.x, cs, acc[0]);
            acc[1] = fma(-w0.x, sn, acc[1]);
            acc[0] = fma(-w0.y, sn, acc[0]);
            acc[1] = fma(-w0.y, cs, acc[1]);
            const double a2 = amp * amp;
#pragma unroll
            for (int d = 0; d < NDET; ++d) acc[AL::kHh + d] = fma(a2, __ldg(tb.ws[d] + k), acc[AL::kHh + d]);
#pragma unroll
            for (int d = 0; d < ND1; ++d) {
              const double2 w = __ldg(tb.wd[d + 1] + k);
              const double rx = R[d].x, ry = R[d].y;
              const double gr = fma(cs, rx, sn * ry);
              const double gi = fma(cs, ry, -(sn * rx));
              acc[AL::kDh + d] = fma(w.x, gr, acc[AL::kDh + d]);
              acc[AL::kDh + d] = fma(w.y, gi, acc[AL::kDh + d]);
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
      continue;
    }
    // -----------------------------------------------------------------------------------------------------------------
    // lane task: lane = particle (PP per thread) over the bins [k0, k1) that lie in the row's merger-ringdown region
    // -----------------------------------------------------------------------------------------------------------------
    const long long grp = task / a.nranges;
    const int rng = (int)(task % a.nranges);
    const int k0 = rng * a.kr, k1 = min(nf, k0 + a.kr);
    double pm[PP][7], am[PP][3], c3[PP], exd[PP];
    double2 Cd[PP][ND1s], St[PP][ND1s];
    double dtq[PP][ND1s];
    int kmr[PP];
    double acc[PP][AL::N];
    int kmin = nf;
#pragma unroll
    for (int j = 0; j < PP; ++j) {
      const long long p = (grp * PP + j) * NT + tid;
      const bool have = p < B;
      const double* cb = a.cbs + (have ? p : 0) * CB_SIZE;
      const bool valid = have && __ldg(cb + CB_VALID) != 0.0;
      kmr[j] = valid ? mr_first_bin(__ldg(cb + CB_FMR), f_min, df, nf) : nf;     // nf: every bin masked
      kmin = min(kmin, kmr[j]);
#pragma unroll
      for (int i = 0; i < 5; ++i) pm[j][i] = 64.0 * __ldg(cb + CB_PM + i);       // quarter turns -> 1/256 turn (exact)
      pm[j][6] = __ldg(cb + CB_PM + 6);                                           // atan argument y = f / fd - f0 / fd
      pm[j][5] = -__ldg(cb + CB_PM + 5) * pm[j][6];
      am[j][0] = __ldg(cb + CB_AM); am[j][1] = __ldg(cb + CB_AM + 1); am[j][2] = __ldg(cb + CB_AM + 2);
      c3[j] = __ldg(cb + CB_AM + 3);
      exd[j] = exp_tab(-c3[j] * df, &mtab);                                       // ex(f - df) = ex(f) exd
#pragma unroll
      for (int d = 0; d < ND1; ++d) {
        Cd[j][d] = make_double2(__ldg(cb + CB_DET + 4 * (d + 1)), __ldg(cb + CB_DET + 4 * (d + 1) + 1));
        dtq[j][d] = __ldg(cb + CB_DET + 4 * (d + 1) + 2);
        double sn, cs;
        sincos_qt(dtq[j][d] * df, sn, cs);
        St[j][d] = make_double2(cs, sn);
      }
#pragma unroll
      for (int i = 0; i < AL::N; ++i) acc[j][i] = 0.0;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) kmin = min(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
    __syncthreads();                       // previous task's readers of sm / s_kmin are done
    if (lane == 0) s_kmin[wrp] = kmin;
    __syncthreads();
    int kmin_cta = s_kmin[0];
#pragma unroll
    for (int w = 1; w < NWARP; ++w) kmin_cta = min(kmin_cta, s_kmin[w]);
    for (int t_lo = k0; t_lo < k1; t_lo += KT) {
      const int n = min(KT, k1 - t_lo);
      if (t_lo + n <= kmin_cta) continue;  // CTA-uniform: the whole tile lies below every row's merger-ringdown region
      __syncthreads();
      for (int i = tid; i < n; i += NT) {
        const int k = t_lo + i;
        sm.f[i] = __ldg(tb.f + k); sm.f34[i] = __ldg(tb.f34 + k); sm.y3[i] = __ldg(tb.t01 + k).y;
#pragma unroll
        for (int d = 0; d < NDET; ++d) { sm.wd[d][i] = __ldg(tb.wd[d] + k); sm.ws[d][i] = __ldg(tb.ws[d] + k); }
      }
      __syncthreads();
      if (t_lo + n <= kmin) continue;      // warp-uniform (no barrier below)
      double ex[PP];
      double2 S[PP][ND1s];
      const double f_top = sm.f[n - 1];
#pragma unroll
      for (int j = 0; j < PP; ++j) {
        ex[j] = exp_tab(c3[j] * (f_top - am[j][0]), &mtab);
#pragma unroll
        for (int d = 0; d < ND1s; ++d) S[j][d] = make_double2(0.0, 0.0);
      }
#pragma unroll 2
      for (int kk = n - 1; kk >= 0; --kk) {
        const double f = sm.f[kk], f34 = sm.f34[kk], y3 = sm.y3[kk];
        double2 w[NDET];
        double wsv[NDET];
#pragma unroll
        for (int d = 0; d < NDET; ++d) { w[d] = sm.wd[d][kk]; wsv[d] = sm.ws[d][kk]; }
#pragma unroll
        for (int j = 0; j < PP; ++j) {
          double q = fma(pm[j][1], f, pm[j][0]);
          q = fma(pm[j][2], y3, q);
          q = fma(pm[j][3], f34, q);
          q = fma(pm[j][4], atan_tab(fma(f, pm[j][6], pm[j][5]), &mtab), q);
          const double fx = f - am[j][0];
          double amp = am[j][1] * rcp_nr1(fma(fx, fx, am[j][2])) * ex[j];
          ex[j] *= exd[j];
          amp = (t_lo + kk >= kmr[j]) ? amp : 0.0;        // bins below the row's merger-ringdown region belong to the low task
          double sn, cs;
          sincos_lut(q, &mtab, sn, cs);
          sn *= amp; cs *= amp;
          acc[j][0] = fma(w[0].x, cs, acc[j][0]);
          acc[j][1] = fma(-w[0].x, sn, acc[j][1]);
          acc[j][0] = fma(-w[0].y, sn, acc[j][0]);
          acc[j][1] = fma(-w[0].y, cs, acc[j][1]);
          const double a2 = amp * amp;
#pragma unroll
          for (int d = 0; d < NDET; ++d) acc[j][AL::kHh + d] = fma(a2, wsv[d], acc[j][AL::kHh + d]);
#pragma unroll
          for (int d = 0; d < ND1; ++d) {
            // Horner in the detector's per-bin phasor rho over the tile's bins in descending order: S <- S rho + conj(wd) E
            const double ax = fma(w[d + 1].x, cs, -(w[d + 1].y * sn));
            const double ay = -fma(w[d + 1].x, sn, w[d + 1].y * cs);
            const double sx = S[j][d].x, sy = S[j][d].y;
            S[j][d].x = fma(sx, St[j][d].x, fma(-sy, St[j][d].y, ax));
            S[j][d].y = fma(sx, St[j][d].y, fma(sy, St[j][d].x, ay));
          }
        }
      }
      // close the tile: dh_d += Re(R_d(f_tlo) S), R_d(f) = C_d exp(i dtq f)
      const double f_lo = sm.f[0];
#pragma unroll
      for (int j = 0; j < PP; ++j)
#pragma unroll
        for (int d = 0; d < ND1; ++d) {
          double sn, cs;
          sincos_qt(dtq[j][d] * f_lo, sn, cs);
          const double rx = Cd[j][d].x * cs - Cd[j][d].y * sn, ry = Cd[j][d].x * sn + Cd[j][d].y * cs;
          acc[j][AL::kDh + d] += fma(rx, S[j][d].x, -(ry * S[j][d].y));
        }
    }
#pragma unroll
    for (int j = 0; j < PP; ++j) {
      const long long p = (grp * PP + j) * NT + tid;
      if (p < B) {
#pragma unroll
        for (int i = 0; i < AL::N; ++i) a.partial[((long long)rng * AL::N + i) * a.stride + p] = acc[j][i];
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
