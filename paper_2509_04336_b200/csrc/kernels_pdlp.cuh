// kernels_pdlp.cuh -- K1 for PhenomD-form, lane = row: k_pd_lp (used for the rows of the worklist walk and for large batches) and
// k_finish_rows (the finishing pass of the TaylorF2 rows of the worklist walk).
// Part of libnsgw (one translation unit): included by nsgw.cu inside its anonymous namespace, after kernels_k1.cuh.
//
// Design.  About 80 % of a row's bins (all above max(f_RD/2, f_peak), CB_FMR) use ONE formula -- phase =
// a + b f + c/f + d f^3/4 + e atan((f - f0)/fd), amplitude = Lorentzian x exponential -- and differ between rows only in the
// coefficients: lane = row, coefficients in registers, the bins' table values broadcast from a shared-memory tile, no cross-lane
// reduction, no per-bin global traffic (the design that took TaylorF2 to 0.63 of the FP64 peak).  Consecutive bins of a lane let the
// expensive functions be CARRIED: atan by atan y' = atan y - atan((y - y') / (1 + y y')) with y - y' = yA df the same for every bin, the
// exponential as a geometric sequence, the detector phasors by Horner's rule -- 54 FP64 instructions per particle-bin against 77 in the
// bins-strided-over-threads k_bins.
// Where the merger-ringdown region starts depends on the row (total mass, final spin), so below the highest start of a warp's rows
// the lanes disagree on the formula: those tiles evaluate the candidate formulas of the regions present and select per lane by the row's
// own boundaries, with the extra coefficients read from a shared-memory block staged per task (conflict-free: consecutive lanes,
// consecutive words).  Three tile classes, chosen per warp and tile: all merger-ringdown (registers only); intermediate or
// merger-ringdown (f >= 0.018/M for every row: + 13 coefficients); any region (+ 25 more and six more table values per bin).
//
// Task = (group of NT x PP rows, range of `kr` bins on the fixed tile grid), persistent CTAs over the task list.  A task writes its rows'
// partial sums to partial[range][N][stride]; the CTA that finishes a group's LAST range (a ticket per group) adds the ranges in range
// order and writes logL -- no finishing launch, and the order of the sum does not depend on which CTA came last.  A row's sums do not
// depend on the rows it shares a warp, a task or a launch with, so the likelihood of a proposal is the same number whatever batch it is
// evaluated in: the walk's chunking stays invisible.
#pragma once

#ifndef NSGW_PD_PP
#define NSGW_PD_PP 1
#define NSGW_PD_OCC 3
#define NSGW_PD_UNR 4
#endif
#ifndef NSGW_PD_KT
#define NSGW_PD_KT 128
#endif
#ifndef NSGW_PD_NT
#define NSGW_PD_NT 128
#endif
constexpr int kPdNT = NSGW_PD_NT;     // threads per CTA
constexpr int kPdPP = NSGW_PD_PP;     // rows per thread
constexpr int kPdKT = NSGW_PD_KT;     // bins per shared-memory tile
constexpr int kPdOCC = NSGW_PD_OCC;   // CTAs per SM
constexpr int kPdUNR = NSGW_PD_UNR;   // bins per unrolled loop body

template <int NDET>
struct PdTile {
  double f[kPdKT], f34[kPdKT], y3[kPdKT], lnf[kPdKT];
  double2 wd[NDET][kPdKT];
  double ws[NDET][kPdKT];
  double y5[kPdKT], y2[kPdKT], y1[kPdKT], x1[kPdKT], xl[kPdKT], x2[kPdKT];   // class-2 tiles only: f^-5/3, f^-2/3, f^-1/3, f^1/3, f^1/3 ln f, f^2/3
};

// Rows to evaluate: `n_rows_dev` (device, optional) overrides n_rows -- the worklist walk sizes its rounds on the device.
struct PdArgs {
  const double* cbs;          // [rows][CB_SIZE]
  long long n_rows;
  const int* n_rows_dev;
  long long stride;           // row stride of `partial` (>= rows)
  int kr;                     // bins per range (multiple of kPdKT)
  int nranges;
  double* partial;            // [nranges][N][stride]
  int* ticket;                // [groups] zero on entry, zero again on exit: ranges of the group finished so far
  double* logl;               // [rows]
  double* parts;              // optional [rows][2 NDET]
};

// Takes a ticket of a row group on behalf of the CTA: one thread, behind a CTA-wide barrier that follows the CTA's stores.  Returns the
// number of tickets taken before.  acq_rel at device scope: the release half orders the CTA's stores (observed through the barrier)
// before the ticket, the acquire half orders the ticket before the loads that follow the next barrier.  (One MEMBAR + one L1
// invalidate by one thread per task; __threadfence() by every thread before and after cost 0.5 % of a config-3 run.)
__device__ __forceinline__ int pd_ticket_take(int* t) {
  int old;
  asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], 1;" : "=r"(old) : "l"(t) : "memory");
  return old;
}

// Odd Taylor coefficients of atan beyond the linear term: -1/3, 1/5, -1/7.
__constant__ double kAtanR[3] = {-1.0 / 3.0, 0.2, -1.0 / 7.0};

// Shared-memory coefficient block of a task, [kPdMixAll][NT PP] (row-minor).  Classes 1 and 2 read the first kPdMix1 entries per row:
// 128 PB0..3 (intermediate phase, 1/512 turn), AH0..6 (intermediate amplitude), FP2, FA2 [Hz]; class 2 also 128 PH0..12 (inspiral phase),
// AI0..9 (inspiral amplitude), FP1, FA1.
constexpr int kPdMix1 = 13, kPdMixAll = 13 + 25;
template <int PP>
constexpr size_t pd_mix_bytes() { return sizeof(double) * kPdMixAll * kPdNT * PP; }

template <int NDET, int PP>
struct PdRow {
  static constexpr int ND1s = NDET > 1 ? NDET - 1 : 1;
  double pm[PP][5], yA[PP], yB[PP], dy[PP], am[PP][3], exd[PP];
  double2 St[PP][ND1s];
  double acc[PP][AccLayout<2, NDET>::N];
  // per tile
  double ex[PP], yp[PP], At[PP];
  double2 S[PP][ND1s];
};

// One tile, bins in descending order.  CLS 0: every row of the warp is in its merger-ringdown region; 1: intermediate or
// merger-ringdown; 2: any region.
template <int NDET, int PP, int CLS>
__device__ __forceinline__ void pd_tile_loop(PdRow<NDET, PP>& r, const PdTile<NDET>& sm, const double* __restrict__ mix, const double2* sc9,
                                             int n, int tid) {
  using AL = AccLayout<2, NDET>;
  constexpr int ND1 = NDET - 1, NR = kPdNT * PP;
#pragma unroll kPdUNR
  for (int kk = n - 1; kk >= 0; --kk) {
    const double f = sm.f[kk], f34 = sm.f34[kk], y3 = sm.y3[kk];
    double2 w[NDET];
    double wsv[NDET];
#pragma unroll
    for (int d = 0; d < NDET; ++d) { w[d] = sm.wd[d][kk]; wsv[d] = sm.ws[d][kk]; }
    double L = 0.0, if3 = 0.0, y5 = 0.0, y2 = 0.0, y1 = 0.0, x1 = 0.0, xl = 0.0, x2 = 0.0, fx = 0.0, fx2 = 0.0, ff = 0.0;
    if (CLS >= 1) { L = sm.lnf[kk]; if3 = y3 * y3 * y3; }
    if (CLS == 2) {
      y5 = sm.y5[kk]; y2 = sm.y2[kk]; y1 = sm.y1[kk]; x1 = sm.x1[kk]; xl = sm.xl[kk]; x2 = sm.x2[kk];
      fx = f * x1; fx2 = fx * x1; ff = f * f;
    }
#pragma unroll
    for (int j = 0; j < PP; ++j) {
      // atan((f - f0)/fd) carried down from the bin above: atan(y') = atan(y) - atan((y - y') / (1 + y y'))
      const double y = fma(f, r.yA[j], r.yB[j]);
      const double t = r.dy[j] * rcp_nr1(fma(y, r.yp[j], 1.0));     // the bins are equally spaced: y' - y = yA df
      r.yp[j] = y;
      const double z = t * t;
      double pa = fma(z, kAtanR[2], kAtanR[1]);     // |t| <= df / fd < 0.03: t^9/9 < 1e-15
      pa = fma(pa, z, kAtanR[0]);
      pa = fma(pa, z, 1.0);
      r.At[j] = fma(-t, pa, r.At[j]);
      double q = fma(r.pm[j][1], f, r.pm[j][0]);
      q = fma(r.pm[j][2], y3, q);
      q = fma(r.pm[j][3], f34, q);
      q = fma(r.pm[j][4], r.At[j], q);
      const double fr = f - r.am[j][0];
      double amp = rcp_nr1(fma(fr, fr, r.am[j][2])) * r.ex[j];       // ex carries the Lorentzian's numerator
      r.ex[j] *= r.exd[j];
      if (CLS >= 1) {
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
        if (CLS == 2) {
          const double* c = m + kPdMix1 * NR;       // PH0..12: y5 y3 y2 y 1 L x xL x2 f | fx fx2 ff
          double qs = fma(c[0 * NR], y5, c[4 * NR]);
          qs = fma(c[1 * NR], y3, qs);
          qs = fma(c[2 * NR], y2, qs);
          qs = fma(c[3 * NR], y1, qs);
          qs = fma(c[5 * NR], L, qs);
          qs = fma(c[6 * NR], x1, qs);
          qs = fma(c[7 * NR], xl, qs);
          qs = fma(c[8 * NR], x2, qs);
          qs = fma(c[9 * NR], f, qs);
          qs = fma(c[10 * NR], fx, qs);
          qs = fma(c[11 * NR], fx2, qs);
          qs = fma(c[12 * NR], ff, qs);
          q = (f < c[23 * NR]) ? qs : q;
          double pi_ = c[22 * NR];                  // AI9..AI0: degree-9 polynomial in x = f^1/3
#pragma unroll
          for (int i = 8; i >= 0; --i) pi_ = fma(pi_, x1, c[(13 + i) * NR]);
          amp = (f < c[24 * NR]) ? pi_ : amp;
        }
      }
      double sn, cs;
      sincos_lut9(q, sc9, sn, cs);
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
  constexpr int NT = kPdNT, PP = kPdPP, KT = kPdKT, ND1 = NDET - 1, ND1s = NDET > 1 ? NDET - 1 : 1, NWARP = NT / 32, NR = NT * PP;
  __shared__ __align__(16) PdTile<NDET> sm;
  __shared__ MathTablesEA mtab;                           // exp_tab / atan_tab at the tile starts
  __shared__ __align__(16) double2 sc9[kSc9N];            // sincos_lut9 in the bin loops
  __shared__ int s_k1[NWARP], s_k2[NWARP], s_last;
  extern __shared__ __align__(16) double mix[];          // [kPdMixAll][NR]
  const DevCfg& cfg = *cfgp;
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const int nf = cfg.n_freq;
  const double f_min = cfg.f_min, df = cfg.df;
  load_math_tables_ea(&mtab, tb.mt, tid, NT);  // built at ns_init: not the previous kernel's output
  load_sc9(sc9, tb.sc9, tid, NT);
  pdl_wait();                                  // the rows (count, coefficient blocks) are
  const long long B = a.n_rows_dev ? (long long)*a.n_rows_dev : a.n_rows;
  if (B <= 0) return;
  const long long ngroups = (B + NR - 1) / NR;
  const long long ntasks = ngroups * a.nranges;
  if (blockIdx.x >= ntasks) return;
  __syncthreads();
  for (long long task = blockIdx.x; task < ntasks; task += gridDim.x) {
    const long long grp = task / a.nranges;
    const int rng = (int)(task % a.nranges);
    const int k0 = rng * a.kr, k1 = min(nf, k0 + a.kr);
    // per row: phase a + b f + c/f + d f^3/4 + e atan(yA f + yB) in 1/512 turn; amplitude g1 / ((f - f_RD)^2 + w^2) x ex(f).
    // An invalid row (unphysical theta: logL = -inf whatever the sums) gets zero coefficients, so nothing undefined is evaluated.
    PdRow<NDET, PP> r;
    double c3[PP], g1[PP];
    int k1max = 0, k2max = 0;          // over this thread's rows: first bin past the inspiral phase region / in the merger-ringdown region
#pragma unroll
    for (int j = 0; j < PP; ++j) {
      const long long p = (grp * PP + j) * NT + tid;
      const double* cb = a.cbs + (p < B ? p : 0) * CB_SIZE;
      const bool valid = p < B && __ldg(cb + CB_VALID) != 0.0;
      k1max = max(k1max, valid ? mr_first_bin(__ldg(cb + CB_FP1), f_min, df, nf) : 0);
      k2max = max(k2max, valid ? mr_first_bin(__ldg(cb + CB_FMR), f_min, df, nf) : 0);
#pragma unroll
      for (int i = 0; i < 5; ++i) r.pm[j][i] = valid ? 128.0 * __ldg(cb + CB_PM + i) : 0.0;    // quarter turns -> 1/512 turn (exact)
      r.yA[j] = valid ? __ldg(cb + CB_PM + 6) : 0.0;
      r.yB[j] = valid ? -__ldg(cb + CB_PM + 5) * r.yA[j] : 0.0;
      r.dy[j] = r.yA[j] * df;                                                                   // y(f + df) - y(f)
      r.am[j][0] = valid ? __ldg(cb + CB_AM) : 0.0;
      g1[j] = valid ? __ldg(cb + CB_AM + 1) : 0.0;
      r.am[j][2] = valid ? __ldg(cb + CB_AM + 2) : 1.0;
      c3[j] = valid ? __ldg(cb + CB_AM + 3) : 0.0;
      r.exd[j] = exp_tab(-c3[j] * df, &mtab);                                                   // ex(f - df) = ex(f) exd
#pragma unroll
      for (int d = 0; d < ND1; ++d) {
        double sn, cs;
        sincos_qt((valid ? __ldg(cb + CB_DET + 4 * (d + 1) + 2) : 0.0) * df, sn, cs);
        r.St[j][d] = make_double2(cs, sn);
      }
#pragma unroll
      for (int i = 0; i < AL::N; ++i) r.acc[j][i] = 0.0;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      k1max = max(k1max, __shfl_xor_sync(0xffffffffu, k1max, o));
      k2max = max(k2max, __shfl_xor_sync(0xffffffffu, k2max, o));
    }
    __syncthreads();                       // previous task's readers of sm / mix / s_k* are done
    if (lane == 0) { s_k1[wrp] = k1max; s_k2[wrp] = k2max; }
    __syncthreads();
    int k1cta = s_k1[0], k2cta = s_k2[0];
#pragma unroll
    for (int w = 1; w < NWARP; ++w) { k1cta = max(k1cta, s_k1[w]); k2cta = max(k2cta, s_k2[w]); }
    if (k0 < k2cta) {                      // CTA-uniform: some tile of this range needs the other regions' coefficients
#pragma unroll
      for (int j = 0; j < PP; ++j) {
        const long long p = (grp * PP + j) * NT + tid;
        const double* cb = a.cbs + (p < B ? p : 0) * CB_SIZE;
        const bool valid = p < B && __ldg(cb + CB_VALID) != 0.0;
        double* m = mix + j * NT + tid;
#pragma unroll
        for (int i = 0; i < 4; ++i) m[i * NR] = valid ? 128.0 * __ldg(cb + CB_PB + i) : 0.0;
#pragma unroll
        for (int i = 0; i < 7; ++i) m[(4 + i) * NR] = valid ? __ldg(cb + CB_AH + i) : 0.0;
        m[11 * NR] = valid ? __ldg(cb + CB_FP2) : 0.0;
        m[12 * NR] = valid ? __ldg(cb + CB_FA2) : 0.0;
        if (k0 < k1cta) {
          double* c = m + kPdMix1 * NR;
#pragma unroll
          for (int i = 0; i < 13; ++i) c[i * NR] = valid ? 128.0 * __ldg(cb + CB_PH + i) : 0.0;
#pragma unroll
          for (int i = 0; i < 10; ++i) c[(13 + i) * NR] = valid ? __ldg(cb + CB_AI + i) : 0.0;
          c[23 * NR] = valid ? __ldg(cb + CB_FP1) : 0.0;
          c[24 * NR] = valid ? __ldg(cb + CB_FA1) : 0.0;
        }
      }
    }
    for (int t_lo = k0; t_lo < k1; t_lo += KT) {
      const int n = min(KT, k1 - t_lo);
      __syncthreads();
      const bool need2 = t_lo < k1cta;     // CTA-uniform: some warp evaluates this tile with the inspiral formulas
      for (int i = tid; i < n; i += NT) {
        const int k = t_lo + i;
        const double2 t01 = __ldg(tb.t01 + k), t45 = __ldg(tb.t45 + k);
        sm.f[i] = __ldg(tb.f + k); sm.f34[i] = __ldg(tb.f34 + k); sm.y3[i] = t01.y; sm.lnf[i] = t45.x;
#pragma unroll
        for (int d = 0; d < NDET; ++d) { sm.wd[d][i] = __ldg(tb.wd[d] + k); sm.ws[d][i] = __ldg(tb.ws[d] + k); }
        if (need2) {
          const double2 t23 = __ldg(tb.t23 + k), t67 = __ldg(tb.t67 + k);
          sm.y5[i] = t01.x; sm.y2[i] = t23.x; sm.y1[i] = t23.y; sm.x1[i] = t45.y; sm.xl[i] = t67.x; sm.x2[i] = t67.y;
        }
      }
      __syncthreads();
      // tile start (top bin, the loop runs downwards): ex by exp_tab, the atan term by atan_tab one bin ABOVE the top, from where
      // it is carried down; the steps have one sign, so a relative error of 2^-40 in the reciprocal is 2^-40 of the tile's total
      // change (<= pi); the next tile starts afresh
      const double f_top = sm.f[n - 1];
#pragma unroll
      for (int j = 0; j < PP; ++j) {
        r.ex[j] = g1[j] * exp_tab(c3[j] * (f_top - r.am[j][0]), &mtab);
        r.yp[j] = fma(f_top + df, r.yA[j], r.yB[j]);
        r.At[j] = atan_tab(r.yp[j], &mtab);
#pragma unroll
        for (int d = 0; d < ND1s; ++d) r.S[j][d] = make_double2(0.0, 0.0);
      }
      if (t_lo >= k2max) pd_tile_loop<NDET, PP, 0>(r, sm, mix, sc9, n, tid);          // warp-uniform choices
      else if (t_lo >= k1max) pd_tile_loop<NDET, PP, 1>(r, sm, mix, sc9, n, tid);
      else pd_tile_loop<NDET, PP, 2>(r, sm, mix, sc9, n, tid);
      // close the tile: dh_d += Re(R_d(f_tlo) S), R_d(f) = C_d exp(i dtq f)
      const double f_lo = sm.f[0];
#pragma unroll
      for (int j = 0; j < PP; ++j) {
        const long long p = (grp * PP + j) * NT + tid;
        const double* cb = a.cbs + (p < B ? p : 0) * CB_SIZE;
        const bool valid = p < B && __ldg(cb + CB_VALID) != 0.0;
#pragma unroll
        for (int d = 0; d < ND1; ++d) {
          const double cr = valid ? __ldg(cb + CB_DET + 4 * (d + 1)) : 0.0, ci = valid ? __ldg(cb + CB_DET + 4 * (d + 1) + 1) : 0.0;
          double sn, cs;
          sincos_qt((valid ? __ldg(cb + CB_DET + 4 * (d + 1) + 2) : 0.0) * f_lo, sn, cs);
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
    // the CTA that finishes the group's last range adds the ranges in range order and writes logL (a ticket per group)
    // (release: the CTA's stores -> barrier -> thread 0's acq_rel ticket; acquire: ticket -> barrier -> the CTA's L2 loads)
    __syncthreads();
    if (tid == 0) s_last = (pd_ticket_take(a.ticket + grp) == a.nranges - 1) ? 1 : 0;
    __syncthreads();
    if (s_last) {
#pragma unroll
      for (int j = 0; j < PP; ++j) {
        const long long p = (grp * PP + j) * NT + tid;
        if (p < B) {
          double sums[AL::N];
#pragma unroll
          for (int i = 0; i < AL::N; ++i) sums[i] = 0.0;
          for (int c = 0; c < a.nranges; ++c)
#pragma unroll
            for (int i = 0; i < AL::N; ++i) sums[i] += __ldcg(a.partial + ((long long)c * AL::N + i) * a.stride + p);
          a.logl[p] = finish_logl<2, NDET>(cfg, a.cbs + p * CB_SIZE, sums, a.parts ? a.parts + p * 2 * NDET : nullptr);
        }
      }
      if (tid == 0) a.ticket[grp] = 0;
    }
  }
}

// Adds a row's partial sums in slot order and finishes logL (R:L1).  n_rows_dev / stride as in PdArgs.
template <int MODEL, int NDET>
__global__ void k_finish_rows(const DevCfg* __restrict__ cfgp, const double* __restrict__ cbs_g, const double* __restrict__ partial, int nslots,
                              long long n_rows, const int* __restrict__ n_rows_dev, long long stride, double* logl, double* parts) {
  pdl_wait();   // (launched as a programmatic dependent of the sweep)
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
