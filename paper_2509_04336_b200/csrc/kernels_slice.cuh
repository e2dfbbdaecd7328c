// kernels_slice.cuh -- hit-and-run slice-sampling inner kernel (reading R:L25): the alternative K2.
// Part of libnsgw (one translation unit): included by nsgw.cu inside its anonymous namespace, after kernels_walk.cuh.
// See include/nsgw.h (ns_slice_batch) for the contract.
#pragma once

struct SliceArgs {
  const double* Lc;      // [D][D] lower-triangular direction factor (unit-cube coordinates)
  double* u;             // [B, D] in/out
  double* logl;          // [B] in/out
  long long B;
  double lstar;
  const double* lstar_dev;     // if non-null overrides lstar (ns_step)
  const long long* iter_dev;   // if non-null: stream_id |= (*iter & 0xFFFFFF)
  int S;                 // slice steps per walker
  uint32_t k0, k1, stream_id;
  long long slot0;
  int* n_eval; int* n_oob; int* n_expand; int* n_shrink; int* n_stuck;
  int* n_moved;                   // optional: S - n_stuck (what the sampler's statistics call accepted steps)
  int* t_evals; double* t_logl;   // optional trace [B, S]
};

constexpr int kSliceMaxExpand = 32, kSliceMaxShrink = 64;

// Direction of step s of walker `slot`: z ~ N(0, I) over the free dims (Box-Muller, Philox blocks 0..7), dir = Lc z / |z|.
__device__ __forceinline__ void slice_direction(const DevCfg& cfg, const SliceArgs& a, uint32_t sid, uint32_t s, uint32_t slot, double* dir) {
  const int D = cfg.ndim;
  int fr[kMaxDim], nfree = 0;
  for (int d = 0; d < D; ++d)
    if (cfg.prior_kind[d] != 4) fr[nfree++] = d;
  double z[kMaxDim];
  for (int i = 0; 2 * i < nfree; ++i) {
    uint32_t w[4];
    philox4x32_10((uint32_t)i, s, slot, sid, a.k0, a.k1, w);
    const double U1 = u01(w[0], w[1]), U2 = u01(w[2], w[3]);
    const double rad = sqrt(-2.0 * log(U1));
    z[2 * i] = rad * cos(2.0 * kPi * U2);
    if (2 * i + 1 < nfree) z[2 * i + 1] = rad * sin(2.0 * kPi * U2);
  }
  double z2 = 0.0;
  for (int i = 0; i < nfree; ++i) z2 += z[i] * z[i];
  const double inv = 1.0 / sqrt(z2);
  for (int d = 0; d < D; ++d) dir[d] = 0.0;
  for (int i = 0; i < nfree; ++i) {
    double acc = 0.0;
    for (int j = 0; j <= i; ++j) acc += a.Lc[(size_t)fr[i] * D + fr[j]] * z[j];
    dir[fr[i]] = acc * inv;
  }
}

// y = x + t dir with periodic wrap; returns false if a non-periodic coordinate leaves (0,1).
__device__ __forceinline__ bool slice_point(const DevCfg& cfg, const double* x, const double* dir, double t, double* y) {
  bool inb = true;
  for (int d = 0; d < cfg.ndim; ++d) {
    if (cfg.prior_kind[d] == 4) { y[d] = x[d]; continue; }
    double v = fma(t, dir[d], x[d]);
    if (cfg.periodic[d]) v = v - floor(v);
    else if (!(v > 0.0 && v < 1.0)) inb = false;
    y[d] = v;
  }
  return inb;
}

__device__ __forceinline__ double slice_shrink_uniform(const SliceArgs& a, uint32_t sid, uint32_t s, uint32_t slot, int k) {
  uint32_t w[4];
  philox4x32_10(9u + (uint32_t)(k / 2), s, slot, sid, a.k0, a.k1, w);
  return (k % 2 == 0) ? u01(w[0], w[1]) : u01(w[2], w[3]);
}

// Bin-less likelihoods (Gaussian toy, cube shell): one thread per walker, the sequential algorithm as stated.
__global__ void k_slice_simple(const DevCfg* __restrict__ cfgp, SliceArgs a) {
  long long row = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (row >= a.B) return;
  const DevCfg& cfg = *cfgp;
  const int D = cfg.ndim;
  const uint32_t slot = (uint32_t)(a.slot0 + row);
  const double lstar = a.lstar_dev ? *a.lstar_dev : a.lstar;
  const uint32_t sid = a.stream_id | (a.iter_dev ? (uint32_t)(*a.iter_dev & 0xFFFFFF) : 0u);
  double x[kMaxDim], y[kMaxDim], dir[kMaxDim];
  for (int d = 0; d < D; ++d) x[d] = a.u[row * D + d];
  double xl = a.logl[row];
  int ne = 0, no = 0, nx = 0, ns = 0, nk = 0;
  for (int s = 0; s < a.S; ++s) {
    const int ne0 = ne;
    slice_direction(cfg, a, sid, (uint32_t)s, slot, dir);
    auto inside = [&](double t, double& lt) -> bool {
      if (!slice_point(cfg, x, dir, t, y)) { ++no; return false; }
      lt = simple_loglike(cfg, y);
      ++ne;
      return lt > lstar;
    };
    uint32_t w8[4];
    philox4x32_10(8u, (uint32_t)s, slot, sid, a.k0, a.k1, w8);
    double l = -u01(w8[0], w8[1]), r = l + 1.0, tmp;
    for (int k = 0; k < kSliceMaxExpand && inside(l, tmp); ++k) { l -= 1.0; ++nx; }
    for (int k = 0; k < kSliceMaxExpand && inside(r, tmp); ++k) { r += 1.0; ++nx; }
    bool moved = false;
    for (int k = 0; k < kSliceMaxShrink; ++k) {
      const double t = l + slice_shrink_uniform(a, sid, (uint32_t)s, slot, k) * (r - l);
      double lt;
      if (inside(t, lt)) {
        for (int d = 0; d < D; ++d) x[d] = y[d];
        xl = lt; moved = true;
        break;
      }
      ++ns;
      if (t < 0.0) l = t; else r = t;
    }
    if (!moved) ++nk;
    if (a.t_evals) a.t_evals[row * a.S + s] = ne - ne0;
    if (a.t_logl) a.t_logl[row * a.S + s] = xl;
  }
  for (int d = 0; d < D; ++d) a.u[row * D + d] = x[d];
  a.logl[row] = xl;
  if (a.n_eval) a.n_eval[row] = ne;
  if (a.n_oob) a.n_oob[row] = no;
  if (a.n_expand) a.n_expand[row] = nx;
  if (a.n_shrink) a.n_shrink[row] = ns;
  if (a.n_stuck) a.n_stuck[row] = nk;
  if (a.n_moved) a.n_moved[row] = a.S - nk;
}

// GW likelihoods: one CTA per walker.  Thread 0 runs the slice step's control flow; the likelihood of its candidate points is
// evaluated by the whole CTA with the same machinery as k_walk_gw (per-candidate set-up by one lane each, then a bin sweep).
// The two ends of the bracket are tested together while stepping out (their tests are independent given x and the direction, so
// the evaluations, counters and results are those of the sequential statement); shrinkage candidates go two at a time, the second
// being the sequential statement's next draw under the assumption that the first is rejected (discarded, uncounted, otherwise).
template <int MODEL, int NDET, int NT>
__global__ void __launch_bounds__(NT, 512 / NT) k_slice_gw(const DevCfg* __restrict__ cfgp, Tables tb, SliceArgs a) {
  using AL = AccLayout<MODEL, NDET>;
  constexpr int NW = NT / 32, PG = 2, ND1 = NDET > 1 ? NDET - 1 : 1;
  __shared__ __align__(16) double cbs[PG * CB_SIZE];
  __shared__ double2 tabL[PG * ND1 * 32], tabW[PG * ND1 * NW], step[PG * ND1];
  __shared__ double red[NW * PG * AL::N], out[PG * AL::N];
  __shared__ MathTables mtab;
  __shared__ bool active[PG];
  __shared__ int slot[PG];
  __shared__ double s_x[kMaxDim], s_dir[kMaxDim], s_y[PG][kMaxDim], s_logl[PG];
  __shared__ int s_flag[PG];      // per candidate: -1 none, 0 out of the cube, 1 in the cube but unphysical theta, 2 to be swept
  __shared__ int s_ctl;           // 0: another round of this step, 1: step finished, 2: walk finished
  const DevCfg& cfg = *cfgp;
  const int D = cfg.ndim;
  const int tid = threadIdx.x;
  const long long row = blockIdx.x;
  const uint32_t wslot = (uint32_t)(a.slot0 + row);
  const double lstar = a.lstar_dev ? *a.lstar_dev : a.lstar;
  const uint32_t sid = a.stream_id | (a.iter_dev ? (uint32_t)(*a.iter_dev & 0xFFFFFF) : 0u);
  load_math_tables(&mtab, tb.mt, tid, NT);
  // thread 0's state
  double xl = 0.0, l = 0.0, r = 0.0, cand_t[PG] = {0.0, 0.0};
  int ne = 0, no = 0, nx = 0, ns = 0, nk = 0, ne0 = 0;
  int s = 0, mode = 0, kl = 0, kr = 0, ksh = 0;
  bool l_act = false, r_act = false, fresh = true;
  if (tid == 0) {
    for (int d = 0; d < D; ++d) s_x[d] = a.u[row * D + d];
    xl = a.logl[row];
    s_ctl = (a.S > 0) ? 0 : 2;
  }
  __syncthreads();
  while (s_ctl != 2) {
    // ---- thread 0: next candidates
    if (tid == 0) {
      if (fresh) {          // new slice step: direction and bracket
        slice_direction(cfg, a, sid, (uint32_t)s, wslot, s_dir);
        uint32_t w8[4];
        philox4x32_10(8u, (uint32_t)s, wslot, sid, a.k0, a.k1, w8);
        l = -u01(w8[0], w8[1]); r = l + 1.0;
        mode = 0; kl = kr = ksh = 0; l_act = r_act = true; ne0 = ne; fresh = false;
      }
      if (mode == 0 && !l_act && !r_act) mode = 1;
      s_flag[0] = s_flag[1] = -1;
      if (mode == 0) {
        if (l_act) { cand_t[0] = l; s_flag[0] = slice_point(cfg, s_x, s_dir, l, s_y[0]) ? 2 : 0; }
        if (r_act) { cand_t[1] = r; s_flag[1] = slice_point(cfg, s_x, s_dir, r, s_y[1]) ? 2 : 0; }
      } else {
        // shrinkage, two candidates per round: the second is the one the sequential statement draws IF the first is rejected
        // (the bracket end on the first one's side moves to it; the draw itself does not depend on any likelihood value)
        cand_t[0] = l + slice_shrink_uniform(a, sid, (uint32_t)s, wslot, ksh) * (r - l);
        s_flag[0] = slice_point(cfg, s_x, s_dir, cand_t[0], s_y[0]) ? 2 : 0;
        if (ksh + 1 < kSliceMaxShrink) {
          const double l2 = (cand_t[0] < 0.0) ? cand_t[0] : l, r2 = (cand_t[0] < 0.0) ? r : cand_t[0];
          cand_t[1] = l2 + slice_shrink_uniform(a, sid, (uint32_t)s, wslot, ksh + 1) * (r2 - l2);
          s_flag[1] = slice_point(cfg, s_x, s_dir, cand_t[1], s_y[1]) ? 2 : 0;
        }
      }
    }
    __syncthreads();
    // ---- set-up of the in-cube candidates, one lane each
    if (tid < PG && s_flag[tid] == 2) {
      double th[11];
#pragma unroll
      for (int d = 0; d < 11; ++d) th[d] = prior_transform_dim(cfg.prior_kind[d], cfg.prior_lo[d], cfg.prior_hi[d], s_y[tid][d]);
      s_flag[tid] = setup_particle<MODEL>(cfg, th, cbs + tid * CB_SIZE) ? 2 : 1;
    }
    __syncthreads();
    const int n_sw = (s_flag[0] == 2 ? 1 : 0) + (s_flag[1] == 2 ? 1 : 0);
    if (n_sw > 0) {
      build_phasor_tables<NDET, NT>(cfg, cbs, PG, tabL, tabW, step);
      if (tid < PG) {
        const int first = (s_flag[0] == 2) ? 0 : 1;
        slot[tid] = (n_sw == 2) ? tid : first;
        active[tid] = (n_sw == 2) || tid == 0;
      }
      __syncthreads();
      if (n_sw == 2) sweep_group<MODEL, NDET, 2, NT>(cfg, tb, cbs, tabL, tabW, step, &mtab, active, slot, red, out);
      else sweep_group<MODEL, NDET, 1, NT>(cfg, tb, cbs, tabL, tabW, step, &mtab, active, slot, red, out);
      if (tid < n_sw) s_logl[slot[tid]] = finish_logl<MODEL, NDET>(cfg, cbs + slot[tid] * CB_SIZE, out + tid * AL::N, nullptr);
      __syncthreads();
    }
    // ---- thread 0: consume the outcomes
    if (tid == 0) {
      auto outcome = [&](int c, double& lt) -> bool {      // inside(candidate c); counts like the sequential statement
        if (s_flag[c] == 0) { ++no; return false; }
        ++ne;
        lt = (s_flag[c] == 2) ? s_logl[c] : -INFINITY;
        return lt > lstar;
      };
      double lt = 0.0;
      bool done = false;
      if (mode == 0) {
        if (l_act) { if (outcome(0, lt)) { l -= 1.0; ++nx; if (++kl == kSliceMaxExpand) l_act = false; } else l_act = false; }
        if (r_act) { if (outcome(1, lt)) { r += 1.0; ++nx; if (++kr == kSliceMaxExpand) r_act = false; } else r_act = false; }
      } else {
        for (int c = 0; c < PG && !done && s_flag[c] >= 0; ++c) {      // in order; the second only if the first was rejected
          if (outcome(c, lt)) {
            for (int d = 0; d < D; ++d) s_x[d] = s_y[c][d];
            xl = lt; done = true;
          } else {
            ++ns;
            if (cand_t[c] < 0.0) l = cand_t[c]; else r = cand_t[c];
            if (++ksh == kSliceMaxShrink) { ++nk; done = true; }
          }
        }
      }
      if (done) {
        if (a.t_evals) a.t_evals[row * a.S + s] = ne - ne0;
        if (a.t_logl) a.t_logl[row * a.S + s] = xl;
        ++s; fresh = true;
      }
      s_ctl = (s >= a.S) ? 2 : (done ? 1 : 0);
    }
    __syncthreads();
  }
  if (tid == 0) {
    for (int d = 0; d < D; ++d) a.u[row * D + d] = s_x[d];
    a.logl[row] = xl;
    if (a.n_eval) a.n_eval[row] = ne;
    if (a.n_oob) a.n_oob[row] = no;
    if (a.n_expand) a.n_expand[row] = nx;
    if (a.n_shrink) a.n_shrink[row] = ns;
    if (a.n_stuck) a.n_stuck[row] = nk;
    if (a.n_moved) a.n_moved[row] = a.S - nk;
  }
}

// Direction factor inside the sampler: lower-triangular Cholesky factor of the covariance of the m survivors (unit-cube
// coordinates, free dims; FIXED dims get zero rows): sequential sums in the survivors' order, 1/(m-1), diagonal (1 + 1e-12).
// One CTA: thread per dimension (means), thread per (a, b) pair (covariances), thread 0 (factorisation).
__global__ void k_cov_chol(const DevCfg* __restrict__ cfgp, const double* __restrict__ pts, int m, double* Lc) {
  __shared__ double mean[kMaxDim], C[kMaxDim][kMaxDim];
  const DevCfg& cfg = *cfgp;
  const int D = cfg.ndim, t = threadIdx.x;
  if (t < D) {
    double acc = 0.0;
    for (int i = 0; i < m; ++i) acc += pts[(size_t)i * D + t];
    mean[t] = acc / m;
  }
  __syncthreads();
  if (t < D * D) {
    const int a_ = t / D, b_ = t % D;
    if (b_ <= a_) {
      double acc = 0.0;
      for (int i = 0; i < m; ++i) acc += (pts[(size_t)i * D + a_] - mean[a_]) * (pts[(size_t)i * D + b_] - mean[b_]);
      C[a_][b_] = acc / (m - 1);
    }
  }
  __syncthreads();
  if (t == 0) {
    for (int i = 0; i < D * D; ++i) Lc[i] = 0.0;
    for (int a_ = 0; a_ < D; ++a_) {
      if (cfg.prior_kind[a_] == 4) continue;
      for (int b_ = 0; b_ <= a_; ++b_) {
        if (cfg.prior_kind[b_] == 4) continue;
        double sum = (a_ == b_) ? C[a_][a_] * (1.0 + 1e-12) : C[a_][b_];
        for (int c = 0; c < b_; ++c) sum -= Lc[a_ * D + c] * Lc[b_ * D + c];
        Lc[a_ * D + b_] = (a_ == b_) ? sqrt(sum) : sum / Lc[b_ * D + b_];
      }
    }
  }
}
