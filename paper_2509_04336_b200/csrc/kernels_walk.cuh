// kernels_walk.cuh -- K2: DE proposal, the thread-per-walker walk for bin-less likelihoods, the speculative-chunk GW walk kernel
// Part of libnsgw (one translation unit): included by nsgw.cu inside its anonymous namespace, after nsgw_device.cuh.
// See include/nsgw.h for the contract and DESIGN.md section 5 for the design of each kernel.
#pragma once

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
  int stage;                // GW PhenomD-form exact sweep: 1 = per-thread LDGSTS staging of the table values (bin_loop)
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
                                            const int* slot, double* red, double* out /*smem [PG][N]*/,
                                            double* stage = nullptr /*smem, see bin_loop*/) {
  using AL = AccLayout<MODEL, NDET>;
  constexpr int NV = PG * AL::N;
  double acc[PG][AL::N];
  bin_loop<MODEL, NDET, PG, NT>(cfg, tb, cbs, tabL, tabW, step, mt, active, slot, acc, stage);
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
// the per-thread table staging slots of bin_loop's merger-ringdown loop (WalkArgs::stage), carved behind the chunk buffers
template <int NDET, int NT>
constexpr size_t walk_stage_bytes() { return sizeof(double) * NT * (3 + 3 * NDET); }

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
  double* stage = (MODEL == 2 && !RB && a.stage) ? cbs + DM * (CB_SIZE + kMaxDim) : nullptr;   // exact PhenomD sweep: table staging
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
        if (ng == PG) sweep_group<MODEL, NDET, PG, NT>(cfg, tb, cbs, tabL, tabW, step, &mtab, active, slot, red, out, stage);
        else sweep_group<MODEL, NDET, 1, NT>(cfg, tb, cbs, tabL, tabW, step, &mtab, active, slot, red, out, stage);
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

