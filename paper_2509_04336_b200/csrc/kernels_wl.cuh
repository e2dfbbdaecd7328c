// kernels_wl.cuh -- K2 as a worklist: the lock-step acceptance walk of a batch in ROUNDS over the whole batch.
// Part of libnsgw (one translation unit): included by nsgw.cu inside its anonymous namespace, after kernels_walk.cuh.
//
// k_walk_gw gives every walker a CTA of its own: with k = 500-700 walkers that is 16-20 warps per SM streaming the bins' table
// values from L2, one barrier-separated phase after the other (measured 0.27 of the FP64 peak on config 3).  Here a round is
//   k_wl_head   (warp per walker)  resolve the walker's previous chunk (first acceptance discards the later steps), then propose
//                                  its next chunk: steps t0, t0+1, .. from the current point until E of them are in bounds (at most
//                                  128 steps), rows for the in-bounds ones allocated from a batch-wide counter, prior transform
//                                  and waveform set-up one row per lane;
//   row sweep   (nsgw.cu)          the likelihood of EVERY row of the batch in one launch of the batched likelihood kernels
//                                  (k x E = 16 000 rows on config 3: the machine is full, tables are reused across rows);
// chained on the stream; round r + 1's kernel publishes the number of walkers that still walked in round r to mapped host memory, the
// host follows the device two rounds behind and stops enqueuing when the number reaches zero (rounds enqueued past the end are no-ops).  Decisions, counters, trace and end points are exactly those of
// the sequential algorithm and of k_walk_gw for every chunk length: a row's logL does not depend on the rows it shares a launch
// with, and the speculative steps after an acceptance are redone from the accepted point with the same Philox counters.
#pragma once

constexpr int kWlWarps = 2;          // warps of a walker's CTA in k_wl_head: warp 0 resolves and proposes, both set the rows up
constexpr int kWlEMax = 64;          // rows per walker and round (cap)

struct WlState {
  int* t0;                // [B] steps consumed
  int* E;                 // [B] in-bounds proposals the walker asks for in its next chunk (adaptive: halved after a chunk with an
                          //     acceptance, doubled after one without; or fixed)
  int* nsteps;            // [B] steps of the pending chunk
  int* nslots;            // [B] in-bounds proposals (rows) of the pending chunk
  int* rowbase;           // [B] first row of the pending chunk in its round's row buffers
  int* cnt;               // [3 B] accepted, evaluated, out-of-bounds
  unsigned char* step;    // [B][kWalkSteps] per step of the pending chunk: 0 out of bounds, else slot + 1
  // per-round row buffers, double-buffered by round parity
  double* row_u[2];       // [R][kMaxDim] proposals
  double* row_cb[2];      // [R][CB_SIZE] coefficient blocks
  double* row_logl[2];    // [R]
  int* n_rows;            // [2] rows of the round (by parity)
  int* n_active;          // [2] walkers that proposed in the round (by parity)
  int* sum_need;          // [3] by round mod 3: rows the batch still needs (sum over walkers of remaining steps x in-bounds fraction)
  int* host_nact;         // [4] pinned host memory the device can write: n_active of round r at [r & 3], published by round r + 1's kernel
  int nact_slot;          // (r - 1) & 3 for the launch of round r
  int e_cap;              // rows per walker and round (<= kWlEMax)
  int r_target;           // rows per round the chunk lengths aim for
  int cap_rows;           // rows the row buffers hold (B x e_cap)
};

template <int MODEL>
__global__ void __launch_bounds__(32 * kWlWarps) k_wl_head(const DevCfg* __restrict__ cfgp, WalkArgs a, WlState st, int round) {
  __shared__ double s_stage[32][kMaxDim];
  __shared__ double s_prop[kWlEMax][kMaxDim];
  __shared__ double s_cur[kMaxDim];
  __shared__ int s_nslots, s_rowbase;
  const DevCfg& cfg = *cfgp;
  const int D = cfg.ndim;
  const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
  const long long row = blockIdx.x;
  const int par = round & 1;
  pdl_wait();   // the sweep of the previous round wrote the rows' logL
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    // the previous round's walker count goes to the host by a store into mapped memory (a copy in the stream between this kernel and
    // the sweep would serialise kernel -> copy engine -> kernel every round); the host reads it behind an event that follows this kernel
    if (round > 0) { st.host_nact[st.nact_slot] = st.n_active[par ^ 1]; __threadfence_system(); }
    st.n_rows[par ^ 1] = 0; st.n_active[par ^ 1] = 0; st.sum_need[(round + 1) % 3] = 0;
  }
  if (wrp == 0) {
  const int W = a.W_dev ? *a.W_dev : a.W;
  const double lstar = a.lstar_dev ? *a.lstar_dev : a.lstar;
  const uint32_t sid = a.stream_id | (a.iter_dev ? (uint32_t)(*a.iter_dev & 0xFFFFFF) : 0u);
  const bool spec_fixed = a.spec_fixed != 0;
  const int spec = max(1, min(st.e_cap, a.spec));
  int t0, E;
  double inb = 0.25;                    // in-bounds fraction of the walker's proposals (estimate: its last chunk)
  if (round == 0) {
    t0 = 0;
    // first chunk: about the number of rows to the first acceptance when the walk length is tuned to naccept acceptances (W / 100 for
    // the usual 60 of a third of the steps in bounds) -- 2 for the short walks of the first iterations, where most chunks end early,
    // near the cap for long walks, where doubling up from 2 costs four half-empty rounds
    E = spec_fixed ? spec : min(spec, max(2, W / 100));
    if (lane < 3) st.cnt[lane * a.B + row] = 0;
  } else {
    // ---- resolve the pending chunk: steps in order, the first acceptance ends it ---------------------------------------
    t0 = st.t0[row];
    E = st.E[row];
    const int nsteps = st.nsteps[row];
    if (nsteps > 0) {
      inb = fmax((double)st.nslots[row], 0.5) / nsteps;
      const int rb = st.rowbase[row];
      const double* rl = st.row_logl[par ^ 1];
      const unsigned char* stp = st.step + row * kWalkSteps;
      int used = nsteps, acc_slot = -1;
      for (int j0 = 0; j0 < nsteps; j0 += 32) {       // first accepted step, 32 steps at a time
        const int j = j0 + lane;
        const int sl = (j < nsteps) ? (int)stp[j] - 1 : -1;
        const bool hit = sl >= 0 && rl[rb + sl] > lstar;
        const unsigned m = __ballot_sync(0xffffffffu, hit);
        if (m) {
          const int first = __ffs(m) - 1;
          used = j0 + first + 1;
          acc_slot = __shfl_sync(0xffffffffu, sl, first);
          break;
        }
      }
      int n_in = 0;
      for (int j0 = 0; j0 < used; j0 += 32) {
        const int j = j0 + lane;
        if (j < used) {
          const int sl = (int)stp[j] - 1;
          const long long t = (long long)row * a.trace_stride + t0 + j;
          if (sl < 0) {
            if (a.tflags) a.tflags[t] = 1;
            if (a.tlogl) a.tlogl[t] = nan("");
          } else {
            ++n_in;
            const double pl = rl[rb + sl];
            if (a.tflags) a.tflags[t] = (j == used - 1 && acc_slot >= 0) ? 6 : 4;
            if (a.tlogl) a.tlogl[t] = pl;
          }
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) n_in += __shfl_xor_sync(0xffffffffu, n_in, o);
      if (acc_slot >= 0) {
        const double* ru = st.row_u[par ^ 1] + (size_t)(rb + acc_slot) * kMaxDim;
        if (lane < D) a.u[row * D + lane] = ru[lane];
        if (lane == 0) a.logl[row] = rl[rb + acc_slot];
      }
      if (lane == 0) {
        st.cnt[0 * a.B + row] += (acc_slot >= 0) ? 1 : 0;
        st.cnt[1 * a.B + row] += n_in;
        st.cnt[2 * a.B + row] += used - n_in;
      }
      t0 += used;
      if (!spec_fixed) E = (acc_slot >= 0) ? max(1, E >> 1) : min(spec, E << 1);
    }
  }
  __syncwarp();
  // ---- propose the next chunk from the current point -----------------------------------------------------------------------
  if (lane < D) s_cur[lane] = a.u[row * D + lane];
  __syncwarp();
  int nslots = 0, nsteps = 0;
  int rowbase = 0;
  if (t0 < W) {
    // Chunk length.  The walkers differ in how many of their W steps are in bounds, i.e. in how many rows they still need; lengths
    // in proportion to that need make them finish in the same round, with about r_target rows per round over the batch (the need
    // of the batch is last round's sum).  The walker's own halve-after-a-hit / double-after-a-miss length caps it: where
    // acceptances are frequent, long chunks are mostly discarded.  Any choice gives the same chain.
    const int need = max(1, (int)ceil((W - t0) * inb));
    if (lane == 0) atomicAdd(&st.sum_need[round % 3], need);
    int emax = E;
    if (!spec_fixed) {
      const double tot = (round == 0) ? 0.25 * (double)W * (double)a.B : (double)st.sum_need[(round + 2) % 3];
      const int e_pol = (int)ceil(need * (double)st.r_target / fmax(tot, (double)st.r_target));
      emax = max(1, min(E, min(spec, e_pol)));
    }
    unsigned char* stp = st.step + row * kWalkSteps;
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
        stp[j] = inb ? (unsigned char)(nslots + rank + 1) : 0;
        if (inb)
          for (int d = 0; d < D; ++d) s_prop[nslots + rank][d] = s_stage[lane][d];
      }
      nslots += min(cnt, room);
      nsteps += consumed;
      __syncwarp();
    }
    // rows for the in-bounds proposals from the batch-wide counter (placement is arbitrary: a row's logL does not depend on it)
    if (lane == 0 && nslots > 0) rowbase = atomicAdd(&st.n_rows[par], nslots);
    rowbase = __shfl_sync(0xffffffffu, rowbase, 0);
    if (rowbase + nslots > st.cap_rows) __trap();   // cannot happen (every walker asks for <= e_cap rows): a bounds check that stays on
    if (lane == 0) atomicAdd(&st.n_active[par], 1);
  }
  if (lane == 0) {
    st.t0[row] = t0; st.E[row] = E; st.nsteps[row] = nsteps; st.nslots[row] = nslots; st.rowbase[row] = rowbase;
    s_nslots = nslots; s_rowbase = rowbase;
  }
  }   // warp 0
  __syncthreads();
  // prior transform and waveform set-up of the chunk's rows, one row per thread of the CTA (the serial set-up chain is the latency
  // of this kernel: 64 lanes take a 64-row chunk in one pass)
  const int nslots_all = s_nslots, rowbase_all = s_rowbase;
  for (int sl = threadIdx.x; sl < nslots_all; sl += 32 * kWlWarps) {
    double* ru = st.row_u[par] + (size_t)(rowbase_all + sl) * kMaxDim;
    double th[11];
#pragma unroll
    for (int d = 0; d < 11; ++d) {
      const double x = s_prop[sl][d];
      ru[d] = x;
      th[d] = prior_transform_dim(cfg.prior_kind[d], cfg.prior_lo[d], cfg.prior_hi[d], x);
    }
    setup_particle<MODEL>(cfg, th, st.row_cb[par] + (size_t)(rowbase_all + sl) * CB_SIZE);
  }
}

// Counters of the finished walk -> the caller's arrays (each may be null).
__global__ void k_wl_counters(const int* __restrict__ cnt, long long B, int* na, int* ne, int* no) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= B) return;
  if (na) na[i] = cnt[i];
  if (ne) ne[i] = cnt[B + i];
  if (no) no[i] = cnt[2 * B + i];
}
