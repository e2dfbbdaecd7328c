// kernels_k3.cuh -- K3: selection (rank), evidence scan, start points, write-back, adaptation, final evidence; FP64 peak probe
// Part of libnsgw (one translation unit): included by nsgw.cu inside its anonymous namespace, after nsgw_device.cuh.
// See include/nsgw.h for the contract and DESIGN.md section 5 for the design of each kernel.
#pragma once

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
// fixed_w > 0 (slice kernel): report that many steps per replacement and leave the walk length alone.
__global__ void k_adapt(DevState* st, const int* __restrict__ na, const int* __restrict__ ne, const int* __restrict__ no, int k,
                        const double* __restrict__ logl, int n, int fixed_w) {
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
    const int W = fixed_w > 0 ? fixed_w : st->W;
    double amean = (double)s_a[0] / k;
    double r = fmax(0.5, amean) / W;
    double walks = fixed_w > 0 ? st->walks : fmin((st->walks * st->delay + st->naccept / r) / (st->delay + 1.0), (double)st->maxmcmc);
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
// lw_out (optional) [n]: the width log w of each live point in ascending-logL order (the rows R:L26 appends to the dead points).
__global__ void k_finalize(const DevState* __restrict__ st, const double* __restrict__ logl, const int* __restrict__ order, int n,
                           double* out, double* lw_out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double logx = st->logx, logz = st->logz, h = st->h, lw;
  for (int i = 0; i < n; ++i) {
    evidence_update(logl[order[i]], (double)(n - i), logx, logz, h, lw);
    if (lw_out) lw_out[i] = lw;
  }
  out[0] = logz; out[1] = h;
}

// Posterior rows (R:L26): the recorded dead points followed by the live points in ascending logL.  theta
// (optional) [N, D] = prior transform of each row; t [N] = logL + log w.
__global__ void k_post_rows(const DevCfg* __restrict__ cfg, const double* __restrict__ dead, long long n_dead,
                            const double* __restrict__ live_u, const double* __restrict__ live_l, const int* __restrict__ order,
                            const double* __restrict__ lw_live, int n, double* theta, double* t) {
  const long long r = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (r >= n_dead + n) return;
  const int D = cfg->ndim;
  const double* u;
  double l, w;
  if (r < n_dead) {
    const double* row = dead + (size_t)r * (D + 3);
    u = row; l = row[D]; w = row[D + 1];
  } else {
    const int j = (int)(r - n_dead), id = order[j];
    u = live_u + (size_t)id * D; l = live_l[id]; w = lw_live[j];
  }
  if (theta)
    for (int d = 0; d < D; ++d)
      theta[(size_t)r * D + d] = prior_transform_dim(cfg->prior_kind[d], cfg->prior_lo[d], cfg->prior_hi[d], u[d]);
  t[r] = l + w;
}

constexpr int kPostThreads = 1024;

// Fixed-order sum (or maximum) over the CTA: strided partials, then a binary tree in shared memory.
template <bool MAX>
__device__ __forceinline__ double post_reduce(double v, double* red) {
  __syncthreads();
  red[threadIdx.x] = v;
  __syncthreads();
  for (int s = kPostThreads / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) red[threadIdx.x] = MAX ? fmax(red[threadIdx.x], red[threadIdx.x + s]) : red[threadIdx.x] + red[threadIdx.x + s];
    __syncthreads();
  }
  return red[0];
}

// Normalises t in place to log p = t - logZ, logZ = log sum exp t (R:L26), and reduces the summaries: out[0] = logZ,
// out[1] = 1 / sum p^2, out[2 + d] = sum p [theta_d < ref_d] (NaN without a reference point).  One CTA, fixed order.
__global__ void __launch_bounds__(kPostThreads) k_post_norm(double* t, long long N, const double* __restrict__ theta, int D,
                                                            const double* __restrict__ ref, double* out) {
  __shared__ double red[kPostThreads];
  const int tid = threadIdx.x;
  double m = -INFINITY;
  for (long long i = tid; i < N; i += kPostThreads) m = fmax(m, t[i]);
  m = post_reduce<true>(m, red);
  double s = 0.0;
  for (long long i = tid; i < N; i += kPostThreads) s += exp(t[i] - m);
  s = post_reduce<false>(s, red);
  const double logz = m + log(s);
  double s2 = 0.0;
  for (long long i = tid; i < N; i += kPostThreads) {
    const double lp = t[i] - logz, p = exp(lp);
    t[i] = lp;
    s2 += p * p;
  }
  s2 = post_reduce<false>(s2, red);
  if (tid == 0) { out[0] = logz; out[1] = 1.0 / s2; }
  for (int d = 0; d < D; ++d) {
    double c = 0.0;
    if (ref && theta)
      for (long long i = tid; i < N; i += kPostThreads)
        if (theta[(size_t)i * D + d] < ref[d]) c += exp(t[i]);
    c = post_reduce<false>(c, red);
    if (tid == 0) out[2 + d] = (ref && theta) ? c : NAN;
  }
}

// Inclusive cumulative sum of p = exp(log p) in row order (R:L27).  One CTA: thread t owns the contiguous rows
// [t L, (t + 1) L), L = ceil(N / kPostThreads); thread 0 scans the partials; fixed order, bit-reproducible.
__global__ void __launch_bounds__(kPostThreads) k_post_cumsum(const double* __restrict__ logp, long long N, double* cum) {
  __shared__ double part[kPostThreads];
  const int tid = threadIdx.x;
  const long long L = (N + kPostThreads - 1) / kPostThreads;
  const long long lo = min(N, tid * L), hi = min(N, lo + L);
  double s = 0.0;
  for (long long i = lo; i < hi; ++i) s += exp(logp[i]);
  part[tid] = s;
  __syncthreads();
  if (tid == 0) {
    double run = 0.0;
    for (int t = 0; t < kPostThreads; ++t) { const double v = part[t]; part[t] = run; run += v; }
  }
  __syncthreads();
  s = part[tid];
  for (long long i = lo; i < hi; ++i) { s += exp(logp[i]); cum[i] = s; }
}

// Systematic resampling (R:L27): draw j sits at t_j = (j + U) / n_out, U = u01 of Philox block (0, 0, 0, 4 << 24) under
// key = seed; its row is the first i with C_i > t_j C_{N-1} (binary search).  idx and / or the gathered theta rows are written.
__global__ void k_post_pick(const double* __restrict__ cum, long long N, long long n_out, uint32_t k0, uint32_t k1, int D,
                            const double* __restrict__ theta, long long* idx, double* theta_out) {
  const long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (j >= n_out) return;
  uint32_t w[4];
  philox4x32_10(0u, 0u, 0u, 4u << 24, k0, k1, w);
  const double U = u01(w[0], w[1]);
  const double v = (((double)j + U) / (double)n_out) * cum[N - 1];
  long long lo = 0, hi = N;            // first i in [0, N) with cum[i] > v; N if none
  while (lo < hi) {
    const long long mid = (lo + hi) >> 1;
    if (cum[mid] > v) hi = mid; else lo = mid + 1;
  }
  const long long i = min(lo, N - 1);
  if (idx) idx[j] = i;
  if (theta_out)
    for (int d = 0; d < D; ++d) theta_out[(size_t)j * D + d] = theta[(size_t)i * D + d];
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
