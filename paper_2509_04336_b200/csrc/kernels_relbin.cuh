// kernels_relbin.cuh -- relative binning (R:L24): bin edges, summary data, batched evaluation
// Part of libnsgw (one translation unit): included by nsgw.cu inside its anonymous namespace, after nsgw_device.cuh.
// See include/nsgw.h for the contract and DESIGN.md section 5 for the design of each kernel.
#pragma once

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

