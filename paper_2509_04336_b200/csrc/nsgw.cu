// nsgw.cu -- host side and C-ABI of libnsgw.so (see include/nsgw.h for the contract, DESIGN.md for the design).
//
// One translation unit; the kernels live in headers included below (inside the anonymous namespace):
//   nsgw_device.cuh      Philox, prior transforms, table-driven sin/cos / exp / atan, detector response, per-particle set-up,
//                        per-bin PhenomD-form evaluation
//   kernels_k1.cuh       k_tables / k_i73 / k_math_tables / k_draw_live / k_prior_transform (ns_init), k_setup, k_bins (CTA per
//                        particle pair), k_bins_lp + k_finish (lane per particle), k_waveform
//   kernels_pdlp.cuh     k_pd_lp (PhenomD-form, lane per row, atan / exp / phasors carried from bin to bin, ticketed finish), k_finish_rows
//   kernels_relbin.cuh   k_rb_delta / k_rb_select / k_rb_summary / k_relbin (relative binning, R:L24)
//   kernels_walk.cuh     de_propose, k_walk_simple, k_walk_gw (speculative chunks; exact or relative-binning likelihood)
//   kernels_wl.cuh       k_wl_head (the walk as batch-wide rounds: resolve + propose + set-up per walker; rows swept by the K1 kernels)
//   kernels_slice.cuh    k_slice_simple, k_slice_gw (hit-and-run slice sampling, R:L25)
//   kernels_k3.cuh       k_rank / k_evidence / k_gather_start / k_writeback / k_adapt / k_finalize, k_dfma_probe
// This file: ns_handle, launch geometry, argument checks and the extern "C" entry points.
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
constexpr int kPostOut = 2 + kMaxDim;                 // ns_posterior summaries: logZ, ESS, CL per parameter
constexpr int kFinDoubles = 2 + kPostOut + kMaxDim;   // d_fin / h_fin: final evidence, posterior summaries, reference point

// ======================================================================================================
// Device state of the sampler
// ======================================================================================================
struct DevState {
  double logx, logz, h, walks, delay, lstar;
  long long iter, n_eval_total;
  int W, naccept, maxmcmc, pad;
  ns_stats stats;
};

#include "kernels_k1.cuh"
#include "kernels_pdlp.cuh"
#include "kernels_relbin.cuh"
#include "kernels_walk.cuh"
#include "kernels_wl.cuh"
#include "kernels_slice.cuh"
#include "kernels_k3.cuh"


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
  double* d_partial = nullptr;  // k_bins_lp / k_pd_lp: per-range partial sums [n_ranges][N][B]
  size_t partial_cap = 0;
  int* d_ticket = nullptr;      // k_pd_lp: ranges finished per row group (zero between launches)
  long long ticket_cap = 0;
  int n_sm = 148;
  int opt_host_zero_copy = 1;   // gw_loglike_batch_host reads / writes pinned buffers in place (NSGW_OPT_HOST_ZERO_COPY)
  int opt_inner = 0;            // 0 acceptance walk, 1 hit-and-run slice sampling inside ns_step
  int opt_slice_steps = 0;      // slice steps per replacement (0: 5 per free dimension)
  double* d_lc = nullptr;       // slice kernel: direction factor [ndim][ndim]
  int opt_like = 0;             // 0 exact likelihood, 1 relative binning (sampler and ns_loglike_u_batch)
  int opt_walk_spec = 0;        // 0 auto (per-walker adaptive), 1..32 fixed speculative chunk length
  int opt_walk_stage = 0;       // PhenomD-form exact walk: LDGSTS staging of the sweep's table values (NSGW_OPT_WALK_STAGE; measured slower)
  int opt_bins_kernel = 0;      // 0 auto, 1 CTA-per-particle (k_bins), 2 lane-per-particle (k_bins_lp / k_pd_lp)
  int opt_walk_kernel = 0;      // 0 auto (3), 1 CTA per walker (k_walk_gw), 2 worklist rounds swept by k_bins, 3 swept by the lane-per-row kernels
  // worklist walk (kernels_wl.cuh): per-walker state, double-buffered row buffers, host-visible progress
  WlState wl{};
  long long wl_cap_b = 0, wl_cap_r = 0;
  int wl_kr = 0;                // bins per range of k_pd_lp on the walk's rows: fixed per handle so a row's logL never depends on the round
  int* h_wl_nact = nullptr;     // pinned, mapped ring [4]: walkers of a round, written by the next round's kernel
  int* d_wl_nact = nullptr;     // its device address
  cudaEvent_t wl_ev[4] = {nullptr, nullptr, nullptr, nullptr};
  long long cb_cap = 0;
  double* d_theta = nullptr;    // scratch theta
  long long theta_cap = 0;
  double* d_hio = nullptr;      // host-entry scratch: theta [B,11] + logl [B]
  long long hio_cap = 0;
  double* d_fin = nullptr;      // 2 doubles (final evidence) + kPostOut (posterior summaries) + kMaxDim (reference point)
  double* d_post_lw = nullptr;  // [n_live] widths of the live points' rows (R:L26)
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
#define NSGW_LP_UNR 2
#define NSGW_LP_OCC 3
#endif
constexpr int kLpNT = NSGW_LP_NT, kLpKR = 256, kLpPP = NSGW_LP_PP, kLpUNR = NSGW_LP_UNR, kLpOCC = NSGW_LP_OCC;
// From kLpBigBatch rows on: ONE CTA of 512 threads per SM instead of three of 128 -- the SM then holds one copy of the 32 KB sin/cos
// table instead of three, a tile serves 1024 rows, and at 124 registers 16 warps are resident instead of 12 (measured, config 2, kernel
// time at 65536 rows: 3 x 128 threads 0.649 ms, 1 x 384 0.631, 1 x 512 0.621, with the loop unrolled by 2 instead of 4 0.616; 448 or 416
// threads -- warps not a multiple of the four sub-partitions -- 0.69 / 0.76; 640 / 768 threads spill: 0.66 / 0.72; 2 x 256 0.630).
#ifndef NSGW_LP_NT_BIG
#define NSGW_LP_NT_BIG 512
#define NSGW_LP_OCC_BIG 1
#endif
constexpr int kLpNTBig = NSGW_LP_NT_BIG, kLpOCCBig = NSGW_LP_OCC_BIG;
constexpr long long kLpBigBatch = 6144;
constexpr long long kLpMinBatch = 1024;   // below this the CTA-per-particle kernel fills the machine better
constexpr long long kPdMinBatch = 16384;  // PhenomD-form: from here k_pd_lp is faster than k_bins (measured: 35.9 vs 34.6 M evals/s at 16384, 44.5 vs 35.9 at 65536)

int ensure_partial(ns_handle* h, size_t n) {
  if (n > h->partial_cap) {
    if (h->d_partial) cudaFree(h->d_partial);
    h->d_partial = nullptr; h->partial_cap = 0;
    CU_CHECK(h, cudaMalloc(&h->d_partial, sizeof(double) * n));
    h->partial_cap = n;
  }
  return 0;
}

// Launch with programmatic stream serialization: the kernel may become resident while the kernel before it on the stream still runs;
// it calls pdl_wait() before it reads what that kernel wrote.
template <class... KArgs, class... Args>
cudaError_t launch_pdl(void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t s, Args... args) {
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3(grid); lc.blockDim = dim3(block); lc.dynamicSmemBytes = smem; lc.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = 1;
  return cudaLaunchKernelEx(&lc, kern, KArgs(args)...);
}

// cbs [B][CB_SIZE]; rows_dev (optional, device) overrides the row count of the task lists (B is then the capacity).
template <int NDET, int NT, int OCC>
int launch_bins_lp_g(ns_handle* h, const double* cbs, long long B, const int* rows_dev, double* logl, double* parts, cudaStream_t s) {
  using AL = AccLayout<1, NDET>;
  constexpr int PP = kLpPP;
  const long long ngroups = (B + NT * PP - 1) / (NT * PP);
  const long long grid_max = (long long)h->n_sm * OCC;
  // bins per task (multiple of the unroll, 32..256): the value that minimises rounds x (bins per task + per-task overhead) x
  // slow-down from sharing the SM, rounds = ceil(tasks / resident CTAs) -- large tiles amortise the per-task set-up, small ones
  // balance the last round; one CTA alone on an SM already runs at ~85 % of the FP64 pipe, so co-resident CTAs divide it
  // (this is what makes few, long tasks the better choice for small batches), plus k_finish's cost per range
  int kr = kLpKR;
  {
    double best = 1e300;
    for (int c = 32; c <= kLpKR; c += kLpUNR) {
      const int nr = (h->cfg.n_freq + c - 1) / c;
      const long long nt = ngroups * nr;
      const long long per_sm = std::min<long long>(OCC, (nt + h->n_sm - 1) / h->n_sm);
      const double cost = (double)((nt + grid_max - 1) / grid_max) * (c + 8) * std::max(1.0, 0.85 * per_sm) + 0.25 * nr;
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
  CU_CHECK(h, cudaFuncSetAttribute(k_bins_lp<NDET, NT, kLpKR, PP, kLpUNR, OCC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kLpDynSmem));
  // programmatic dependent launches: the sweep behind k_setup / k_wl_head (its table copy runs under their tail), the finish behind the sweep
  CU_CHECK(h, launch_pdl(k_bins_lp<NDET, NT, kLpKR, PP, kLpUNR, OCC>, (unsigned)grid, NT, kLpDynSmem, s, (const DevCfg*)h->d_cfg, h->tb, cbs,
                         (long long)B, rows_dev, kr, nranges, (long long)ntasks, h->d_partial));
  if (e0) { cudaEventRecord(e1, s); h->prof_ev.emplace_back(e0, e1); }
  LAUNCH_CHECK(h);
  if (rows_dev) {
    const long long gfin = std::min<long long>((B + 127) / 128, (long long)h->n_sm * 8);
    CU_CHECK(h, launch_pdl(k_finish_rows<1, NDET>, (unsigned)gfin, 128, 0, s, (const DevCfg*)h->d_cfg, cbs, (const double*)h->d_partial, nranges,
                           (long long)B, rows_dev, (long long)B, logl, parts));
  } else {
    CU_CHECK(h, launch_pdl(k_finish<1, NDET>, (unsigned)((B + 127) / 128), 128, 0, s, (const DevCfg*)h->d_cfg, cbs, (const double*)h->d_partial,
                           nranges, (long long)B, logl, parts));
  }
  LAUNCH_CHECK(h);
  return 0;
}
// (with rows_dev, B is the row CAPACITY of a round of the worklist walk and the rows are several times fewer: the small geometry's
// finer tasks -- measured on `extras.walk`, 16384 walkers: 27.2 against 22.2 M evaluations/s)
template <int NDET>
int launch_bins_lp(ns_handle* h, const double* cbs, long long B, const int* rows_dev, double* logl, double* parts, cudaStream_t s) {
  if (B >= kLpBigBatch && !rows_dev) return launch_bins_lp_g<NDET, kLpNTBig, kLpOCCBig>(h, cbs, B, rows_dev, logl, parts, s);
  return launch_bins_lp_g<NDET, kLpNT, kLpOCC>(h, cbs, B, rows_dev, logl, parts, s);
}

// Bins per range of k_pd_lp for `rows` rows (multiple of the tile length): the value that minimises rounds x (range + per-task
// overhead) over the persistent grid, rounds = ceil(tasks / CTA slots).
int pd_pick_kr(const ns_handle* h, long long rows) {
  const long long ngroups = (rows + kPdNT * kPdPP - 1) / (kPdNT * kPdPP);
  const long long slots = (long long)h->n_sm * kPdOCC;
  int kr = kPdKT;
  double best = 1e300;
  for (int c = 2 * kPdKT; c <= 384; c += kPdKT) {
    const int nr = (h->cfg.n_freq + c - 1) / c;
    const long long nt = ngroups * nr;
    const double cost = (double)((nt + slots - 1) / slots) * (c + 24) + 0.25 * nr;
    if (cost < best - 1e-9) { best = cost; kr = c; }
  }
  return kr;
}

// Scratch of k_pd_lp for `rows` rows: per-range partial sums and one ticket per row group.
int ensure_pd_scratch(ns_handle* h, long long rows, int nranges, int nacc, cudaStream_t s) {
  int rc = ensure_partial(h, (size_t)rows * nranges * nacc);
  if (rc) return rc;
  const long long ngroups = (rows + kPdNT * kPdPP - 1) / (kPdNT * kPdPP);
  if (ngroups > h->ticket_cap) {
    if (h->d_ticket) cudaFree(h->d_ticket);
    h->d_ticket = nullptr; h->ticket_cap = 0;
    CU_CHECK(h, cudaMalloc(&h->d_ticket, sizeof(int) * (size_t)ngroups));
    CU_CHECK(h, cudaMemsetAsync(h->d_ticket, 0, sizeof(int) * (size_t)ngroups, s));   // the kernel leaves every ticket at zero again
    h->ticket_cap = ngroups;
  }
  return 0;
}

// PhenomD-form rows -> logL through k_pd_lp (which also finishes).  cbs [rows][CB_SIZE]; rows_dev (optional, device) overrides `rows`
// for the task list (then `rows` is the capacity the buffers and the grid are sized for); kr: bins per range (0: by pd_pick_kr).
template <int NDET>
int launch_pd_lp(ns_handle* h, const double* cbs, long long rows, const int* rows_dev, int kr, double* logl, double* parts, cudaStream_t s) {
  using AL = AccLayout<2, NDET>;
  if (kr <= 0) kr = pd_pick_kr(h, rows);
  const int nranges = (h->cfg.n_freq + kr - 1) / kr;
  int rc = ensure_pd_scratch(h, rows, nranges, AL::N, s);
  if (rc) return rc;
  const long long ngroups = (rows + kPdNT * kPdPP - 1) / (kPdNT * kPdPP);
  PdArgs a;
  a.cbs = cbs; a.n_rows = rows; a.n_rows_dev = rows_dev; a.stride = rows; a.kr = kr; a.nranges = nranges; a.partial = h->d_partial;
  a.ticket = h->d_ticket; a.logl = logl; a.parts = parts;
  const long long ntasks = ngroups * nranges;
  const long long grid = std::min<long long>(ntasks, (long long)h->n_sm * kPdOCC);
  CU_CHECK(h, cudaFuncSetAttribute(k_pd_lp<NDET>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pd_mix_bytes<kPdPP>()));
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (h->prof && h->prof_ev.size() < 4096) {
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0, s);
  }
  // programmatic dependent launch behind k_wl_head (a round of the worklist walk) or k_setup (a batch): the tables are copied under its tail
  CU_CHECK(h, launch_pdl(k_pd_lp<NDET>, (unsigned)grid, kPdNT, pd_mix_bytes<kPdPP>(), s, (const DevCfg*)h->d_cfg, h->tb, a));
  if (e0) { cudaEventRecord(e1, s); h->prof_ev.emplace_back(e0, e1); }
  LAUNCH_CHECK(h);
  return 0;
}

template <int MODEL, int NDET>
int launch_bins_nd(ns_handle* h, long long B, double* logl, double* parts, cudaStream_t s) {
  if (MODEL == 1 && (h->opt_bins_kernel == 2 || (h->opt_bins_kernel == 0 && B >= kLpMinBatch)))
    return launch_bins_lp<NDET>(h, h->d_cb, B, nullptr, logl, parts, s);
  if (MODEL == 2 && (h->opt_bins_kernel == 2 || (h->opt_bins_kernel == 0 && B >= kPdMinBatch)))
    return launch_pd_lp<NDET>(h, h->d_cb, B, nullptr, 0, logl, parts, s);
  int P = pick_p(B);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (h->prof && h->prof_ev.size() < 4096) {
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0, s);
  }
  if (P == 2) {
    CU_CHECK(h, launch_pdl(k_bins<MODEL, NDET, 2>, (unsigned)((B + 1) / 2), kBinsThreads, 0, s, (const DevCfg*)h->d_cfg, h->tb, (const double*)h->d_cb,
                           (long long)B, (const int*)nullptr, logl, parts));
  } else {
    CU_CHECK(h, launch_pdl(k_bins<MODEL, NDET, 1>, (unsigned)B, kBinsThreads, 0, s, (const DevCfg*)h->d_cfg, h->tb, (const double*)h->d_cb, (long long)B,
                           (const int*)nullptr, logl, parts));
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

// theta_mapped: theta_dev is the device address of mapped host memory (read through k_setup_staged).
int loglike_theta(ns_handle* h, const double* theta_dev, long long B, double* logl, double* parts, cudaStream_t s, bool theta_mapped = false) {
  if (B == 0) return 0;
  int rc = ensure_cb(h, B);
  if (rc) return rc;
  unsigned g = (unsigned)((B + 127) / 128);
  if (h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2) {
    if (theta_mapped) k_setup_staged<1><<<g, 128, 0, s>>>(h->d_cfg, theta_dev, B, h->d_cb);
    else k_setup<1><<<g, 128, 0, s>>>(h->d_cfg, theta_dev, B, h->d_cb);
    LAUNCH_CHECK(h);
    return launch_bins<1>(h, B, logl, parts, s);
  }
  if (theta_mapped) k_setup_staged<2><<<g, 128, 0, s>>>(h->d_cfg, theta_dev, B, h->d_cb);
  else k_setup<2><<<g, 128, 0, s>>>(h->d_cfg, theta_dev, B, h->d_cb);
  LAUNCH_CHECK(h);
  return launch_bins<2>(h, B, logl, parts, s);
}

// Device address of a host buffer the device can access directly (pinned and mapped: cudaHostAlloc / cudaMallocHost / cudaHostRegister
// memory under unified addressing), or null for pageable memory.
void* mapped_device_ptr(const void* host) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, host) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return (at.type == cudaMemoryTypeHost) ? at.devicePointer : nullptr;
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
  // (per launch: the attribute is per device and per function, and a process may drive several devices and threads)
  CU_CHECK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)(walk_smem_bytes<NDET, NT>(kWalkDMax) + extra + walk_stage_bytes<NDET, NT>())));
  a.spec_cap = dm;
  a.spec = std::min(a.spec, dm);
  const size_t stage = (MODEL == 2 && !RB && a.stage) ? walk_stage_bytes<NDET, NT>() : 0;
  kern<<<(unsigned)a.B, NT, walk_smem_bytes<NDET, NT>(dm) + extra + stage, s>>>(h->d_cfg, h->tb, a, h->rb);
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
  const size_t extra = h->opt_like == 1 ? sizeof(double) * NT * 2 * NDET
                                        : (h->opt_walk_stage && h->cfg.like_kind != NSGW_LIKE_GW_TAYLORF2 ? walk_stage_bytes<NDET, NT>() : 0);
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

// ---- the walk as batch-wide rounds (kernels_wl.cuh) -----------------------------------------------------------------------
// Buffers for B walkers and R = B x e_cap rows per round.  One allocation per kind (int state, step maps, row doubles, counters).
int ensure_wl(ns_handle* h, long long B, long long R) {
  if (!h->h_wl_nact) {
    CU_CHECK(h, cudaHostAlloc((void**)&h->h_wl_nact, sizeof(int) * 4, cudaHostAllocMapped));
    CU_CHECK(h, cudaHostGetDevicePointer((void**)&h->d_wl_nact, h->h_wl_nact, 0));
    for (auto& e : h->wl_ev) CU_CHECK(h, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    CU_CHECK(h, cudaMalloc(&h->wl.n_rows, sizeof(int) * 8));
    h->wl.n_active = h->wl.n_rows + 2;
    h->wl.sum_need = h->wl.n_rows + 4;
  }
  if (B > h->wl_cap_b) {
    cudaFree(h->wl.t0); cudaFree(h->wl.step);
    h->wl.t0 = nullptr; h->wl.step = nullptr; h->wl_cap_b = 0;
    CU_CHECK(h, cudaMalloc(&h->wl.t0, sizeof(int) * 8 * (size_t)B));
    CU_CHECK(h, cudaMalloc(&h->wl.step, (size_t)B * kWalkSteps));
    h->wl.E = h->wl.t0 + B; h->wl.nsteps = h->wl.t0 + 2 * B; h->wl.rowbase = h->wl.t0 + 3 * B; h->wl.nslots = h->wl.t0 + 4 * B;
    h->wl.cnt = h->wl.t0 + 5 * B;
    h->wl_cap_b = B;
  }
  if (R > h->wl_cap_r) {
    cudaFree(h->wl.row_u[0]);
    h->wl.row_u[0] = nullptr; h->wl_cap_r = 0;
    const size_t per = (size_t)R * (kMaxDim + CB_SIZE + 1);
    CU_CHECK(h, cudaMalloc(&h->wl.row_u[0], sizeof(double) * 2 * per));
    for (int i = 0; i < 2; ++i) {
      double* base = h->wl.row_u[0] + i * per;
      h->wl.row_u[i] = base; h->wl.row_cb[i] = base + (size_t)R * kMaxDim; h->wl.row_logl[i] = base + (size_t)R * (kMaxDim + CB_SIZE);
    }
    h->wl_cap_r = R;
  }
  return 0;
}

// logL of the rows of one round (cbs [R cap][CB_SIZE], count on the device) with the batched K1 kernels.
template <int MODEL, int NDET>
int sweep_rows(ns_handle* h, const double* cbs, long long R, const int* rows_dev, bool lane, double* logl, cudaStream_t s) {
  if (MODEL == 2 && lane) return launch_pd_lp<NDET>(h, cbs, R, rows_dev, h->wl_kr, logl, nullptr, s);
  if (MODEL == 1 && lane && R >= kLpMinBatch) return launch_bins_lp<NDET>(h, cbs, R, rows_dev, logl, nullptr, s);
  if (R >= 4096)
    CU_CHECK(h, launch_pdl(k_bins<MODEL, NDET, 2>, (unsigned)((R + 1) / 2), kBinsThreads, 0, s, (const DevCfg*)h->d_cfg, h->tb, cbs, (long long)R, rows_dev,
                           logl, (double*)nullptr));
  else
    CU_CHECK(h, launch_pdl(k_bins<MODEL, NDET, 1>, (unsigned)R, kBinsThreads, 0, s, (const DevCfg*)h->d_cfg, h->tb, cbs, (long long)R, rows_dev, logl,
                           (double*)nullptr));
  LAUNCH_CHECK(h);
  return 0;
}

// rows per walker and round: up to 64 while that keeps a round near 64 Ki rows (large batches fill the machine with short chunks)
int wl_e_cap(long long B) { return (int)std::max<long long>(1, std::min<long long>(kWlEMax, 65536 / std::max<long long>(B, 1))); }

// Buffers of the worklist walk for B walkers (and the lane kernel's scratch for PhenomD-form), so that the first walk of a handle does
// not pay for allocations.
int wl_prepare(ns_handle* h, long long B, cudaStream_t s) {
  const long long R = B * wl_e_cap(B);
  int rc = ensure_wl(h, B, R);
  if (rc) return rc;
  // about 32 ranges per row group whatever the band (measured on configs 3 and 4: 8 and 127 ranges are 10-25 % slower): the rows of a
  // round vary, many tasks keep the persistent grid balanced; fixed per handle, so a row's sums never depend on the round
  if (h->wl_kr == 0) h->wl_kr = std::max(kPdKT, (h->cfg.n_freq / 32 + kPdKT - 1) / kPdKT * kPdKT);
  if (h->cfg.like_kind == NSGW_LIKE_GW_PHENOMD_FORM && h->opt_walk_kernel != 2)
    return ensure_pd_scratch(h, R, (h->cfg.n_freq + h->wl_kr - 1) / h->wl_kr, 2 + (h->cfg.n_det - 1) + h->cfg.n_det, s);
  return 0;
}

template <int MODEL, int NDET>
int run_walk_wl(ns_handle* h, const WalkArgs& a, cudaStream_t s) {
  const long long B = a.B;
  const int e_cap = wl_e_cap(B);
  const long long R = B * e_cap;
  int rc = wl_prepare(h, B, s);
  if (rc) return rc;
  // Which kernel sweeps the rows: the lane-per-row kernels win once a round holds enough rows (persistent grid, a lane walks 128 bins
  // serially), the CTA-per-row-pair kernel below that.  Rows per round are known on the device only, so the choice is made once per
  // call from what the host knows -- walkers x expected chunk length, the chunk length following the acceptance rate the walk length
  // is tuned to (naccept accepted steps per W): a function of (B, W, naccept), so a call's results do not depend on its chunking.
  bool lane = h->opt_walk_kernel == 3;
  if (h->opt_walk_kernel == 0) {
    int W = a.W;
    if (a.W_dev) {
      CU_CHECK(h, cudaMemcpyAsync(h->h_wl_nact, a.W_dev, sizeof(int), cudaMemcpyDeviceToHost, s));
      CU_CHECK(h, cudaStreamSynchronize(s));
      W = h->h_wl_nact[0];
    }
    const double chunk = std::min<double>(e_cap, std::max(1.0, 0.3 * W / std::max(1, h->cfg.naccept)));
    lane = (double)B * chunk >= 12000.0;
  }
  WlState st = h->wl;
  st.host_nact = h->d_wl_nact;
  st.e_cap = e_cap;
  st.cap_rows = (int)R;
  st.r_target = (int)std::min<long long>(R, std::max<long long>(16384, 24 * B));
  CU_CHECK(h, cudaMemsetAsync(st.n_rows, 0, sizeof(int) * 8, s));
  const unsigned gh = (unsigned)B;   // one CTA (kWlWarps warps) per walker
  for (long long r = 0;; ++r) {
    const int par = (int)(r & 1);
    st.nact_slot = (int)((r + 3) & 3);
    const int rcode = (int)std::min<long long>(r, 6 + r % 6);   // first round or not, parity and round mod 3 matter
    if (r == 0) k_wl_head<MODEL><<<gh, 32 * kWlWarps, 0, s>>>(h->d_cfg, a, st, rcode);
    else CU_CHECK(h, launch_pdl(k_wl_head<MODEL>, gh, 32 * kWlWarps, 0, s, (const DevCfg*)h->d_cfg, a, st, rcode));   // behind the sweep
    LAUNCH_CHECK(h);
    CU_CHECK(h, cudaEventRecord(h->wl_ev[r & 3], s));
    rc = sweep_rows<MODEL, NDET>(h, st.row_cb[par], R, st.n_rows + par, lane, st.row_logl[par], s);
    if (rc) return rc;
    if (r >= 2) {   // round r - 1's kernel published the walkers of round r - 2; the host runs ahead of what it has seen, and rounds
                    // enqueued after the last walker finished are no-ops
      CU_CHECK(h, cudaEventSynchronize(h->wl_ev[(r - 1) & 3]));
      if (h->h_wl_nact[(r - 2) & 3] == 0) break;
    }
  }
  if (a.n_accept || a.n_eval || a.n_oob) {
    k_wl_counters<<<(unsigned)((B + 255) / 256), 256, 0, s>>>(st.cnt, B, a.n_accept, a.n_eval, a.n_oob);
    LAUNCH_CHECK(h);
  }
  return 0;
}

int launch_walk(ns_handle* h, const WalkArgs& a, cudaStream_t s) {
  if (a.B == 0) return 0;
  if (!is_gw(h->cfg.like_kind)) {
    k_walk_simple<<<(unsigned)((a.B + 63) / 64), 64, 0, s>>>(h->d_cfg, a);
    LAUNCH_CHECK(h);
    return 0;
  }
  const int nd = h->cfg.n_det;
  if (h->opt_like == 0 && h->opt_walk_kernel != 1) {   // exact likelihood: batch-wide rounds (kernels_wl.cuh)
    if (h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2) {
      if (nd == 1) return run_walk_wl<1, 1>(h, a, s);
      if (nd == 2) return run_walk_wl<1, 2>(h, a, s);
      if (nd == 3) return run_walk_wl<1, 3>(h, a, s);
    } else {
      if (nd == 1) return run_walk_wl<2, 1>(h, a, s);
      if (nd == 2) return run_walk_wl<2, 2>(h, a, s);
      if (nd == 3) return run_walk_wl<2, 3>(h, a, s);
    }
  }
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
  cudaFree(h->d_cur_l); cudaFree(h->d_cnt); cudaFree(h->d_cb); cudaFree(h->d_partial); cudaFree(h->d_ticket); cudaFree(h->d_theta); cudaFree(h->d_fin); cudaFree(h->d_post_lw); cudaFree(h->d_hio);
  if (h->s_own) cudaStreamDestroy(h->s_own);
  cudaFree(h->d_rb_edge); cudaFree(h->d_rb_buf); cudaFree(h->d_lc);
  cudaFree(h->wl.t0); cudaFree(h->wl.step); cudaFree(h->wl.row_u[0]); cudaFree(h->wl.n_rows);
  if (h->h_wl_nact) cudaFreeHost(h->h_wl_nact);
  for (auto& e : h->wl_ev) if (e) cudaEventDestroy(e);
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
    static_assert(sizeof(MathTables) % sizeof(double2) == 0, "the 512-entry table follows the struct, 16-byte aligned");
    INIT_CHECK(cudaMalloc(&h->d_mtab, sizeof(MathTables) + sizeof(double2) * (kSc9N + kSc11N)), -2);
    double2* sc9 = reinterpret_cast<double2*>(reinterpret_cast<char*>(h->d_mtab) + sizeof(MathTables));
    h->tb.sc11 = sc9 + kSc9N;
    k_math_tables<<<1, 256, 0, s>>>(h->d_mtab, sc9, sc9 + kSc9N);
    g_launches.fetch_add(1);
    h->tb.mt = h->d_mtab;
    h->tb.sc9 = sc9;
    k_i73<<<1, 256, 0, s>>>(h->d_cfg, h->d_ws);
    g_launches.fetch_add(1);
    INIT_CHECK(cudaGetLastError(), -2);
  }

  // ---- sampler state
  INIT_CHECK(cudaMalloc(&h->d_state, sizeof(DevState)), -2);
  INIT_CHECK(cudaMalloc(&h->d_fin, sizeof(double) * kFinDoubles), -2);
  INIT_CHECK(cudaMallocHost(&h->h_stats, sizeof(ns_stats)), -2);
  INIT_CHECK(cudaMallocHost(&h->h_fin, sizeof(double) * kFinDoubles), -2);
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
    INIT_CHECK(cudaMalloc(&h->d_post_lw, sizeof(double) * (size_t)n), -2);
    INIT_CHECK(cudaMalloc(&h->d_surv, sizeof(double) * (size_t)(n - k) * D), -2);
    INIT_CHECK(cudaMalloc(&h->d_cur_u, sizeof(double) * (size_t)k * D), -2);
    INIT_CHECK(cudaMalloc(&h->d_cur_l, sizeof(double) * (size_t)k), -2);
    INIT_CHECK(cudaMalloc(&h->d_cnt, sizeof(int) * 3 * (size_t)k), -2);
    INIT_CHECK(cudaMalloc(&h->d_lc, sizeof(double) * (size_t)D * D), -2);
    if (live_u_dev) {
      INIT_CHECK(cudaMemcpyAsync(h->d_live_u, live_u_dev, sizeof(double) * (size_t)n * D, cudaMemcpyDeviceToDevice, s), -2);
    } else {
      k_draw_live<<<(n + 127) / 128, 128, 0, s>>>(D, n, (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32), h->d_live_u);
      g_launches.fetch_add(1);
    }
    int rc = loglike_u(h, h->d_live_u, n, h->d_live_l, s);
    if (rc) return bail(rc);
    if (gw) {
      rc = wl_prepare(h, k, s);
      if (rc) return bail(rc);
    }
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
  // Pinned (mapped) buffers: no copies at all -- the set-up kernel reads theta over the host link while it computes, the finishing code
  // writes logL straight into the caller's buffer; what is saved is the set-up's own time and the copy engine's turn at both ends
  // (measured at B = 65536 on one box: 0.778 ms against 0.792 with the copies, the device-resident call 0.650: the 5.8 MB of theta
  // take 0.115 ms over the link either way, and they cannot be hidden under the sweep, which needs every row's coefficient block).
  // Pageable buffers take the copies below.
  if (h->opt_host_zero_copy) {
    const double* th_m = static_cast<const double*>(mapped_device_ptr(theta_host));
    double* lg_m = static_cast<double*>(mapped_device_ptr(logl_host));
    if (th_m && lg_m) {
      int rc = loglike_theta(h, th_m, B, lg_m, nullptr, s, true);
      if (rc) return rc;
      CU_CHECK(h, cudaStreamSynchronize(s));
      return 0;
    }
  }
  if (B > h->hio_cap) {
    if (h->d_hio) cudaFree(h->d_hio);
    h->d_hio = nullptr; h->hio_cap = 0;
    CU_CHECK(h, cudaMalloc(&h->d_hio, sizeof(double) * 12 * (size_t)B));
    h->hio_cap = B;
  }
  double* th = h->d_hio;
  double* lg = h->d_hio + 11 * (size_t)B;
  // One copy in, the kernels, one copy out, all on the caller's stream.  Measured alternatives (B = 65536, pinned buffers, B200 on
  // PCIe gen 5): the same through copy streams of the handle's own with event dependencies, 0.76-0.79 of the device-resident rate;
  // two or three chunks with the copies of chunk i+1 behind the kernels of chunk i, 0.66-0.69 (the chunks' launches are less
  // efficient than one launch over the batch and every cross-stream dependency costs more than the 0.1 ms copy it hides); this
  // form, 0.83-0.86.
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
  a.spec = h->opt_walk_spec > 0 ? h->opt_walk_spec : kWlEMax;   // (k_walk_gw clamps it to its own 32-slot buffers)
  a.spec_fixed = h->opt_walk_spec > 0;
  a.stage = h->opt_walk_stage;
  return launch_walk(h, a, (cudaStream_t)stream);
}

}  // extern "C"

namespace {
// Slice kernel launch (bin-less likelihoods: thread per walker; GW: CTA per walker).
int launch_slice(ns_handle* h, const SliceArgs& a, cudaStream_t s) {
  if (a.B == 0) return 0;
  if (!is_gw(h->cfg.like_kind)) {
    k_slice_simple<<<(unsigned)((a.B + 63) / 64), 64, 0, s>>>(h->d_cfg, a);
    LAUNCH_CHECK(h);
    return 0;
  }
  const bool tf2 = h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2;
  const int nd = h->cfg.n_det;
#define SLICE_GW(M, N) k_slice_gw<M, N, 128><<<(unsigned)a.B, 128, 0, s>>>(h->d_cfg, h->tb, a)
  if (tf2) { if (nd == 1) SLICE_GW(1, 1); else if (nd == 2) SLICE_GW(1, 2); else SLICE_GW(1, 3); }
  else { if (nd == 1) SLICE_GW(2, 1); else if (nd == 2) SLICE_GW(2, 2); else SLICE_GW(2, 3); }
#undef SLICE_GW
  LAUNCH_CHECK(h);
  return 0;
}

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
  a.spec = h->opt_walk_spec > 0 ? h->opt_walk_spec : kWlEMax;
  a.spec_fixed = h->opt_walk_spec > 0;
  a.stage = h->opt_walk_stage;
  a.k0 = k0; a.k1 = k1; a.stream_id = 0u; a.slot0 = 0;
  a.n_accept = h->d_cnt; a.n_eval = h->d_cnt + k; a.n_oob = h->d_cnt + 2 * k;
  int rc = 0;
  if (h->opt_inner == 1) {
    // hit-and-run slice sampling (R:L25): directions from the survivors' covariance, a fixed number of steps, no adaptation
    k_cov_chol<<<1, 256, 0, s>>>(h->d_cfg, h->d_surv, m, h->d_lc);
    LAUNCH_CHECK(h);
    SliceArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.Lc = h->d_lc; sa.u = h->d_cur_u; sa.logl = h->d_cur_l; sa.B = k;
    sa.lstar_dev = &h->d_state->lstar; sa.iter_dev = &h->d_state->iter;
    sa.S = h->opt_slice_steps > 0 ? h->opt_slice_steps : 5 * h->n_free;
    sa.k0 = k0; sa.k1 = k1; sa.stream_id = 0u; sa.slot0 = 0;
    sa.n_moved = h->d_cnt; sa.n_eval = h->d_cnt + k; sa.n_oob = h->d_cnt + 2 * k;
    rc = launch_slice(h, sa, s);
  } else {
    rc = launch_walk(h, a, s);
  }
  if (rc) return rc;
  k_writeback<<<(k + 127) / 128, 128, 0, s>>>(h->d_order, k, D, h->d_cur_u, h->d_cur_l, h->d_live_u, h->d_live_l);
  LAUNCH_CHECK(h);
  k_adapt<<<1, 256, 0, s>>>(h->d_state, h->d_cnt, h->d_cnt + k, h->d_cnt + 2 * k, k, h->d_live_l, n,
                            h->opt_inner == 1 ? (h->opt_slice_steps > 0 ? h->opt_slice_steps : 5 * h->n_free) : 0);
  LAUNCH_CHECK(h);
  return 0;
}
}  // namespace

extern "C" {

int ns_slice_batch(ns_handle* h, const double* lc_dev, double* u_dev, double* logl_dev, int64_t B, double logl_star, int32_t n_steps,
                   uint64_t seed, uint32_t stream_id, int64_t slot0, int32_t* n_eval_dev, int32_t* n_oob_dev, int32_t* n_expand_dev,
                   int32_t* n_shrink_dev, int32_t* n_stuck_dev, int32_t* trace_evals_dev, double* trace_logl_dev, void* stream) {
  if (!h) return -3;
  if (B < 0 || n_steps < 0 || !lc_dev || (B > 0 && (!u_dev || !logl_dev))) return fail(h, -1, "bad arguments");
  if (h->opt_like == 1) return fail(h, -5, "the slice kernel evaluates the exact likelihood only");
  if (B == 0) return 0;
  cudaStream_t s = (cudaStream_t)stream;
  SliceArgs a;
  memset(&a, 0, sizeof(a));
  a.Lc = lc_dev; a.u = u_dev; a.logl = logl_dev; a.B = B; a.lstar = logl_star; a.S = n_steps;
  a.k0 = (uint32_t)(seed & 0xFFFFFFFFull); a.k1 = (uint32_t)(seed >> 32); a.stream_id = stream_id; a.slot0 = slot0;
  a.n_eval = n_eval_dev; a.n_oob = n_oob_dev; a.n_expand = n_expand_dev; a.n_shrink = n_shrink_dev; a.n_stuck = n_stuck_dev;
  a.t_evals = trace_evals_dev; a.t_logl = trace_logl_dev;
  return launch_slice(h, a, s);
}

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
  // the runs step on streams of their own (non-blocking): everything the caller enqueued before -- on whatever stream -- must be
  // complete first; the call returns with every run's stream idle
  if (cudaDeviceSynchronize() != cudaSuccess) return fail(hs[0], -2, "cudaDeviceSynchronize");
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
  // the new set-up is built in buffers of its own and swapped into the handle only on success: a failed call leaves the earlier
  // set-up (and a sampler that is using it, NSGW_OPT_LIKELIHOOD = 1) untouched
  int* new_edge = nullptr;
  double* new_buf = nullptr;
  auto drop = [&](int rc) { cudaFree(new_edge); cudaFree(new_buf); return rc; };
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
#define RB_CHECK(expr)                                                                            \
  do {                                                                                            \
    cudaError_t e_ = (expr);                                                                      \
    if (e_ != cudaSuccess)                                                                        \
      return drop(fail(h, e_ == cudaErrorMemoryAllocation ? -4 : -2, std::string(#expr) + ": " + cudaGetErrorString(e_))); \
  } while (0)
  RB_CHECK(cudaMalloc(&new_edge, sizeof(int) * (nb + 1)));
  RB_CHECK(cudaMalloc(&new_buf, sizeof(double) * n_buf));
  double* b = new_buf;
  double2* A0 = reinterpret_cast<double2*>(b); b += (size_t)nd * nb * 2;
  double2* A1 = reinterpret_cast<double2*>(b); b += (size_t)nd * nb * 2;
  double2* ig0 = reinterpret_cast<double2*>(b); b += (size_t)nd * (nb + 1) * 2;
  double* B0 = b; b += (size_t)nd * nb;
  double* B1 = b; b += (size_t)nd * nb;
  double* inv_w = b; b += nb;
  double* cb0 = b; b += CB_SIZE;
  double* th0 = b;
  RB_CHECK(cudaMemcpyAsync(new_edge, edge.data(), sizeof(int) * (nb + 1), cudaMemcpyHostToDevice, s));
  RB_CHECK(cudaMemcpyAsync(th0, theta0_host, sizeof(double) * 11, cudaMemcpyHostToDevice, s));
  const bool tf2 = h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2;
  if (tf2) k_setup<1><<<1, 32, 0, s>>>(h->d_cfg, th0, 1, cb0);
  else k_setup<2><<<1, 32, 0, s>>>(h->d_cfg, th0, 1, cb0);
  g_launches.fetch_add(1);
#define RB_SUMMARY(M, N) k_rb_summary<M, N><<<nb, 128, 0, s>>>(h->d_cfg, h->tb, cb0, new_edge, nb, A0, A1, B0, B1, ig0, inv_w)
  if (tf2) { if (nd == 1) RB_SUMMARY(1, 1); else if (nd == 2) RB_SUMMARY(1, 2); else RB_SUMMARY(1, 3); }
  else { if (nd == 1) RB_SUMMARY(2, 1); else if (nd == 2) RB_SUMMARY(2, 2); else RB_SUMMARY(2, 3); }
#undef RB_SUMMARY
  g_launches.fetch_add(1);
  RB_CHECK(cudaGetLastError());
  double valid = 0.0;
  RB_CHECK(cudaMemcpyAsync(&valid, cb0 + CB_VALID, sizeof(double), cudaMemcpyDeviceToHost, s));
  RB_CHECK(cudaStreamSynchronize(s));
#undef RB_CHECK
  if (valid == 0.0) return drop(fail(h, -1, "fiducial theta0 is unphysical"));
  cudaFree(h->d_rb_edge); cudaFree(h->d_rb_buf);
  h->d_rb_edge = new_edge; h->d_rb_buf = new_buf;
  h->rb_nb = nb;
  h->rb.edge = h->d_rb_edge; h->rb.A0 = A0; h->rb.A1 = A1; h->rb.B0 = B0; h->rb.B1 = B1; h->rb.ig0 = ig0; h->rb.inv_w = inv_w; h->rb.nb = nb;
  if (n_bins_host) *n_bins_host = nb;
  if (h->opt_like == 1 && h->cfg.n_live > 0) {   // a sampler already on relative binning: its live logL must refer to the new summary data
    int rc = loglike_u(h, h->d_live_u, h->cfg.n_live, h->d_live_l, s);
    if (rc) return rc;
    CU_CHECK(h, cudaStreamSynchronize(s));
  }
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
  k_finalize<<<1, 32, 0, s>>>(h->d_state, h->d_live_l, h->d_order, n, h->d_fin, nullptr);
  LAUNCH_CHECK(h);
  CU_CHECK(h, cudaMemcpyAsync(h->h_fin, h->d_fin, sizeof(double) * 2, cudaMemcpyDeviceToHost, s));
  CU_CHECK(h, cudaStreamSynchronize(s));
  const double neff = k / std::log((double)n / (double)(n - k));
  if (logz_host) *logz_host = h->h_fin[0];
  if (h_host) *h_host = h->h_fin[1];
  if (logz_err_host) *logz_err_host = std::sqrt(std::max(h->h_fin[1], 0.0) / neff);
  return 0;
}

int ns_posterior(ns_handle* h, const double* dead_dev, int64_t n_dead, double* theta_dev, double* logp_dev, const double* theta_ref_host,
                 double* summary_host, void* stream) {
  if (!h) return -3;
  if (h->cfg.n_live <= 0) return fail(h, -3, "handle has no live set");
  if (n_dead < 0 || (n_dead > 0 && !dead_dev) || !logp_dev) return fail(h, -1, "bad arguments");
  if (theta_ref_host && !theta_dev) return fail(h, -1, "credible levels need theta_dev");
  cudaStream_t s = (cudaStream_t)stream;
  const int n = h->cfg.n_live, D = h->cfg.ndim;
  const long long N = n_dead + n;
  double* d_out = h->d_fin + 2;
  double* d_ref = h->d_fin + 2 + kPostOut;
  if (theta_ref_host) CU_CHECK(h, cudaMemcpyAsync(d_ref, theta_ref_host, sizeof(double) * D, cudaMemcpyHostToDevice, s));
  k_rank<<<(n + 255) / 256, 256, 0, s>>>(h->d_live_l, n, h->d_order);
  LAUNCH_CHECK(h);
  k_finalize<<<1, 32, 0, s>>>(h->d_state, h->d_live_l, h->d_order, n, h->d_fin, h->d_post_lw);
  LAUNCH_CHECK(h);
  k_post_rows<<<(unsigned)((N + 255) / 256), 256, 0, s>>>(h->d_cfg, dead_dev, n_dead, h->d_live_u, h->d_live_l, h->d_order, h->d_post_lw, n,
                                                         theta_dev, logp_dev);
  LAUNCH_CHECK(h);
  k_post_norm<<<1, kPostThreads, 0, s>>>(logp_dev, N, theta_dev, D, theta_ref_host ? d_ref : nullptr, d_out);
  LAUNCH_CHECK(h);
  if (summary_host) {
    CU_CHECK(h, cudaMemcpyAsync(h->h_fin + 2, d_out, sizeof(double) * (2 + D), cudaMemcpyDeviceToHost, s));
    CU_CHECK(h, cudaStreamSynchronize(s));
    for (int i = 0; i < 2 + D; ++i) summary_host[i] = h->h_fin[2 + i];
  }
  return 0;
}

int ns_posterior_resample(ns_handle* h, const double* logp_dev, const double* theta_dev, int64_t N, int64_t n_out, uint64_t seed,
                          double* cum_dev, int64_t* idx_dev, double* theta_out_dev, void* stream) {
  if (!h) return -3;
  if (N <= 0 || n_out < 0 || !logp_dev || !cum_dev || (!idx_dev && !theta_out_dev) || (theta_out_dev && !theta_dev))
    return fail(h, -1, "bad arguments");
  cudaStream_t s = (cudaStream_t)stream;
  k_post_cumsum<<<1, kPostThreads, 0, s>>>(logp_dev, N, cum_dev);
  LAUNCH_CHECK(h);
  if (n_out == 0) return 0;
  k_post_pick<<<(unsigned)((n_out + 255) / 256), 256, 0, s>>>(cum_dev, N, n_out, (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32),
                                                             h->cfg.ndim, theta_dev, reinterpret_cast<long long*>(idx_dev), theta_out_dev);
  LAUNCH_CHECK(h);
  return 0;
}

int nsgw_set_option(ns_handle* h, int32_t key, int32_t value) {
  if (!h) return -3;
  if (key == NSGW_OPT_BINS_KERNEL && value >= 0 && value <= 2) { h->opt_bins_kernel = value; return 0; }
  if (key == NSGW_OPT_WALK_SPEC && value >= 0 && value <= kWalkDMax) { h->opt_walk_spec = value; return 0; }
  if (key == NSGW_OPT_WALK_STAGE && (value == 0 || value == 1)) { h->opt_walk_stage = value; return 0; }
  if (key == NSGW_OPT_WALK_KERNEL && value >= 0 && value <= 3) { h->opt_walk_kernel = value; return 0; }
  if (key == NSGW_OPT_HOST_ZERO_COPY && (value == 0 || value == 1)) { h->opt_host_zero_copy = value; return 0; }
  if (key == NSGW_OPT_INNER_KERNEL && (value == 0 || value == 1)) {
    if (value == 1 && h->opt_like == 1) return fail(h, -5, "the slice kernel evaluates the exact likelihood only");
    h->opt_inner = value;
    return 0;
  }
  if (key == NSGW_OPT_SLICE_STEPS && value >= 0) { h->opt_slice_steps = value; return 0; }
  if (key == NSGW_OPT_LIKELIHOOD && value == 1 && h->opt_inner == 1) return fail(h, -5, "the slice kernel evaluates the exact likelihood only");
  if (key == NSGW_OPT_LIKELIHOOD && (value == 0 || value == 1)) {
    if (!is_gw(h->cfg.like_kind)) return fail(h, -3, "handle has no GW likelihood");
    if (value == 1 && h->rb_nb <= 0) return fail(h, -3, "ns_relbin_setup has not been called");
    h->opt_like = value;
    if (h->cfg.n_live > 0) {   // the live points' logL must come from the likelihood the sampler will compare against
      CU_CHECK(h, cudaDeviceSynchronize());   // the call has no stream argument: order it after all pending work on any stream
      int rc = loglike_u(h, h->d_live_u, h->cfg.n_live, h->d_live_l, nullptr);
      if (rc) return rc;
      CU_CHECK(h, cudaDeviceSynchronize());
    }
    return 0;
  }
  return fail(h, -1, "unknown option or value");
}

int ns_get_state(ns_handle* h, ns_state* state_host, double* live_u_dev, double* live_logl_dev, void* stream) {
  if (!h) return -3;
  if (h->cfg.n_live <= 0) return fail(h, -3, "handle has no live set");
  if (!state_host) return fail(h, -1, "null argument");
  cudaStream_t s = (cudaStream_t)stream;
  DevState ds;
  CU_CHECK(h, cudaMemcpyAsync(&ds, h->d_state, sizeof(DevState), cudaMemcpyDeviceToHost, s));
  int rc = ns_get_live(h, live_u_dev, live_logl_dev, stream);
  if (rc) return rc;
  CU_CHECK(h, cudaStreamSynchronize(s));
  memset(state_host, 0, sizeof(*state_host));
  state_host->struct_version = NSGW_STRUCT_VERSION;
  state_host->iteration = ds.iter; state_host->n_eval_total = ds.n_eval_total;
  state_host->logx = ds.logx; state_host->logz = ds.logz; state_host->h = ds.h; state_host->walks = ds.walks;
  state_host->seed = h->seed;
  return 0;
}

int ns_set_state(ns_handle* h, const ns_state* state_host, const double* live_u_dev, const double* live_logl_dev, void* stream) {
  if (!h) return -3;
  if (h->cfg.n_live <= 0) return fail(h, -3, "handle has no live set");
  if (!state_host || !live_u_dev || !live_logl_dev) return fail(h, -1, "null argument");
  if (state_host->struct_version != NSGW_STRUCT_VERSION || state_host->iteration < 0 || !(state_host->walks >= 1.0))
    return fail(h, -1, "bad state");
  cudaStream_t s = (cudaStream_t)stream;
  const size_t n = h->cfg.n_live, D = h->cfg.ndim;
  DevState ds;
  CU_CHECK(h, cudaMemcpyAsync(&ds, h->d_state, sizeof(DevState), cudaMemcpyDeviceToHost, s));
  CU_CHECK(h, cudaStreamSynchronize(s));
  ds.iter = state_host->iteration; ds.n_eval_total = state_host->n_eval_total;
  ds.logx = state_host->logx; ds.logz = state_host->logz; ds.h = state_host->h; ds.walks = state_host->walks;
  h->seed = state_host->seed;
  CU_CHECK(h, cudaMemcpyAsync(h->d_state, &ds, sizeof(DevState), cudaMemcpyHostToDevice, s));
  CU_CHECK(h, cudaMemcpyAsync(h->d_live_u, live_u_dev, sizeof(double) * n * D, cudaMemcpyDeviceToDevice, s));
  CU_CHECK(h, cudaMemcpyAsync(h->d_live_l, live_logl_dev, sizeof(double) * n, cudaMemcpyDeviceToDevice, s));
  CU_CHECK(h, cudaStreamSynchronize(s));
  return 0;
}

}  // extern "C"

namespace {
template <class K>
int occ_of(K kern, int threads, size_t smem, long long grid, int n_sm, double* frac, int32_t* ctas) {
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem) != cudaSuccess) return -2;
  const double resident = std::min<double>((double)per_sm, (double)grid / n_sm);
  if (frac) *frac = resident * threads / 2048.0;
  if (ctas) *ctas = per_sm;
  return 0;
}
template <int NDET>
int occ_lp(long long rows, int n_sm, double* frac, int32_t* ctas) {   // the walk's rounds are swept with the small geometry
  auto kern = k_bins_lp<NDET, kLpNT, kLpKR, kLpPP, kLpUNR, kLpOCC>;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kLpDynSmem);
  const long long grid = std::min<long long>((rows + kLpNT * kLpPP - 1) / (kLpNT * kLpPP) * 16, (long long)n_sm * kLpOCC);
  return occ_of(kern, kLpNT, kLpDynSmem, grid, n_sm, frac, ctas);
}
}  // namespace

extern "C" {

int nsgw_sweep_occupancy(ns_handle* h, int64_t rows, double* warps_active_host, int32_t* ctas_per_sm_host) {
  if (!h) return -3;
  if (!is_gw(h->cfg.like_kind) || rows < 1) return fail(h, -1, "bad arguments");
  const int nd = h->cfg.n_det, n_sm = h->n_sm;
  const bool tf2 = h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2;
  if (tf2 && rows >= kLpMinBatch && (h->opt_walk_kernel == 3 || (h->opt_walk_kernel == 0 && rows >= 12000))) {
    if (nd == 1) return occ_lp<1>(rows, n_sm, warps_active_host, ctas_per_sm_host);
    if (nd == 2) return occ_lp<2>(rows, n_sm, warps_active_host, ctas_per_sm_host);
    return occ_lp<3>(rows, n_sm, warps_active_host, ctas_per_sm_host);
  }
  if (!tf2 && (h->opt_walk_kernel == 3 || (h->opt_walk_kernel == 0 && rows >= 12000))) {
    const int kr = h->wl_kr > 0 ? h->wl_kr : std::max(kPdKT, (h->cfg.n_freq / 32 + kPdKT - 1) / kPdKT * kPdKT);
    const long long grid = std::min<long long>((rows + kPdNT * kPdPP - 1) / (kPdNT * kPdPP) * ((h->cfg.n_freq + kr - 1) / kr), (long long)n_sm * kPdOCC);
    const size_t dyn = pd_mix_bytes<kPdPP>();
    if (nd == 1) { cudaFuncSetAttribute(k_pd_lp<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn); return occ_of(k_pd_lp<1>, kPdNT, dyn, grid, n_sm, warps_active_host, ctas_per_sm_host); }
    if (nd == 2) { cudaFuncSetAttribute(k_pd_lp<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn); return occ_of(k_pd_lp<2>, kPdNT, dyn, grid, n_sm, warps_active_host, ctas_per_sm_host); }
    cudaFuncSetAttribute(k_pd_lp<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn);
    return occ_of(k_pd_lp<3>, kPdNT, dyn, grid, n_sm, warps_active_host, ctas_per_sm_host);
  }
  const bool p2 = rows >= 4096;
  const long long grid = p2 ? (rows + 1) / 2 : rows;
#define OCC_BINS(M, N)                                                                                                          \
  return p2 ? occ_of(k_bins<M, N, 2>, kBinsThreads, 0, grid, n_sm, warps_active_host, ctas_per_sm_host)                          \
            : occ_of(k_bins<M, N, 1>, kBinsThreads, 0, grid, n_sm, warps_active_host, ctas_per_sm_host)
  if (tf2) { if (nd == 1) OCC_BINS(1, 1); if (nd == 2) OCC_BINS(1, 2); OCC_BINS(1, 3); }
  if (nd == 1) OCC_BINS(2, 1);
  if (nd == 2) OCC_BINS(2, 2);
  OCC_BINS(2, 3);
#undef OCC_BINS
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

// ======================================================================================================
// gw_loglike_batch_noalloc: the batched likelihood for callers that cannot allocate (include/nsgw.h)
// ======================================================================================================
// The coefficient blocks, the per-range partial sums and the tickets of k_bins_lp / k_pd_lp live in ONE file-scope device array of
// fixed size instead of the handle's grow-on-demand buffers.  Every device that loads the library holds the array until exit; every
// call on a device shares it.  In host code `g_na_scratch` is a host-side stand-in, not a device address: the address the kernels
// get comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr long long kNaMaxRows = NSGW_NOALLOC_MAX_ROWS;
constexpr int kNaMaxBins = NSGW_NOALLOC_MAX_BINS;
constexpr int kNaKr = 256;                                    // bins per range in this entry point (both kernels)
constexpr int kNaMaxRanges = (kNaMaxBins + kNaKr - 1) / kNaKr;
constexpr int kNaMaxAcc = 7;                                  // AccLayout<2, 3>::N, the widest row of partial sums
constexpr int kNaTickets = 64;                                // ints; >= row groups of kNaMaxRows rows
constexpr size_t kNaCbDoubles = (size_t)kNaMaxRows * CB_SIZE;
constexpr size_t kNaPartialDoubles = (size_t)kNaMaxRows * kNaMaxRanges * kNaMaxAcc;
constexpr size_t kNaDoubles = kNaCbDoubles + kNaPartialDoubles + kNaTickets / 2;
static_assert(AccLayout<2, 3>::N == kNaMaxAcc && AccLayout<1, 3>::N <= kNaMaxAcc, "partial-sum width");
static_assert((kNaMaxRows + kPdNT * kPdPP - 1) / (kPdNT * kPdPP) <= kNaTickets, "tickets");
static_assert(kNaKr % kPdKT == 0 && kNaKr <= kLpKR && kNaKr % kLpUNR == 0, "range length fits both kernels");
static_assert(kNaDoubles * sizeof(double) <= (size_t)NSGW_NOALLOC_SCRATCH_BYTES, "scratch size stated in nsgw.h");

static __device__ __align__(256) double g_na_scratch[kNaDoubles];   // 16.1 MiB: [rows][CB_SIZE] | [ranges][N][rows] | tickets

namespace {

constexpr int kNaMaxDevices = 64;
std::atomic<double*> g_na_ptr[kNaMaxDevices];   // device address of g_na_scratch per device ordinal (null: not asked yet)

// Device address of the current device's copy of g_na_scratch.
int na_scratch(ns_handle* h, double** out) {
  int dev = -1;
  CU_CHECK(h, cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNaMaxDevices) return fail(h, -5, "gw_loglike_batch_noalloc: device ordinal beyond 63");
  double* p = g_na_ptr[dev].load(std::memory_order_acquire);
  if (!p) {
    CU_CHECK(h, cudaGetSymbolAddress((void**)&p, g_na_scratch));
    if (!p) return fail(h, -2, "gw_loglike_batch_noalloc: cudaGetSymbolAddress returned a null address");
    g_na_ptr[dev].store(p, std::memory_order_release);   // two first callers get the same address: the race is benign
  }
  *out = p;
  return 0;
}

template <int NDET>
int na_launch(ns_handle* h, const double* theta_dev, long long B, double* logl, cudaStream_t s, double* scratch) {
  const bool tf2 = h->cfg.like_kind == NSGW_LIKE_GW_TAYLORF2;
  double* cbs = scratch;
  double* partial = scratch + kNaCbDoubles;
  int* ticket = reinterpret_cast<int*>(scratch + kNaCbDoubles + kNaPartialDoubles);
  const int nranges = (h->cfg.n_freq + kNaKr - 1) / kNaKr;
  const unsigned gs = (unsigned)((B + 127) / 128);
  if (tf2) {
    constexpr int NT = kLpNT, PP = kLpPP;
    const long long ngroups = (B + NT * PP - 1) / (NT * PP);
    const long long ntasks = ngroups * nranges;
    const long long grid = std::min<long long>(ntasks, (long long)h->n_sm * kLpOCC);
    k_setup<1><<<gs, 128, 0, s>>>(h->d_cfg, theta_dev, B, cbs);
    LAUNCH_CHECK(h);
    // every (range, sum, row < B) entry of `partial` the finishing pass reads is written by this launch: nothing to clear
    CU_CHECK(h, cudaFuncSetAttribute(k_bins_lp<NDET, NT, kLpKR, PP, kLpUNR, kLpOCC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kLpDynSmem));
    k_bins_lp<NDET, NT, kLpKR, PP, kLpUNR, kLpOCC><<<(unsigned)grid, NT, kLpDynSmem, s>>>(h->d_cfg, h->tb, cbs, B, nullptr, kNaKr, nranges, ntasks, partial);
    LAUNCH_CHECK(h);
    k_finish<1, NDET><<<gs, 128, 0, s>>>(h->d_cfg, cbs, partial, nranges, B, logl, nullptr);
    LAUNCH_CHECK(h);
    return 0;
  }
  const long long ngroups = (B + kPdNT * kPdPP - 1) / (kPdNT * kPdPP);
  const long long ntasks = ngroups * nranges;
  const long long grid = std::min<long long>(ntasks, (long long)h->n_sm * kPdOCC);
  // the tickets must start at zero; the array keeps whatever the last call (possibly an aborted one) left
  CU_CHECK(h, cudaMemsetAsync(ticket, 0, sizeof(int) * kNaTickets, s));
  k_setup<2><<<gs, 128, 0, s>>>(h->d_cfg, theta_dev, B, cbs);
  LAUNCH_CHECK(h);
  PdArgs a;
  a.cbs = cbs; a.n_rows = B; a.n_rows_dev = nullptr; a.stride = B; a.kr = kNaKr; a.nranges = nranges; a.partial = partial;
  a.ticket = ticket; a.logl = logl; a.parts = nullptr;
  CU_CHECK(h, cudaFuncSetAttribute(k_pd_lp<NDET>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pd_mix_bytes<kPdPP>()));
  k_pd_lp<NDET><<<(unsigned)grid, kPdNT, pd_mix_bytes<kPdPP>(), s>>>(h->d_cfg, h->tb, a);
  LAUNCH_CHECK(h);
  return 0;
}

}  // namespace

extern "C" {

int gw_loglike_batch_noalloc(ns_handle* h, const double* theta_dev, int64_t B, double* logl_dev, void* stream) {
  if (!h) return -3;
  if (!is_gw(h->cfg.like_kind)) return fail(h, -3, "handle has no GW likelihood");
  if (B < 0 || (B > 0 && (!theta_dev || !logl_dev))) return fail(h, -1, "bad arguments");
  if (B > kNaMaxRows)
    return fail(h, -5, "gw_loglike_batch_noalloc: B = " + std::to_string((long long)B) + " rows exceed NSGW_NOALLOC_MAX_ROWS = " +
                           std::to_string(kNaMaxRows) + " (split the batch, or use gw_loglike_batch)");
  if (h->cfg.n_freq > kNaMaxBins)
    return fail(h, -5, "gw_loglike_batch_noalloc: n_freq = " + std::to_string(h->cfg.n_freq) + " bins exceed NSGW_NOALLOC_MAX_BINS = " +
                           std::to_string(kNaMaxBins) + " (use gw_loglike_batch)");
  if (B == 0) return 0;
  double* scratch = nullptr;
  int rc = na_scratch(h, &scratch);
  if (rc) return rc;
  cudaStream_t s = (cudaStream_t)stream;
  switch (h->cfg.n_det) {
    case 1: return na_launch<1>(h, theta_dev, B, logl_dev, s, scratch);
    case 2: return na_launch<2>(h, theta_dev, B, logl_dev, s, scratch);
    case 3: return na_launch<3>(h, theta_dev, B, logl_dev, s, scratch);
    default: return fail(h, -5, "n_det must be 1..3 for the GW kernels");
  }
}

}  // extern "C"
