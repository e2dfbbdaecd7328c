#!/usr/bin/env python
"""bench.py -- throughput of the batched GW log-likelihood hot path on B200.

Metric (BASELINE.json): GW log-likelihood evaluations per second.  Workload at N=1: BASELINE.json configs[1] --
TaylorF2 3.5PN aligned-spin, H1+L1, 4 s at 2048 Hz (4017 complex128 bins per detector), B = 65536 parameter rows drawn
from the config-3 prior box; one "step" = one gw_loglike_batch call over the whole batch (set-up kernel + bin-sweep kernel).
Extra objects report the lock-step walk (ns_walk_batch) and a full nested-sampling run on the same machine.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--batch B] [--quick]

One JSON line on stdout (rank 0).  --impl reference times the CPU oracle (oracle/) on the host cores instead.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz = 37.2
METRIC = "gw_loglike_evals_per_sec"
UNIT = "evals/s"


def alg_flops_per_bin(n_det, model="taylorf2"):
    """Algorithmic fp64 flops per (particle, bin) of the minimal formulation the kernel implements,
    FMA = 2: 9-FMA phase (18); table-driven sincos with k_bins_lp's 2048-entry table: exact reduction (F2I, I2F on the
    conversion pipe + 1 subtraction), r^2 (1), sin 1 FMA + 1 mul (3), cos 1 FMA (2), complex product with the table entry (6) = 13
    (k_pd_lp's 512-entry table needs one more cos term: 15; the 256-entry table of the other kernels one more each: 19);
    detector 0: 4 FMA (8); every further detector: conj(wd) E (6) and one complex Horner step in the detector's per-bin
    phasor (4 FMA = 8) = 14."""
    if model == "phenomd":
        # merger-ringdown bin (about 80 % of the bins) as k_bins evaluates it (bins strided over threads): phase 47,
        # amplitude 32 + 3, table-driven sincos 21, detector 0: 10, every further detector 18
        return 47 + 35 + 21 + 10 + 18 * (n_det - 1)
    if model == "phenomd_lane":
        # the same bin as k_pd_lp evaluates it (lane per row, consecutive bins: the cheaper formulation, so this is the model its
        # fractions are quoted on): atan carried by the subtraction formula with a constant step 18, phase 8, Lorentzian with the
        # exponential as a geometric sequence 9, table-driven sincos 15 + scaling by the amplitude 2, detector 0: 8 + <h,h> 3, every
        # further detector: Horner step 14 + <h,h> 2
        return 18 + 8 + 9 + 17 + 11 + 16 * (n_det - 1)
    assert model == "taylorf2"
    return 18 + 13 + 8 + 14 * (n_det - 1)


def _profile_key(name):
    m = __import__("re").match(r"r(\d+)([a-z]*)_", name)
    return (int(m.group(1)), len(m.group(2)), m.group(2)) if m else (-1, 0, "")


def traffic_from_profile(kernel="k_bins_lp"):
    """DRAM bytes per launch of the dominant kernel (dram__bytes_read.sum + dram__bytes_write.sum) read from the newest committed
    `ncu --set full` summary of it under profiles/ (text; the file's first line is the command that made it).  (bytes, file)."""
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_{kernel}_ncu_full.txt")), key=lambda q: _profile_key(os.path.basename(q)))
    if not files:
        return None, None
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    tot, seen = 0.0, 0
    for line in open(files[-1]):
        f = line.split()
        if len(f) == 3 and f[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum") and f[1] in unit:
            tot += float(f[2]) * unit[f[1]]
            seen += 1
    return (tot, os.path.relpath(files[-1], ROOT)) if seen == 2 else (None, None)


def spawn_command(n_gpus, argv, port=None):
    """`bench.py --gpus N` started without a launcher re-executes itself under torch.distributed.run, one rank per GPU."""
    port = port or (29500 + os.getpid() % 2000)
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}", "--master-addr", "127.0.0.1",
            "--master-port", str(port), os.path.join(ROOT, "bench.py")] + list(argv)


def resolve_world(args, environ):
    """What --gpus means, for both arms: the number of ranks of the job.  Returns "run" (this process is a rank of a job of that
    size, or N = 1), "spawn" (N > 1 and no launcher: start N ranks) or raises SystemExit when the flag contradicts the launcher."""
    ws = environ.get("WORLD_SIZE")
    if ws is None:
        return "run" if args.gpus <= 1 else "spawn"
    if int(ws) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={ws} ranks")
    return "run"


class ClockSampler:
    """Samples SM clock and throttle reasons while the timed region runs (NVML every 20 ms; nvidia-smi as a fallback)."""

    def __init__(self, index=0):
        self.samples, self.reasons, self.max_mhz, self.how = [], set(), None, None
        self._stop = threading.Event()
        self.index = index
        self._t = threading.Thread(target=self._run, daemon=True)

    def _run_nvml(self):
        import pynvml as N
        N.nvmlInit()
        h = N.nvmlDeviceGetHandleByIndex(self.index)
        self.max_mhz = float(N.nvmlDeviceGetMaxClockInfo(h, N.NVML_CLOCK_SM))
        bits = {"hw_slowdown": N.nvmlClocksThrottleReasonHwSlowdown, "hw_thermal_slowdown": N.nvmlClocksThrottleReasonHwThermalSlowdown,
                "sw_thermal_slowdown": N.nvmlClocksThrottleReasonSwThermalSlowdown, "sw_power_cap": N.nvmlClocksThrottleReasonSwPowerCap}
        self.how = "nvml"
        while not self._stop.is_set():
            self.samples.append(float(N.nvmlDeviceGetClockInfo(h, N.NVML_CLOCK_SM)))
            r = N.nvmlDeviceGetCurrentClocksThrottleReasons(h)
            for n, b in bits.items():
                if r & b:
                    self.reasons.add(n)
            self._stop.wait(0.02)

    def _run_smi(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        self.how = "nvidia-smi"
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip().splitlines()[0]
                f = [x.strip() for x in out.split(",")]
                self.samples.append(float(f[0]))
                self.max_mhz = float(f[1])
                for n, v in zip(names, f[2:]):
                    if v.lower().startswith("active"):
                        self.reasons.add(n)
            except Exception:
                pass
            self._stop.wait(0.1)

    def _run(self):
        try:
            self._run_nvml()
        except Exception:
            self._run_smi()

    def __enter__(self):
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples), "how": self.how}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    return json.load(open(p)) if os.path.exists(p) else {}


# --------------------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle as it stands
# --------------------------------------------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    from paper_2509_04336_b200 import workloads as W
    spec = W.config2(lambda s, th: O.OracleProblem(s).waveform(th))
    P = O.OracleProblem(spec)
    cores = os.cpu_count()
    B = args.ref_batch
    theta = P.prior_transform(W.uniform_rows(0, B, 11, seed=2))
    for _ in range(args.warmup):
        P.gw_loglike(theta[: max(64, B // 8)])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        P.gw_loglike(theta)
    dt = time.perf_counter() - t0
    val = args.steps * B / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config2 gw_loglike_batch TaylorF2 H1+L1 4017 bins, bounded sample of {B} rows per step (CPU oracle)"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{B} rows per step x {args.steps} steps, OpenMP over rows"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2509_04336_b200 import dist as D, nsgw, workloads as W

    rank, world, local = D.env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local)
    D.init("nccl", torch.device("cuda", local))

    def barrier():
        D.barrier("cuda")

    # ---- workload: config 2.  The injected signal comes from the CUDA library itself (gw_waveform).
    def wf_cuda(spec, th):
        tmp = dict(spec)
        tmp["strain"] = np.zeros((spec["n_det"], spec["n_freq"], 2))
        hh = nsgw.Handle(tmp)
        out = hh.gw_waveform(torch.as_tensor(th).cuda()).cpu().numpy()
        hh.close()
        return out

    spec = W.config2(wf_cuda)
    h = nsgw.Handle(spec)
    B = args.batch
    n_det, n_freq = spec["n_det"], spec["n_freq"]
    # weak scaling, no data-path collective: rank r owns rows [r B, (r+1) B) of one index-keyed stream of unit-cube rows
    u = torch.as_tensor(W.uniform_rows(rank * B, (rank + 1) * B, 11, seed=2)).cuda()
    theta = h.prior_transform_batch(u)
    logl = torch.empty(B, dtype=torch.float64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()

    def timed(nrows, steps, clocks=False):
        """`steps` timed gw_loglike_batch calls over the first nrows rows: L2 flushed before every call (outside its event pair),
        CUDA events on the launching stream, max over ranks.  Returns (ms total, dominant-kernel ms total, its launches, library
        launches, clock summary)."""
        th_n, out_n = theta[:nrows], logl[:nrows]
        for _ in range(max(args.warmup, 3)):
            h.gw_loglike_batch(th_n, out=out_n)
        barrier()
        n0 = nsgw.launch_count()
        h.profile_enable(True)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        with ClockSampler(local) as clk:
            barrier()
            for a, b in ev:
                flush.zero_()                       # L2 flush between timed iterations (outside the event pair)
                a.record(stream)
                h.gw_loglike_batch(th_n, out=out_n)
                b.record(stream)
            barrier()
        h.profile_enable(False)
        nl = nsgw.launch_count() - n0
        t = D.max_over_ranks(sum(a.elapsed_time(b) for a, b in ev), "cuda")
        k_ms, k_n = h.profile_read()
        return t, k_ms, k_n, nl, clk.summary()

    # batch sizes BASELINE.json lists for config 2, same method each; the largest is the headline step
    sweep_B = sorted({b for b in (1024, 16384, 65536) if b < B} | {B})
    sweep_raw = {}
    for b in sweep_B:
        sweep_raw[b] = timed(b, args.steps if b == B else max(20, args.steps // 2))
    ms, kern_ms, kern_n, launches, clocks = sweep_raw[B]
    value = world * B * args.steps / (ms * 1e-3)

    # ---- end to end through the host-buffer C-ABI call: pinned theta -> H2D -> set-up + bin sweep -> D2H logL, all timed
    th_host = theta.cpu().pin_memory()
    out_host = torch.empty(B, dtype=torch.float64).pin_memory()

    def e2e_step():
        h.gw_loglike_batch_host(th_host, out_host)       # synchronises

    for _ in range(3):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    barrier()
    e2e_s = D.max_over_ranks(time.perf_counter() - t0, "cuda")
    e2e_val = world * B * args.steps / e2e_s
    e2e_diff = float((out_host - logl.cpu()).abs().max())
    assert e2e_diff == 0.0, e2e_diff        # same kernels, same launch geometry: the identical numbers

    line = None
    fp64_burst = nsgw.measure_fp64_peak(1 << 17) if rank == 0 else None
    if rank == 0:
        peaks = measured_peaks()
        flops_launch = float(B) * n_freq * alg_flops_per_bin(n_det)
        ach = flops_launch / (kern_ms / kern_n * 1e-3) / 1e12
        # DRAM bytes per launch of the dominant kernel: dram__bytes_read.sum + dram__bytes_write.sum of the committed
        # `ncu --set full` capture of this same command (profiles/r01ad_k_bins_lp_ncu_full.txt); only valid for the default batch
        traffic, traffic_file = traffic_from_profile("k_bins_lp") if (B == 65536 and n_freq == 4017) else (None, None)
        roof = {"bound": "alu", "achieved": ach, "peak": fp64_burst, "unit": "TFLOP/s", "frac": ach / fp64_burst,
                "traffic": traffic, "traffic_unit": "bytes per launch (ncu dram read+write) from %s; algorithmic 96 B x B = %d" % (traffic_file, 96 * B), "kernel": "k_bins_lp<2det> (lane per particle, one CTA of 512 threads x 2 particles per SM from 6144 rows, three of 128 below; 256-bin tiles)", "kernel_ms": kern_ms / kern_n,
                "flops_per_particle_bin": alg_flops_per_bin(n_det),
                "model_note": "the flop model follows the kernel's formulation down: 53 per particle-bin (2 detectors) since k_bins_lp takes sin/cos "
                              "from a 2048-entry table (three FMAs fewer), 59 before; on the 59-flop yardstick of BENCH_r01 this run is at %.3f"
                              % (ach * (alg_flops_per_bin(n_det) + 6.0) / alg_flops_per_bin(n_det) / fp64_burst),
                "peak_source": "measured here: nsgw_measure_fp64_peak (8 independent DFMA chains/thread, 8 CTAs x 256 thr per SM), burst",
                "frac_of_nominal_37.2": ach / NOMINAL_FP64_TFLOPS,
                "hbm_peak_gbs_measured": peaks.get("hbm_gbs")}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"config2 gw_loglike_batch TaylorF2 H1+L1 {n_freq} bins x {n_det} det, B={B} rows per GPU",
                           "l2": "flushed between timed iterations (256 MiB write)", "parallelism": f"rows sharded x{world}, no collective"},
                "clocks": clocks,
                "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": B * 11 * 8, "d2h_bytes_per_step": B * 8,
                        "max_abs_dlogl_vs_device_call": e2e_diff,
                        "how": "gw_loglike_batch_host on pinned host buffers: the set-up kernel fetches theta over the host link, the finishing code "
                               "stores logL into the host buffer (the same bytes cross the link as with copies; nsgw_set_option(NSGW_OPT_HOST_ZERO_COPY, 0) "
                               "restores cudaMemcpyAsync H2D / D2H around the kernels)"},
                "gpu_launches": int(launches), "roofline": roof}
        bs = []
        for b in sweep_B:
            t, k_ms, k_n, _, ck = sweep_raw[b]
            nst = args.steps if b == B else max(20, args.steps // 2)
            fl = float(b) * n_freq * alg_flops_per_bin(n_det)
            bs.append({"B": b, "ms_per_step": t / nst, "evals_per_s": world * b * nst / (t * 1e-3), "sweep_kernel_ms": k_ms / max(k_n, 1),
                       "frac_fp64_peak_step": fl / (t / nst * 1e-3) / 1e12 / fp64_burst,
                       "frac_fp64_peak_sweep_kernel": fl / (k_ms / max(k_n, 1) * 1e-3) / 1e12 / fp64_burst, "sm_mhz": ck["sm_mhz"]})
        line["batch_sweep"] = {"what": "config 2 (BASELINE.json: B in {1024, 16384, 65536}); same flush + CUDA-event method per size; "
                                       "fractions of the FP64 peak measured in this run, %d flops per particle-bin" % alg_flops_per_bin(n_det),
                               "points": bs}

    # ---- extras (rank 0, N=1 only): walk throughput and one full nested-sampling run
    if rank == 0 and world == 1 and not args.quick:
        extras = {}
        # lock-step walk on the same data: B_w walkers, W steps
        Bw, Wl = 16384, 20
        P_u = torch.as_tensor(W.uniforms(2 * Bw, 11, 9)).cuda()
        ll = h.loglike_u_batch(P_u)
        order = torch.argsort(ll)
        donors = P_u[order[Bw:]].contiguous()
        lstar = float(ll[order[Bw - 1]])
        uw = donors[torch.arange(Bw, device="cuda") % donors.shape[0]].clone()
        lw = ll[order[Bw:]][torch.arange(Bw, device="cuda") % donors.shape[0]].clone()
        for rep in range(2):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            cnt = h.walk_batch(donors, uw, lw, lstar, Wl, 1234, 7 + rep)
            b.record(stream)
            torch.cuda.synchronize()
        ne = int(cnt["n_eval"].sum())
        wms = a.elapsed_time(b)
        extras["walk"] = {"workload": f"ns_walk_batch config2 data, B={Bw}, W={Wl}", "evals_per_s": ne / (wms * 1e-3), "ms": wms,
                          "evals": ne, "accept_mean": float(cnt["n_accept"].double().mean()),
                          "accept_min": int(cnt["n_accept"].min()), "accept_max": int(cnt["n_accept"].max()),
                          "oob_frac": float(cnt["n_oob"].sum()) / (Bw * Wl)}
        # full run: config 3 (PhenomD-form, H1+L1, n_live 1000, k 500, naccept 60, dlogz < 0.1)
        spec3, smp3 = W.config3(wf_cuda_for(nsgw, torch))
        # PhenomD-form batched likelihood on the config-3 data (the model of configs 3-5), B = 65536 prior rows: both sweep kernels
        hp = nsgw.Handle(spec3)
        th3 = hp.prior_transform_batch(u)
        o3 = torch.empty(B, dtype=torch.float64, device="cuda")
        pd = {}
        for name, kern in (("k_bins_cta_per_row_pair", 1), ("k_pd_lp_lane_per_row", 2)):
            hp.set_option(0, kern)
            for _ in range(3):
                hp.gw_loglike_batch(th3, out=o3)
            evp = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(20)]
            for a, b in evp:
                flush.zero_()
                a.record(stream)
                hp.gw_loglike_batch(th3, out=o3)
                b.record(stream)
            torch.cuda.synchronize()
            pms = sum(a.elapsed_time(b) for a, b in evp) / len(evp)
            mdl = "phenomd" if kern == 1 else "phenomd_lane"
            pd[name] = {"ms_per_step": pms, "evals_per_s": B / (pms * 1e-3), "flops_per_particle_bin_model": alg_flops_per_bin(2, mdl),
                        "frac_fp64_peak": B * n_freq * alg_flops_per_bin(2, mdl) / (pms * 1e-3) / 1e12 / fp64_burst}
        extras["phenomd_batch_config3_B65536"] = pd
        hp.close()
        h3 = nsgw.Handle(spec3, smp3, seed=1)
        t0 = time.perf_counter()
        nit, st = h3.run(smp3["term_kind"], smp3["term_tol"], 4000)
        logz, err, H = h3.finalize_evidence()
        wall = time.perf_counter() - t0
        extras["ns_run_config3"] = {"wall_s": wall, "iterations": nit, "n_eval_total": st["n_eval_total"], "logz": logz, "logz_err": err,
                                    "H": H, "walk_len_last": st["walk_len"], "accept_mean_last": st["accept_mean"],
                                    "evals_per_s": st["n_eval_total"] / wall}
        h3.close()
        # config 4: longer segment (8 s at 4096 Hz, 16225 bins), n_live 1400, k 700, live-evidence-fraction rule
        spec4, smp4 = W.config4(wf_cuda_for(nsgw, torch))
        h4 = nsgw.Handle(spec4, smp4, seed=1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        nit, st = h4.run(smp4["term_kind"], smp4["term_tol"], 4000)
        logz, err, H = h4.finalize_evidence()
        wall = time.perf_counter() - t0
        extras["ns_run_config4"] = {"wall_s": wall, "iterations": nit, "n_eval_total": st["n_eval_total"], "logz": logz,
                                    "logz_err": err, "H": H, "walk_len_last": st["walk_len"],
                                    "accept_mean_last": st["accept_mean"], "evals_per_s": st["n_eval_total"] / wall}
        h4.close()
        # first iteration of both runs alone (same seed, same live set: the step the oracle is timed on below)
        first = {}
        for name, sp_, sm_ in (("config3", spec3, smp3), ("config4", spec4, smp4)):
            hf = nsgw.Handle(sp_, sm_, seed=1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            stf = hf.step()
            first[name] = {"ms": 1e3 * (time.perf_counter() - t0), "walk_len": stf["walk_len"], "n_eval": stf["n_eval"], "n_oob": stf["n_oob"]}
            hf.close()
        extras["ns_step_first_iteration"] = first
        # config 5: divergence and saturation sweep (H1+L1+V1, 16 s at 4096 Hz, 32449 bins): B walkers against a live set of 2B
        # points scattered about the injection, the lower half deleted, W in {20, 60, 200}, no adaptation.  The whole grid of
        # BASELINE.json (10 batch sizes x 3 walk lengths); a point is skipped only if the time budget of the sweep runs out.
        spec5 = W.config5(wf_cuda_for(nsgw, torch))
        h5 = nsgw.Handle(spec5)
        fl5 = alg_flops_per_bin(3, "phenomd_lane") * spec5["n_freq"]
        sweep, skipped = [], []
        t_sweep = time.perf_counter()
        for Bw in (256, 512, 1024, 2048, 4096, 8192, 16384, 32768, 65536, 131072):
            u5 = torch.as_tensor(W.config5_live(spec5, 2 * Bw)).cuda()
            l5 = h5.loglike_u_batch(u5)
            order = torch.argsort(l5)
            donors = u5[order[Bw:]].contiguous()
            lstar = float(l5[order[Bw - 1]])
            for Wl in (20, 60, 200):
                if time.perf_counter() - t_sweep > args.sweep_budget_s:
                    skipped.append([Bw, Wl])
                    continue
                # rows a round is expected to hold (the library's own estimate: walkers x chunk length from W and naccept = 60)
                occ, ctas = h5.sweep_occupancy(int(Bw * max(1.0, min(64.0, 65536.0 / Bw, 0.3 * Wl / 60.0))))
                if Wl == 20:        # the first walk of a batch size allocates the round buffers: not part of the timed call
                    h5.walk_batch(donors, donors.clone(), l5[order[Bw:]].clone(), lstar, 2, 4321, 8)
                uw, lw = donors.clone(), l5[order[Bw:]].clone()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                cnt = h5.walk_batch(donors, uw, lw, lstar, Wl, 4321, 9)
                b.record(stream)
                torch.cuda.synchronize()
                ne, na = int(cnt["n_eval"].sum()), cnt["n_accept"].double()
                wms = a.elapsed_time(b)
                sweep.append({"B": Bw, "W": Wl, "ms": wms, "evals": ne, "evals_per_s": ne / (wms * 1e-3),
                              "accept_mean": float(na.mean()), "accept_std": float(na.std()), "accept_min": int(na.min()),
                              "accept_max": int(na.max()), "oob_frac": float(cnt["n_oob"].sum()) / (Bw * Wl),
                              "warps_active_sweep_kernel": occ, "frac_fp64_peak": ne * fl5 / (wms * 1e-3) / 1e12 / fp64_burst})
        extras["config5_sweep"] = {"what": "ns_walk_batch, PhenomD-form, 3 detectors x 32449 bins; warps_active = resident warps / 64 of "
                                           "the row-sweep kernel (occupancy API x grid fill at the rows of a full round); frac_fp64_peak = "
                                           "%d model flops per particle-bin (k_pd_lp's formulation; k_bins' costs %d) x bins x evaluations / time / measured peak" % (alg_flops_per_bin(3, "phenomd_lane"), alg_flops_per_bin(3, "phenomd")),
                                   "points": sweep, "skipped_for_time": skipped}
        h5.close()
        if args.full_extras:
            # config 3 on the relative-binning likelihood (fiducial = the injection, eps = 0.5), and the batched
            # relative-binning evaluation on the config-2 data
            h3r = nsgw.Handle(spec3, smp3, seed=1)
            nbins = h3r.relbin_setup(W.INJ_C3)
            h3r.set_option(2, 1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            nit, st = h3r.run(smp3["term_kind"], smp3["term_tol"], 4000)
            logz, err, H = h3r.finalize_evidence()
            wall = time.perf_counter() - t0
            extras["ns_run_config3_relbin"] = {"wall_s": wall, "iterations": nit, "n_eval_total": st["n_eval_total"], "logz": logz,
                                               "logz_err": err, "H": H, "n_bins": nbins, "walk_len_last": st["walk_len"],
                                               "accept_mean_last": st["accept_mean"], "evals_per_s": st["n_eval_total"] / wall}
            # posterior post-processing of such a run (ns_posterior + ns_posterior_resample; R:L26-27), timed with CUDA events
            k3, D3 = smp3["n_delete"], 11
            h3p = nsgw.Handle(spec3, smp3, seed=1)
            h3p.relbin_setup(W.INJ_C3)
            h3p.set_option(2, 1)
            dead3 = torch.empty((200 * k3, D3 + 3), dtype=torch.float64, device="cuda")
            nit, st = h3p.run(smp3["term_kind"], smp3["term_tol"], 200, dead=dead3)
            rows3 = dead3[: nit * k3].contiguous()
            for _ in range(3):
                post = h3p.posterior(rows3, theta_ref=W.INJ_C3)
                h3p.posterior_resample(post["logp"], 10000, 1, theta=post["theta"])
            a, b, c = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            a.record(stream)
            for _ in range(10):
                post = h3p.posterior(rows3, theta_ref=W.INJ_C3)
            b.record(stream)
            for _ in range(10):
                h3p.posterior_resample(post["logp"], 10000, 1, theta=post["theta"])
            c.record(stream)
            torch.cuda.synchronize()
            extras["posterior_config3_relbin"] = {"rows": int(rows3.shape[0]) + smp3["n_live"], "ns_posterior_ms": a.elapsed_time(b) / 10,
                                                  "resample_10000_ms": b.elapsed_time(c) / 10, "ess": post["ess"], "logz_rows": post["logz"],
                                                  "cl_injection": [round(float(x), 4) for x in post["cl"]]}
            h3p.close()
            h3r.close()
            nb2 = h.relbin_setup(W.INJ_C3)
            rb_out = torch.empty(B, dtype=torch.float64, device="cuda")
            for _ in range(3):
                h.gw_loglike_relbin_batch(theta, out=rb_out)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for _ in range(20):
                h.gw_loglike_relbin_batch(theta, out=rb_out)
            b.record(stream)
            torch.cuda.synchronize()
            rms = a.elapsed_time(b) / 20
            extras["relbin_batch_config2"] = {"n_bins": nb2, "ms": rms, "evals_per_s": B / (rms * 1e-3)}
            # four config-3 runs with different seeds at once (ns_run_many): the runs' walk kernels share the SMs
            hs = [nsgw.Handle(spec3, smp3, seed=sd) for sd in (1, 2, 3, 4)]
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            its, sts = nsgw.run_many(hs, smp3["term_kind"], smp3["term_tol"], 4000)
            fins = [hh.finalize_evidence() for hh in hs]
            wall = time.perf_counter() - t0
            ev = sum(st_["n_eval_total"] for st_ in sts)
            extras["ns_run_many_4x_config3"] = {"wall_s": wall, "iterations": its, "n_eval_total": ev, "evals_per_s": ev / wall,
                                                "logz": [f_[0] for f_ in fins], "logz_err": [f_[1] for f_ in fins],
                                                "wall_s_per_run": wall / len(hs)}
            for hh in hs:
                hh.close()
            # slice-sampling inner kernel against the acceptance walk from the same mid-run state of config 3:
            # survivors as donors / covariance source, k = 500 replacements
            hs3 = nsgw.Handle(spec3, smp3, seed=1)
            for _ in range(40):
                hs3.step(want_stats=False)
            u_l, l_l = hs3.get_live()
            order = torch.argsort(l_l)
            kk = smp3["n_delete"]
            donors = u_l[order[kk:]].contiguous()
            ld = l_l[order[kk:]].contiguous()
            lstar = float(l_l[order[kk - 1]])
            lc = torch.linalg.cholesky(torch.cov(donors.T) + 1e-12 * torch.eye(11, dtype=torch.float64, device="cuda")).contiguous()
            idx = torch.arange(kk, device="cuda") % donors.shape[0]
            res = {}
            for S_ in (11, 55):
                uw, lw = donors[idx].clone(), ld[idx].clone()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                cnt = hs3.slice_batch(lc, uw, lw, lstar, S_, 777, (6 << 24) | 1, trace=True)
                b.record(stream)
                torch.cuda.synchronize()
                ne = cnt["n_eval"].double()
                te = cnt["trace_evals"].double()
                res[f"S={S_}"] = {"ms": a.elapsed_time(b), "evals": int(ne.sum()), "evals_per_s": float(ne.sum()) / (a.elapsed_time(b) * 1e-3),
                                  "evals_per_step_mean": float(te.mean()), "evals_per_step_std": float(te.std()),
                                  "evals_per_step_max": int(te.max()), "evals_per_walker_min": int(ne.min()),
                                  "evals_per_walker_max": int(ne.max()), "expand_per_step": float(cnt["n_expand"].double().mean()) / S_,
                                  "shrink_per_step": float(cnt["n_shrink"].double().mean()) / S_, "stuck": int(cnt["n_stuck"].sum())}
            uw, lw = donors[idx].clone(), ld[idx].clone()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            cw = hs3.walk_batch(donors, uw, lw, lstar, 5000, 777, 3)
            b.record(stream)
            torch.cuda.synchronize()
            res["acceptance_walk_W=5000"] = {"ms": a.elapsed_time(b), "evals": int(cw["n_eval"].sum()),
                                             "evals_per_s": float(cw["n_eval"].sum()) / (a.elapsed_time(b) * 1e-3),
                                             "accept_mean": float(cw["n_accept"].double().mean())}
            extras["slice_vs_walk_config3_midrun"] = res
            hs3.close()
            # full config-3 run with the slice kernel inside the sampler (55 = 5 x 11 steps per replacement)
            hsl = nsgw.Handle(spec3, smp3, seed=1)
            hsl.set_option(4, 55)
            hsl.set_option(3, 1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            nit, st = hsl.run(smp3["term_kind"], smp3["term_tol"], 4000)
            logz, err, H = hsl.finalize_evidence()
            wall = time.perf_counter() - t0
            extras["ns_run_config3_slice"] = {"wall_s": wall, "iterations": nit, "n_eval_total": st["n_eval_total"], "logz": logz,
                                              "logz_err": err, "H": H, "slice_steps": st["walk_len"], "moved_mean_last": st["accept_mean"],
                                              "evals_per_s": st["n_eval_total"] / wall}
            hsl.close()
            # sequential limit: config 1 with k = 1 against the batched k = 50 (same n_live, same rule)
            spec1, smp1, logz_true = W.config1()
            seq = {}
            for kdel in (50, 1):
                smp_k = dict(smp1, n_delete=kdel)
                hk = nsgw.Handle(spec1, smp_k, seed=1)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                nit, st = hk.run(smp1["term_kind"], smp1["term_tol"], 200000)
                lz, le, _ = hk.finalize_evidence()
                seq[f"k={kdel}"] = {"wall_s": time.perf_counter() - t0, "iterations": nit, "n_eval_total": st["n_eval_total"],
                                    "logz": lz, "logz_err": le, "walk_len_last": st["walk_len"], "accept_mean_last": st["accept_mean"]}
                hk.close()
            seq["logz_closed_form"] = logz_true["logz_exact"]
            extras["config1_sequential_limit"] = seq
            # the same on a GW problem that both settings finish (PhenomD-form, H1+L1, 20-128 Hz = 433 bins, SNR 10; Mc, q, dL, tc
            # free, n_live 400): k = 200 against k = 1 (one CTA walks at a time: the sequential bilby-like limit on this machine);
            # and config 3 itself with k = 1, first 2000 iterations only
            wfc = wf_cuda_for(nsgw, torch)
            spec_s = W.fix_dims(W.make_data(W.gw_spec(W.LIKE_PHENOMD, ["H1", "L1"], 4.0, 128.0, (20.0, 40.0)), W.INJ_C3, 10.0, wfc),
                                (0, 1, 4, 8), W.INJ_C3)
            gseq = {}
            for kdel in (200, 1):
                smp_k = dict(n_live=400, n_delete=kdel, naccept=20, maxmcmc=2000, walks0=50.0, delay=-1.0)
                hk = nsgw.Handle(spec_s, smp_k, seed=1)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                nit, st = hk.run(0, 0.1, 200000)
                lz, le, _ = hk.finalize_evidence()
                wall = time.perf_counter() - t0
                gseq[f"k={kdel}"] = {"wall_s": wall, "iterations": nit, "n_eval_total": st["n_eval_total"], "logz": lz, "logz_err": le,
                                     "walk_len_last": st["walk_len"], "evals_per_s": st["n_eval_total"] / wall}
                hk.close()
            hk = nsgw.Handle(spec3, dict(smp3, n_delete=1), seed=1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            nit, st = hk.run(smp3["term_kind"], smp3["term_tol"], 2000)
            wall = time.perf_counter() - t0
            gseq["config3_k=1_first_2000_iterations"] = {"wall_s": wall, "iterations": nit, "n_eval_total": st["n_eval_total"],
                                                         "walk_len_last": st["walk_len"], "evals_per_s": st["n_eval_total"] / wall,
                                                         "logx": st["logx"]}
            hk.close()
            extras["gw_sequential_limit"] = gseq
            # PP test (stand-in for the paper's 100-injection study): config-3 shape, priors, PSD and sampler
            # settings; injections drawn from the prior, each in its own noise; credible levels of the injected values from the
            # weighted posterior (ns_posterior); KS test of uniformity per parameter
            from paper_2509_04336_b200 import pp

            def pt_cuda(s, uu):
                tmp = dict(s)
                tmp["strain"] = np.zeros((s["n_det"], s["n_freq"], 2))
                hh = nsgw.Handle(tmp)
                out = hh.prior_transform_batch(torch.as_tensor(uu).cuda()).cpu().numpy()
                hh.close()
                return out

            specs_pp, th_pp = W.pp_problem_set(spec3, args.pp_injections, 9001, wf_cuda_for(nsgw, torch), pt_cuda)
            # the same with the distance prior cut to [200, 800] Mpc (SNR 20-80 for the config-3 masses): the regime relative
            # binning is made for (eps 0.1: the tolerance has to shrink as the SNR grows)
            spec3n = dict(spec3)
            spec3n["prior_lo"], spec3n["prior_hi"] = list(spec3["prior_lo"]), list(spec3["prior_hi"])
            spec3n["prior_lo"][4], spec3n["prior_hi"][4] = 200.0, 800.0
            specs_pn, th_pn = W.pp_problem_set(spec3n, args.pp_injections, 9002, wf_cuda_for(nsgw, torch), pt_cuda)
            for label, kw in (("exact", {}), ("relbin", {"relbin_eps": 0.5}), ("near_exact", {}), ("near_relbin", {"relbin_eps": 0.1})):
                if label.startswith("near"):
                    specs_pp, th_pp = specs_pn, th_pn
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                res = pp.credible_levels(specs_pp, th_pp, smp3, smp3["term_kind"], smp3["term_tol"], 400, seed0=500, group=4, **kw)
                wall = time.perf_counter() - t0
                ks = [pp.ks_uniform(res["cl"][:, d]) for d in range(11)]
                extras["pp_config3_" + label] = {
                    "injections": args.pp_injections, "wall_s": wall, "n_eval_total": int(res["evals"].sum()),
                    "iterations_mean": float(res["iters"].mean()), "ess_median": float(np.median(res["ess"])),
                    "ks_D": [round(k_[0], 4) for k_ in ks], "ks_p": [round(k_[1], 4) for k_ in ks],
                    "cl_mean": [round(float(x), 4) for x in res["cl"].mean(axis=0)],
                    "cl_var": [round(float(x), 4) for x in res["cl"].var(axis=0)]}
        line["extras"] = extras

    # ---- CPU baseline: the oracle as it stands on the host cores, bounded sample of the same rows (rank 0, N=1)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as O
        Pc = O.OracleProblem(spec)
        nb = args.cpu_rows
        th_np = theta[:nb].cpu().numpy()
        Pc.gw_loglike(th_np[:64])
        t0 = time.perf_counter()
        for _ in range(args.cpu_passes):
            lo = Pc.gw_loglike(th_np)
        dt = (time.perf_counter() - t0) / args.cpu_passes
        lg = logl[:nb].cpu().numpy()
        line["cpu_baseline"] = {"value": nb / dt, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                                "sample": f"first {nb} of the {B} rows x {args.cpu_passes} passes, OpenMP over rows, {dt * args.cpu_passes:.1f} s of CPU work",
                                "max_abs_dlogl_vs_gpu": float(np.max(np.abs(lg - lo)))}
        if not args.quick:
            # the oracle's sampler on the first iteration of configs 3 and 4 (same seed: same live set, walk length and proposals as
            # the device step above), and its full runs EXTRAPOLATED from that rate to the device runs' evaluation counts
            ex = line["extras"]
            steps = {}
            for name, sp_, sm_, run in (("config3", spec3, smp3, ex["ns_run_config3"]), ("config4", spec4, smp4, ex["ns_run_config4"])):
                Po = O.OracleProblem(sp_)
                t0 = time.perf_counter()
                So = O.OracleSampler(Po, sm_["n_live"], sm_["n_delete"], sm_["naccept"], sm_["maxmcmc"], sm_["walks0"], sm_["delay"], seed=1)
                t_init = time.perf_counter() - t0
                t0 = time.perf_counter()
                so = So.step()
                t_step = time.perf_counter() - t0
                rate = so["n_eval"] / t_step
                dev = ex["ns_step_first_iteration"][name]
                steps[name] = {"oracle_step_s": t_step, "oracle_init_live_s": t_init, "walk_len": so["walk_len"], "n_eval": so["n_eval"],
                               "oracle_evals_per_s": rate, "device_step_ms": dev["ms"],
                               "same_step_as_device": [so["walk_len"], so["n_eval"], so["n_oob"]] == [dev["walk_len"], dev["n_eval"], dev["n_oob"]],
                               "device_run_wall_s": run["wall_s"], "device_run_evals": run["n_eval_total"],
                               "oracle_run_wall_s_extrapolated": run["n_eval_total"] / rate,
                               "note": "extrapolation: device run's likelihood evaluations / oracle evaluations per second on this step"}
            gold = os.path.join(ROOT, "tests", "golden", "config3_oracle_run.json")
            if os.path.exists(gold):
                g = json.load(open(gold))
                steps["config3"]["oracle_full_run_stored"] = {"wall_s": g["wall_s"], "threads": g["threads"], "iterations": g["iterations"],
                                                              "n_eval_total": g["n_eval_total"], "logz": g["logz"], "logz_err": g["logz_err"],
                                                              "file": "tests/golden/config3_oracle_run.json (oracle/make_baseline.py; another machine's cores)"}
            line["cpu_baseline"]["ns_step"] = steps
    if rank == 0:
        print(json.dumps(line), flush=True)
    h.close()
    D.finalize()


def wf_cuda_for(nsgw, torch):
    def wf(spec, th):
        tmp = dict(spec)
        tmp["strain"] = np.zeros((spec["n_det"], spec["n_freq"], 2))
        hh = nsgw.Handle(tmp)
        out = hh.gw_waveform(torch.as_tensor(th).cuda()).cpu().numpy()
        hh.close()
        return out
    return wf


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--batch", type=int, default=65536)
    ap.add_argument("--ref-batch", type=int, default=1024)
    ap.add_argument("--cpu-rows", type=int, default=65536)
    ap.add_argument("--cpu-passes", type=int, default=3)
    ap.add_argument("--quick", action="store_true", help="skip the walk / full-run extras")
    ap.add_argument("--full-extras", action="store_true", help="also: relative binning, posterior, concurrent runs, slice kernel, sequential limit, PP tests")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--pp-injections", type=int, default=100, help="injections of the PP leg of --full-extras")
    ap.add_argument("--sweep-budget-s", type=float, default=90.0, help="time cap of the config-5 sweep (points past it are listed as skipped)")
    args = ap.parse_args()
    if resolve_world(args, os.environ) == "spawn":       # `bench.py --gpus N` by itself: start the N ranks
        os.execvp(sys.executable, spawn_command(args.gpus, sys.argv[1:]))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
