"""Writes the stored full-run baselines under tests/golden/ -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Runs the CPU oracle's nested sampler (oracle.cpp: orc_step, readings R:L6-L18) on a full-size BASELINE.json config, one seed,
and stores what the GPU-vs-oracle run test compares (SURVEY 8c-T "Full runs", 8(d) "config 3 one seed with all cores (cache
logZ, sigma, posterior quantiles and wall-clock)"; the paper's own validation has this form: posterior overlap P:198, logZ within
error P:256, KS P:276):

  logZ, sigma(logZ), H, iterations, likelihood evaluations, the per-iteration trajectory (walk length, mean / min / max accepted
  steps, evaluations, out-of-bounds proposals, logL*, logZ), n_post equal-weight posterior rows (R:L26 weights, R:L27
  systematic resampling), wall-clock and thread count.

Imports oracle/ and the input generators (paper_2509_04336_b200.workloads: inputs only) and nothing else of the package;
no value in the output comes from the CUDA path.

  python -m oracle.make_baseline --config 3 --seed 1 --threads 8 --out tests/golden/config3_oracle_run.json
  python -m oracle.make_baseline --config 4 --seed 1 --max-iter 2 --out tests/golden/config4_oracle_steps.json   (first steps only)
"""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle as O                                   # noqa: E402
from paper_2509_04336_b200 import workloads as W                 # noqa: E402  (seeded inputs only)

TRAJ_KEYS = ("walk_len", "walks_next", "accept_mean", "accept_min", "accept_max", "n_eval", "n_oob", "n_stuck", "logl_star",
             "logx", "logz", "h", "dlogz", "live_frac_log")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=3, choices=[3, 4])
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--threads", type=int, default=0, help="OpenMP threads over walkers (0 = all cores)")
    ap.add_argument("--max-iter", type=int, default=4000)
    ap.add_argument("--n-post", type=int, default=2000)
    ap.add_argument("--out", required=True)
    ap.add_argument("--progress", default=None, help="optional file that receives one line per iteration")
    args = ap.parse_args()

    wf = lambda s, th: O.OracleProblem(s).waveform(th)
    spec, smp = (W.config3 if args.config == 3 else W.config4)(wf)
    P = O.OracleProblem(spec)
    threads = args.threads if args.threads > 0 else (os.cpu_count() or 1)
    t_start = time.perf_counter()
    S = O.OracleSampler(P, smp["n_live"], smp["n_delete"], smp["naccept"], smp["maxmcmc"], smp["walks0"], smp["delay"],
                        seed=args.seed, threads=threads)
    traj = {k: [] for k in TRAJ_KEYS}
    step_s, dead_rows = [], []
    done_by_rule = False
    it = 0
    while it < args.max_iter:
        t0 = time.perf_counter()
        st, dead = S.step(want_dead=True)
        step_s.append(time.perf_counter() - t0)
        dead_rows.append(dead)
        for k in TRAJ_KEYS:
            traj[k].append(st[k])
        it += 1
        if args.progress:
            with open(args.progress, "a") as f:
                f.write(json.dumps({"it": it, "t": time.perf_counter() - t_start, **{k: st[k] for k in TRAJ_KEYS}}) + "\n")
        # the termination rule of orc_run (R:L18)
        if smp["term_kind"] == 0 and st["dlogz"] < smp["term_tol"]:
            done_by_rule = True
            break
        if smp["term_kind"] == 1 and st["live_frac_log"] < np.log(smp["term_tol"]):
            done_by_rule = True
            break
    wall = time.perf_counter() - t_start
    logz, err, H = S.finalize()
    out = {
        "what": "CPU oracle nested-sampling run (oracle/make_baseline.py); compared statistically with the CUDA path",
        "config": args.config, "seed": args.seed, "sampler": smp, "n_freq": spec["n_freq"], "n_det": spec["n_det"],
        "terminated_by_rule": done_by_rule, "iterations": it, "n_eval_total": int(st["n_eval_total"]),
        "logz": logz, "logz_err": err, "H": H, "wall_s": wall, "threads": threads, "step_s": [round(x, 3) for x in step_s],
        "trajectory": traj,
    }
    if done_by_rule and args.n_post > 0:
        u_l, l_l = S.live()
        post = O.posterior(P, np.concatenate(dead_rows), u_l, l_l, st["logx"], theta_ref=spec["theta_inj"])
        idx, _ = O.posterior_resample(post["logp"], args.n_post, args.seed)
        out["posterior"] = {"n_rows": int(post["logp"].size), "ess": post["ess"], "logz_rows": post["logz"],
                            "cl_injection": [float(x) for x in post["cl"]],
                            "theta_equal_weight": [[float("%.12g" % v) for v in row] for row in post["theta"][idx]]}
    os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
    with open(args.out, "w") as f:
        json.dump(out, f)
        f.write("\n")
    print(json.dumps({k: out[k] for k in ("config", "iterations", "n_eval_total", "logz", "logz_err", "H", "wall_s", "threads")}))


if __name__ == "__main__":
    main()
