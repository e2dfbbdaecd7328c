"""PP-test harness (the paper's 100-injection study): one nested-sampling run per injection, several
at a time through ns_run_many, and the credible level of the injected value under each run's weighted posterior (ns_posterior).
If sampler, likelihood and priors are consistent, the levels of every parameter are uniform on (0, 1).  Everything numerical
runs in the CUDA library; this module only loops over injections."""
import math

import numpy as np
import torch

from . import nsgw


def credible_levels(specs, thetas, sampler, term_kind, term_tol, max_iter, seed0=1, group=4, relbin_eps=None, slice_kernel=False):
    """specs[i]: problem with the i-th injection's strain; thetas[i]: its injected parameters.  Returns a dict of NumPy arrays:
    cl [n, ndim] (NaN columns are never produced: FIXED parameters give level 0), ess [n], logz [n], iters [n], evals [n]."""
    n, D, k = len(specs), specs[0]["ndim"], sampler["n_delete"]
    cl, ess, logz = np.empty((n, D)), np.empty(n), np.empty(n)
    iters, evals = np.empty(n, np.int64), np.empty(n, np.int64)
    for g0 in range(0, n, group):
        idx = list(range(g0, min(n, g0 + group)))
        hs, dead = [], []
        for i in idx:
            h = nsgw.Handle(specs[i], sampler, seed=seed0 + i)
            if relbin_eps is not None:
                h.relbin_setup(thetas[i], 1.0, relbin_eps)
                h.set_option(nsgw.OPT_LIKELIHOOD, 1)
            if slice_kernel:
                h.set_option(nsgw.OPT_INNER_KERNEL, 1)
            hs.append(h)
            dead.append(torch.empty((max_iter * k, D + 3), dtype=torch.float64, device="cuda"))
        its, sts = nsgw.run_many(hs, term_kind, term_tol, max_iter, dead=dead)
        for j, i in enumerate(idx):
            out = hs[j].posterior(dead[j][: its[j] * k].contiguous(), theta_ref=thetas[i], want_theta=True)
            cl[i], ess[i], logz[i] = out["cl"], out["ess"], out["logz"]
            iters[i], evals[i] = its[j], sts[j]["n_eval_total"]
        del hs, dead
    return {"cl": cl, "ess": ess, "logz": logz, "iters": iters, "evals": evals}


def ks_uniform(x):
    """One-sample Kolmogorov-Smirnov test of x against U(0, 1): (D, asymptotic p-value with Stephens' small-sample factor)."""
    x = np.sort(np.asarray(x, dtype=np.float64))
    n = x.size
    d = max(float(np.max(np.arange(1, n + 1) / n - x)), float(np.max(x - np.arange(0, n) / n)))
    lam = (math.sqrt(n) + 0.12 + 0.11 / math.sqrt(n)) * d
    if lam < 0.2:
        return d, 1.0
    p = 2.0 * sum((-1.0) ** (j - 1) * math.exp(-2.0 * j * j * lam * lam) for j in range(1, 101))
    return d, min(1.0, max(0.0, p))
