"""Shared helpers of the parity tests: build a workload's trace with the ORACLE
(the oracle plays the paper's 'CPU solver that synthesises the experimental
trace') and marshal the same workload dict for both sides.
No arithmetic of the method lives here."""
import json
import os

import numpy as np

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm


def oracle_trace(wl, truths=None, noise=True):
    """[n_traces][W] trace: oracle window of the ground truth (+ seeded noise)."""
    M = orc.model_from(wl)
    T = wl["n_traces"]
    if truths is None:
        truths = [wl["truth"]] if wl["truth"] is not None else wlm.pixel_truths(wl)
    truths = np.asarray(truths, dtype=np.float64).reshape(T, wl["n_params"])
    out = np.empty((T, wl["n_window"]))
    for s in range(T):
        bad, w = orc.window(M, truths[s], wl["z0"], wl["v0"])
        assert bad == 0
        out[s] = w
    if noise:
        out = out + wlm.trace_noise(wl, n_traces=T)
    return out


def rel_err(a, b):
    """Element-wise relative error with inf == inf counted as 0."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    both_inf = np.isinf(a) & np.isinf(b) & (np.sign(a) == np.sign(b))
    with np.errstate(invalid="ignore", divide="ignore"):
        e = np.abs(a - b) / np.maximum(np.abs(b), np.finfo(np.float64).tiny)
    e = np.where(both_inf, 0.0, e)
    e = np.where((a == b), 0.0, e)
    return e


def record_parity(label, precision, e, tol, n_above, n_excused_repo, n_excused_c15):
    """Append one row of parity statistics to the file named by $AFM_PARITY_STATS
    (profiles/r3_parity_stats.md is made from such a run); no-op when it is unset.
    e: relative errors of the sample; n_above: how many are >= tol; n_excused_*: how
    many of those the repository's R15 rule and SURVEY.md c-15's one-ulp rule excuse."""
    path = os.environ.get("AFM_PARITY_STATS")
    if not path:
        return
    e = np.asarray(e, dtype=np.float64)
    fin = e[np.isfinite(e)]
    row = dict(label=label, precision=precision, n=int(e.size), tol=tol,
               median=float(np.median(fin)), p99=float(np.percentile(fin, 99)),
               max=float(fin.max()), above_tol=int(n_above),
               excused_repo_rule=int(n_excused_repo), excused_c15_one_ulp=int(n_excused_c15))
    with open(path, "a") as f:
        f.write(json.dumps(row) + "\n")
