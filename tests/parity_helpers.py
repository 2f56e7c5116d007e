"""Shared helpers of the parity tests: build a workload's trace with the ORACLE
(the oracle plays the paper's 'CPU solver that synthesises the experimental
trace') and marshal the same workload dict for both sides.
No arithmetic of the method lives here."""
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
