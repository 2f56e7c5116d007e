"""afm_forward_batch_noalloc: the forward batch for callers that cannot let the
library allocate device memory.

Who that is: the acquisition loop of a running microscope (the paper's "near
real-time" use), which cannot absorb the stall of a cudaMalloc or
cudaFree in the middle of a scan line -- both take driver-wide locks and may wait
for the whole device -- and a process whose device memory has been handed to
another component's pool, where an allocation made behind that pool's back can
fail or take memory the pool counts on.  For them the library carries a 4 MiB
scratch array inside its own device image (include/afm.h, AFM_NOALLOC_MAX_ROWS
rows of the time-tile stream) and this entry point uses that instead of the
grow-only workspace.

What is checked here: the misfits equal those of afm_forward_batch, the ordinary
path, within the tolerances of the other parity tests (1e-9 relative in FP64,
1e-3 in FP32), on calls made back to back -- the array is shared by all calls and
never cleared, so a call must not be able to see what the one before it left
behind (a longer solve, another law, another precision) -- and that a batch
beyond the built-in size is refused with a message instead of overrunning it.

This file is named to be collected last: `pytest -x` stops at the first failure
and a failure here must not hide the parity tests proper.  It passes on its own in
a fresh process (the first call below is then the first CUDA call of the library)
and after the rest of the suite (the workspace of the ordinary path is then
already large, options have been set and reset).
"""
import ctypes as C

import numpy as np
import pytest

from paper_1109_0334_b200 import workloads as wlm
from parity_helpers import oracle_trace, rel_err

TOL = {0: 1e-9, 1: 1e-3}    # afm_precision -> relative tolerance of the parity tests


@pytest.fixture(scope="module")
def afm():
    import torch
    assert torch.cuda.is_available()
    from paper_1109_0334_b200 import afm as m
    m.lib()  # fails loudly if the CUDA library is missing
    return m


def _case(wl, n, seed, phases=False, truths=None):
    """Seeded inputs of one batch: (workload, params [n][D], trace, z0v0 or None)."""
    trace = oracle_trace(wl, truths=truths)
    params = wlm.draw_params(wl, n, seed=seed)
    z0v0 = wlm.draw_initial_states(wl, n, seed=seed + 1) if phases else None
    return wl, params, trace, z0v0


def _both_paths(afm, case, precision):
    """(misfit of afm_forward_batch, misfit of afm_forward_batch_noalloc) on the
    same device tensors, same stream, the no-allocation call second."""
    import torch
    wl, params, trace, z0v0 = case
    cfg = afm.cfg_from(wl, precision=precision)
    p = torch.as_tensor(np.ascontiguousarray(params), device="cuda")
    t = torch.as_tensor(np.ascontiguousarray(trace), device="cuda")
    zv = None if z0v0 is None else torch.as_tensor(np.ascontiguousarray(z0v0), device="cuda")
    ref = afm.afm_forward_batch(p, t, cfg, z0v0=zv)
    out = torch.full((p.shape[0],), -1.0, dtype=torch.float64, device="cuda")
    got = afm.afm_forward_batch_noalloc(p, t, cfg, out, z0v0=zv)
    assert got.data_ptr() == out.data_ptr()      # the caller's buffer, nothing new
    torch.cuda.synchronize()
    return ref.cpu().numpy(), out.cpu().numpy()


def _agree(ref, got, precision):
    assert np.all(got >= 0)                      # every particle was written
    assert np.isfinite(ref).any()
    assert np.array_equal(np.isinf(ref), np.isinf(got))
    assert rel_err(got, ref).max() < TOL[precision]


@pytest.mark.gpu
@pytest.mark.parametrize("precision", [0, 1])
def test_noalloc_matches_the_ordinary_path_on_consecutive_calls(afm, precision):
    """Three calls in a row through the one shared array: a short DMT solve, then a
    longer DMT + viscoelastic solve with three traces that overwrites five times as
    many rows, then the first batch again.  Each equals the ordinary path; the
    third also equals the first bit for bit, so nothing of the second call's rows
    leaked into it."""
    short = _case(wlm.scaled(wlm.config(0), n_cycles=12, n_skip_cycles=6), 131, seed=31)
    wl2 = wlm.scaled(wlm.config(2), n_cycles=8, n_skip_cycles=4, n_traces=3)
    truths = wlm.draw_params(wl2, 3, seed=41)
    longer = _case(wl2, 3 * 70, seed=33, truths=truths)
    assert longer[0]["n_traces"] * longer[0]["n_steps"] > 4 * short[0]["n_steps"]

    ref_a, got_a = _both_paths(afm, short, precision)
    _agree(ref_a, got_a, precision)
    ref_b, got_b = _both_paths(afm, longer, precision)
    _agree(ref_b, got_b, precision)
    ref_c, got_c = _both_paths(afm, short, precision)
    _agree(ref_c, got_c, precision)
    assert np.array_equal(got_c, got_a)


@pytest.mark.gpu
def test_noalloc_after_the_other_precision_and_with_initial_states(afm):
    """FP32 rows (16 bytes each) written over FP64 rows (32 bytes) and back, with
    per-particle initial states (configs[1]'s random phases), several warps."""
    wl = wlm.scaled(wlm.config(1), n_cycles=10, n_skip_cycles=5)
    case = _case(wl, 517, seed=51, phases=True)
    for precision in (0, 1, 0):
        ref, got = _both_paths(afm, case, precision)
        _agree(ref, got, precision)


@pytest.mark.gpu
def test_noalloc_takes_a_batch_of_exactly_the_built_in_size(afm):
    """n_traces * N == AFM_NOALLOC_MAX_ROWS: the last row of the array is used."""
    wl = wlm.scaled(wlm.config(0), steps_per_cycle=128, n_cycles=1024, n_skip_cycles=1020)
    assert wl["n_steps"] == afm.NOALLOC_MAX_ROWS
    ref, got = _both_paths(afm, _case(wl, 40, seed=61), 0)
    _agree(ref, got, 0)


def test_noalloc_refuses_more_rows_than_the_built_in_array():
    """One row too many is AFM_EINVAL with the sizes in the message, decided before
    any device is touched (so this one runs on the CPU box too)."""
    from paper_1109_0334_b200 import afm, build
    build.build()
    lib = afm.lib()
    wl = wlm.scaled(wlm.config(0), steps_per_cycle=afm.NOALLOC_MAX_ROWS // 2 + 1,
                    n_cycles=2, n_skip_cycles=1)
    cfg = afm.cfg_from(wl)
    rc = lib.afm_forward_batch_noalloc(C.c_void_p(16), 4, C.c_void_p(16), C.byref(cfg),
                                       None, C.c_void_p(16), None)
    assert rc == afm.EINVAL
    msg = lib.afm_last_error().decode()
    assert str(afm.NOALLOC_MAX_ROWS) in msg and str(wl["n_steps"]) in msg
    # the count is over all traces: three traces of a third of the array each, plus
    # one cycle, no longer fit
    wl3 = wlm.scaled(wlm.config(0), steps_per_cycle=128, n_cycles=342, n_skip_cycles=1,
                     n_traces=3)
    assert wl3["n_steps"] <= afm.NOALLOC_MAX_ROWS < 3 * wl3["n_steps"]
    cfg3 = afm.cfg_from(wl3)
    rc = lib.afm_forward_batch_noalloc(C.c_void_p(16), 6, C.c_void_p(16), C.byref(cfg3),
                                       None, C.c_void_p(16), None)
    assert rc == afm.EINVAL
    assert str(3 * wl3["n_steps"]) in lib.afm_last_error().decode()
