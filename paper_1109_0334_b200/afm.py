"""Thin ctypes binding of libafm_b200.so (include/afm.h).

Argument marshalling only: every step of the hot path runs in the library's
CUDA kernels.  PyTorch appears here as the owner of device memory and of the
CUDA stream, nothing else.  There is no CPU fallback: loading fails loudly if
the library has not been built (`python -m paper_1109_0334_b200.build`), and
every compute call raises AfmError when no sm_100 device is present.

Function names and argument order follow include/afm.h.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libafm_b200.so")

LAW_NONE, LAW_DMT, LAW_DMT_VISC, LAW_LJ_EXP, LAW_HOOKE, LAW_KELVIN_VOIGT = 0, 1, 2, 3, 4, 5
F64, F32 = 0, 1
OK, EINVAL, ECUDA, EUNSUPPORTED = 0, -1, -2, -3

# every symbol include/afm.h declares (tests check the library exports them all)
SYMBOLS = (
    "afm_forward_batch", "afm_forward_batch_host", "afm_forward_batch_noalloc",
    "afm_pso_invert", "afm_pso_invert_host", "afm_pso_step", "afm_pso_step_host", "afm_pso_init",
    "afm_kernel_times", "afm_queue_status", "afm_last_integrate_kernel",
    "afm_pso_shard_init", "afm_pso_shard_eval", "afm_pso_shard_move",
    "afm_beam_modes", "afm_beam_forward_batch", "afm_beam_pso_invert",
    "afm_beam_trajectory", "afm_philox4x32_10", "afm_trajectory", "afm_fma_peak",
    "afm_launch_count",
    "afm_reset_launch_count", "afm_set_option", "afm_last_error",
    "afm_version", "afm_shutdown",
)


class BeamCfg(C.Structure):
    _fields_ = [("L", C.c_double), ("E", C.c_double), ("I", C.c_double),
                ("mu", C.c_double), ("Q", C.c_double), ("f_drive", C.c_double),
                ("A_base", C.c_double), ("A_ref", C.c_double), ("z_c", C.c_double),
                ("R", C.c_double), ("a0", C.c_double), ("law", C.c_int32),
                ("n_params", C.c_int32), ("n_modes", C.c_int32),
                ("n_points", C.c_int32), ("steps_per_cycle", C.c_int32),
                ("n_cycles", C.c_int32), ("n_skip_cycles", C.c_int32),
                ("n_traces", C.c_int32)]

    @property
    def n_steps(self):
        return self.steps_per_cycle * self.n_cycles

    @property
    def n_window(self):
        return self.steps_per_cycle * (self.n_cycles - self.n_skip_cycles)


class AfmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("afm error %d: %s" % (code, msg))
        self.code = code


class Cfg(C.Structure):
    _fields_ = [("k", C.c_double), ("f0", C.c_double), ("Q", C.c_double),
                ("f_drive", C.c_double), ("A0", C.c_double),
                ("z_c", C.c_double), ("R", C.c_double), ("a0", C.c_double),
                ("z0", C.c_double), ("v0", C.c_double),
                ("law", C.c_int32), ("n_params", C.c_int32),
                ("steps_per_cycle", C.c_int32), ("n_cycles", C.c_int32),
                ("n_skip_cycles", C.c_int32), ("n_traces", C.c_int32),
                ("precision", C.c_int32), ("reserved_", C.c_int32)]

    @property
    def n_steps(self):
        return self.steps_per_cycle * self.n_cycles

    @property
    def n_window(self):
        return self.steps_per_cycle * (self.n_cycles - self.n_skip_cycles)


class Bounds(C.Structure):
    _fields_ = [("lo", C.c_double * 4), ("hi", C.c_double * 4),
                ("log10_scale", C.c_int32 * 4)]


class SwarmCfg(C.Structure):
    _fields_ = [("n_particles", C.c_int32), ("n_iters", C.c_int32),
                ("w", C.c_double), ("c1", C.c_double), ("c2", C.c_double),
                ("j_target", C.c_double), ("topology", C.c_int32),
                ("async_chunk", C.c_int32)]


_lib = None


def lib():
    """The loaded library; raises if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                "%s is missing: build it with `python -m paper_1109_0334_b200.build` "
                "(there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp, dp, i32, i64, u64 = C.c_void_p, C.c_void_p, C.c_int32, C.c_int64, C.c_uint64
        L.afm_forward_batch.argtypes = [dp, i64, dp, C.POINTER(Cfg), dp, dp, vp]
        L.afm_forward_batch_host.argtypes = [dp, i64, dp, C.POINTER(Cfg), dp, dp, vp]
        L.afm_forward_batch_noalloc.argtypes = [dp, i64, dp, C.POINTER(Cfg), dp, dp, vp]
        L.afm_forward_batch_noalloc.restype = C.c_int
        L.afm_pso_invert.argtypes = [C.POINTER(Bounds), C.POINTER(SwarmCfg), u64, dp,
                                     C.POINTER(Cfg), dp, dp, dp, dp,
                                     C.POINTER(i32), vp]
        L.afm_pso_invert_host.argtypes = [C.POINTER(Bounds), C.POINTER(SwarmCfg), u64,
                                          dp, C.POINTER(Cfg), dp, dp,
                                          C.POINTER(i32), vp]
        L.afm_pso_step.argtypes = [C.POINTER(Bounds), C.POINTER(SwarmCfg), i32, i32,
                                   u64, i32, i32, dp, dp, dp, dp, dp, dp, dp, vp]
        L.afm_pso_step_host.argtypes = L.afm_pso_step.argtypes
        L.afm_pso_step_host.restype = C.c_int
        L.afm_kernel_times.argtypes = [C.POINTER(C.c_double), i32, C.POINTER(i32)]
        L.afm_kernel_times.restype = C.c_int
        L.afm_last_integrate_kernel.argtypes = []
        L.afm_last_integrate_kernel.restype = C.c_char_p
        L.afm_queue_status.argtypes = [vp]
        L.afm_queue_status.restype = C.c_int
        L.afm_pso_init.argtypes = [C.POINTER(Bounds), C.POINTER(SwarmCfg), i32, i32,
                                   u64, dp, dp, dp, dp, dp, dp, vp]
        L.afm_pso_shard_init.argtypes = [C.POINTER(Bounds), C.POINTER(SwarmCfg), i32,
                                         i32, u64, i64, dp, dp, dp, dp, dp, dp, vp]
        L.afm_pso_shard_eval.argtypes = [C.POINTER(Bounds), C.POINTER(SwarmCfg), dp,
                                         C.POINTER(Cfg), i64, dp, dp, dp, dp, dp, vp]
        L.afm_pso_shard_move.argtypes = [C.POINTER(Bounds), C.POINTER(SwarmCfg), i32,
                                         i32, u64, i32, i32, i64, dp, i32, i32, i64, dp,
                                         dp, dp, dp, dp, dp, dp, dp, vp]
        L.afm_beam_modes.argtypes = [C.POINTER(BeamCfg), dp, dp, dp, dp, dp, vp]
        L.afm_beam_forward_batch.argtypes = [dp, i64, dp, C.POINTER(BeamCfg),
                                             C.POINTER(Bounds), dp, vp]
        L.afm_beam_pso_invert.argtypes = [C.POINTER(Bounds), C.POINTER(SwarmCfg), u64, dp,
                                          C.POINTER(BeamCfg), dp, dp, dp, dp,
                                          C.POINTER(i32), vp]
        L.afm_beam_trajectory.argtypes = [dp, C.POINTER(BeamCfg), dp, dp, vp]
        for name in ("afm_beam_modes", "afm_beam_forward_batch", "afm_beam_pso_invert",
                     "afm_beam_trajectory"):
            getattr(L, name).restype = C.c_int
        L.afm_philox4x32_10.argtypes = [dp, i64, C.POINTER(C.c_uint32), dp, vp]
        L.afm_trajectory.argtypes = [dp, C.POINTER(Cfg), C.c_double, C.c_double,
                                     dp, dp, vp]
        L.afm_fma_peak.argtypes = [i32, C.c_double, C.POINTER(C.c_double), vp]
        for name in ("afm_forward_batch", "afm_forward_batch_host", "afm_pso_invert",
                     "afm_pso_invert_host", "afm_pso_step", "afm_pso_step_host", "afm_pso_init",
    "afm_kernel_times",
                     "afm_philox4x32_10", "afm_trajectory", "afm_fma_peak",
                     "afm_pso_shard_init", "afm_pso_shard_eval",
                     "afm_pso_shard_move"):
            getattr(L, name).restype = C.c_int
        L.afm_launch_count.restype = i64
        L.afm_launch_count.argtypes = []
        L.afm_reset_launch_count.restype = None
        L.afm_set_option.argtypes = [C.c_char_p, i64]
        L.afm_set_option.restype = C.c_int
        L.afm_last_error.restype = C.c_char_p
        L.afm_version.restype = C.c_char_p
        L.afm_shutdown.restype = None
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise AfmError(rc, lib().afm_last_error().decode("utf-8", "replace"))


# ---- marshalling from the workload dictionaries ------------------------------

def cfg_from(wl, precision=F64, **over):
    """afm_cfg from a paper_1109_0334_b200.workloads dict."""
    c = wl["cantilever"]
    cfg = Cfg(k=c["k"], f0=c["f0"], Q=c["Q"], f_drive=c["f_drive"], A0=c["A0"],
              z_c=c["z_c"], R=c["R"], a0=c["a0"], z0=wl["z0"], v0=wl["v0"],
              law=wl["law"], n_params=wl["n_params"],
              steps_per_cycle=wl["steps_per_cycle"], n_cycles=wl["n_cycles"],
              n_skip_cycles=wl["n_skip_cycles"], n_traces=wl["n_traces"],
              precision=precision, reserved_=0)
    for k, v in over.items():
        setattr(cfg, k, v)
    return cfg


def bounds_from(wl):
    b = Bounds()
    for j in range(wl["n_params"]):
        b.lo[j] = wl["bounds"]["lo"][j]
        b.hi[j] = wl["bounds"]["hi"][j]
        b.log10_scale[j] = int(wl["bounds"]["log10"][j])
    return b


def swarm_from(wl, j_target=0.0, **over):
    s = wl["swarm"]
    sc = SwarmCfg(n_particles=s["n_particles"], n_iters=s["n_iters"], w=s["w"],
                  c1=s["c1"], c2=s["c2"], j_target=j_target,
                  topology=s.get("topology", 0), async_chunk=s.get("async_chunk", 0))
    for k, v in over.items():
        setattr(sc, k, v)
    return sc


# ---- device-buffer helpers (torch = allocator + stream) ---------------------

def _torch():
    import torch
    return torch


def _stream_ptr(stream):
    if stream is None:
        return _torch().cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _dev_f64(t, name):
    torch = _torch()
    if not isinstance(t, torch.Tensor):
        t = torch.as_tensor(np.ascontiguousarray(t, dtype=np.float64), device="cuda")
    if not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError("%s must be a contiguous CUDA float64 tensor" % name)
    return t


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _host_f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _hptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


# ---- the calls of include/afm.h -------------------------------------------------

def afm_forward_batch(params, trace, cfg, z0v0=None, misfit=None, stream=None):
    """misfit[p] = J(theta_p) (device tensors in, device tensor out; async)."""
    torch = _torch()
    params = _dev_f64(params, "params")
    trace = _dev_f64(trace, "trace")
    P = params.shape[0]
    if params.numel() != P * max(cfg.n_params, 0) and cfg.n_params > 0:
        raise ValueError("params must be [P][D]")
    if trace.numel() != cfg.n_traces * cfg.n_window:
        raise ValueError("trace must hold n_traces * W = %d samples"
                         % (cfg.n_traces * cfg.n_window))
    if z0v0 is not None:
        z0v0 = _dev_f64(z0v0, "z0v0")
        if z0v0.numel() != 2 * P:
            raise ValueError("z0v0 must be [P][2]")
    if misfit is None:
        misfit = torch.empty(P, dtype=torch.float64, device=params.device)
    else:
        misfit = _dev_f64(misfit, "misfit")
    _check(lib().afm_forward_batch(_ptr(params), P, _ptr(trace), C.byref(cfg),
                                   _ptr(z0v0), _ptr(misfit), _stream_ptr(stream)))
    return misfit


# Rows (one per trace and RK4 step) of the scratch array built into the library
# for afm_forward_batch_noalloc: AFM_NOALLOC_MAX_ROWS of include/afm.h.
NOALLOC_MAX_ROWS = 131072


def afm_forward_batch_noalloc(params, trace, cfg, misfit, z0v0=None, stream=None):
    """afm_forward_batch for callers that must not let the library allocate device
    memory (an instrument's acquisition loop that cannot absorb the stall of a
    cudaMalloc/cudaFree; a process whose device memory is owned by another pool).
    The library's only scratch sits in a 4 MiB array inside its own device image,
    so cfg.n_traces * cfg.n_steps may not exceed NOALLOC_MAX_ROWS (AfmError
    otherwise).  All tensors, `misfit` included, are the caller's: nothing is
    created here.  Make the first call on each device at start-up (it looks up the
    array's device address); calls must not overlap on the GPU, they share the
    array.  See include/afm.h."""
    params = _dev_f64(params, "params")
    trace = _dev_f64(trace, "trace")
    misfit = _dev_f64(misfit, "misfit")
    P = params.shape[0]
    if params.numel() != P * max(cfg.n_params, 0) and cfg.n_params > 0:
        raise ValueError("params must be [P][D]")
    if trace.numel() != cfg.n_traces * cfg.n_window:
        raise ValueError("trace must hold n_traces * W = %d samples"
                         % (cfg.n_traces * cfg.n_window))
    if misfit.numel() != P:
        raise ValueError("misfit must be [P]")
    if z0v0 is not None:
        z0v0 = _dev_f64(z0v0, "z0v0")
        if z0v0.numel() != 2 * P:
            raise ValueError("z0v0 must be [P][2]")
    _check(lib().afm_forward_batch_noalloc(_ptr(params), P, _ptr(trace), C.byref(cfg),
                                           _ptr(z0v0), _ptr(misfit),
                                           _stream_ptr(stream)))
    return misfit


def afm_forward_batch_host(params, trace, cfg, z0v0=None, misfit=None, stream=None):
    """Same with host (numpy) buffers; copies inside the call; synchronous."""
    params = _host_f64(params)
    trace = _host_f64(trace)
    P = params.shape[0]
    if trace.size != cfg.n_traces * cfg.n_window:
        raise ValueError("trace must hold n_traces * W samples")
    z0v0 = None if z0v0 is None else _host_f64(z0v0)
    if misfit is None:
        misfit = np.empty(P, dtype=np.float64)
    _check(lib().afm_forward_batch_host(_hptr(params), P, _hptr(trace), C.byref(cfg),
                                        _hptr(z0v0), _hptr(misfit),
                                        _stream_ptr(stream)))
    return misfit


def afm_pso_invert(bounds, swarm, seed, trace, cfg, dump=False, hist=False,
                   stream=None):
    """Returns dict(theta_star [T][D], J_star [T], n_iters_done, dump, gbest_hist);
    dump / gbest_hist are device tensors or None; rows of batches a cost cutoff left
    unrun are not written."""
    torch = _torch()
    trace = _dev_f64(trace, "trace")
    if trace.numel() != cfg.n_traces * cfg.n_window:
        raise ValueError("trace must hold n_traces * W samples")
    D, T = cfg.n_params, cfg.n_traces
    PT = swarm.n_particles * T
    th = np.empty((T, D), dtype=np.float64)
    Js = np.empty(T, dtype=np.float64)
    if isinstance(dump, torch.Tensor):          # caller-owned [n_iters][PT][3D+2]
        dmp = _dev_f64(dump, "dump")
        if dmp.numel() != swarm.n_iters * PT * (3 * D + 2):
            raise ValueError("dump must be [n_iters][PT][3D+2]")
    else:
        dmp = (torch.empty((swarm.n_iters, PT, 3 * D + 2), dtype=torch.float64,
                           device=trace.device) if dump else None)
    gh = (torch.empty((swarm.n_iters, T, D + 1), dtype=torch.float64,
                      device=trace.device) if hist else None)
    done = C.c_int32(0)
    _check(lib().afm_pso_invert(C.byref(bounds), C.byref(swarm), int(seed),
                                _ptr(trace), C.byref(cfg), _hptr(th), _hptr(Js),
                                _ptr(dmp), _ptr(gh), C.byref(done),
                                _stream_ptr(stream)))
    return dict(theta_star=th, J_star=Js, n_iters_done=done.value, dump=dmp,
                gbest_hist=gh)


def afm_pso_invert_host(bounds, swarm, seed, trace, cfg, stream=None):
    trace = _host_f64(trace)
    if trace.size != cfg.n_traces * cfg.n_window:
        raise ValueError("trace must hold n_traces * W samples")
    D, T = cfg.n_params, cfg.n_traces
    th = np.empty((T, D), dtype=np.float64)
    Js = np.empty(T, dtype=np.float64)
    done = C.c_int32(0)
    _check(lib().afm_pso_invert_host(C.byref(bounds), C.byref(swarm), int(seed),
                                     _hptr(trace), C.byref(cfg), _hptr(th),
                                     _hptr(Js), C.byref(done), _stream_ptr(stream)))
    return dict(theta_star=th, J_star=Js, n_iters_done=done.value)


def afm_pso_init(bounds, swarm, n_dims, n_traces, seed, stream=None):
    """Allocates and fills the swarm state; returns a dict of device tensors."""
    torch = _torch()
    PT = swarm.n_particles * n_traces
    kw = dict(dtype=torch.float64, device="cuda")
    st = dict(x=torch.empty((PT, n_dims), **kw), v=torch.empty((PT, n_dims), **kw),
              pbest=torch.empty((PT, n_dims), **kw), pbestJ=torch.empty(PT, **kw),
              gbest=torch.empty((n_traces, n_dims), **kw),
              gbestJ=torch.empty(n_traces, **kw))
    _check(lib().afm_pso_init(C.byref(bounds), C.byref(swarm), n_dims, n_traces,
                              int(seed), _ptr(st["x"]), _ptr(st["v"]),
                              _ptr(st["pbest"]), _ptr(st["pbestJ"]),
                              _ptr(st["gbest"]), _ptr(st["gbestJ"]),
                              _stream_ptr(stream)))
    return st


def afm_pso_step(bounds, swarm, n_dims, n_traces, seed, iteration, do_move, J, st,
                 stream=None):
    J = _dev_f64(J, "J")
    _check(lib().afm_pso_step(C.byref(bounds), C.byref(swarm), n_dims, n_traces,
                              int(seed), int(iteration), int(bool(do_move)), _ptr(J),
                              _ptr(st["x"]), _ptr(st["v"]), _ptr(st["pbest"]),
                              _ptr(st["pbestJ"]), _ptr(st["gbest"]),
                              _ptr(st["gbestJ"]), _stream_ptr(stream)))
    return st


def afm_pso_step_host(bounds, swarm, n_dims, n_traces, seed, iteration, do_move, J, st,
                      stream=None):
    """afm_pso_step on HOST (numpy) state: st is a dict of contiguous float64 arrays
    x, v, pbest [PT][D], pbestJ [PT], gbest [T][D], gbestJ [T], updated in place."""
    for k in ("x", "v", "pbest", "pbestJ", "gbest", "gbestJ"):
        a = st[k]
        if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous):
            raise TypeError("st[%r] must be a contiguous float64 numpy array" % k)
    J = _host_f64(J)
    _check(lib().afm_pso_step_host(C.byref(bounds), C.byref(swarm), n_dims, n_traces,
                                   int(seed), int(iteration), int(bool(do_move)), _hptr(J),
                                   _hptr(st["x"]), _hptr(st["v"]), _hptr(st["pbest"]),
                                   _hptr(st["pbestJ"]), _hptr(st["gbest"]),
                                   _hptr(st["gbestJ"]), _stream_ptr(stream)))
    return st


def afm_queue_status(stream=None):
    """Waits for `stream` and raises AfmError if a segment-queue worker has given up
    since the last check: call it after the asynchronous device-tensor calls
    (afm_forward_batch, afm_beam_forward_batch, afm_pso_shard_eval) before trusting
    their outputs."""
    _check(lib().afm_queue_status(_stream_ptr(stream)))


def afm_last_integrate_kernel():
    """Name of the integrate kernel the last compute call of this thread launched."""
    return lib().afm_last_integrate_kernel().decode()


def afm_kernel_times(max_n=64):
    """Durations (ms, oldest first) of the last integrate-kernel launches recorded
    since afm_set_option("kernel_events", 1)."""
    buf = (C.c_double * max_n)()
    n = C.c_int32(0)
    _check(lib().afm_kernel_times(buf, max_n, C.byref(n)))
    return [buf[i] for i in range(n.value)]


def shard_row_doubles(n_dims, topology):
    """Doubles per trace in a shard's candidate row (include/afm.h): D + 2, or 3 D + 4
    with the ring topology (edge particles' personal bests ride along)."""
    return 3 * n_dims + 4 if topology == 1 else n_dims + 2


def afm_pso_shard_init(bounds, swarm, n_dims, n_traces, seed, first_particle,
                       stream=None):
    """Swarm state of a shard: swarm.n_particles local particles
    per local trace, global index = first_particle + local index."""
    torch = _torch()
    PT = swarm.n_particles * n_traces
    kw = dict(dtype=torch.float64, device="cuda")
    st = dict(x=torch.empty((PT, n_dims), **kw), v=torch.empty((PT, n_dims), **kw),
              pbest=torch.empty((PT, n_dims), **kw), pbestJ=torch.empty(PT, **kw),
              gbest=torch.empty((n_traces, n_dims), **kw),
              gbestJ=torch.empty(n_traces, **kw), J=torch.empty(PT, **kw),
              cand=torch.empty((n_traces, shard_row_doubles(n_dims, swarm.topology)), **kw),
              theta_star=torch.empty((n_traces, n_dims), **kw),
              J_star=torch.empty(n_traces, **kw))
    _check(lib().afm_pso_shard_init(C.byref(bounds), C.byref(swarm), n_dims, n_traces,
                                    int(seed), int(first_particle), _ptr(st["x"]),
                                    _ptr(st["v"]), _ptr(st["pbest"]),
                                    _ptr(st["pbestJ"]), _ptr(st["gbest"]),
                                    _ptr(st["gbestJ"]), _stream_ptr(stream)))
    return st


def afm_pso_shard_eval(bounds, swarm, trace, cfg, first_particle, st, stream=None):
    """Forward batch + personal bests of the shard; returns st["cand"]
    [n_traces][R] = (pbestJ, global index, pbest x[D][, edge particles' bests]) for the
    exchange."""
    trace = _dev_f64(trace, "trace")
    if trace.numel() != cfg.n_traces * cfg.n_window:
        raise ValueError("trace must hold n_traces * W samples")
    _check(lib().afm_pso_shard_eval(C.byref(bounds), C.byref(swarm), _ptr(trace),
                                    C.byref(cfg), int(first_particle), _ptr(st["x"]),
                                    _ptr(st["J"]), _ptr(st["pbest"]),
                                    _ptr(st["pbestJ"]), _ptr(st["cand"]),
                                    _stream_ptr(stream)))
    return st["cand"]


def afm_pso_shard_move(bounds, swarm, n_dims, n_traces, seed, iteration, do_move,
                       first_particle, gathered, st, rank=0, swarm_particles=None,
                       stream=None):
    """Global best from the gathered candidates [n_ranks][n_traces][R], then the
    Eq. 8 move of the shard.  rank: this process's block in `gathered`;
    swarm_particles: particles per trace of the whole swarm (default: the shard's)."""
    gathered = _dev_f64(gathered, "gathered")
    R = shard_row_doubles(n_dims, swarm.topology)
    n_ranks = gathered.numel() // (n_traces * R)
    if n_ranks * n_traces * R != gathered.numel():
        raise ValueError("gathered must be [n_ranks][n_traces][%d]" % R)
    total = swarm.n_particles if swarm_particles is None else int(swarm_particles)
    _check(lib().afm_pso_shard_move(C.byref(bounds), C.byref(swarm), n_dims, n_traces,
                                    int(seed), int(iteration), int(bool(do_move)),
                                    int(first_particle), _ptr(gathered), n_ranks,
                                    int(rank), total,
                                    _ptr(st["x"]), _ptr(st["v"]), _ptr(st["pbest"]),
                                    _ptr(st["pbestJ"]),
                                    _ptr(st["gbest"]), _ptr(st["gbestJ"]),
                                    _ptr(st["theta_star"]), _ptr(st["J_star"]),
                                    _stream_ptr(stream)))
    return st


def beam_cfg_from(wl, **over):
    """afm_beam_cfg of a workloads.beam_workload() dictionary."""
    b = wl["beam"]
    kw = dict(L=b["L"], E=b["E"], I=b["I"], mu=b["mu"], Q=b["Q"], f_drive=b["f_drive"],
              A_base=b["A_base"], A_ref=b["A_ref"], z_c=b["z_c"], R=b["R"], a0=b["a0"],
              law=wl["law"], n_params=wl["n_params"], n_modes=b["n_modes"],
              n_points=b["n_points"], steps_per_cycle=wl["steps_per_cycle"],
              n_cycles=wl["n_cycles"], n_skip_cycles=wl["n_skip_cycles"],
              n_traces=wl["n_traces"])
    kw.update(over)
    return BeamCfg(**kw)


def afm_beam_modes(cfg, stream=None):
    """dict of host arrays [n_modes]: beta_L, omega, phi_L, participation, compliance."""
    m = cfg.n_modes
    out = {k: np.empty(m) for k in ("beta_L", "omega", "phi_L", "participation",
                                    "compliance")}
    _check(lib().afm_beam_modes(C.byref(cfg), _hptr(out["beta_L"]), _hptr(out["omega"]),
                                _hptr(out["phi_L"]), _hptr(out["participation"]),
                                _hptr(out["compliance"]), _stream_ptr(stream)))
    return out


def afm_beam_forward_batch(params, trace, cfg, bounds=None, misfit=None, stream=None):
    torch = _torch()
    params = _dev_f64(params, "params")
    trace = _dev_f64(trace, "trace")
    P = params.shape[0]
    if trace.numel() != cfg.n_traces * cfg.n_window:
        raise ValueError("trace must hold n_traces * W samples")
    if misfit is None:
        misfit = torch.empty(P, dtype=torch.float64, device=params.device)
    _check(lib().afm_beam_forward_batch(_ptr(params), P, _ptr(trace), C.byref(cfg),
                                        None if bounds is None else C.byref(bounds),
                                        _ptr(misfit), _stream_ptr(stream)))
    return misfit


def afm_beam_pso_invert(bounds, swarm, seed, trace, cfg, dump=False, hist=False,
                        stream=None):
    torch = _torch()
    trace = _dev_f64(trace, "trace")
    if trace.numel() != cfg.n_traces * cfg.n_window:
        raise ValueError("trace must hold n_traces * W samples")
    D, T = cfg.n_params, cfg.n_traces
    PT = swarm.n_particles * T
    th = np.empty((T, D), dtype=np.float64)
    Js = np.empty(T, dtype=np.float64)
    dmp = (torch.empty((swarm.n_iters, PT, 3 * D + 2), dtype=torch.float64,
                       device=trace.device) if dump else None)
    gh = (torch.empty((swarm.n_iters, T, D + 1), dtype=torch.float64,
                      device=trace.device) if hist else None)
    done = C.c_int32(0)
    _check(lib().afm_beam_pso_invert(C.byref(bounds), C.byref(swarm), int(seed),
                                     _ptr(trace), C.byref(cfg), _hptr(th), _hptr(Js),
                                     _ptr(dmp), _ptr(gh), C.byref(done),
                                     _stream_ptr(stream)))
    return dict(theta_star=th, J_star=Js, n_iters_done=done.value, dump=dmp,
                gbest_hist=gh)


def afm_beam_trajectory(theta, cfg, stream=None):
    """(tip_u[N+1], tip_v[N+1]) of one particle, as numpy arrays."""
    torch = _torch()
    theta = _host_f64(theta)
    N = cfg.n_steps
    u = torch.empty(N + 1, dtype=torch.float64, device="cuda")
    v = torch.empty(N + 1, dtype=torch.float64, device="cuda")
    _check(lib().afm_beam_trajectory(_hptr(theta), C.byref(cfg), _ptr(u), _ptr(v),
                                     _stream_ptr(stream)))
    torch.cuda.synchronize()
    return u.cpu().numpy(), v.cpu().numpy()


def afm_philox4x32_10(ctr, key, stream=None):
    """ctr [n][4] uint32 (numpy) -> [n][4] uint32 (numpy), computed on the device."""
    torch = _torch()
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    n = ctr.shape[0]
    d_in = torch.as_tensor(ctr.view(np.int32), device="cuda")
    d_out = torch.empty_like(d_in)
    k = (C.c_uint32 * 2)(int(key[0]), int(key[1]))
    _check(lib().afm_philox4x32_10(_ptr(d_in), n, k, _ptr(d_out), _stream_ptr(stream)))
    return d_out.cpu().numpy().view(np.uint32)


def afm_trajectory(theta, cfg, z0, v0, stream=None):
    """(zs[N+1], vs[N+1]) of one particle, as numpy arrays."""
    torch = _torch()
    theta = _host_f64(theta)
    N = cfg.n_steps
    zs = torch.empty(N + 1, dtype=torch.float64, device="cuda")
    vs = torch.empty(N + 1, dtype=torch.float64, device="cuda")
    _check(lib().afm_trajectory(_hptr(theta), C.byref(cfg), float(z0), float(v0),
                                _ptr(zs), _ptr(vs), _stream_ptr(stream)))
    torch.cuda.synchronize()
    return zs.cpu().numpy(), vs.cpu().numpy()


def afm_fma_peak(precision, seconds=0.2, stream=None):
    """Measured register-only FMA rate in TFLOP/s (2 flops per FMA)."""
    out = C.c_double(0.0)
    _check(lib().afm_fma_peak(int(precision), float(seconds), C.byref(out),
                              _stream_ptr(stream)))
    return out.value


def afm_launch_count():
    return int(lib().afm_launch_count())


def afm_reset_launch_count():
    lib().afm_reset_launch_count()


def afm_set_option(name, value):
    _check(lib().afm_set_option(name.encode(), int(value)))


def afm_last_error():
    return lib().afm_last_error().decode("utf-8", "replace")


def afm_version():
    return lib().afm_version().decode()


def afm_shutdown():
    lib().afm_shutdown()
