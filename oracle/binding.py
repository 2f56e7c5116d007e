"""ctypes view of oracle/libafm_oracle*.so (TEST INFRASTRUCTURE, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It imports nothing from the
CUDA package.  Argument marshalling only; all arithmetic is in afm_oracle.c.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))

LAW_NONE, LAW_DMT, LAW_DMT_VISC, LAW_LJ_EXP, LAW_HOOKE, LAW_KELVIN_VOIGT = 0, 1, 2, 3, 4, 5


class Model(C.Structure):
    _fields_ = [("k", C.c_double), ("f0", C.c_double), ("Q", C.c_double),
                ("f_drive", C.c_double), ("A0", C.c_double),
                ("z_c", C.c_double), ("R", C.c_double), ("a0", C.c_double),
                ("law", C.c_int32), ("n_theta", C.c_int32), ("S", C.c_int32),
                ("n_cycles", C.c_int32), ("n_skip", C.c_int32),
                ("pad_", C.c_int32)]


class Consts(C.Structure):
    _fields_ = [("w0", C.c_double), ("w", C.c_double), ("m", C.c_double),
                ("c", C.c_double), ("r", C.c_double), ("F0", C.c_double),
                ("dt", C.c_double), ("N", C.c_int64), ("W", C.c_int64)]


class Box(C.Structure):
    _fields_ = [("lo", C.c_double * 4), ("hi", C.c_double * 4),
                ("log10", C.c_int32 * 4)]


class Swarm(C.Structure):
    _fields_ = [("n_particles", C.c_int32), ("n_iters", C.c_int32),
                ("w", C.c_double), ("c1", C.c_double), ("c2", C.c_double),
                ("j_target", C.c_double), ("topology", C.c_int32),
                ("async_chunk", C.c_int32)]


# cost callback of orc_pso_core: double eval(ctx, theta[D], trace_s[W])
EVAL_FN = C.CFUNCTYPE(C.c_double, C.c_void_p, C.POINTER(C.c_double),
                      C.POINTER(C.c_double))


class Beam(C.Structure):
    _fields_ = [("L", C.c_double), ("E", C.c_double), ("I", C.c_double),
                ("mu", C.c_double), ("Q", C.c_double), ("f_drive", C.c_double),
                ("A_base", C.c_double), ("A_ref", C.c_double), ("z_c", C.c_double),
                ("R", C.c_double), ("a0", C.c_double), ("law", C.c_int32),
                ("n_theta", C.c_int32), ("n_modes", C.c_int32),
                ("n_points", C.c_int32), ("S", C.c_int32), ("n_cycles", C.c_int32),
                ("n_skip", C.c_int32), ("literal_eq7", C.c_int32)]


class BeamModes(C.Structure):
    _fields_ = [(n, C.c_double * 8) for n in ("bL", "omega", "phiL", "norm", "intphi",
                                              "gain", "fgain")] + \
               [("w", C.c_double), ("dt", C.c_double), ("N", C.c_int64), ("W", C.c_int64)]


_dp = C.POINTER(C.c_double)
_libs = {}


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def lib(openmp=False):
    """Load (building if stale) the single-threaded or the OpenMP oracle."""
    key = bool(openmp)
    if key not in _libs:
        paths = _build.build()
        L = C.CDLL(paths[1] if openmp else paths[0])
        L.orc_constants.argtypes = [C.POINTER(Model), C.POINTER(Consts)]
        L.orc_constants.restype = None
        L.orc_force.argtypes = [C.POINTER(Model), _dp, C.c_double, C.c_double]
        L.orc_force.restype = C.c_double
        L.orc_rhs.argtypes = [C.POINTER(Model), _dp, C.c_double, C.c_double,
                              C.c_double, _dp, _dp]
        L.orc_rhs.restype = None
        L.orc_rk4_step.argtypes = [C.POINTER(Model), _dp, C.c_double,
                                   C.c_double, _dp, _dp]
        L.orc_rk4_step.restype = None
        L.orc_integrate.argtypes = [C.POINTER(Model), _dp, C.c_double,
                                    C.c_double, _dp, _dp]
        L.orc_integrate.restype = C.c_int
        L.orc_window.argtypes = [C.POINTER(Model), _dp, C.c_double, C.c_double,
                                 _dp]
        L.orc_window.restype = C.c_int
        L.orc_misfit.argtypes = [C.POINTER(Model), _dp, C.c_double, C.c_double,
                                 _dp]
        L.orc_misfit.restype = C.c_double
        L.orc_forward_batch.argtypes = [C.POINTER(Model), _dp, C.c_int64, _dp,
                                        C.c_int32, _dp, C.c_double, C.c_double,
                                        _dp]
        L.orc_forward_batch.restype = None
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32),
                                        C.POINTER(C.c_uint32),
                                        C.POINTER(C.c_uint32)]
        L.orc_philox4x32_10.restype = None
        L.orc_pso_uniforms.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32,
                                       C.c_uint32, C.c_int32, _dp, _dp]
        L.orc_pso_uniforms.restype = None
        L.orc_theta_of_x.argtypes = [C.POINTER(Box), C.c_int32, _dp, _dp]
        L.orc_theta_of_x.restype = None
        L.orc_pso_invert.argtypes = [C.POINTER(Model), C.POINTER(Box),
                                     C.POINTER(Swarm), C.c_uint64, _dp,
                                     C.c_int32, C.c_double, C.c_double, _dp,
                                     _dp, _dp, _dp]
        L.orc_pso_invert.restype = C.c_int32
        L.orc_pso_core.argtypes = [EVAL_FN, C.c_void_p, C.c_int64, C.c_int32,
                                   C.POINTER(Box), C.POINTER(Swarm), C.c_uint64,
                                   _dp, C.c_int32, _dp, _dp, _dp, _dp]
        L.orc_pso_core.restype = C.c_int32
        L.orc_beam_setup.argtypes = [C.POINTER(Beam), C.POINTER(BeamModes)]
        L.orc_beam_setup.restype = None
        L.orc_beam_shape.argtypes = [C.POINTER(Beam), C.POINTER(BeamModes), C.c_int32,
                                     C.c_double]
        L.orc_beam_shape.restype = C.c_double
        L.orc_beam_integrate.argtypes = [C.POINTER(Beam), _dp, _dp, _dp, _dp, _dp]
        L.orc_beam_integrate.restype = C.c_int
        L.orc_beam_window.argtypes = [C.POINTER(Beam), _dp, _dp]
        L.orc_beam_window.restype = C.c_int
        L.orc_beam_misfit.argtypes = [C.POINTER(Beam), _dp, _dp]
        L.orc_beam_misfit.restype = C.c_double
        L.orc_beam_forward_batch.argtypes = [C.POINTER(Beam), _dp, C.c_int64, _dp,
                                             C.c_int32, _dp]
        L.orc_beam_forward_batch.restype = None
        L.orc_beam_pso_invert.argtypes = [C.POINTER(Beam), C.POINTER(Box),
                                          C.POINTER(Swarm), C.c_uint64, _dp, C.c_int32,
                                          _dp, _dp, _dp, _dp]
        L.orc_beam_pso_invert.restype = C.c_int32
        _libs[key] = L
    return _libs[key]


# ---- marshalling from the workload dictionaries (inputs module) ------------

def model_from(wl, law=None, n_cycles=None, S=None, n_skip=None):
    """Build a Model from a workload dict (see paper_1109_0334_b200.workloads)."""
    c = wl["cantilever"]
    return Model(k=c["k"], f0=c["f0"], Q=c["Q"], f_drive=c["f_drive"],
                 A0=c["A0"], z_c=c["z_c"], R=c["R"], a0=c["a0"],
                 law=wl["law"] if law is None else law,
                 n_theta=wl["n_params"],
                 S=wl["steps_per_cycle"] if S is None else S,
                 n_cycles=wl["n_cycles"] if n_cycles is None else n_cycles,
                 n_skip=wl["n_skip_cycles"] if n_skip is None else n_skip,
                 pad_=0)


def box_from(wl):
    b = Box()
    for j in range(wl["n_params"]):
        b.lo[j] = wl["bounds"]["lo"][j]
        b.hi[j] = wl["bounds"]["hi"][j]
        b.log10[j] = int(wl["bounds"]["log10"][j])
    return b


def swarm_from(wl, n_particles=None, n_iters=None, topology=None, j_target=0.0,
               async_chunk=0):
    s = wl["swarm"]
    return Swarm(n_particles=s["n_particles"] if n_particles is None else n_particles,
                 n_iters=s["n_iters"] if n_iters is None else n_iters,
                 w=s["w"], c1=s["c1"], c2=s["c2"], j_target=j_target,
                 topology=s.get("topology", 0) if topology is None else topology,
                 async_chunk=async_chunk)


# ---- thin calls -------------------------------------------------------------

def constants(M):
    c = Consts()
    lib().orc_constants(C.byref(M), C.byref(c))
    return c


def force(M, theta, d, v=0.0):
    th = _f64(theta)
    return lib().orc_force(C.byref(M), _ptr(th), float(d), float(v))


def rhs(M, theta, t, z, v):
    th = _f64(theta)
    dz, dv = C.c_double(), C.c_double()
    lib().orc_rhs(C.byref(M), _ptr(th), t, z, v, C.byref(dz), C.byref(dv))
    return dz.value, dv.value


def rk4_step(M, theta, t, dt, z, v):
    th = _f64(theta)
    zz, vv = C.c_double(z), C.c_double(v)
    lib().orc_rk4_step(C.byref(M), _ptr(th), t, dt, C.byref(zz), C.byref(vv))
    return zz.value, vv.value


def integrate(M, theta, z0, v0):
    """Full trajectory: (diverged, zs[N+1], vs[N+1])."""
    th = _f64(theta)
    N = constants(M).N
    zs = np.empty(N + 1)
    vs = np.empty(N + 1)
    bad = lib().orc_integrate(C.byref(M), _ptr(th), z0, v0, _ptr(zs), _ptr(vs))
    return bad, zs, vs


def window(M, theta, z0, v0):
    th = _f64(theta)
    w = np.empty(constants(M).W)
    bad = lib().orc_window(C.byref(M), _ptr(th), z0, v0, _ptr(w))
    return bad, w


def misfit(M, theta, z0, v0, trace):
    th, tr = _f64(theta), _f64(trace)
    assert tr.size == constants(M).W
    return lib().orc_misfit(C.byref(M), _ptr(th), z0, v0, _ptr(tr))


def forward_batch(M, params, trace, z0v0=None, z0=0.0, v0=0.0, n_traces=1,
                  openmp=False):
    params = _f64(params)
    P = params.shape[0]
    assert params.shape[1] == M.n_theta and P % n_traces == 0
    tr = _f64(trace)
    assert tr.size == n_traces * constants(M).W
    zv = None if z0v0 is None else _f64(z0v0)
    out = np.empty(P)
    lib(openmp).orc_forward_batch(C.byref(M), _ptr(params), P, _ptr(tr),
                                  n_traces, _ptr(zv), z0, v0, _ptr(out))
    return out


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def pso_uniforms(seed, gp, it, purpose, D):
    a = np.zeros(4)
    b = np.zeros(4)
    lib().orc_pso_uniforms(seed, gp, it, purpose, D, _ptr(a), _ptr(b))
    return a[:D].copy(), b[:D].copy()


def theta_of_x(B, D, x):
    x = _f64(x)
    th = np.empty(D)
    lib().orc_theta_of_x(C.byref(B), D, _ptr(x), _ptr(th))
    return th


def pso_invert(M, B, Sw, seed, trace, z0, v0, n_traces=1, dump=False,
               openmp=False):
    """Returns dict(theta_star [T][D], J_star [T], dump [it][PT][3D+2] or None,
    gbest_hist [it][T][D+1], n_iters_done); rows of unrun batches are NaN."""
    D = M.n_theta
    PT = Sw.n_particles * n_traces
    tr = _f64(trace)
    assert tr.size == n_traces * constants(M).W
    th = np.empty((n_traces, D))
    Js = np.empty(n_traces)
    dmp = np.empty((Sw.n_iters, PT, 3 * D + 2)) if dump else None
    gh = np.empty((Sw.n_iters, n_traces, D + 1))
    done = lib(openmp).orc_pso_invert(C.byref(M), C.byref(B), C.byref(Sw), seed,
                                      _ptr(tr), n_traces, z0, v0, _ptr(th), _ptr(Js),
                                      _ptr(dmp), _ptr(gh))
    return dict(theta_star=th, J_star=Js, dump=dmp, gbest_hist=gh, n_iters_done=int(done))


def pso_core(cost, D, B, Sw, seed, trace, n_traces=1):
    """The oracle's PSO loop around a PYTHON cost function cost(theta[D], U_s[W]) ->
    float (the pins of the cutoff and chunk rules use hand-made costs).  trace is
    [n_traces][W].  Single-threaded.  Same outputs as pso_invert, dump included."""
    tr = _f64(trace).reshape(n_traces, -1)
    Wn = tr.shape[1]
    PT = Sw.n_particles * n_traces

    def _cb(_ctx, th, U):
        return float(cost(np.array([th[j] for j in range(D)]),
                          np.ctypeslib.as_array(U, shape=(Wn,))))

    th = np.empty((n_traces, D))
    Js = np.empty(n_traces)
    dmp = np.empty((Sw.n_iters, PT, 3 * D + 2))
    gh = np.empty((Sw.n_iters, n_traces, D + 1))
    done = lib().orc_pso_core(EVAL_FN(_cb), None, Wn, D, C.byref(B), C.byref(Sw), seed,
                              _ptr(tr), n_traces, _ptr(th), _ptr(Js), _ptr(dmp), _ptr(gh))
    return dict(theta_star=th, J_star=Js, dump=dmp, gbest_hist=gh, n_iters_done=int(done))


# ---- the multi-mode Euler-Bernoulli beam (afm_oracle_beam.h) ------------------

def beam_from(wl, **over):
    b = wl["beam"]
    kw = dict(L=b["L"], E=b["E"], I=b["I"], mu=b["mu"], Q=b["Q"], f_drive=b["f_drive"],
              A_base=b["A_base"], A_ref=b["A_ref"], z_c=b["z_c"], R=b["R"], a0=b["a0"],
              law=wl["law"], n_theta=wl["n_params"], n_modes=b["n_modes"],
              n_points=b["n_points"], S=wl["steps_per_cycle"], n_cycles=wl["n_cycles"],
              n_skip=wl["n_skip_cycles"], literal_eq7=0)
    kw.update(over)
    return Beam(**kw)


def beam_setup(B):
    mo = BeamModes()
    lib().orc_beam_setup(C.byref(B), C.byref(mo))
    return mo


def beam_shape(B, mo, i, x):
    return lib().orc_beam_shape(C.byref(B), C.byref(mo), int(i), float(x))


def beam_integrate(B, theta, eta0=None, want_eta=False):
    """(diverged, tip_u[N+1], tip_v[N+1], eta[N+1][2m] or None)."""
    th = _f64(theta)
    mo = beam_setup(B)
    u, v = np.empty(mo.N + 1), np.empty(mo.N + 1)
    eta = np.empty((mo.N + 1, 2 * B.n_modes)) if want_eta else None
    e0 = None if eta0 is None else _f64(eta0)
    bad = lib().orc_beam_integrate(C.byref(B), _ptr(th), _ptr(e0), _ptr(u), _ptr(v),
                                   _ptr(eta))
    return bad, u, v, eta


def beam_window(B, theta):
    th = _f64(theta)
    w = np.empty(beam_setup(B).W)
    bad = lib().orc_beam_window(C.byref(B), _ptr(th), _ptr(w))
    return bad, w


def beam_forward_batch(B, params, trace, n_traces=1, openmp=False):
    params = _f64(params)
    tr = _f64(trace)
    assert tr.size == n_traces * beam_setup(B).W
    out = np.empty(params.shape[0])
    lib(openmp).orc_beam_forward_batch(C.byref(B), _ptr(params), params.shape[0],
                                       _ptr(tr), n_traces, _ptr(out))
    return out


def beam_pso_invert(B, Bx, Sw, seed, trace, n_traces=1, dump=False, openmp=False):
    D = B.n_theta
    PT = Sw.n_particles * n_traces
    tr = _f64(trace)
    th = np.empty((n_traces, D))
    Js = np.empty(n_traces)
    dmp = np.empty((Sw.n_iters, PT, 3 * D + 2)) if dump else None
    gh = np.empty((Sw.n_iters, n_traces, D + 1))
    done = lib(openmp).orc_beam_pso_invert(C.byref(B), C.byref(Bx), C.byref(Sw), seed,
                                           _ptr(tr), n_traces, _ptr(th), _ptr(Js),
                                           _ptr(dmp), _ptr(gh))
    return dict(theta_star=th, J_star=Js, dump=dmp, gbest_hist=gh, n_iters_done=int(done))
