"""Host logic of paper_1109_0334_b200/sharded.py at world_size 2 over gloo (CPU).

sharded.py holds no arithmetic: it partitions index ranges, all-gathers one
candidate row per rank and calls three compute entry points.  Here those entry
points are a TEST DOUBLE built on the CPU oracle's primitives (its Philox
uniforms, its coordinate map, its forward batch), so that what is checked is
exactly the sharding logic: the slices, the global particle offsets fed to the
random streams, the exchange, the lowest-global-index tie-break -- a 2-rank run
must reproduce the oracle's single-process inversion bit for bit.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm
from paper_1109_0334_b200.sharded import ShardedSwarm, split_even
from parity_helpers import oracle_trace


class _Cfg:            # the fields of afm.Cfg that sharded.py touches
    def __init__(self, wl):
        self.n_params, self.n_traces = wl["n_params"], wl["n_traces"]
        self.n_window = wl["n_window"]


class _Swarm:
    def __init__(self, wl):
        s = wl["swarm"]
        self.n_particles, self.n_iters = s["n_particles"], s["n_iters"]
        self.w, self.c1, self.c2 = s["w"], s["c1"], s["c2"]
        self.topology = s.get("topology", 0)


class OracleDouble:
    """init / eval / move with the oracle's primitives on CPU tensors (readings
    R10, R11 of DESIGN.md restated; test infrastructure only)."""

    def __init__(self, wl):
        self.wl = wl
        self.M = orc.model_from(wl)
        self.B = orc.box_from(wl)
        b = wl["bounds"]
        self.lo, self.hi = np.array(b["lo"]), np.array(b["hi"])

    def init(self, bounds, swarm, D, T, seed, first):
        PT = swarm.n_particles * T
        x, v = np.empty((PT, D)), np.empty((PT, D))
        for i in range(PT):
            a, b = orc.pso_uniforms(seed, first + i, 0, 0, D)
            span = self.hi - self.lo
            x[i] = self.lo + a * span
            v[i] = 0.5 * ((self.lo + b * span) - x[i])
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a))
        return dict(x=t(x), v=t(v), pbest=t(x.copy()), pbestJ=t(np.full(PT, np.inf)),
                    gbest=t(x[::swarm.n_particles].copy()), gbestJ=t(np.full(T, np.inf)),
                    J=t(np.empty(PT)),
                    cand=t(np.empty((T, 3 * D + 4 if swarm.topology == 1 else D + 2))),
                    theta_star=t(np.empty((T, D))), J_star=t(np.empty(T)))

    def eval(self, bounds, swarm, trace, cfg, first, st):
        D, T, per = cfg.n_params, cfg.n_traces, swarm.n_particles
        x = st["x"].numpy()
        th = np.stack([orc.theta_of_x(self.B, D, xi) for xi in x])
        J = orc.forward_batch(self.M, th, trace.numpy(), z0=self.wl["z0"],
                              v0=self.wl["v0"], n_traces=T)
        st["J"].copy_(torch.from_numpy(J))
        pb, pbJ = st["pbest"].numpy(), st["pbestJ"].numpy()
        better = J < pbJ
        pbJ[better] = J[better]
        pb[better] = x[better]
        cand = st["cand"].numpy()
        for s in range(T):
            seg = pbJ[s * per:(s + 1) * per]
            i = int(np.argmin(seg)) if np.isfinite(seg).any() else 0   # first minimum
            if not np.isfinite(seg).any():
                cand[s, 0], cand[s, 1] = np.inf, float(2 ** 62)
                cand[s, 2:D + 2] = pb[s * per]
            else:
                cand[s, 0], cand[s, 1] = seg[i], float(first + s * per + i)
                cand[s, 2:D + 2] = pb[s * per + i]
            if swarm.topology == 1:            # edge particles' personal bests ride along
                for k, q in enumerate((s * per, s * per + per - 1)):
                    e = D + 2 + k * (D + 1)
                    cand[s, e] = pbJ[q]
                    cand[s, e + 1:e + 1 + D] = pb[q]
        return st["cand"]

    def move(self, bounds, swarm, D, T, seed, it, do_move, first, gathered, st, rank=0,
             swarm_particles=None):
        R = 3 * D + 4 if swarm.topology == 1 else D + 2
        g = gathered.numpy().reshape(-1, T, R)
        gb, gbJ = st["gbest"].numpy(), st["gbestJ"].numpy()
        for s in range(T):
            order = sorted(range(g.shape[0]), key=lambda r: (g[r, s, 0], g[r, s, 1]))
            r = order[0]
            if g[r, s, 0] < gbJ[s]:
                gbJ[s] = g[r, s, 0]
                gb[s] = g[r, s, 2:D + 2]
            st["theta_star"].numpy()[s] = orc.theta_of_x(self.B, D, gb[s])
            st["J_star"].numpy()[s] = gbJ[s]
        if not do_move:
            return st
        x, v, pb = st["x"].numpy(), st["v"].numpy(), st["pbest"].numpy()
        pbJ = st["pbestJ"].numpy()
        per = swarm.n_particles
        total = per if swarm_particles is None else swarm_particles
        off = first % total
        n_ranks = g.shape[0]
        for i in range(x.shape[0]):
            r1, r2 = orc.pso_uniforms(seed, first + i, it, 1, D)
            s = i // per
            social = gb[s]
            if swarm.topology == 1:
                # ring of three over in-swarm indices; a neighbour outside this shard
                # is the last particle of the rank before / the first of the rank after
                gi = off + (i - s * per)

                def best_of(c):
                    lc = c - off
                    if 0 <= lc < per:
                        return pbJ[s * per + lc], pb[s * per + lc]
                    if c == (gi - 1) % total:
                        row = g[(rank - 1) % n_ranks, s, D + 2 + (D + 1):]
                    else:
                        row = g[(rank + 1) % n_ranks, s, D + 2:D + 2 + (D + 1)]
                    return row[0], row[1:1 + D]
                cands = [(gi - 1) % total, gi, (gi + 1) % total]
                best = min(cands, key=lambda c: (best_of(c)[0], c))
                social = best_of(best)[1]
            vn = (swarm.w * v[i] + (swarm.c1 * r1) * (pb[i] - x[i])) + \
                 (swarm.c2 * r2) * (social - x[i])
            xn = x[i] + vn
            low, high = xn < self.lo, xn > self.hi
            xn = np.where(low, self.lo, np.where(high, self.hi, xn))
            vn = np.where(low | high, 0.0, vn)
            x[i], v[i] = xn, vn
        return st


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, wl, trace, shard, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        sw = ShardedSwarm(None, _Swarm(wl), wl["pso_seed"], torch.from_numpy(trace),
                          _Cfg(wl), shard=shard, backend=OracleDouble(wl))
        th, Js = sw.run()
        out[rank] = (th.numpy().copy(), Js.numpy().copy(), sw.first,
                     sw.swarm.n_particles, sw.n_traces)
    finally:
        dist.destroy_process_group()


def _run(world, wl, trace, shard):
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), wl, trace, shard, out), nprocs=world,
             join=True)
    return [out[r] for r in range(world)]


def test_split_even_covers_everything():
    for n, w in ((10, 3), (64, 2), (7, 7), (5, 2), (256, 8)):
        parts = [split_even(n, w, r) for r in range(w)]
        assert parts[0][0] == 0 and sum(c for _, c in parts) == n
        for (f0, c0), (f1, _) in zip(parts, parts[1:]):
            assert f1 == f0 + c0
        assert max(c for _, c in parts) - min(c for _, c in parts) <= 1


def test_particle_sharding_world2_replays_the_single_process_oracle():
    """One swarm of 41 particles (ragged split 21 + 20) over 2 gloo ranks."""
    wl = wlm.scaled(wlm.config(0), n_cycles=6, n_skip_cycles=3, n_particles=41,
                    n_iters=5)
    trace = oracle_trace(wl)
    o = orc.pso_invert(orc.model_from(wl), orc.box_from(wl), orc.swarm_from(wl),
                       wl["pso_seed"], trace, wl["z0"], wl["v0"])
    res = _run(2, wl, trace, "particles")
    assert (res[0][2], res[0][3]) == (0, 21) and (res[1][2], res[1][3]) == (21, 20)
    for th, Js, *_ in res:                       # identical on both ranks
        assert np.array_equal(th, o["theta_star"])
        assert np.array_equal(Js, o["J_star"])


def test_ring_topology_sharded_over_2_ranks_replays_the_oracle():
    """topology = 1 on a swarm of 23 particles split 12 + 11: the edge particles'
    personal bests travel in the all-gathered rows (3 D + 4 doubles per rank), the
    ring wraps from the last rank to the first; and with whole traces per rank."""
    wl = wlm.scaled(wlm.config(0), n_cycles=6, n_skip_cycles=3, n_particles=23,
                    n_iters=6)
    wl["swarm"]["topology"] = 1
    trace = oracle_trace(wl)
    o = orc.pso_invert(orc.model_from(wl), orc.box_from(wl), orc.swarm_from(wl),
                       wl["pso_seed"], trace, wl["z0"], wl["v0"])
    ref = orc.pso_invert(orc.model_from(wl), orc.box_from(wl),
                         orc.swarm_from(wl, topology=0), wl["pso_seed"], trace, wl["z0"],
                         wl["v0"])
    assert not np.array_equal(o["theta_star"], ref["theta_star"])
    for th, Js, *_ in _run(2, wl, trace, "particles"):
        assert np.array_equal(th, o["theta_star"])
        assert np.array_equal(Js, o["J_star"])
    w4 = wlm.scaled(wlm.config(4), n_cycles=4, n_skip_cycles=2, n_traces=3,
                    n_particles=9, n_iters=4, steps_per_cycle=64)
    w4["swarm"]["topology"] = 1
    tr4 = oracle_trace(w4, truths=wlm.pixel_truths(w4))
    o4 = orc.pso_invert(orc.model_from(w4), orc.box_from(w4), orc.swarm_from(w4),
                        w4["pso_seed"], tr4, w4["z0"], w4["v0"], n_traces=3)
    for th, Js, *_ in _run(2, w4, tr4, "traces"):
        assert np.array_equal(th, o4["theta_star"])
        assert np.array_equal(Js, o4["J_star"])


def test_trace_sharding_world2_needs_no_exchange_and_matches():
    """Three pixels over 2 ranks (2 + 1), each pixel its own swarm."""
    wl = wlm.scaled(wlm.config(4), n_cycles=4, n_skip_cycles=2, n_traces=3,
                    n_particles=12, n_iters=4, steps_per_cycle=64)
    trace = oracle_trace(wl, truths=wlm.pixel_truths(wl))
    o = orc.pso_invert(orc.model_from(wl), orc.box_from(wl), orc.swarm_from(wl),
                       wl["pso_seed"], trace, wl["z0"], wl["v0"], n_traces=3)
    res = _run(2, wl, trace, "traces")
    assert res[0][4] == 2 and res[1][4] == 1
    assert res[1][2] == 2 * 12                   # first global particle of rank 1
    for th, Js, *_ in res:
        assert np.array_equal(th, o["theta_star"])
        assert np.array_equal(Js, o["J_star"])


def test_default_backend_fails_loudly_without_the_library(monkeypatch):
    """No CPU fallback: without libafm_b200.so the default backend raises."""
    from paper_1109_0334_b200 import afm, sharded
    monkeypatch.setattr(afm, "_lib", None)
    monkeypatch.setattr(afm, "LIB_PATH", "/nonexistent/libafm_b200.so")
    with pytest.raises(ImportError):
        sharded.CudaBackend()
