"""GPU: the shard entry points (afm_pso_shard_init / _eval / _move) replay the
single-process afm_pso_invert bit for bit when the shards of one swarm are
stepped side by side on ONE device (no process group: the exchange is a
torch.cat of the candidate rows -- the multi-process exchange itself is covered
on CPU by tests/test_sharded_gloo.py)."""
import copy

import numpy as np
import pytest

from paper_1109_0334_b200 import workloads as wlm
from parity_helpers import oracle_trace

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def afm():
    import torch
    assert torch.cuda.is_available()
    from paper_1109_0334_b200 import afm as m
    m.lib()
    return m


def _shards_side_by_side(afm, wl, trace, cuts, precision=0):
    """Step the particle shards [cuts[i], cuts[i+1]) of a one-trace swarm."""
    import torch
    D = wl["n_params"]
    total = cuts[-1]
    cfg = afm.cfg_from(wl, precision=precision)
    b = afm.bounds_from(wl)
    t = torch.as_tensor(trace, device="cuda")
    sws, sts = [], []
    for lo, hi in zip(cuts, cuts[1:]):
        sw = afm.swarm_from(wl, n_particles=hi - lo)
        sws.append(sw)
        sts.append(afm.afm_pso_shard_init(b, sw, D, 1, wl["pso_seed"], lo))
    for st in sts[1:]:
        st["gbest"].copy_(sts[0]["gbest"])
    n_it = wl["swarm"]["n_iters"]
    xs = []
    for it in range(n_it):
        xs.append(torch.cat([st["x"] for st in sts]).cpu().numpy())
        cands = [afm.afm_pso_shard_eval(b, sw, t, cfg, lo, st).clone()
                 for sw, st, lo in zip(sws, sts, cuts)]
        gathered = torch.stack(cands)            # [n_ranks][1][R]
        for r, (sw, st, lo) in enumerate(zip(sws, sts, cuts)):
            afm.afm_pso_shard_move(b, sw, D, 1, wl["pso_seed"], it, it + 1 < n_it, lo,
                                   gathered, st, rank=r, swarm_particles=total)
    torch.cuda.synchronize()
    return sts, np.stack(xs)


def test_particle_shards_replay_the_unsharded_swarm(afm):
    import torch
    wl = wlm.scaled(wlm.config(2), n_cycles=10, n_skip_cycles=5, n_particles=100,
                    n_iters=6)
    trace = oracle_trace(wl)
    g = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), wl["pso_seed"],
                           torch.as_tensor(trace, device="cuda"), afm.cfg_from(wl),
                           dump=True)
    D = wl["n_params"]
    dump = g["dump"].cpu().numpy()
    sts, xs = _shards_side_by_side(afm, wl, trace, [0, 53, 77, 100])
    assert np.array_equal(xs, dump[:, :, 0:D])           # every iteration's positions
    for st in sts:                                        # same answer on every shard
        assert np.array_equal(st["theta_star"].cpu().numpy(), g["theta_star"])
        assert np.array_equal(st["J_star"].cpu().numpy(), g["J_star"])
    pbJ = torch.cat([st["pbestJ"] for st in sts]).cpu().numpy()
    assert np.array_equal(pbJ, dump[-1, :, 3 * D + 1])


@pytest.mark.parametrize("cuts", [[0, 53, 77, 100], [0, 1, 99, 100], [0, 100]])
def test_ring_topology_across_particle_shards(afm, cuts):
    """topology = 1 with the swarm cut into shards: the ring neighbours of a shard's
    first and last particle live on the adjacent shards and travel in the candidate
    rows (3 D + 4 doubles); one-particle shards and the wrap from the last shard to
    the first included.  Same swarm as the unsharded ring, bit for bit."""
    import torch
    wl = wlm.scaled(wlm.config(2), n_cycles=10, n_skip_cycles=5, n_particles=100,
                    n_iters=6)
    wl["swarm"]["topology"] = 1
    trace = oracle_trace(wl)
    g = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), wl["pso_seed"],
                           torch.as_tensor(trace, device="cuda"), afm.cfg_from(wl),
                           dump=True)
    D = wl["n_params"]
    dump = g["dump"].cpu().numpy()
    sts, xs = _shards_side_by_side(afm, wl, trace, cuts)
    assert sts[0]["cand"].shape[1] == 3 * D + 4
    assert np.array_equal(xs, dump[:, :, 0:D])
    for st in sts:
        assert np.array_equal(st["theta_star"].cpu().numpy(), g["theta_star"])
        assert np.array_equal(st["J_star"].cpu().numpy(), g["J_star"])
    # and it is the ring, not the global best
    wl0 = wlm.scaled(wl)
    wl0["swarm"]["topology"] = 0
    _, xs0 = _shards_side_by_side(afm, wl0, trace, cuts)
    assert not np.array_equal(xs0[3], xs[3])


def test_particle_shards_fp32_kernel(afm):
    import torch
    wl = wlm.scaled(wlm.config(0), n_cycles=8, n_skip_cycles=4, n_particles=70,
                    n_iters=4)
    trace = oracle_trace(wl)
    g = afm.afm_pso_invert(afm.bounds_from(wl), afm.swarm_from(wl), wl["pso_seed"],
                           torch.as_tensor(trace, device="cuda"),
                           afm.cfg_from(wl, precision=afm.F32))
    sts, _ = _shards_side_by_side(afm, wl, trace, [0, 33, 70], precision=afm.F32)
    assert np.array_equal(sts[0]["theta_star"].cpu().numpy(), g["theta_star"])
    assert np.array_equal(sts[1]["J_star"].cpu().numpy(), g["J_star"])


def test_trace_shards_and_world1_driver(afm):
    """configs[4] shape: 3 pixels.  (a) ShardedSwarm at world size 1 == the
    unsharded call; (b) the pixel shards [0,2) and [2,3) with their global
    particle offsets give the same per-pixel answers."""
    import torch
    from paper_1109_0334_b200.sharded import ShardedSwarm
    wl = wlm.scaled(wlm.config(4), n_cycles=8, n_skip_cycles=4, n_traces=3,
                    n_particles=40, n_iters=5)
    trace = oracle_trace(wl, truths=wlm.pixel_truths(wl))
    t = torch.as_tensor(trace, device="cuda")
    b, sw, cfg = afm.bounds_from(wl), afm.swarm_from(wl), afm.cfg_from(wl)
    g = afm.afm_pso_invert(b, sw, wl["pso_seed"], t, cfg)
    th, Js = ShardedSwarm(b, sw, wl["pso_seed"], t, cfg, shard="traces").run()
    assert np.array_equal(th.numpy(), g["theta_star"])
    assert np.array_equal(Js.numpy(), g["J_star"])
    # the ring topology through the driver, whole traces per shard
    swr = afm.swarm_from(wl, topology=1)
    gr = afm.afm_pso_invert(b, swr, wl["pso_seed"], t, cfg)
    thr, Jsr = ShardedSwarm(b, swr, wl["pso_seed"], t, cfg, shard="traces").run()
    assert np.array_equal(thr.numpy(), gr["theta_star"]) and np.array_equal(Jsr.numpy(), gr["J_star"])
    assert not np.array_equal(gr["J_star"], g["J_star"])
    D, per = wl["n_params"], 40
    for t0, tn in ((0, 2), (2, 1)):
        c = copy.copy(cfg)
        c.n_traces = tn
        st = afm.afm_pso_shard_init(b, sw, D, tn, wl["pso_seed"], t0 * per)
        tt = t[t0:t0 + tn].contiguous()
        for it in range(5):
            cand = afm.afm_pso_shard_eval(b, sw, tt, c, t0 * per, st)
            afm.afm_pso_shard_move(b, sw, D, tn, wl["pso_seed"], it, it < 4, t0 * per,
                                   cand.reshape(1, tn, D + 2), st)
        torch.cuda.synchronize()
        assert np.array_equal(st["theta_star"].cpu().numpy(), g["theta_star"][t0:t0 + tn])
        assert np.array_equal(st["J_star"].cpu().numpy(), g["J_star"][t0:t0 + tn])
