"""Pins for the oracle's Philox generator and PSO loop (Eq. 8).

Philox is pinned by published known-answer vectors.  The PSO is pinned by
invariants, by a hand replay of Eq. 8 on the recorded swarm state, and by
recovery of a known ground truth from a noise-free trace on a tiny swarm
(north_star).  The bound rule, the update order and the tie-break are design
readings (R10) pinned on a closed form and on scripted ties in
tests/test_oracle_pso_rules.py; the v0 rule and the counter layout (R10/R11) are
"parity unpinned" beyond oracle = GPU.
"""
import math
import os

import numpy as np
import pytest

from oracle import binding as orc
from paper_1109_0334_b200 import workloads as wlm

KAT = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers():
    n = 0
    for line in open(KAT):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert orc.philox4x32_10(w[0:4], w[4:6]) == w[6:10], line
        n += 1
    assert n == 3


def test_pso_uniform_layout_and_range():
    """counter = (particle, iteration, block + 16*purpose, particle>>32), key = seed;
    words (a0, b0, a1, b1) per block of two dimensions; u = (word >> 8) * 2^-24."""
    seed, gp, it = 0x0123456789ABCDEF, 77, 5
    a, b = orc.pso_uniforms(seed, gp, it, 1, 4)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for blk in range(2):
        o = orc.philox4x32_10([gp, it, blk + 16, 0], key)
        u = [(x >> 8) / 2.0 ** 24 for x in o]
        assert [a[2 * blk], b[2 * blk], a[2 * blk + 1], b[2 * blk + 1]] == u
    a0, b0 = orc.pso_uniforms(seed, gp, it, 0, 3)           # purpose 0, odd D
    o = orc.philox4x32_10([gp, it, 1, 0], key)
    assert a0[2] == (o[0] >> 8) / 2.0 ** 24 and b0[2] == (o[1] >> 8) / 2.0 ** 24
    # every value is a multiple of 2^-24 in [0, 1): exact in FP32 too
    us = np.concatenate([np.concatenate(orc.pso_uniforms(3, p, 0, 1, 4)) for p in range(2000)])
    assert us.min() >= 0.0 and us.max() < 1.0
    assert np.array_equal(us, us.astype(np.float32).astype(np.float64))
    assert np.array_equal(us * 2 ** 24, np.round(us * 2 ** 24))
    assert abs(us.mean() - 0.5) < 4 / math.sqrt(12 * us.size)
    assert abs(us.var() - 1 / 12) < 0.004


def test_theta_of_x():
    wl = wlm.config(2)
    B = orc.box_from(wl)
    th = orc.theta_of_x(B, 3, [-19.0, 9.0, 100.0])
    assert th[0] == pytest.approx(1e-19, rel=1e-14, abs=0.0)
    assert th[1] == pytest.approx(1e9, rel=1e-14, abs=0.0)
    assert th[2] == 100.0                                    # eta is a linear coordinate


def _tiny(noise=False, n_particles=24, n_iters=12):
    wl = wlm.scaled(wlm.config(2), n_cycles=8, n_skip_cycles=4, steps_per_cycle=64,
                    n_particles=n_particles, n_iters=n_iters)
    M, B, Sw = orc.model_from(wl), orc.box_from(wl), orc.swarm_from(wl)
    bad, clean = orc.window(M, wl["truth"], wl["z0"], wl["v0"])
    assert bad == 0
    trace = clean + (wlm.trace_noise(wl)[0] if noise else 0.0)
    return wl, M, B, Sw, trace


def test_pso_invariants_and_hand_replay_of_eq8():
    wl, M, B, Sw, trace = _tiny(noise=True)
    D, P, seed = 3, Sw.n_particles, 11
    out = orc.pso_invert(M, B, Sw, seed, trace, wl["z0"], wl["v0"], dump=True)
    dump, gh = out["dump"], out["gbest_hist"]
    x, v, pb = dump[:, :, 0:D], dump[:, :, D:2 * D], dump[:, :, 2 * D:3 * D]
    J, pbJ = dump[:, :, 3 * D], dump[:, :, 3 * D + 1]
    lo, hi = np.array(wl["bounds"]["lo"]), np.array(wl["bounds"]["hi"])
    # initialisation: x0 = lo + a (hi - lo), v0 = ((lo + b (hi - lo)) - x0) / 2
    for p in range(P):
        a, b = orc.pso_uniforms(seed, p, 0, 0, D)
        assert np.array_equal(x[0, p], lo + a * (hi - lo))
        assert np.array_equal(v[0, p], 0.5 * ((lo + b * (hi - lo)) - x[0, p]))
    # positions stay in the box; J is the misfit of x; personal bests never get worse
    assert np.all(x >= lo) and np.all(x <= hi)
    assert np.all(np.diff(pbJ, axis=0) <= 0)
    assert np.all(pbJ <= J)
    for it in (0, 5, Sw.n_iters - 1):
        for p in (0, 7, P - 1):
            th = orc.theta_of_x(B, D, x[it, p])
            assert J[it, p] == orc.misfit(M, th, wl["z0"], wl["v0"], trace)
            # the personal best is the best position visited so far (first visit on ties)
            k = int(np.argmin(J[:it + 1, p]))
            assert pbJ[it, p] == J[k, p] and np.array_equal(pb[it, p], x[k, p])
    # global best = min over personal bests, lowest index on ties, non-increasing
    for it in range(Sw.n_iters):
        k = int(np.argmin(pbJ[it]))
        assert gh[it, 0, D] == pbJ[it, k]
        assert np.array_equal(gh[it, 0, :D], pb[it, k])
    assert np.all(np.diff(gh[:, 0, D]) <= 0)
    # Eq. 8 by hand, then x <- x + v, then clamp-and-zero
    n_clamped = 0
    for it in range(Sw.n_iters - 1):
        g = gh[it, 0, :D]
        for p in range(P):
            r1, r2 = orc.pso_uniforms(seed, p, it, 1, D)
            vn = Sw.w * v[it, p] + Sw.c1 * r1 * (pb[it, p] - x[it, p]) + Sw.c2 * r2 * (g - x[it, p])
            xn = x[it, p] + vn
            out_lo, out_hi = xn < lo, xn > hi
            n_clamped += int(np.sum(out_lo | out_hi))
            xn = np.where(out_lo, lo, np.where(out_hi, hi, xn))
            vn = np.where(out_lo | out_hi, 0.0, vn)
            assert np.allclose(x[it + 1, p], xn, rtol=1e-14, atol=0)
            assert np.allclose(v[it + 1, p], vn, rtol=1e-12, atol=1e-18)
    assert n_clamped > 0            # the bound rule was exercised
    # results
    assert out["J_star"][0] == gh[-1, 0, D]
    assert np.array_equal(out["theta_star"][0], orc.theta_of_x(B, D, gh[-1, 0, :D]))


def test_pso_is_deterministic_in_the_seed_and_differs_across_seeds():
    wl, M, B, Sw, trace = _tiny(noise=True, n_particles=8, n_iters=4)
    a = orc.pso_invert(M, B, Sw, 5, trace, wl["z0"], wl["v0"], dump=True)
    b = orc.pso_invert(M, B, Sw, 5, trace, wl["z0"], wl["v0"], dump=True)
    c = orc.pso_invert(M, B, Sw, 6, trace, wl["z0"], wl["v0"], dump=True)
    assert np.array_equal(a["dump"], b["dump"])
    assert not np.array_equal(a["dump"][0], c["dump"][0])


def test_pso_segments_are_independent_swarms():
    """n_traces swarms in one call = the same swarms run one by one, with
    particle indices offset (global index = trace * P + p)."""
    wl, M, B, Sw, trace = _tiny(noise=True, n_particles=6, n_iters=5)
    other = trace[::-1].copy()
    both = orc.pso_invert(M, B, Sw, 3, np.stack([trace, other]), wl["z0"], wl["v0"],
                          n_traces=2, dump=True, openmp=True)
    first = orc.pso_invert(M, B, Sw, 3, trace, wl["z0"], wl["v0"], dump=True)
    assert np.array_equal(both["dump"][:, :6], first["dump"])
    assert both["J_star"][0] == first["J_star"][0]
    assert both["J_star"][1] != first["J_star"][0]
    assert np.all(np.diff(both["gbest_hist"][:, 1, -1]) <= 0)


def test_pso_recovers_ground_truth_from_noise_free_trace():
    """north_star: 'recovery of known ground-truth theta from noise-free
    synthetic traces on tiny swarms' (configs[0] sizes, more iterations)."""
    wl = wlm.scaled(wlm.config(0), n_iters=100)
    M, B, Sw = orc.model_from(wl), orc.box_from(wl), orc.swarm_from(wl)
    bad, clean = orc.window(M, wl["truth"], wl["z0"], wl["v0"])
    out = orc.pso_invert(M, B, Sw, wl["pso_seed"], clean, wl["z0"], wl["v0"])
    rel = np.abs(out["theta_star"][0] / np.array(wl["truth"]) - 1.0)
    assert np.all(rel < 1e-3), (out["theta_star"], rel)
    assert out["J_star"][0] < 1e-6 * np.sum(clean ** 2)


def test_ring_topology_by_hand_replay():
    """topology = 1 (R23): the social attractor of
    particle p is the best personal best among p-1, p, p+1 (wrapping inside the
    swarm, lowest index among equal minima).  Replayed here in numpy from the
    oracle's own dump: same uniforms, same Eq. 8, only the attractor differs;
    the reported result is still the best over the whole swarm."""
    wl = wlm.scaled(wlm.config(0), n_cycles=6, n_skip_cycles=3, n_particles=9, n_iters=5)
    M = orc.model_from(wl)
    bad, win = orc.window(M, wl["truth"], wl["z0"], wl["v0"])
    sw = orc.swarm_from(wl, topology=1)
    o = orc.pso_invert(M, orc.box_from(wl), sw, 3, win[None, :], wl["z0"], wl["v0"], dump=True)
    g = orc.pso_invert(M, orc.box_from(wl), orc.swarm_from(wl), 3, win[None, :], wl["z0"],
                       wl["v0"], dump=True)
    d, D, P = o["dump"], 2, 9
    lo, hi = np.array(wl["bounds"]["lo"]), np.array(wl["bounds"]["hi"])
    assert np.array_equal(d[0], g["dump"][0])           # same start, same first batch
    assert not np.array_equal(d[2], g["dump"][2])       # another swarm afterwards
    for it in range(4):
        x, v, pb, pbJ = d[it, :, 0:2], d[it, :, 2:4], d[it, :, 4:6], d[it, :, 7]
        for p in range(P):
            cand = [(p - 1) % P, p, (p + 1) % P]
            best = min(cand, key=lambda c: (pbJ[c], c))
            r1, r2 = orc.pso_uniforms(3, p, it, 1, D)
            vn = sw.w * v[p] + sw.c1 * r1 * (pb[p] - x[p]) + sw.c2 * r2 * (pb[best] - x[p])
            xn = x[p] + vn
            low, high = xn < lo, xn > hi
            xn = np.where(low, lo, np.where(high, hi, xn))
            vn = np.where(low | high, 0.0, vn)
            assert np.array_equal(d[it + 1, p, 0:2], xn), (it, p)
            assert np.array_equal(d[it + 1, p, 2:4], vn), (it, p)
    assert o["J_star"][0] == d[:, :, 6].min()
