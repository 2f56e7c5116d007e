"""Pins for the two swarm rules the oracle states beyond Eq. 8:

* the cost cutoff (R24; "generations to convergence", 236
  "convergence cutoff", 264 "cutoff convergence threshold of J_L2 = 0.0005"), and
* the asynchronous, chunked swarm (R25).

Both are pinned on HAND-MADE cost functions handed to the oracle's own PSO loop
(orc_pso_core): the cost of the k-th evaluation of a swarm is read from a script,
whatever the position, so the batch at which the run must stop, the particle that
must win and the attractor every particle must have seen are written down here by
hand and do not come from the oracle.  Positions are made hand-computable by
switching terms of Eq. 8 off (w = c1 = c2 = 0 freezes the swarm at x0, and
w = c1 = 0 leaves x <- x + c2 r2 (g - x)); x0 and r2 come from the Philox stream,
which has its own known-answer pin (tests/test_oracle_pso.py).
"""
import numpy as np

from oracle import binding as orc


def _box(lo=0.0, hi=10.0, D=1):
    b = orc.Box()
    for j in range(D):
        b.lo[j], b.hi[j], b.log10[j] = lo, hi, 0
    return b


def _swarm(P, n_iters, w=0.0, c1=0.0, c2=0.0, j_target=0.0, topology=0, async_chunk=0):
    return orc.Swarm(n_particles=P, n_iters=n_iters, w=w, c1=c1, c2=c2, j_target=j_target,
                     topology=topology, async_chunk=async_chunk)


class Script:
    """cost(theta, U): U[0] is the trace index s; the k-th call for trace s returns
    script[s][k] (k = batch * P + particle in every mode) and records theta."""

    def __init__(self, rows):
        self.rows = [np.asarray(r, dtype=float).ravel() for r in rows]
        self.k = [0] * len(rows)
        self.seen = [[] for _ in rows]

    def __call__(self, theta, U):
        s = int(U[0])
        k = self.k[s]
        self.k[s] += 1
        self.seen[s].append(theta.copy())
        return self.rows[s][k]


def _x0(seed, gp, lo=0.0, hi=10.0):
    a, _ = orc.pso_uniforms(seed, gp, 0, 0, 1)
    return lo + a[0] * (hi - lo)


def _r2(seed, gp, it):
    _, b = orc.pso_uniforms(seed, gp, it, 1, 1)
    return b[0]


# --------------------------------------------------------------------------- cutoff

def test_cutoff_stops_after_the_first_batch_at_or_below_target():
    """One trace, 3 frozen particles, 6 batches allowed.  Scripted costs per batch:
        batch 0: 9 8 7      best 7
        batch 1: 6 9 9      best 6
        batch 2: 9 9 2.5    best 2.5 <= 3  -> the run ends here: 3 batches
        batch 3: 1 ...      never evaluated
    so n_iters_done = 3, J* = 2.5, theta* = the position of particle 2, and exactly
    9 cost evaluations happen."""
    seed = 7
    rows = [[9, 8, 7, 6, 9, 9, 9, 9, 2.5, 1, 1, 1, 1, 1, 1, 1, 1, 1]]
    sc = Script(rows)
    out = orc.pso_core(sc, 1, _box(), _swarm(3, 6, j_target=3.0), seed, [[0.0]])
    assert out["n_iters_done"] == 3
    assert sc.k[0] == 9
    assert out["J_star"][0] == 2.5
    assert out["theta_star"][0, 0] == _x0(seed, 2)         # frozen swarm: x = x0
    gh = out["gbest_hist"]
    assert list(gh[:3, 0, 1]) == [7.0, 6.0, 2.5]
    assert [gh[0, 0, 0], gh[1, 0, 0], gh[2, 0, 0]] == [_x0(seed, 2), _x0(seed, 0), _x0(seed, 2)]
    assert np.all(np.isnan(gh[3:])) and np.all(np.isnan(out["dump"][3:]))
    assert not np.any(np.isnan(out["dump"][:3]))


def test_cutoff_equal_to_target_stops_and_target_off_runs_everything():
    rows = [[5, 4, 3, 3, 3, 3, 2, 2, 2]]
    # J == target counts as reached (<=): best 4 -> no, 3 -> stop after batch 1
    out = orc.pso_core(Script(rows), 1, _box(), _swarm(2, 4, j_target=3.0), 1, [[0.0]])
    assert out["n_iters_done"] == 2 and out["J_star"][0] == 3.0
    # target 0 and negative targets switch the rule off, even when J reaches 0
    for jt in (0.0, -1.0):
        sc = Script([[5, 0, 0, 0, 0, 0, 0, 0]])
        out = orc.pso_core(sc, 1, _box(), _swarm(2, 4, j_target=jt), 1, [[0.0]])
        assert out["n_iters_done"] == 4 and sc.k[0] == 8
    # a target that is never reached, and costs that are never finite
    out = orc.pso_core(Script(rows), 1, _box(), _swarm(2, 4, j_target=1.0), 1, [[0.0]])
    assert out["n_iters_done"] == 4 and out["J_star"][0] == 2.0
    inf = float("inf")
    out = orc.pso_core(Script([[inf] * 4 + [float("nan")] * 4]), 1, _box(),
                       _swarm(2, 4, j_target=1e300), 1, [[0.0]])
    assert out["n_iters_done"] == 4 and out["J_star"][0] == inf


def test_cutoff_waits_for_every_trace():
    """Two traces, 2 particles each, target 3.  Trace 0 is below target from batch 1
    on, trace 1 only at batch 3: the run ends after batch 3 (4 batches), and trace 0
    kept being evaluated and improved meanwhile (its J* is the batch-3 value 0.5)."""
    rows = [[9, 9, 2, 9, 9, 1, 0.5, 9, 0.1, 0.1],
            [9, 9, 9, 8, 7, 9, 9, 2.9, 0.1, 0.1]]
    sc = Script(rows)
    out = orc.pso_core(sc, 1, _box(), _swarm(2, 5, j_target=3.0), 3, [[0.0], [1.0]],
                       n_traces=2)
    assert out["n_iters_done"] == 4
    assert sc.k == [8, 8]
    assert list(out["J_star"]) == [0.5, 2.9]
    assert list(out["gbest_hist"][:4, 0, 1]) == [9.0, 2.0, 1.0, 0.5]
    assert list(out["gbest_hist"][:4, 1, 1]) == [9.0, 8.0, 7.0, 2.9]
    # global particle index = trace * P + p: trace 1's winner is its particle 1
    assert out["theta_star"][1, 0] == _x0(3, 2 + 1)
    assert out["theta_star"][0, 0] == _x0(3, 0)


def test_no_move_follows_the_stopping_batch():
    """With the swarm free to move (w = 1: ballistic, x <- x + v0), the dump row of the
    stopping batch holds the positions that were evaluated in it, and the state after
    it is never produced: the same run without a target has the same rows up to
    there and goes on."""
    rows = [list(range(20, 0, -1))]
    kw = dict(w=1.0)
    cut = orc.pso_core(Script(rows), 1, _box(), _swarm(2, 6, j_target=15.0, **kw), 5, [[0.0]])
    full = orc.pso_core(Script(rows), 1, _box(), _swarm(2, 6, **kw), 5, [[0.0]])
    # best per batch: 19, 17, 15 -> stop after batch 2
    assert cut["n_iters_done"] == 3 and full["n_iters_done"] == 6
    assert np.array_equal(cut["dump"][:3], full["dump"][:3])
    assert cut["J_star"][0] == 15.0 and full["J_star"][0] == 9.0
    # ballistic positions by hand: x_it = x0 + it v0 while inside the box
    for p in range(2):
        a, b = orc.pso_uniforms(5, p, 0, 0, 1)
        x0, v0 = 10.0 * a[0], 0.5 * (10.0 * b[0] - 10.0 * a[0])
        for it in range(3):
            x = x0
            for _ in range(it):
                x = x + v0
                if x < 0.0 or x > 10.0:
                    break
            else:
                assert cut["dump"][it, p, 0] == x


# --------------------------------------------------------------------- asynchronous

def test_async_chunks_see_the_best_of_earlier_chunks_of_the_same_batch():
    """4 particles, chunks of 2, w = c1 = 0, c2 = 1: x <- x + r2 (g - x).
    Batch 0 costs: 5 6 | 1 9.
      chunk {0, 1}: best so far is particle 0 (J = 5): particle 0 stays where it is,
                    particle 1 moves towards x0[0];
      chunk {2, 3}: now particle 2 (J = 1) is the best: 2 stays, 3 moves towards x0[2].
    The synchronous swarm would send 0, 1 and 3 towards x0[2].
    Batch 1 costs: 9 9 | 9 0.5: chunk {0, 1} is evaluated at its moved positions and
    moves towards x0[2] (still the best); then particle 3 wins at its moved position."""
    seed, P = 11, 4
    rows = [[5, 6, 1, 9, 9, 9, 9, 0.5, 9, 9, 9, 9]]
    sc = Script(rows)
    out = orc.pso_core(sc, 1, _box(), _swarm(P, 3, c2=1.0, async_chunk=2), seed, [[0.0]])
    x0 = [_x0(seed, p) for p in range(P)]
    x = out["dump"][:, :, 0]
    assert list(x[0]) == x0
    x1 = [x0[0] + _r2(seed, 0, 0) * (x0[0] - x0[0]),
          x0[1] + _r2(seed, 1, 0) * (x0[0] - x0[1]),
          x0[2] + _r2(seed, 2, 0) * (x0[2] - x0[2]),
          x0[3] + _r2(seed, 3, 0) * (x0[2] - x0[3])]
    assert list(x[1]) == x1
    # the cost function saw exactly those positions, in that order
    assert [t[0] for t in sc.seen[0][:8]] == x0 + x1
    # batch 1: chunk {0, 1} moves towards x0[2]; then particle 3 takes over (J = 0.5)
    # and chunk {2, 3} moves towards x1[3]
    x2 = [x1[0] + _r2(seed, 0, 1) * (x0[2] - x1[0]),
          x1[1] + _r2(seed, 1, 1) * (x0[2] - x1[1]),
          x1[2] + _r2(seed, 2, 1) * (x1[3] - x1[2]),
          x1[3] + _r2(seed, 3, 1) * (x1[3] - x1[3])]
    assert list(x[2]) == x2
    assert out["J_star"][0] == 0.5 and out["theta_star"][0, 0] == x1[3]
    assert list(out["gbest_hist"][:, 0, 1]) == [1.0, 0.5, 0.5]
    assert out["n_iters_done"] == 3
    # the synchronous swarm on the same script differs from batch 1 on
    sync = orc.pso_core(Script(rows), 1, _box(), _swarm(P, 3, c2=1.0), seed, [[0.0]])
    assert sync["dump"][1, 0, 0] == x0[0] + _r2(seed, 0, 0) * (x0[2] - x0[0])
    assert sync["dump"][1, 0, 0] != x1[0]


def test_async_chunk_covering_the_swarm_is_the_synchronous_swarm():
    rows = [np.linspace(9.0, 1.0, 40)]
    ref = orc.pso_core(Script(rows), 1, _box(), _swarm(5, 8, w=0.7, c1=1.5, c2=1.5), 2, [[0.0]])
    for B in (0, 5, 6, 1000):
        out = orc.pso_core(Script(rows), 1, _box(),
                           _swarm(5, 8, w=0.7, c1=1.5, c2=1.5, async_chunk=B), 2, [[0.0]])
        assert np.array_equal(out["dump"], ref["dump"]), B
    one = orc.pso_core(Script(rows), 1, _box(),
                       _swarm(5, 8, w=0.7, c1=1.5, c2=1.5, async_chunk=2), 2, [[0.0]])
    assert not np.array_equal(one["dump"], ref["dump"])


def test_async_ragged_last_chunk_two_traces_and_cutoff():
    """5 particles in chunks of 2 (2 + 2 + 1), two traces with their own swarms.
    Trace 1's costs are trace 0's in reverse particle order within a batch, so its
    winner differs.  The cutoff is still tested once per batch, after the last chunk:
    target 2.5 is first met by both traces at batch 1."""
    P, seed = 5, 4
    r0 = [9, 8, 7, 6, 5, 4, 3, 2, 1, 0.5, 0.1, 0.1, 0.1, 0.1, 0.1]
    r1 = [5, 6, 7, 8, 9, 0.5, 1, 2, 3, 4, 0.1, 0.1, 0.1, 0.1, 0.1]
    sc = Script([r0, r1])
    out = orc.pso_core(sc, 1, _box(), _swarm(P, 3, c2=1.0, j_target=2.5, async_chunk=2),
                       seed, [[0.0], [1.0]], n_traces=2)
    assert out["n_iters_done"] == 2 and sc.k == [10, 10]
    assert list(out["J_star"]) == [0.5, 0.5]
    x = out["dump"][:, :, 0]
    x0 = [[_x0(seed, s * P + p) for p in range(P)] for s in range(2)]
    assert list(x[0]) == x0[0] + x0[1]
    # trace 0, batch 0: best so far after chunk {0,1} is 1 (J=8), after {2,3} is 3, after {4} is 4
    g0 = [1, 1, 3, 3, 4]
    # trace 1, batch 0: particle 0 (J=5) stays the best throughout
    g1 = [0, 0, 0, 0, 0]
    for s, g in ((0, g0), (1, g1)):
        for p in range(P):
            gp = s * P + p
            want = x0[s][p] + _r2(seed, gp, 0) * (x0[s][g[p]] - x0[s][p])
            assert x[1, gp] == want, (s, p)
    # winners of batch 1: trace 0 particle 4 (0.5), trace 1 particle 0 (0.5)
    assert out["theta_star"][0, 0] == x[1, 4] and out["theta_star"][1, 0] == x[1, 5]


def test_async_ring_uses_the_neighbours_bests_known_when_the_chunk_moves():
    """Ring of three with chunks of 2 on 4 particles, batch 0 costs 5 6 | 1 9.
    When chunk {0, 1} moves, particles 2 and 3 have not been evaluated yet (their
    personal bests are still +Inf): particle 0 looks at {3, 0, 1} -> 0; particle 1 at
    {0, 1, 2} -> 0.  When chunk {2, 3} moves everything is known: particle 2 looks at
    {1, 2, 3} -> 2; particle 3 at {2, 3, 0} -> 2."""
    seed, P = 13, 4
    rows = [[5, 6, 1, 9, 9, 9, 9, 9]]
    out = orc.pso_core(Script(rows), 1, _box(),
                       _swarm(P, 2, c2=1.0, topology=1, async_chunk=2), seed, [[0.0]])
    x0 = [_x0(seed, p) for p in range(P)]
    att = [0, 0, 2, 2]
    for p in range(P):
        assert out["dump"][1, p, 0] == x0[p] + _r2(seed, p, 0) * (x0[att[p]] - x0[p])
    # the synchronous ring on the same costs: particle 1 looks at {0,1,2} -> 2
    sync = orc.pso_core(Script(rows), 1, _box(), _swarm(P, 2, c2=1.0, topology=1), seed,
                        [[0.0]])
    assert sync["dump"][1, 1, 0] == x0[1] + _r2(seed, 1, 0) * (x0[2] - x0[1])


# ------------------------------------------------------------ closed forms and ties

def test_inertia_only_swarm_follows_the_geometric_series_and_sticks_to_the_bounds():
    """c1 = c2 = 0 leaves v <- w v, x <- x + v (PAPER.md:209-214 with both attractor
    terms off): a closed form.  Inside the box x_t = x_0 + v_0 (w + w^2 + ... + w^t)
    -- the velocity is updated BEFORE the position, so the first move is w v_0, not
    v_0 -- and the first time that leaves the box the particle is put on the bound
    it crossed with zero velocity, where it then stays for good (reading R10).  The
    expectation below is that series and that absorbing bound, written out; x_0 and
    v_0 are read from the first dump row.  Also the initial-state rule: x_0 in the
    box and |v_0| <= (hi - lo) / 2."""
    P, n_iters, D, w = 64, 12, 2, 0.9
    lo, hi = [0.0, -3.0], [10.0, 5.0]
    b = orc.Box()
    for j in range(D):
        b.lo[j], b.hi[j], b.log10[j] = lo[j], hi[j], 0
    r = orc.pso_core(lambda th, U: 1.0, D, b, _swarm(P, n_iters, w=w), 7, np.zeros((1, 1)))
    dmp = r["dump"]
    x0, v0 = dmp[0, :, 0:D], dmp[0, :, D:2 * D]
    lo, hi = np.asarray(lo), np.asarray(hi)
    assert np.all(x0 >= lo) and np.all(x0 <= hi)
    assert np.all(np.abs(v0) <= 0.5 * (hi - lo))
    assert np.abs(v0).max() > 0.25 * (hi - lo).min()      # not a degenerate start
    stuck = np.zeros((P, D), bool)
    where = np.zeros((P, D))
    n_stuck_seen = 0
    for t in range(1, n_iters):
        series = sum(w ** k for k in range(1, t + 1))
        free = x0 + v0 * series
        out_lo, out_hi = (free < lo) & ~stuck, (free > hi) & ~stuck
        where = np.where(out_lo, lo, np.where(out_hi, hi, where))
        stuck |= out_lo | out_hi
        want_x = np.where(stuck, where, free)
        want_v = np.where(stuck, 0.0, v0 * w ** t)
        np.testing.assert_allclose(dmp[t, :, 0:D], want_x, rtol=0, atol=1e-12)
        np.testing.assert_allclose(dmp[t, :, D:2 * D], want_v, rtol=0, atol=1e-12)
        n_stuck_seen = int(stuck.sum())
    assert 10 < n_stuck_seen < P * D          # both regimes are exercised


def test_equal_costs_the_lowest_index_wins_and_a_tie_never_replaces_a_best():
    """Scripted costs with exact ties (reading R10): among equal minima the particle
    with the lowest index is the global best; a later cost EQUAL to a personal or
    global best replaces neither (strict <).  Frozen swarm (w = c1 = c2 = 0), so
    every position is x_0 and the expected winner is written down by hand."""
    P = 5
    script = Script([[5, 3, 3, 7, 3,        # batch 0: three-way tie at 3 -> particle 1
                      3, 3, 3, 3, 3,        # batch 1: everybody ties with the best
                      4, 2, 9, 2, 2]])      # batch 2: three-way tie at 2 -> particle 1
    r = orc.pso_core(script, 1, _box(), _swarm(P, 3), 11, np.zeros((1, 1)))
    x0 = np.array([_x0(11, p) for p in range(P)])
    gh = r["gbest_hist"]
    assert gh[0, 0, 0] == x0[1] and gh[0, 0, 1] == 3.0
    assert gh[1, 0, 0] == x0[1] and gh[1, 0, 1] == 3.0      # ties replace nothing
    assert gh[2, 0, 0] == x0[1] and gh[2, 0, 1] == 2.0      # 1 before 3 and 4
    np.testing.assert_array_equal(r["dump"][1, :, -1], [3, 3, 3, 3, 3])   # pbestJ
    np.testing.assert_array_equal(r["dump"][2, :, -1], [3, 2, 3, 2, 2])
    # a second script where the tie is between the last two particles only
    script = Script([[9, 9, 9, 1, 1]])
    r = orc.pso_core(script, 1, _box(), _swarm(P, 1), 11, np.zeros((1, 1)))
    assert r["theta_star"][0, 0] == x0[3] and r["J_star"][0] == 1.0
