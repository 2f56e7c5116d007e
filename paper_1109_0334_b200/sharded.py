"""One swarm (or one line scan) sharded over the ranks of a torch.distributed
group: one process per GPU.

Two ways to shard, both with every arithmetic step inside the CUDA library:

* ``shard="particles"`` -- one trace, the particles split into contiguous
  slices.  Per iteration each rank evaluates its slice (afm_pso_shard_eval),
  the ranks all-gather ONE candidate row each (D + 2 doubles; 3 D + 4 with the
  ring topology, whose rows also carry the personal bests of the slice's first
  and last particle, the ring neighbours of the adjacent slices) -- the only
  data exchange; NCCL over NVLink on GPUs, gloo in the CPU tests -- and every
  rank picks the same global best and moves its slice (afm_pso_shard_move).
* ``shard="traces"`` -- configs[4]: whole pixels per rank, no collective in the
  loop at all; the per-pixel results are gathered once at the end.

Philox counters and the tie-break use GLOBAL particle indices, so a sharded
run replays the single-process afm_pso_invert: bit for bit while both run the
same form of the FP64 kernel (include/afm.h, option "form"; the auto choice
depends on the local particle count), otherwise with misfits equal to ~1e-15
relative and the same swarm unless two misfits tie at that level.

This module holds no arithmetic of the method: it partitions index ranges and
moves candidate rows.  The compute calls go through a backend object with the
three shard entry points; the default backend is the CUDA library and raises
if it is missing -- there is no CPU fallback (the CPU tests inject their own
test double, tests/test_sharded_gloo.py).
"""
import copy


def split_even(n, world, rank):
    """Contiguous slice [first, first + count) of n items for this rank; the
    first n % world ranks get one item more."""
    base, extra = divmod(int(n), int(world))
    count = base + (1 if rank < extra else 0)
    first = rank * base + min(rank, extra)
    return first, count


class CudaBackend:
    """The three shard entry points of libafm_b200.so on torch CUDA tensors."""

    def __init__(self):
        from . import afm
        afm.lib()       # raises ImportError if the library has not been built
        self.afm = afm

    def init(self, bounds, swarm, n_dims, n_traces, seed, first):
        return self.afm.afm_pso_shard_init(bounds, swarm, n_dims, n_traces, seed, first)

    def eval(self, bounds, swarm, trace, cfg, first, st):
        return self.afm.afm_pso_shard_eval(bounds, swarm, trace, cfg, first, st)

    def move(self, bounds, swarm, n_dims, n_traces, seed, it, do_move, first,
             gathered, st, rank=0, swarm_particles=None):
        return self.afm.afm_pso_shard_move(bounds, swarm, n_dims, n_traces, seed, it,
                                           do_move, first, gathered, st, rank=rank,
                                           swarm_particles=swarm_particles)

    def status(self):
        """Raises if a segment-queue kernel of this run lost a chain (afm_queue_status)."""
        self.afm.afm_queue_status()


class ShardedSwarm:
    """PSO inversion of `trace` with the swarm sharded over `group`.

    bounds, swarm, cfg: the GLOBAL problem (afm.Bounds, afm.SwarmCfg with
    n_particles per trace, afm.Cfg with the global n_traces).
    trace: [n_traces][W] tensor on this rank's device (every rank passes the
    whole trace array; a rank reads only its own traces).
    """

    def __init__(self, bounds, swarm, seed, trace, cfg, shard="particles",
                 group=None, backend=None, time_exchange=False):
        import torch.distributed as dist
        self.exchange_events = [] if time_exchange else None   # CUDA event pairs
        self.dist = dist
        self.group = group
        on = dist.is_available() and dist.is_initialized()
        self.world = dist.get_world_size(group) if on else 1
        self.rank = dist.get_rank(group) if on else 0
        self.backend = backend if backend is not None else CudaBackend()
        self.bounds, self.seed = bounds, int(seed)
        self.D = cfg.n_params
        self.n_iters = swarm.n_iters
        self.shard = shard
        self.global_traces = cfg.n_traces
        self.global_per = swarm.n_particles
        self.swarm = copy.copy(swarm)
        self.cfg = copy.copy(cfg)
        W = cfg.n_window
        trace = trace.reshape(cfg.n_traces, W)
        if shard == "particles":
            if cfg.n_traces != 1:
                raise ValueError('shard="particles" needs exactly one trace; '
                                 'use shard="traces" for a line scan')
            first, count = split_even(swarm.n_particles, self.world, self.rank)
            if count < 1:
                raise ValueError("more ranks than particles")
            self.first = first
            self.swarm.n_particles = count
            self.n_traces = 1
            self.trace = trace
            self.exchange = self.world > 1
        elif shard == "traces":
            t0, tn = split_even(cfg.n_traces, self.world, self.rank)
            if tn < 1:
                raise ValueError("more ranks than traces")
            self.trace_first = t0
            self.first = t0 * swarm.n_particles
            self.n_traces = tn
            self.cfg.n_traces = tn
            self.trace = trace[t0:t0 + tn].contiguous()
            self.exchange = False
        else:
            raise ValueError('shard must be "particles" or "traces"')
        self.state = self.backend.init(self.bounds, self.swarm, self.D, self.n_traces,
                                       self.seed, self.first)
        if self.exchange:
            # afm_pso_shard_init seeds gbest with the first LOCAL particle; the
            # unsharded rule is the first GLOBAL particle: rank 0's.
            dist.broadcast(self.state["gbest"], src=self._global_rank(0), group=group)
        self.iteration = 0

    def _global_rank(self, group_rank):
        if self.group is None:
            return group_rank
        return self.dist.get_global_rank(self.group, group_rank)

    def step(self, do_move=True):
        """One iteration: evaluate, exchange the candidate rows, move."""
        import torch
        st = self.state
        cand = self.backend.eval(self.bounds, self.swarm, self.trace, self.cfg,
                                 self.first, st)
        if self.exchange:
            # rows of rank r land at [r * n_traces, (r + 1) * n_traces)
            gathered = torch.empty((self.world * cand.shape[0], cand.shape[1]),
                                   dtype=cand.dtype, device=cand.device)
            timed = self.exchange_events is not None and cand.is_cuda
            if timed:
                e0 = torch.cuda.Event(enable_timing=True)
                e1 = torch.cuda.Event(enable_timing=True)
                e0.record()
            self.dist.all_gather_into_tensor(gathered, cand.contiguous(),
                                             group=self.group)
            if timed:
                e1.record()
                self.exchange_events.append((e0, e1))
        else:
            gathered = cand.reshape((1,) + tuple(cand.shape))
        self.backend.move(self.bounds, self.swarm, self.D, self.n_traces, self.seed,
                          self.iteration, do_move, self.first, gathered, st,
                          rank=self.rank if self.exchange else 0,
                          swarm_particles=self.global_per)
        self.iteration += 1
        return st

    def exchange_ms(self):
        """Durations of the recorded all-gathers (time_exchange=True), device time."""
        import torch
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in (self.exchange_events or [])]

    def run(self):
        """All swarm.n_iters iterations (the last one without a move, as
        afm_pso_invert).  Returns (theta_star [n_traces][D], J_star [n_traces])
        for the GLOBAL problem as CPU tensors, identical on every rank."""
        import torch
        for it in range(self.n_iters):
            self.step(do_move=(it + 1 < self.n_iters))
        if hasattr(self.backend, "status"):
            self.backend.status()   # the shard calls are asynchronous: check once, at the end
        th, Js = self.state["theta_star"], self.state["J_star"]
        if self.shard == "traces" and self.world > 1:
            # once, outside the loop: collect every rank's pixels
            counts = [split_even(self.global_traces, self.world, r)[1]
                      for r in range(self.world)]
            pad = max(counts)
            buf = torch.zeros((pad, self.D + 1), dtype=th.dtype, device=th.device)
            buf[:self.n_traces, :self.D] = th
            buf[:self.n_traces, self.D] = Js
            out = torch.empty((self.world * pad, self.D + 1), dtype=th.dtype,
                              device=th.device)
            self.dist.all_gather_into_tensor(out, buf, group=self.group)
            out = out.reshape(self.world, pad, self.D + 1)
            rows = torch.cat([out[r, :counts[r]] for r in range(self.world)], dim=0)
            th, Js = rows[:, :self.D], rows[:, self.D]
        return th.cpu(), Js.cpu()
