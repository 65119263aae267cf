"""Sharded DD-4DVar: one process per GPU, each owning a contiguous block of time windows.

Within an outer iteration the local problems are independent (eq (37)); the one exchange step per outer
iteration (Alg 1) is what crosses processes.  Spatial neighbours of a subdomain lie in its own window,
so with whole windows per process only two control-shaped arrays cross: the frozen controls (a window's successor
term (25c) reads the NEXT window's controls) and the predecessor end states (read by the next window).  Every process
holds the whole problem (22 GB of 180 GB at the 0.25 deg config) and moves only what it owns.  An owned window reads
from other ranks only the controls of the window after its block and the end states of the window before it, so the
exchange of an iteration is point-to-point with the ranks r +- 1 (`exchange_neighbours`: 2 x one window's slice per block
boundary, 2 x 28 MB per rank at the 0.25 deg config on 8 GPUs), plus two scalar reductions for the history and one broadcast
of window 0's controls at the end of a run for the gather.  `exchange` (every owner broadcasts its whole block) is kept
as the plain-collective form and for the tests.  No arithmetic of the method lives here.
"""
from __future__ import annotations

import numpy as np


def window_blocks(q_time: int, world: int):
    """Contiguous blocks of windows, [j0, j1) per rank (ranks beyond q_time own nothing: j0 == j1)."""
    return [((r * q_time) // world, ((r + 1) * q_time) // world) for r in range(world)]


def exchange_plan(offsets, p12: int, q_time: int, world: int):
    """Element ranges [lo, hi) of the control-shaped exchange buffers that each rank OWNS.
    offsets: control offsets of the nsub + 1 subdomains (subdomain order: window-major).
    Buffer 0 (frozen controls): rank r owns its windows [j0, j1).  Buffer 1 (predecessor end states): the entry of
    subdomain k is the end state of the window before k's, so rank r owns the entries of the windows [j0 + 1, j1 + 1)."""
    plan = []
    for (j0, j1) in window_blocks(q_time, world):
        a0, a1 = offsets[j0 * p12], offsets[j1 * p12]
        b0, b1 = offsets[min(j0 + 1, q_time) * p12], offsets[min(j1 + 1, q_time) * p12]
        if j0 == j1:
            a0 = a1 = b0 = b1 = 0
        plan.append(((a0, a1), (b0, b1)))
    return plan


def exchange(buffers, plan, dist=None):
    """Complete the exchange: every rank broadcasts the ranges it owns.  buffers: (frozen controls, predecessor end states)
    as 1-D tensors (device tensors with NCCL, host tensors with gloo)."""
    if dist is None:
        import torch.distributed as dist
    for r, ranges in enumerate(plan):
        for buf, (lo, hi) in zip(buffers, ranges):
            if hi > lo:
                dist.broadcast(buf[lo:hi], src=r)


def neighbour_plan(offsets, p12: int, q_time: int, world: int):
    """What an owned window really reads from another rank: its successor term (25c) reads the controls of the NEXT window,
    its predecessor term the end states of the window BEFORE it.  With contiguous blocks of windows that is one window's
    slice per block boundary and direction.  -> list of (buffer, lo, hi, src, dst): at the boundary window j between rank a
    (owns j - 1) and rank b (owns j), the frozen controls of window j go b -> a and the end states of window j - 1, which
    are stored at the entries of window j, go a -> b."""
    blocks = window_blocks(q_time, world)
    owners = [r for r, (j0, j1) in enumerate(blocks) if j1 > j0]
    ops = []
    for a, b in zip(owners[:-1], owners[1:]):
        j = blocks[b][0]
        lo, hi = offsets[j * p12], offsets[(j + 1) * p12]
        ops.append((0, lo, hi, b, a))
        ops.append((1, lo, hi, a, b))
    return ops


def exchange_neighbours(buffers, ops, rank: int, dist=None):
    """The exchange of one outer iteration as point-to-point transfers between ranks r and r +- 1 (2 x one window per
    boundary instead of every rank's whole block to everyone; config 3 on 8 GPUs: 2 x 28 MB per rank against 2 x 226 MB).
    After it a rank holds valid frozen data for the windows it owns and the two windows next to them, nothing else."""
    if dist is None:
        import torch.distributed as dist
    reqs = []
    for which, lo, hi, src, dst in ops:
        if rank == src:
            reqs.append(dist.P2POp(dist.isend, buffers[which][lo:hi], dst))
        elif rank == dst:
            reqs.append(dist.P2POp(dist.irecv, buffers[which][lo:hi], src))
    if reqs:
        for w in dist.batch_isend_irecv(reqs):
            w.wait()


class ShardedDD4DVar:
    """Algorithm 1 with the windows sharded over the ranks of the default process group."""

    def __init__(self, workload, device=None, **kw):
        import torch
        import torch.distributed as dist
        from .binding import DD4DVar
        self.dist = dist
        self.rank = dist.get_rank() if dist.is_initialized() else 0
        self.world = dist.get_world_size() if dist.is_initialized() else 1
        self.g = DD4DVar.from_workload(workload, device=device or f"cuda:{torch.cuda.current_device()}", **kw)
        g = self.g
        self.p12 = workload.p_lon * workload.p_lat
        self.q = workload.q_time
        self.j0, self.j1 = window_blocks(self.q, self.world)[self.rank]
        if self.world > 1:
            if self.j0 == self.j1:
                raise ValueError("more ranks than time windows")
            g.set_owned_windows(self.j0, self.j1)
            g.set_history_global(False)
        self.plan = exchange_plan(g.offsets, self.p12, self.q, self.world)
        self.nb_ops = neighbour_plan(g.offsets, self.p12, self.q, self.world)
        self.owned = np.zeros(g.nsub, dtype=bool)
        self.owned[self.j0 * self.p12:self.j1 * self.p12] = True

    def set_background(self, xb, sigma_b):
        self.g.set_background(xb, sigma_b)

    def set_observations(self, obs):
        self.g.set_observations(obs)

    def run(self, outer_iters):
        """-> analysis (on every rank), history [(outer_iters + 1)][2]: sum_ji J_ji at the end of iteration l and
        delta_l (row 0: zeros)."""
        import torch
        g = self.g
        hist = np.zeros((outer_iters + 1, 2))
        for l in range(1, outer_iters + 1):
            g.run(1)
            if self.world > 1:
                # The broadcasts are queued behind torch's CURRENT stream; the library works on g.stream, which need not
                # be the same one.  Order them explicitly on both sides: the collectives after this iteration's kernels,
                # the next iteration's kernels after the collectives (not left to the host-blocking reductions below).
                cur = torch.cuda.current_stream(g.device)
                cur.wait_stream(g.stream)
                exchange_neighbours((g.exchange_view(0), g.exchange_view(1)), self.nb_ops, self.rank, self.dist)
                g.stream.wait_stream(cur)
            J, dm = g.local_stats()
            red = torch.tensor([J[self.owned].sum()], dtype=torch.float64, device=g.device)
            mx = torch.tensor([dm[self.owned].max() if self.owned.any() else 0.0], dtype=torch.float64, device=g.device)
            if self.world > 1:
                self.dist.all_reduce(red, op=self.dist.ReduceOp.SUM)
                self.dist.all_reduce(mx, op=self.dist.ReduceOp.MAX)
            hist[l, 0] = float(red[0]); hist[l, 1] = float(mx[0])
        if self.world > 1:
            # the analysis (eq (12)-(13)) is gathered from the frozen controls of window 0, which only its owner and that
            # owner's neighbour hold after neighbour exchanges: one broadcast of that window's slice at the end of the run
            cur = torch.cuda.current_stream(g.device)
            cur.wait_stream(g.stream)
            self.dist.broadcast(g.exchange_view(0)[g.offsets[0]:g.offsets[self.p12]], src=0)
            g.stream.wait_stream(cur)
        return g.gather_analysis(), hist

    def close(self):
        self.g.close()
