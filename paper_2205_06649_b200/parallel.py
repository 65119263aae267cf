"""Sharded DD-4DVar: one process per GPU, each owning a contiguous block of time windows.

Within an outer iteration the local problems are independent (eq (37)); the one exchange step per outer
iteration (Alg 1) is what crosses processes.  Spatial neighbours of a subdomain lie in its own window,
so with whole windows per process only two control-shaped arrays cross: the frozen controls (a window's successor
term (25c) reads the NEXT window's controls) and the predecessor end states (read by the next window).  Every process
holds the whole problem (22 GB of 180 GB at the 0.25 deg config) and moves only what it owns, so the exchange is one
broadcast per owner and array (NCCL over NVLink: 2 x 226 MB per outer iteration at the 0.25 deg config against
~70 ms of sweeps), plus two scalar reductions for the history.  No arithmetic of the method lives here.
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
                exchange((g.exchange_view(0), g.exchange_view(1)), self.plan, self.dist)
                g.stream.wait_stream(cur)
            J, dm = g.local_stats()
            red = torch.tensor([J[self.owned].sum()], dtype=torch.float64, device=g.device)
            mx = torch.tensor([dm[self.owned].max() if self.owned.any() else 0.0], dtype=torch.float64, device=g.device)
            if self.world > 1:
                self.dist.all_reduce(red, op=self.dist.ReduceOp.SUM)
                self.dist.all_reduce(mx, op=self.dist.ReduceOp.MAX)
            hist[l, 0] = float(red[0]); hist[l, 1] = float(mx[0])
        return g.gather_analysis(), hist

    def close(self):
        self.g.close()
