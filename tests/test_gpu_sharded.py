"""Sharded runs (dd4dvar_set_owned_windows) on ONE GPU: two handles in one process play the two
ranks, each owning a block of time windows; after every outer iteration the test copies the owned ranges of the two
exchange buffers between them (what parallel.exchange does with broadcasts).  The result must be the single-handle
run bit for bit: the sharded iteration is the same arithmetic on the same data."""
import numpy as np
import pytest

from paper_2205_06649_b200 import parallel
from helpers import oracle_problem, gpu_problem, small_workload
from test_gpu_parity import LAYOUTS

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,path", [("cfg0", 0), ("ragged3x2x3_o2", 0), ("wave_k2", 0), ("ragged3x2x3_o2", 1)])
def test_two_window_blocks_reproduce_the_single_run(name, path):
    w = small_workload(**LAYOUTS[name])
    o, prob = oracle_problem(w)
    L = 3
    single = gpu_problem(w, prob, path=path)
    an_s, hist_s = single.run(L)
    world = 2
    ranks = [gpu_problem(w, prob, path=path) for _ in range(world)]
    blocks = parallel.window_blocks(w.q_time, world)
    plan = parallel.exchange_plan(ranks[0].offsets, w.p_lon * w.p_lat, w.q_time, world)
    p12 = w.p_lon * w.p_lat
    for r, g in enumerate(ranks):
        g.set_owned_windows(*blocks[r])
        g.set_history_global(False)
    for l in range(1, L + 1):
        for g in ranks:
            g.run(1)
        views = [(g.exchange_view(0), g.exchange_view(1)) for g in ranks]
        for src in range(world):
            for dst in range(world):
                if dst != src:
                    for b in range(2):
                        lo, hi = plan[src][b]
                        views[dst][b][lo:hi].copy_(views[src][b][lo:hi])
        sumJ = 0.0; delta = 0.0
        for r, g in enumerate(ranks):
            J, dm = g.local_stats()
            own = slice(blocks[r][0] * p12, blocks[r][1] * p12)
            sumJ += J[own].sum(); delta = max(delta, dm[own].max())
        assert abs(sumJ - hist_s[l, 1]) <= 1e-13 * abs(hist_s[l, 1])
        assert delta == hist_s[l, 2]
    for g in ranks:
        assert np.array_equal(g.gather_analysis().cpu().numpy(), an_s.cpu().numpy())
        assert np.array_equal(g.get_controls().cpu().numpy(), single.get_controls().cpu().numpy())


def test_sharded_driver_with_one_rank_is_the_plain_run():
    w = small_workload(**LAYOUTS["cfg0"])
    o, prob = oracle_problem(w)
    single = gpu_problem(w, prob)
    an_s, hist_s = single.run(2)
    sh = parallel.ShardedDD4DVar(w)
    sh.set_background(prob.xb, prob.sigma_b); sh.set_observations(prob.obs)
    an, hist = sh.run(2)
    assert np.array_equal(an.cpu().numpy(), an_s.cpu().numpy())
    assert np.allclose(hist[1:, 0], hist_s[1:, 1], rtol=1e-13) and np.array_equal(hist[1:, 1], hist_s[1:, 2])


def test_two_ranks_over_nccl_reproduce_the_single_run():
    """The same statement over NCCL with one process per GPU, the library on a stream that is not torch's current
    stream (parallel.ShardedDD4DVar orders the broadcasts against it).  Needs two GPUs; skipped on a one-GPU box."""
    import os
    import subprocess
    import sys
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    worker = os.path.join(os.path.dirname(os.path.abspath(__file__)), "nccl_shard_worker.py")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29547", worker],
                       capture_output=True, text=True, timeout=900)
    assert r.returncode == 0 and "nccl shard worker ok" in r.stdout, r.stdout[-3000:] + r.stderr[-3000:]


def test_sharded_driver_on_a_side_stream_with_one_rank():
    """One rank, library on a side stream: the driver and its stream ordering code run (no exchange with one rank)."""
    import torch
    w = small_workload(**LAYOUTS["wave_k2"])
    o, prob = oracle_problem(w)
    single = gpu_problem(w, prob)
    an_s, _ = single.run(2)
    sh = parallel.ShardedDD4DVar(w, stream=torch.cuda.Stream())
    sh.set_background(prob.xb, prob.sigma_b); sh.set_observations(prob.obs)
    an, _ = sh.run(2)
    assert np.array_equal(an.cpu().numpy(), an_s.cpu().numpy())
