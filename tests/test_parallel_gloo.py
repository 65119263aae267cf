"""The N > 1 path of the sharded driver (paper_2205_06649_b200/parallel.py) on CPU with two gloo ranks: the window
blocks, the ownership ranges of the two exchange buffers (computed from the library's own geometry, which
needs no GPU) and the broadcasts that complete the exchange.  The kernels are not involved."""
import ctypes
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2205_06649_b200 import binding, parallel  # noqa: E402


def geometry(p_lon, p_lat, q_time, nlon=40, nlat=23, nsteps=17, overlap=2):
    """Control offsets and windows of every subdomain from the C-ABI (host only)."""
    lib = binding.load_library()
    g = binding.Grid(nlon, nlat, 6.371e6, 7.292e-5, 9.806, float(np.cos(np.deg2rad(50.0))), 0.02)
    d = binding.Decomp(p_lon, p_lat, q_time, overlap, 1.0, 1.0)
    w = binding.Window(600.0, nsteps)
    h = ctypes.c_void_p()
    assert lib.dd4dvar_create(ctypes.byref(g), ctypes.byref(d), ctypes.byref(w), None, None, ctypes.byref(h)) == 0
    n = lib.dd4dvar_num_subdomains(h)
    offs = [lib.dd4dvar_control_offset(h, k) for k in range(n + 1)]
    out = (ctypes.c_int * 16)()
    jw = []
    for k in range(n):
        assert lib.dd4dvar_subdomain_info(h, k, out) == 0
        jw.append(out[2])
    lib.dd4dvar_destroy(h)
    return offs, jw


def test_window_blocks_cover_the_windows_once():
    for q in (1, 2, 3, 8):
        for world in (1, 2, 3, 8):
            blocks = parallel.window_blocks(q, world)
            assert blocks[0][0] == 0 and blocks[-1][1] == q
            assert all(a[1] == b[0] for a, b in zip(blocks, blocks[1:]))


def test_exchange_plan_matches_the_owner_rule():
    p_lon, p_lat, q = 3, 2, 3
    offs, jw = geometry(p_lon, p_lat, q)
    p12 = p_lon * p_lat
    for world in (1, 2, 3):
        plan = parallel.exchange_plan(offs, p12, q, world)
        blocks = parallel.window_blocks(q, world)
        own0 = np.full(offs[-1], -1); own1 = np.full(offs[-1], -1)
        for r, ((a0, a1), (b0, b1)) in enumerate(plan):
            assert np.all(own0[a0:a1] == -1) and np.all(own1[b0:b1] == -1)       # ranges do not overlap
            own0[a0:a1] = r; own1[b0:b1] = r
        for k in range(len(jw)):
            r_own = next(r for r, (j0, j1) in enumerate(blocks) if j0 <= jw[k] < j1)
            assert np.all(own0[offs[k]:offs[k + 1]] == r_own)
            if jw[k] == 0:
                assert np.all(own1[offs[k]:offs[k + 1]] == -1)                   # no predecessor window: nobody sends it
            else:
                r_pred = next(r for r, (j0, j1) in enumerate(blocks) if j0 <= jw[k] - 1 < j1)
                assert np.all(own1[offs[k]:offs[k + 1]] == r_pred)


WORKER = r'''
import os, sys
sys.path.insert(0, %r)
OUT = %r
import numpy as np, torch
import torch.distributed as dist
sys.path.insert(0, os.path.join(%r, "tests"))
from test_parallel_gloo import geometry
from paper_2205_06649_b200 import parallel
dist.init_process_group("gloo")
r, world = dist.get_rank(), dist.get_world_size()
p_lon, p_lat, q = 3, 2, 3
offs, jw = geometry(p_lon, p_lat, q)
plan = parallel.exchange_plan(offs, p_lon * p_lat, q, world)
n = offs[-1]
truth = [torch.from_numpy(np.random.default_rng(7 + b).standard_normal(n)) for b in range(2)]
bufs = [torch.full((n,), float(-1 - r), dtype=torch.float64) for _ in range(2)]      # what this rank does not own: junk
for b in range(2):
    lo, hi = plan[r][b]
    bufs[b][lo:hi] = truth[b][lo:hi]
parallel.exchange(bufs, plan, dist)
assert torch.equal(bufs[0], truth[0])
first = offs[p_lon * p_lat]                 # entries of window 0 have no owner in buffer 1
assert torch.equal(bufs[1][first:], truth[1][first:]) and torch.all(bufs[1][:first] == float(-1 - r))
dist.barrier()
dist.destroy_process_group()
open(os.path.join(OUT, "rank%%d.ok" %% r), "w").write("ok")
'''


def test_exchange_between_two_gloo_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % (ROOT, str(tmp_path), ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    p = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29531", str(script)],
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stdout + p.stderr
    assert (tmp_path / "rank0.ok").exists() and (tmp_path / "rank1.ok").exists()
