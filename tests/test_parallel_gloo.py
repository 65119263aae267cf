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


def test_neighbour_plan_sends_exactly_what_the_owned_windows_read():
    """Def of the reads: window j's successor term reads the controls of window j + 1, its predecessor term the end states
    of window j - 1 (buffer-1 entries of window j).  For every rank, what it owns plus what the plan delivers must cover
    exactly those reads that it does not own, and nothing is sent to a rank that owns it already."""
    p_lon, p_lat, q = 3, 2, 5
    offs, jw = geometry(p_lon, p_lat, q, nsteps=20)
    p12 = p_lon * p_lat
    for world in (1, 2, 3, 5):
        blocks = parallel.window_blocks(q, world)
        ops = parallel.neighbour_plan(offs, p12, q, world)
        for r, (j0, j1) in enumerate(blocks):
            need0 = {j + 1 for j in range(j0, j1) if j + 1 < q and not (j0 <= j + 1 < j1)}      # controls of foreign successor windows
            need1 = {j for j in range(j0, j1) if j > 0 and not (j0 <= j - 1 < j1)}              # entries of own windows filled by a foreign predecessor
            got0 = set(); got1 = set()
            for which, lo, hi, src, dst in ops:
                assert src != dst and abs(src - dst) == 1
                j = next(k for k in range(q) if offs[k * p12] == lo)
                assert hi == offs[(j + 1) * p12]
                if dst == r:
                    (got0 if which == 0 else got1).add(j)
                if which == 0:
                    assert blocks[src][0] <= j < blocks[src][1]                 # the owner of window j sends its controls
                else:
                    assert blocks[src][0] <= j - 1 < blocks[src][1]             # the owner of window j - 1 sends its end states
            assert got0 == need0 and got1 == need1, (world, r, got0, need0, got1, need1)


NB_WORKER = r'''
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
p_lon, p_lat, q = 3, 2, 5
p12 = p_lon * p_lat
offs, jw = geometry(p_lon, p_lat, q, nsteps=20)
blocks = parallel.window_blocks(q, world)
plan = parallel.exchange_plan(offs, p12, q, world)
ops = parallel.neighbour_plan(offs, p12, q, world)
n = offs[-1]
truth = [torch.from_numpy(np.random.default_rng(7 + b).standard_normal(n)) for b in range(2)]
junk = float(-1 - r)
bufs = [torch.full((n,), junk, dtype=torch.float64) for _ in range(2)]
for b in range(2):
    lo, hi = plan[r][b]
    bufs[b][lo:hi] = truth[b][lo:hi]
parallel.exchange_neighbours(bufs, ops, r, dist)
j0, j1 = blocks[r]
for j in range(q):
    sl = slice(offs[j * p12], offs[(j + 1) * p12])
    # buffer 0: own windows and the successor of the last one; buffer 1: the entries of own windows (j > 0) and of window j1 (own end states)
    have0 = j0 <= j < j1 or j == j1
    have1 = (j0 <= j < j1 and j > 0) or (j == j1 and j < q)
    assert torch.equal(bufs[0][sl], truth[0][sl]) == have0, (r, j, "controls")
    assert torch.equal(bufs[1][sl], truth[1][sl]) == have1, (r, j, "end states")
    if not have0: assert torch.all(bufs[0][sl] == junk)
    if not have1: assert torch.all(bufs[1][sl] == junk)
dist.barrier()
dist.destroy_process_group()
open(os.path.join(OUT, "nb_rank%%d.ok" %% r), "w").write("ok")
'''


def test_neighbour_exchange_between_three_gloo_ranks(tmp_path):
    """Three ranks, five windows: the middle rank has a neighbour on either side.  After the exchange every rank holds the
    true data exactly where its own windows read it and its own junk everywhere else."""
    script = tmp_path / "nb_worker.py"
    script.write_text(NB_WORKER % (ROOT, str(tmp_path), ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    p = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=3",
                        "--master-addr", "127.0.0.1", "--master-port", "29533", str(script)],
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stdout[-3000:] + p.stderr[-3000:]
    assert all((tmp_path / f"nb_rank{r}.ok").exists() for r in range(3))
