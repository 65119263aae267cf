"""Shared test helpers: build one seeded problem and feed the SAME inputs to the CPU oracle and
to the CUDA library (inputs come from paper_2205_06649_b200.synth, which holds no method
arithmetic; the truth trajectory used to sample observations is the oracle's)."""
import numpy as np

from paper_2205_06649_b200 import synth


def oracle_problem(w, **kw):
    from oracle import Oracle
    o = Oracle.from_workload(w, **kw)
    prob = synth.make_problem(w, o.forecast)
    o.set_background(prob.xb, prob.sigma_b)
    o.set_observations(prob.obs)
    return o, prob


def gpu_problem(w, prob, overlap_levels=False, **kw):
    from paper_2205_06649_b200.binding import DD4DVar
    g = DD4DVar.from_workload(w, **kw)
    if overlap_levels:
        g.set_overlap_levels(True)
    g.set_background(prob.xb, prob.sigma_b)
    if prob.obs is not None:
        g.set_observations(prob.obs)
    return g


def rel(a, b):
    """||a - b||_2 / ||b||_2 (0 if both vanish)."""
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    nb = np.linalg.norm(b.ravel())
    na = np.linalg.norm((a - b).ravel())
    return 0.0 if na == 0.0 else na / max(nb, 1e-300)


def small_workload(nlon=36, nlat=18, dt=600.0, nsteps=16, p_lon=2, p_lat=2, q_time=2, overlap=1,
                   nbumps=3, obs_frac=0.5, obs_every=2, outer=3, cfg=0, **kw):
    return synth.Workload(cfg, nlon, nlat, dt, nsteps, nbumps, obs_frac, obs_every, p_lon, p_lat, q_time,
                          overlap, outer, name="test", **kw)
