"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (fused path).

Config 1 (1 deg, 64 subdomains): every subdomain's cost / gradient, and two outer iterations.
Config 3 (0.25 deg, 2048 subdomains, the roofline headline): the oracle evaluates a SAMPLE of
subdomains one by one (pole tiles, interior tiles, first / middle / last window); properties that
hold at any size are checked on all of them (eq (19): sum of local costs at the background =
J(x_b); the observation-free cost of a window-0 subdomain at the background is zero).
"""
import numpy as np
import pytest

from paper_2205_06649_b200 import synth
from helpers import oracle_problem, gpu_problem, rel

pytestmark = pytest.mark.gpu
TOL_EVAL = 1e-10
TOL_AN = 1e-8


def perturbed(o, prob, ks, seed, amp=0.5):
    sb = prob.sigma_b[:, None, None]
    return {k: o.get_control(k) + amp * sb * synth.random_fields(o.sub_shape(k), seed + k) for k in ks}


def test_config1_all_subdomains_and_two_outer_iterations():
    w = synth.CONFIGS[1]
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob)
    assert g.active_path in (2, 4) and g.nsub == 64
    xs = perturbed(o, prob, range(o.nsub), 77)
    costs, parts, grads = g.eval_local(g.pack([xs[k] for k in range(o.nsub)]))
    gl = [t.cpu().numpy() for t in g.split(grads)]
    for k in range(o.nsub):
        po, go, _ = o.eval_local(k, xs[k])
        assert abs(costs[k] - po[0]) <= TOL_EVAL * abs(po[0]), k
        assert rel(gl[k], go) <= TOL_EVAL, (k, rel(gl[k], go))
    an_o, hist_o = o.run(2)
    an_g, hist_g = g.run(2)
    an_g = an_g.cpu().numpy()
    for f in range(3):
        assert rel(an_g[f], an_o[f]) <= TOL_AN, f
    assert np.all(np.abs(hist_g[:, :2] - hist_o[:, :2]) <= 1e-8 * np.abs(hist_o[:, :2]) + 1e-300)
    # generic kernels agree with the fused ones on the same problem
    g1 = gpu_problem(w, prob, path=1)
    c1, _, gr1 = g1.eval_local(g1.pack([xs[k] for k in range(o.nsub)]))
    g2 = gpu_problem(w, prob, path=2)
    c2, _, gr2 = g2.eval_local(g2.pack([xs[k] for k in range(o.nsub)]))
    assert np.max(np.abs(c1 - c2) / np.abs(c1)) <= 1e-12
    assert rel(gr2.cpu().numpy(), gr1.cpu().numpy()) <= 1e-12


def test_config3_sampled_subdomains_and_invariants():
    w = synth.CONFIGS[3]
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob)
    assert g.active_path in (2, 4) and g.nsub == 2048
    p12 = w.p_lon * w.p_lat
    sample = [0, 15, 8 * 16 + 7, 15 * 16 + 15, 3 * p12 + 5 * 16 + 9, 7 * p12 + 0, 7 * p12 + 15 * 16 + 3, 4 * p12 + 16 * 8]
    # at the background controls: eq (19) and per-subdomain costs on the sample
    ctr = g.get_controls()
    costs, parts, grads = g.eval_local(ctr)
    Jb, _ = g.eval_global(prob.xb, want_grad=False)
    assert abs(costs.sum() - Jb) <= 1e-9 * Jb
    assert np.all(parts[:, 2:] == 0.0)                 # no overlap mismatch at the background
    gl = g.split(grads)
    for k in sample:
        po, go, _ = o.eval_local(k, o.get_control(k))
        assert abs(costs[k] - po[0]) <= TOL_EVAL * abs(po[0]), k
        assert rel(gl[k].cpu().numpy(), go) <= TOL_EVAL, k
    # perturbed controls on the sample (the other subdomains stay at the background)
    xs = perturbed(o, prob, sample, 5)
    flat = ctr.clone()
    for k in sample:
        n = int(np.prod(g.sub_shape(k)))
        flat[g.offsets[k]:g.offsets[k] + n] = g._dev(xs[k]).reshape(-1)
    costs, parts, grads = g.eval_local(flat)
    gl = g.split(grads)
    for k in sample:
        po, go, tr = o.eval_local(k, xs[k], want_traj=True)
        assert abs(costs[k] - po[0]) <= TOL_EVAL * abs(po[0]), k
        for q in range(5):
            assert abs(parts[k, q] - po[1 + q]) <= TOL_EVAL * abs(po[0]), (k, q)
        assert rel(gl[k].cpu().numpy(), go) <= TOL_EVAL, (k, rel(gl[k].cpu().numpy(), go))
        assert rel(g.get_local_trajectory(k).cpu().numpy(), tr) <= 1e-12, k


def test_config4_large_tile_layout_follows_the_oracle_iteration():
    """Config 4, layout 2x2x2 overlap 1 on the 0.5 deg problem (tiles 362x181: generic step
    kernels, many 32x16 blocks per tile): cost / gradient of every subdomain and the history of the
    first two outer iterations equal the oracle's (this layout's J_global rises - both sides agree)."""
    w = synth.CONFIGS[2].with_layout(2, 2, 2, 1)
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob)
    assert g.active_path == 1 and g.nsub == 8
    xs = perturbed(o, prob, range(o.nsub), 41)
    costs, parts, grads = g.eval_local(g.pack([xs[k] for k in range(o.nsub)]))
    gl = g.split(grads)
    for k in range(o.nsub):
        po, go, _ = o.eval_local(k, xs[k])
        assert abs(costs[k] - po[0]) <= TOL_EVAL * abs(po[0]), k
        assert rel(gl[k].cpu().numpy(), go) <= TOL_EVAL, k
    an_o, hist_o = o.run(2)
    an_g, hist_g = g.run(2)
    assert np.all(np.abs(hist_g[:, :2] - hist_o[:, :2]) <= 1e-8 * np.abs(hist_o[:, :2]))
    for f in range(3):
        assert rel(an_g.cpu().numpy()[f], an_o[f]) <= TOL_AN


def test_config2_one_outer_iteration():
    """Config 2 (0.5 deg, 8x8x8 = 512 subdomains, wavenumber-4 perturbation): one outer iteration
    of Algorithm 1 against the oracle, and sampled evaluations with the exchanged data."""
    w = synth.CONFIGS[2]
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob)
    assert g.active_path in (2, 4) and g.nsub == 512
    an_o, hist_o = o.run(1)
    an_g, hist_g = g.run(1)
    an_g = an_g.cpu().numpy()
    for f in range(3):
        assert rel(an_g[f], an_o[f]) <= TOL_AN, f
    assert np.all(np.abs(hist_g[:, :2] - hist_o[:, :2]) <= 1e-8 * np.abs(hist_o[:, :2]))
    assert abs(hist_g[1, 2] - hist_o[1, 2]) <= 1e-6 * hist_o[1, 2]
    sample = [0, 63, 64 * 3 + 27, 64 * 7 + 63]
    ctr = g.get_controls()
    costs, parts, grads = g.eval_local(ctr)
    for k in sample:
        po, go, _ = o.eval_local(k, o.get_control(k))
        assert abs(costs[k] - po[0]) <= 1e-8 * abs(po[0]), k
        assert rel(g.split(grads)[k].cpu().numpy(), go) <= 1e-8, k
