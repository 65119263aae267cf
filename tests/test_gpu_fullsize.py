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
TOL_MAX = 1e-9          # largest single-element gradient error relative to the largest element


def check_sample(o, g, prob, sample, seed, tol=TOL_EVAL, tol_max=TOL_MAX, traj=False):
    """Perturbed controls on a sample of subdomains (the others keep their current controls):
    cost, the five parts, gradient (2-norm and element-wise) and optionally the stored trajectory."""
    xs = perturbed(o, prob, sample, seed)
    flat = g.get_controls().clone()
    for k in sample:
        n = int(np.prod(g.sub_shape(k)))
        flat[g.offsets[k]:g.offsets[k] + n] = g._dev(xs[k]).reshape(-1)
    costs, parts, grads = g.eval_local(flat)
    gl = g.split(grads)
    for k in sample:
        po, go, tr = o.eval_local(k, xs[k], want_traj=traj)
        gk = gl[k].cpu().numpy()
        assert abs(costs[k] - po[0]) <= tol * abs(po[0]), k
        for q in range(5):
            assert abs(parts[k, q] - po[1 + q]) <= tol * abs(po[0]), (k, q)
        assert rel(gk, go) <= tol, (k, rel(gk, go))
        assert np.abs(gk - go).max() <= tol_max * np.abs(go).max(), (k, np.abs(gk - go).max() / np.abs(go).max())
        if traj:
            assert rel(g.get_local_trajectory(k).cpu().numpy(), tr) <= 1e-12, k


def perturbed(o, prob, ks, seed, amp=0.5):
    sb = prob.sigma_b[:, None, None]
    return {k: o.get_control(k) + amp * sb * synth.random_fields(o.sub_shape(k), seed + k) for k in ks}


def test_config1_all_subdomains_and_two_outer_iterations():
    w = synth.CONFIGS[1]
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob)
    assert g.active_path == 5 and g.nsub == 64
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
    assert g.active_path == 5 and g.nsub == 2048
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
    # the host-buffer entry point in the configuration bench.py times for `e2e` (six chunks of 1 + 2 + 4 + 4 + 2 + 1
    # rounds of 148 subdomains, copies overlapped with the masked sweeps): bit for bit what the one-sweep call returned
    import torch
    h_ctrl = flat.cpu().pin_memory()
    h_grad = torch.zeros_like(h_ctrl).pin_memory()
    h_cost = np.zeros(g.nsub)
    g.eval_local_host(h_ctrl, h_cost, h_grad)
    assert np.array_equal(h_cost, costs)
    assert np.array_equal(h_grad.numpy(), grads.cpu().numpy())


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
    assert g.active_path == 5 and g.nsub == 512
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


def test_config3_two_outer_iterations_and_exchanged_data():
    """The headline config through Algorithm 1: run(2) against the oracle (analysis 1e-8 per field,
    history 1e-8, step norm 1e-6), then 16 sampled subdomains re-evaluated on the EXCHANGED data:
    pole-row tiles, tiles across the clamp latitude (50 deg: tile rows 3 and 12 of 16), first,
    middle and last windows."""
    w = synth.CONFIGS[3]
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob)
    assert g.active_path == 5 and g.nsub == 2048
    an_o, hist_o = o.run(2)
    an_g, hist_g = g.run(2)
    an_g = an_g.cpu().numpy()
    for f in range(3):
        assert rel(an_g[f], an_o[f]) <= TOL_AN, (f, rel(an_g[f], an_o[f]))
    assert rel(an_g - prob.xb, an_o - prob.xb) <= 1e-6
    assert np.all(np.abs(hist_g[:, :2] - hist_o[:, :2]) <= 1e-8 * np.abs(hist_o[:, :2]) + 1e-300), (hist_g, hist_o)
    assert np.all(np.abs(hist_g[:, 2] - hist_o[:, 2]) <= 1e-6 * np.abs(hist_o[:, 2]) + 1e-12)
    p12 = w.p_lon * w.p_lat
    tile = lambda a, b: b * w.p_lon + a
    sample = [0 * p12 + tile(0, 0), 0 * p12 + tile(9, 3), 0 * p12 + tile(15, 15), 1 * p12 + tile(4, 12),
              2 * p12 + tile(7, 8), 3 * p12 + tile(0, 15), 3 * p12 + tile(11, 3), 4 * p12 + tile(8, 0),
              4 * p12 + tile(15, 7), 5 * p12 + tile(2, 12), 5 * p12 + tile(13, 1), 6 * p12 + tile(6, 14),
              7 * p12 + tile(0, 0), 7 * p12 + tile(15, 15), 7 * p12 + tile(5, 4), 7 * p12 + tile(10, 11)]
    check_sample(o, g, prob, sample, 91, tol=1e-8, tol_max=1e-7)


def test_config2_three_outer_iterations():
    w = synth.CONFIGS[2]
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob)
    an_o, hist_o = o.run(3)
    an_g, hist_g = g.run(3)
    an_g = an_g.cpu().numpy()
    for f in range(3):
        assert rel(an_g[f], an_o[f]) <= TOL_AN, (f, rel(an_g[f], an_o[f]))
    assert np.all(np.abs(hist_g[:, :2] - hist_o[:, :2]) <= 1e-8 * np.abs(hist_o[:, :2]) + 1e-300)
    assert np.all(np.abs(hist_g[:, 2] - hist_o[:, 2]) <= 1e-6 * np.abs(hist_o[:, 2]) + 1e-12)


SWEEP_LAYOUTS = [(1, 1, 1, 0), (2, 2, 2, 2), (4, 4, 4, 1), (4, 4, 4, 2), (8, 8, 8, 1), (8, 8, 8, 2),
                 (16, 16, 8, 1), (16, 16, 8, 2)]


@pytest.mark.parametrize("lay", SWEEP_LAYOUTS, ids=lambda l: "%dx%dx%d_o%d" % l)
def test_config4_every_layout_at_full_size(lay):
    """BASELINE.json configs[4]: every layout of the decomposition sweep on the 720x360 / 128-step
    problem, whichever kernel family serves it (generic for the large tiles, wavefront / row-marching
    for the small ones, incl. the ragged 22/23-row tiles of 16x16x8): sampled subdomains at perturbed
    controls, cost / parts / gradient element-wise / stored trajectory."""
    w = synth.CONFIGS[2].with_layout(*lay)
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob)
    n = o.nsub
    sample = sorted(set([0, n - 1, n // 2, n // 3 + 1, (2 * n) // 3, n // 5]))[:6] if n > 8 else list(range(n))
    check_sample(o, g, prob, sample, 17 + lay[0], traj=n > 1)
    if n == 1:      # the undecomposed layout is plain global 4D-Var: eval_global agrees as well
        x = prob.xb + 0.3 * prob.sigma_b[:, None, None] * synth.random_fields(prob.xb.shape, 3)
        Jo, go, _ = o.eval_global(x)
        Jg, gg = g.eval_global(x)
        assert abs(Jg - Jo) <= TOL_EVAL * abs(Jo) and rel(gg.cpu().numpy(), go) <= TOL_EVAL


def test_config3_gauss_newton_operator_on_sampled_subdomains():
    """SURVEY.md 8(f1) at the headline size: H_GN p (TLM sweep + adjoint sweep + control-level terms) of
    sampled subdomains of config 3 against the oracle, first / middle / last window, pole and interior tiles."""
    w = synth.CONFIGS[3]
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob)
    assert g.active_path == 5
    p12 = w.p_lon * w.p_lat
    sample = [0, 5 * 16 + 7, 3 * p12 + 15 * 16 + 15, 4 * p12 + 8 * 16 + 3, 7 * p12 + 2, 7 * p12 + 15 * 16]
    xs = g.get_controls()
    flat_p = g.torch.zeros_like(xs)
    ps = {}
    for k in sample:
        ps[k] = synth.random_fields(o.sub_shape(k), 500 + k)
        flat_p[g.offsets[k]:g.offsets[k + 1]] = g.torch.from_numpy(ps[k].reshape(-1)).to(flat_p.device)
    Hp = g.gn_hessvec(xs, flat_p)
    for k in sample:
        ref = o.gn_hessvec(k, o.get_control(k), ps[k])
        got = Hp[g.offsets[k]:g.offsets[k + 1]].cpu().numpy().reshape(ref.shape)
        assert rel(got, ref) <= 1e-10, (k, rel(got, ref))
        assert np.abs(got - ref).max() <= 1e-9 * np.abs(ref).max(), k


def test_config4_layout_with_the_overlap_penalty_on_every_level():
    """SURVEY.md 8(f4) at full size: the 4x4x4 o2 layout of config 4 (720x360, 32-step windows) with the spatial
    overlap penalty on every level of the window (generic kernels), sampled subdomains against the oracle."""
    w = synth.CONFIGS[2].with_layout(4, 4, 4, 2)
    o, prob = oracle_problem(w)
    o.set_overlap_levels(True)
    g = gpu_problem(w, prob, overlap_levels=True, path=1)
    check_sample(o, g, prob, [0, 5, 21, 38, 47, 63], 71)
