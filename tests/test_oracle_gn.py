"""Pins of the oracle's Gauss-Newton local minimiser (oracle/dd4dvar_oracle.c O11):
incremental Gauss-Newton (Alg 5, Alg 6) with the normal equations
(42)-(43) PAPER.md:620-626 solved by CG in w = V^+ (u - u^b) (eq (44)-(46) PAPER.md:630-649).

What the mathematics fixes, none of it taken from the oracle's own output:
  * H_GN = 2 grad F^T grad F is symmetric: <H p, q> = <p, H q>;
  * where every residual vanishes the Gauss-Newton Hessian IS the Hessian of J_ji, so H_GN p equals the
    centred difference of the (already pinned) adjoint gradient;
  * with the identity model (dt = 0, kappa = 0) J is quadratic and separable, and one Gauss-Newton
    iteration with enough CG iterations reaches the BLUE / optimal-interpolation closed form cell by cell;
  * CG with k iterations minimises the quadratic model over the k-th Krylov space: the model value
    is non-increasing in k, and J_ji decreases on the real problem.
"""
import copy

import numpy as np

from paper_2205_06649_b200 import synth
from helpers import oracle_problem, small_workload, rel


def w_dot(a, b):
    return float(np.sum(a * b))


def test_gn_hessvec_is_symmetric_on_every_kind_of_subdomain():
    # 3x2x3 ragged layout: tiles with pole walls, first / middle / last window (predecessor, successor terms)
    w = small_workload(nlon=40, nlat=23, nsteps=17, p_lon=3, p_lat=2, q_time=3, overlap=2)
    o, prob = oracle_problem(w)
    sb = prob.sigma_b[:, None, None]
    for k in (0, 4, 8, 11, 13, 17):
        x = o.get_control(k) + 0.7 * sb * synth.random_fields(o.sub_shape(k), 100 + k)
        p = synth.random_fields(o.sub_shape(k), 200 + k)
        q = synth.random_fields(o.sub_shape(k), 300 + k)
        Hp, Hq = o.gn_hessvec(k, x, p), o.gn_hessvec(k, x, q)
        a, b = w_dot(Hp, q), w_dot(p, Hq)
        assert abs(a - b) <= 1e-12 * max(abs(a), abs(b)), (k, a, b)
        assert w_dot(p, Hp) > 0.0               # positive definite: mu > 0 or the background term


def test_gn_hessian_equals_hessian_of_J_where_all_residuals_vanish():
    """Observations sampled WITHOUT noise from the background's own trajectory: at iteration 0 the
    control u^b(s_j), the frozen neighbour data and the observations are all consistent, F_ji = 0, and the
    second-order term sum F_i Hess(F_i) that Gauss-Newton drops (Remark 3) vanishes.  Then
    H_GN p = d/d eps grad J(w + eps p), here by centred differences of the adjoint gradient."""
    w = small_workload(nlon=36, nlat=18, nsteps=12, p_lon=2, p_lat=2, q_time=3, overlap=1)
    o, prob = oracle_problem(w)
    obs = copy.copy(prob.obs)
    tb = o.forecast(prob.xb, obs.levels)
    vals = [tb[t].reshape(-1)[obs.index[obs.offsets[t]:obs.offsets[t + 1]]] for t in range(len(obs.levels))]
    obs.value = np.concatenate(vals)
    o.set_observations(obs)
    sb = prob.sigma_b[:, None, None]
    for k in (0, 3, 5, 6, 9, 11):
        x0 = o.get_control(k)
        parts, g0, _ = o.eval_local(k, x0)
        assert parts[0] <= 1e-18 * np.sum((x0 / sb) ** 2) and np.abs(g0).max() <= 1e-9 * np.abs(1.0 / sb).max()
        p = synth.random_fields(o.sub_shape(k), 400 + k)
        Hp = o.gn_hessvec(k, x0, p)
        eps = 1e-3
        gp = sb * o.eval_local(k, x0 + eps * sb * p)[1]
        gm = sb * o.eval_local(k, x0 - eps * sb * p)[1]
        fd = (gp - gm) / (2 * eps)
        assert rel(Hp, fd) <= 2e-6, (k, rel(Hp, fd))
        # element-wise too: a wrong weight on a few overlap cells cannot hide under the norm
        assert np.abs(Hp - fd).max() <= 1e-5 * np.abs(fd).max(), k


def test_one_gauss_newton_iteration_reaches_the_blue_closed_form_for_the_identity_model():
    """dt = 0 and kappa = 0: Phi = identity, H = selection.  Undecomposed layout (eq (6)):
    J(x) = sum (x - x_b)^2 / s_b^2 + sum_levels sum_obs (x[idx] - y)^2 / s_o^2 is separable, minimised by
    x* = (x_b / s_b^2 + sum_k y_k / s_o^2) / (1 / s_b^2 + n_k / s_o^2) in observed cells, x_b elsewhere.
    H_GN in w-space is diagonal; the gradient at x_b lives on the observed cells, where H_GN takes three
    distinct values (one per field: the ratios s_b / s_o differ), so 3 CG iterations solve it exactly."""
    w = small_workload(nlon=24, nlat=12, dt=0.0, nsteps=6, p_lon=1, p_lat=1, q_time=1, overlap=0, obs_frac=0.4,
                       obs_every=2)
    o, prob = oracle_problem(w, diffusion=0.0)
    obs = copy.copy(prob.obs)
    obs.sigma_o = prob.obs.sigma_o * np.array([1.0, 2.0, 3.5])      # three distinct ratios s_b / s_o
    o.set_observations(obs)
    num = prob.xb / prob.sigma_b[:, None, None] ** 2
    den = np.ones_like(prob.xb) / prob.sigma_b[:, None, None] ** 2
    ncell = w.nlon * w.nlat
    for t in range(len(obs.levels)):
        idx = obs.index[obs.offsets[t]:obs.offsets[t + 1]]
        so2 = obs.sigma_o[idx // ncell] ** 2
        np.add.at(num.reshape(-1), idx, obs.value[obs.offsets[t]:obs.offsets[t + 1]] / so2)
        np.add.at(den.reshape(-1), idx, 1.0 / so2)
    xstar = num / den
    x1, J0, J1 = o.gn_local(0, prob.xb, 1, 6)
    assert rel(x1, xstar) <= 1e-12
    assert np.abs(x1 - xstar).max() <= 1e-10 * np.abs(xstar).max()
    assert J1 < J0
    g1 = o.eval_local(0, x1)[1]
    assert np.abs(g1 * prob.sigma_b[:, None, None]).max() <= 1e-8 * np.sqrt(J0)
    # with too few CG iterations the step is the Krylov minimiser, not x*
    x2, _, J2 = o.gn_local(0, prob.xb, 1, 1)
    assert rel(x2 - prob.xb, xstar - prob.xb) > 1e-3 and J1 < J2 < J0
    x3, _, J3 = o.gn_local(0, prob.xb, 1, 3)
    assert rel(x3, xstar) <= 1e-12


def test_gauss_newton_decreases_J_and_dd_iteration_with_it_decreases_the_global_cost():
    w = synth.CONFIGS[0]
    o, prob = oracle_problem(w)
    sb = prob.sigma_b[:, None, None]
    for k in range(o.nsub):
        x0 = o.get_control(k)
        _, Ja, Jb = o.gn_local(k, x0, 1, 3)
        _, _, Jc = o.gn_local(k, x0, 2, 6)
        assert Jb < Ja and Jc <= Jb * (1 + 1e-12), (k, Ja, Jb, Jc)
    an, hist = o.run_gn(3, 2, 5)
    assert np.all(np.isfinite(hist))
    assert hist[-1, 0] < hist[0, 0]
    # zero Gauss-Newton iterations leave the background in place
    o2, _ = oracle_problem(w)
    an0, h0 = o2.run_gn(1, 0, 5)
    assert rel(an0, prob.xb) <= 1e-15 and h0[1, 2] == 0.0
