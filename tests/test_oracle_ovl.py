"""Pins of the oracle's all-level overlap penalty (option `set_overlap_levels`): eq (25c) case 1
with the overlapping operator O_ik of eq (21) PAPER.md:300 read literally, i.e. acting on every level of the
window Delta_j and not on the control level only (R12 is the default).

Fixed by the mathematics, not by the oracle's output:
  * identity model (dt = 0, kappa = 0): every level equals the control, so the all-level term is exactly
    (W + 1) times the control-level term, for any control;
  * consistent data (iteration 0, control = background): the local trajectory IS the background trajectory on
    the extended tile, every overlap residual vanishes on every level;
  * the gradient is the derivative of the cost (centred differences), the Gauss-Newton operator the Hessian
    where the residuals vanish.
"""
import copy

import numpy as np

from paper_2205_06649_b200 import synth
from helpers import oracle_problem, small_workload, rel


def test_identity_model_all_level_term_is_w_plus_one_times_the_control_level_term():
    w = small_workload(nlon=36, nlat=18, dt=0.0, nsteps=12, p_lon=3, p_lat=2, q_time=2, overlap=2)
    o, prob = oracle_problem(w, diffusion=0.0)
    sb = prob.sigma_b[:, None, None]
    for k in range(o.nsub):
        x = o.get_control(k) + 0.8 * sb * synth.random_fields(o.sub_shape(k), 7 + k)
        W = o.subs[k]["e"] - o.subs[k]["s"]
        o.set_overlap_levels(False); p0, g0, _ = o.eval_local(k, x)
        o.set_overlap_levels(True); p1, g1, _ = o.eval_local(k, x)
        assert p0[3] > 0
        assert abs(p1[3] - (W + 1) * p0[3]) <= 1e-12 * p1[3], (k, p1[3], p0[3])
        for q in (1, 2, 4, 5):
            assert p1[q] == p0[q]
        assert abs(p1[0] - p0[0] - W * p0[3]) <= 1e-12 * p1[0]


def test_consistent_data_have_no_overlap_residual_on_any_level():
    w = small_workload(nlon=40, nlat=23, nsteps=17, p_lon=3, p_lat=2, q_time=3, overlap=2)
    o, prob = oracle_problem(w)
    o.set_overlap_levels(True)
    for k in range(o.nsub):
        parts, _, _ = o.eval_local(k, o.get_control(k))
        assert parts[3] <= 1e-20 * parts[0], (k, parts)
    # after an exchange the frozen trajectories come from the neighbours' stores (traj_prev): with controls that
    # do not move (n_inner = 0) they are again the background trajectory
    o2, _ = oracle_problem(w, n_inner=0)
    o2.set_overlap_levels(True)
    o2.run(1)
    for k in range(o2.nsub):
        parts, _, _ = o2.eval_local(k, o2.get_control(k))
        assert parts[3] <= 1e-20 * parts[0], (k, parts)


def test_gradient_with_all_level_overlap_matches_centred_differences():
    w = small_workload(nlon=36, nlat=18, nsteps=8, p_lon=2, p_lat=2, q_time=2, overlap=2)
    o, prob = oracle_problem(w)
    o.set_overlap_levels(True)
    sb = prob.sigma_b[:, None, None]
    for k in (0, 3, 5, 6):
        x = o.get_control(k) + 0.5 * sb * synth.random_fields(o.sub_shape(k), 21 + k)
        parts, g, _ = o.eval_local(k, x)
        assert parts[3] > 0.02 * parts[0]           # the overlap term matters in this test
        for seed in (1, 2):
            d = sb * synth.random_fields(o.sub_shape(k), 50 + seed)
            eps = 1e-5
            Jp = o.eval_local(k, x + eps * d, want_grad=False)[0][0]
            Jm = o.eval_local(k, x - eps * d, want_grad=False)[0][0]
            fd = (Jp - Jm) / (2 * eps)
            an = float(np.sum(g * d))
            assert abs(fd - an) <= 2e-7 * abs(an), (k, fd, an)


def test_gauss_newton_operator_with_all_level_overlap_is_the_hessian_where_residuals_vanish():
    w = small_workload(nlon=36, nlat=18, nsteps=12, p_lon=2, p_lat=2, q_time=3, overlap=1)
    o, prob = oracle_problem(w)
    o.set_overlap_levels(True)
    obs = copy.copy(prob.obs)
    tb = o.forecast(prob.xb, obs.levels)
    obs.value = np.concatenate([tb[t].reshape(-1)[obs.index[obs.offsets[t]:obs.offsets[t + 1]]]
                                for t in range(len(obs.levels))])
    o.set_observations(obs)
    sb = prob.sigma_b[:, None, None]
    for k in (0, 5, 11):
        x0 = o.get_control(k)
        p = synth.random_fields(o.sub_shape(k), 400 + k)
        Hp = o.gn_hessvec(k, x0, p)
        o.set_overlap_levels(False); Hp_off = o.gn_hessvec(k, x0, p); o.set_overlap_levels(True)
        assert rel(Hp, Hp_off) > 1e-3              # the option changes the operator
        eps = 1e-3
        fd = (sb * o.eval_local(k, x0 + eps * sb * p)[1] - sb * o.eval_local(k, x0 - eps * sb * p)[1]) / (2 * eps)
        assert rel(Hp, fd) <= 2e-6, (k, rel(Hp, fd))
