"""GPU-vs-oracle parity with the spatial overlap penalty on every level of the window (eq (21)
PAPER.md:300 read literally; option dd4dvar_set_overlap_levels, generic kernels)."""
import numpy as np
import pytest

from paper_2205_06649_b200 import synth
from helpers import oracle_problem, gpu_problem, rel, small_workload
from test_gpu_parity import LAYOUTS, check_eval_local, perturbed_controls

pytestmark = pytest.mark.gpu


def pair(name, path):
    w = small_workload(**LAYOUTS[name])
    o, prob = oracle_problem(w)
    o.set_overlap_levels(True)
    g = gpu_problem(w, prob, overlap_levels=True, path=path)
    return w, o, prob, g


@pytest.mark.parametrize("path", [1, 3])
@pytest.mark.parametrize("name", ["cfg0", "ragged3x2x3_o2", "cols4x1x1_o1", "wave_k2"])
def test_eval_local_with_all_level_overlap_matches_oracle(name, path):
    w, o, prob, g = pair(name, path)
    check_eval_local(o, g, [o.get_control(k) for k in range(o.nsub)])
    xs = perturbed_controls(o, prob, 11)
    check_eval_local(o, g, xs)
    # the option is switched on: the spatial-overlap part differs from the control-level reading
    o.set_overlap_levels(False)
    off = sum(o.eval_local(k, xs[k], want_grad=False)[0][3] for k in range(o.nsub))
    o.set_overlap_levels(True)
    on = sum(o.eval_local(k, xs[k], want_grad=False)[0][3] for k in range(o.nsub))
    assert on > 1.5 * off


@pytest.mark.parametrize("name", ["cfg0", "ragged3x2x3_o2"])
def test_run_with_all_level_overlap_matches_oracle(name):
    w, o, prob, g = pair(name, 1)
    an_o, hist_o = o.run(2)
    an_g, hist_g = g.run(2)
    an_g = an_g.cpu().numpy()
    for f in range(3):
        assert rel(an_g[f], an_o[f]) <= 1e-8, (f, rel(an_g[f], an_o[f]))
    assert np.all(np.abs(hist_g[:, :2] - hist_o[:, :2]) <= 1e-8 * np.abs(hist_o[:, :2]) + 1e-300), (hist_g, hist_o)
    assert np.all(np.abs(hist_g[:, 2] - hist_o[:, 2]) <= 1e-6 * np.abs(hist_o[:, 2]) + 1e-12)
    # evaluations on the exchanged data: the overlap store was refreshed from the neighbours' new trajectories
    check_eval_local(o, g, perturbed_controls(o, prob, 23, amp=0.3))


def test_option_is_refused_where_it_is_not_served():
    w = small_workload(**LAYOUTS["cfg0"])
    o, prob = oracle_problem(w)
    from paper_2205_06649_b200.binding import DD4DVar
    g = DD4DVar.from_workload(w)            # default path: wavefront kernels
    with pytest.raises(Exception) as e:
        g.set_overlap_levels(True)
    assert getattr(e.value, "code", 0) == -2
    g.set_background(prob.xb, prob.sigma_b)
    with pytest.raises(Exception) as e:
        g.set_overlap_levels(False)
    assert getattr(e.value, "code", 0) == -3


def test_gauss_newton_entry_points_refuse_the_all_level_overlap_penalty():
    """include/dd4dvar.h: dd4dvar_run_gn and dd4dvar_gn_hessvec return -2 while dd4dvar_set_overlap_levels is on
    (there is no Gauss-Newton path for the all-level penalty; running it would silently drop the term's curvature)."""
    from paper_2205_06649_b200.binding import DD4DVarError
    w = small_workload()
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob, overlap_levels=True, path=1)
    x = g.get_controls()
    with pytest.raises(DD4DVarError) as e1:
        g.gn_hessvec(x, x)
    with pytest.raises(DD4DVarError) as e2:
        g.run_gn(1, 1, 1)
    assert e1.value.code == -2 and e2.value.code == -2
    assert "overlap_levels" in str(e1.value)
    g.run(1)                                   # the L-BFGS driver still serves it
    g.close()
