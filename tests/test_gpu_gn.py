"""GPU-vs-oracle parity of the Gauss-Newton local minimiser (Alg 5-7)
through the C-ABI: the operator H_GN (tangent-linear sweep + adjoint sweep + control-level terms) at 1e-10,
the DD iteration driven by it at the tolerances of the L-BFGS path (analysis 1e-8)."""
import numpy as np
import pytest

from paper_2205_06649_b200 import synth
from helpers import oracle_problem, gpu_problem, rel, small_workload
from test_gpu_parity import LAYOUTS

pytestmark = pytest.mark.gpu

GN_LAYOUTS = ["cfg0", "wave_fit100", "wave_px76", "wave_k2"]


def pair(name, path=0):
    w = small_workload(**LAYOUTS[name])
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob, path=path)
    assert g.active_path == (path or 5)
    return w, o, prob, g


GENERIC = [("ragged3x2x3_o2", 1), ("bands1x3x2", 1), ("undecomposed", 1), ("cfg0", 3), ("time_only", 1)]


@pytest.mark.parametrize("name", GN_LAYOUTS)
def test_gn_operator_matches_oracle(name):
    w, o, prob, g = pair(name)
    sb = prob.sigma_b[:, None, None]
    xs = [o.get_control(k) + 0.6 * sb * synth.random_fields(o.sub_shape(k), 31 + k) for k in range(o.nsub)]
    ps = [synth.random_fields(o.sub_shape(k), 77 + k) for k in range(o.nsub)]
    Hp = [t.cpu().numpy() for t in g.split(g.gn_hessvec(g.pack(xs), g.pack(ps)))]
    for k in range(o.nsub):
        ref = o.gn_hessvec(k, xs[k], ps[k])
        assert rel(Hp[k], ref) <= 1e-10, (k, rel(Hp[k], ref))
        assert np.abs(Hp[k] - ref).max() <= 1e-9 * np.abs(ref).max(), k
    # symmetry on the GPU side as well (oracle-independent)
    qs = [synth.random_fields(o.sub_shape(k), 99 + k) for k in range(o.nsub)]
    Hq = [t.cpu().numpy() for t in g.split(g.gn_hessvec(g.pack(xs), g.pack(qs)))]
    for k in range(o.nsub):
        a, b = float(np.sum(Hp[k] * qs[k])), float(np.sum(ps[k] * Hq[k]))
        assert abs(a - b) <= 1e-11 * max(abs(a), abs(b)), (k, a, b)


@pytest.mark.parametrize("name", GN_LAYOUTS)
def test_run_gn_matches_oracle(name):
    w, o, prob, g = pair(name)
    an_o, hist_o = o.run_gn(2, 2, 4)
    an_g, hist_g = g.run_gn(2, 2, 4)
    an_g = an_g.cpu().numpy()
    for f in range(3):
        assert rel(an_g[f], an_o[f]) <= 1e-8, (f, rel(an_g[f], an_o[f]))
    assert rel(an_g - prob.xb, an_o - prob.xb) <= 1e-6
    assert np.all(np.abs(hist_g[:, :2] - hist_o[:, :2]) <= 1e-8 * np.abs(hist_o[:, :2]) + 1e-300), (hist_g, hist_o)
    assert np.all(np.abs(hist_g[:, 2] - hist_o[:, 2]) <= 1e-6 * np.abs(hist_o[:, 2]) + 1e-12)
    ctr = [t.cpu().numpy() for t in g.split(g.get_controls())]
    for k in range(o.nsub):
        assert rel(ctr[k], o.get_control(k)) <= 1e-8, k


@pytest.mark.parametrize("name,path", GENERIC)
def test_gn_on_generic_layouts_matches_oracle(name, path):
    """Any layout through the generic kernels: the operator and the driver."""
    w, o, prob, g = pair(name, path)
    sb = prob.sigma_b[:, None, None]
    xs = [o.get_control(k) + 0.6 * sb * synth.random_fields(o.sub_shape(k), 31 + k) for k in range(o.nsub)]
    ps = [synth.random_fields(o.sub_shape(k), 77 + k) for k in range(o.nsub)]
    Hp = [t.cpu().numpy() for t in g.split(g.gn_hessvec(g.pack(xs), g.pack(ps)))]
    for k in range(o.nsub):
        ref = o.gn_hessvec(k, xs[k], ps[k])
        assert rel(Hp[k], ref) <= 1e-10, (k, rel(Hp[k], ref))
        assert np.abs(Hp[k] - ref).max() <= 1e-9 * np.abs(ref).max(), k
    an_o, hist_o = o.run_gn(2, 2, 3)
    an_g, hist_g = g.run_gn(2, 2, 3)
    an_g = an_g.cpu().numpy()
    for f in range(3):
        assert rel(an_g[f], an_o[f]) <= 1e-8, (f, rel(an_g[f], an_o[f]))
    assert np.all(np.abs(hist_g[:, :2] - hist_o[:, :2]) <= 1e-8 * np.abs(hist_o[:, :2]) + 1e-300), (hist_g, hist_o)


def test_run_gn_refuses_the_row_marching_paths():
    w = small_workload(**LAYOUTS["cfg0"])
    o, prob = oracle_problem(w)
    g = gpu_problem(w, prob, path=2)
    with pytest.raises(Exception) as e:
        g.run_gn(1, 1, 1)
    assert getattr(e.value, "code", 0) == -2
