"""Fixtures under tests/golden: values the paper prints, and the oracle's regression pin."""
import os

import numpy as np

from oracle import Oracle
from paper_2205_06649_b200 import synth

G = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def rows(name):
    return [l.split() for l in open(os.path.join(G, name)) if l.strip() and not l.startswith("#")]


def test_paper_table3_problem_sizes_from_the_oracle_geometry():
    """Table 3 (l.1045-1047): QP subdomains of n_loc = 32 give QP*3*32^2 unknowns."""
    layouts = {2: (2, 1, 1), 4: (2, 2, 1), 8: (2, 2, 2), 16: (4, 2, 2), 32: (4, 4, 2), 64: (4, 4, 4)}
    for qp, printed in rows("paper_table3_problem_sizes.txt"):
        p1, p2, q = layouts[int(qp)]
        o = Oracle(32 * p1, 32 * p2, 100.0, 4 * q, p1, p2, q, 0)
        owned = sum(3 * (s["oi1"] - s["oi0"]) * (s["oj1"] - s["oj0"]) for s in o.subs)
        assert o.nsub == int(qp) and owned == int(qp) * 3 * 32 * 32
        assert float("%.1e" % owned) == float(printed) or abs(owned - float(printed)) <= 0.05 * float(printed)


def test_paper_def4_weights():
    """Def 4 (l.164-170) in the 1-D-space picture: a 1 x p_lat band layout with 2 windows."""
    o = Oracle(36, 20, 100.0, 8, 1, 2, 2, 1)
    seen = {}
    for k in range(o.nsub):
        s = o.subs[k]
        for level in (s["s"], s["s"] + 1, s["e"]):
            wt = o.sub_weight(k, level)
            mt = 2 if level == 4 else 1
            for lj in range(s["ey"]):
                gj = s["ej0"] + lj
                ms = 2 if 9 <= gj <= 10 else 1
                seen[(mt, ms)] = wt[lj, 0]
    for mt, ms, wgt in rows("paper_def4_weights.txt"):
        assert seen[(int(mt), int(ms))] == float(wgt)


def test_oracle_config0_history_regression():
    w = synth.CONFIGS[0]
    o = Oracle.from_workload(w)
    prob = synth.make_problem(w, o.forecast)
    o.set_background(prob.xb, prob.sigma_b)
    o.set_observations(prob.obs)
    an, hist = o.run(3)
    ref = np.array([[float(v) for v in r] for r in rows("oracle_config0_history.txt")])
    assert np.allclose(hist, ref[:-1], rtol=1e-9, atol=0)
    assert np.allclose([np.linalg.norm(an[k]) for k in range(3)], ref[-1], rtol=1e-11)
