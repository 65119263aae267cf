"""Writes tests/golden/oracle_config0_history.txt.  Calls only oracle/ and the seeded input
generator; nothing here touches the CUDA path."""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from oracle import Oracle  # noqa: E402
from paper_2205_06649_b200 import synth  # noqa: E402


def main():
    w = synth.CONFIGS[0]
    o = Oracle.from_workload(w)
    prob = synth.make_problem(w, o.forecast)
    o.set_background(prob.xb, prob.sigma_b)
    o.set_observations(prob.obs)
    an, hist = o.run(3)
    with open(os.path.join(HERE, "oracle_config0_history.txt"), "w") as f:
        f.write("# oracle.run(3) on BASELINE.json configs[0]: J(gathered analysis), sum_ji J_ji, delta_l; "
                "last line: ||analysis||_2 per field (h,u,v)\n")
        for row in hist:
            f.write(" ".join(repr(float(v)) for v in row) + "\n")
        f.write(" ".join(repr(float(np.linalg.norm(an[k]))) for k in range(3)) + "\n")


if __name__ == "__main__":
    main()
