"""Worker of tests/test_gpu_sharded.py::test_two_ranks_over_nccl_reproduce_the_single_run (launched with torchrun, one
process per GPU): the window-sharded driver over NCCL must return the single-GPU run bit for bit."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)

from paper_2205_06649_b200 import parallel, synth  # noqa: E402
from paper_2205_06649_b200.binding import DD4DVar  # noqa: E402
from helpers import small_workload  # noqa: E402
from test_gpu_parity import LAYOUTS  # noqa: E402


def main():
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    dist.init_process_group("nccl", device_id=torch.device(dev))
    for name in ("wave_k2", "ragged3x2x3_o2"):
        w = small_workload(**LAYOUTS[name])
        single = DD4DVar.from_workload(w, device=dev)
        prob = synth.make_problem(w, single.forecast)
        single.set_background(prob.xb, prob.sigma_b); single.set_observations(prob.obs)
        an_s, hist_s = single.run(3)
        # the library on a stream of its own, not torch's current stream: the exchange must order itself against it
        side = torch.cuda.Stream(device=dev)
        sh = parallel.ShardedDD4DVar(w, device=dev, stream=side)
        sh.set_background(prob.xb, prob.sigma_b); sh.set_observations(prob.obs)
        an, hist = sh.run(3)
        assert np.array_equal(an.cpu().numpy(), an_s.cpu().numpy()), name
        assert np.allclose(hist[1:, 0], hist_s[1:, 1], rtol=1e-13) and np.array_equal(hist[1:, 1], hist_s[1:, 2]), name
        sh.close(); single.close()
    dist.barrier()
    if dist.get_rank() == 0:
        print("nccl shard worker ok")
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
