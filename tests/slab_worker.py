"""Worker of tests/test_slab_gpu.py: one rank of a z-slab run under torchrun.  gloo: two ranks share cuda:0 (safe: no
kernel waits on another rank, the exchange is staged through the host).  nccl: ONE rank, which is its own neighbour
above and below, so that the stream-ordered NCCL transport (slab.ring_transfer on the communication stream, no host
synchronisation) runs for real on one GPU."""
import math
import os
import sys

import numpy as np
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2012_08758_b200 import binding, inputs, slab  # noqa: E402


def main():
    out_dir = sys.argv[1]
    backend = sys.argv[2] if len(sys.argv) > 2 else "gloo"
    transport = sys.argv[3] if len(sys.argv) > 3 else "buffers"
    if backend == "nccl":
        import torch
        torch.cuda.set_device(0)
        dist.init_process_group("nccl", device_id=torch.device("cuda", 0))
    else:
        dist.init_process_group("gloo")
    shape = (32, 24, 32)
    lengths = (2 * math.pi, 1.5 * math.pi, 3.0 * math.pi)
    state = inputs.smooth_strong_state(shape, 41)
    rk = slab.SlabRank(shape, lengths, dist, binding.AC_F64, transport=transport, nu=5e-3, eta=4e-3, cs=1.0, k_f=3,
                       helicity=1.0)
    rk.load_state(state)
    dt = 2e-3
    for s in range(2):
        f = rk.forcing_from_draws(0.3 + 0.1 * s, 0.6, 0.2, dt, 0.02)       # of the global box
        rk.step(dt, f)
    d = rk.reduce()
    np.save(os.path.join(out_dir, "slab_%d.npy" % rk.rank), rk.slab.ctx.ac_store_state())
    if rk.rank == 0:
        np.save(os.path.join(out_dir, "diag.npy"), np.array([d["urms"], d["brms"], d["umax"], d["bmax"], d["dt_cfl"]]))
    dist.barrier()
    rk.free()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
