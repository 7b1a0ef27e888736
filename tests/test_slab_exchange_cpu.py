"""Host logic of the z-slab halo exchange (paper_2012_08758_b200/slab.py) with gloo on the CPU, world_size 2 and 3:
every rank's lower ghost planes receive the upper boundary planes of the rank below and vice versa (periodic ring),
for all 7 fields, and the combined diagnostics follow the sum / max rules."""
import math
import os

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2012_08758_b200 import slab


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    n = 3 * 5 * 4                                           # 3 planes of a 5 x 4 padded plane
    mk = lambda tag: [torch.full((n,), float(100 * rank + 10 * q + tag), dtype=torch.float64) for q in range(7)]
    send_up, send_dn = mk(1), mk(2)
    recv_lo = [torch.zeros(n, dtype=torch.float64) for _ in range(7)]
    recv_hi = [torch.zeros(n, dtype=torch.float64) for _ in range(7)]
    slab.ring_exchange(send_up, send_dn, recv_lo, recv_hi, dist, rank, world)
    out[rank] = ([float(t[0]) for t in recv_lo], [float(t[-1]) for t in recv_hi])
    dist.barrier()
    dist.destroy_process_group()


def _run(world, port):
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    for r in range(world):
        below, above = (r - 1) % world, (r + 1) % world
        lo, hi = out[r]
        assert lo == [100.0 * below + 10 * q + 1 for q in range(7)]     # the rank below sent its "up" planes
        assert hi == [100.0 * above + 10 * q + 2 for q in range(7)]     # the rank above sent its "down" planes


def test_ring_exchange_world2():
    _run(2, 29541)


def test_ring_exchange_world3():
    _run(3, 29543)


def test_combine_raw_and_rank_forcing():
    raws = [(1.0, 0.25, 2.0, 0.5, -0.1, 0.2), (3.0, 0.16, 6.0, 0.75, -0.3, 0.1)]
    d = slab.combine_raw(raws, 8, 0.1, 1e-3, 2e-3, 1.0)
    assert d["urms"] == math.sqrt(4.0 / 8) and d["brms"] == math.sqrt(8.0 / 8)
    assert d["umax"] == 0.5 and d["bmax"] == math.sqrt(0.75)
    assert d["lnrho_min"] == -0.3 and d["lnrho_max"] == 0.2
    assert d["dt_cfl"] == min(0.4 * 0.1 / 1.5, 0.25 * 0.01 / 2e-3)
    f = ((1.0, 2.0, 3.0), 0.5, (1, 0, 0), (0, 1, 0))
    assert slab.rank_forcing(f, 2.0) == ((1.0, 2.0, 3.0), 0.5 + 6.0, (1, 0, 0), (0, 1, 0))
    assert slab.rank_forcing(None, 1.0) is None
    assert slab.local_lengths((1.0, 2.0, 6.0), 3) == (1.0, 2.0, 2.0)
