"""Host logic of the z-slab decomposition (paper_2012_08758_b200/slab.py) on the CPU.

1. The transport: ring_transfer with gloo at world_size 2 and 4: every rank's recv_lo holds the send_hi buffer of the
   rank below and its recv_hi the send_lo buffer of the rank above (periodic ring).
2. The schedule (Fig. 3: pack -> inner part beside the transfer -> unpack -> outer part): slab.py
   drives a numpy stand-in for binding.Context that implements the same calls (ac_set_slab, ac_halo_pack / unpack,
   ac_substep / ac_substep_part, ac_reduce_raw, ac_diag_combine) for a toy update with the path's data dependences: a
   radius-3 periodic stencil along z, a 2N register rebuilt from the previous buffer, a z-dependent forcing phase.
   The decomposed run (in one process and as 2 and 4 gloo ranks, with and without the inner / outer split) must
   equal the single-domain run bit for bit.  A wrong order of the calls (outer before the halo has landed, a missing
   exchange before the reductions, a stale send buffer) fails here without a GPU."""
import math
import os

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2012_08758_b200 import binding, slab

R = 3
W = np.array([0.05, -0.2, 0.6, 0.1, 0.6, -0.2, 0.05])      # any radius-3 stencil


class ToyContext:
    """numpy stand-in for binding.Context: state (7, nz, 1, 1) with z ghost planes; u_new = u + a (u - prev) +
    dt (sum_m W_m u(z + m) + cos(kz z + phase)); the calls and their ordering rules mirror include/ac_mhd.h."""

    def __init__(self, shape, lengths, dtype, device="cpu", **kw):
        self.nz = shape[0]
        self.lz = lengths[2]
        self.device = "cpu"
        self.stream = slab._HostStream()
        self.z0, self.nzg = 0, self.nz
        self.buf = [np.zeros((7, self.nz + 2 * R)), np.zeros((7, self.nz + 2 * R))]
        self.cur, self.next_substep, self.inner_done = 0, 0, -1
        self.halo_fresh = True

    def ac_set_variant(self, v):
        pass

    def ac_set_slab(self, z0, nzg):
        self.z0, self.nzg = z0, nzg

    def ac_halo_bytes(self):
        return 7 * R * 8

    def ac_load_state(self, state):
        self.buf[0][:, R:-R] = state.reshape(7, self.nz)
        self._wrap(0)
        self.cur, self.next_substep, self.inner_done = 0, 0, -1
        self.halo_fresh = self.nzg == self.nz

    def _wrap(self, b):
        if self.nzg == self.nz:                      # an ordinary periodic box fills its own ghost planes
            self.buf[b][:, :R] = self.buf[b][:, -2 * R:-R]
            self.buf[b][:, -R:] = self.buf[b][:, R:2 * R]

    def ac_halo_pack(self, lo, hi, stream=None):
        assert self.inner_done == -1
        u = self.buf[self.cur]
        lo.view(torch.float64).copy_(torch.from_numpy(u[:, R:2 * R].copy().ravel()))
        hi.view(torch.float64).copy_(torch.from_numpy(u[:, -2 * R:-R].copy().ravel()))

    def ac_halo_unpack(self, lo, hi, stream=None):
        u = self.buf[self.cur]
        u[:, :R] = lo.view(torch.float64).numpy().reshape(7, R)
        u[:, -R:] = hi.view(torch.float64).numpy().reshape(7, R)
        self.halo_fresh = True

    def _update(self, s, dt, forcing, z_lo, z_hi):
        u, prev = self.buf[self.cur], self.buf[1 - self.cur]
        a = [0.0, -0.4, -0.7][s]
        h = self.lz / self.nz
        for z in range(z_lo, z_hi):
            if z < R or z >= self.nz - R:
                assert self.halo_fresh, "boundary planes updated before the halo of this state has landed"
            rhs = (W * u[:, z:z + 2 * R + 1]).sum(axis=1)
            if forcing is not None:
                rhs = rhs + math.cos(forcing[0] * ((z + self.z0) * h) + forcing[1])
            prev[:, z + R] = u[:, z + R] + a * (u[:, z + R] - prev[:, z + R]) + dt * rhs

    def _finish(self, s):
        self.cur = 1 - self.cur
        self._wrap(self.cur)
        self.next_substep = (s + 1) % 3
        self.inner_done = -1
        self.halo_fresh = self.nzg == self.nz

    def ac_substep(self, s, dt, forcing):
        assert s == self.next_substep and self.inner_done == -1
        self._update(s, dt, forcing, 0, self.nz)
        self._finish(s)

    def ac_substep_part(self, s, dt, forcing, part):
        assert s == self.next_substep
        if part == binding.AC_PART_INNER:
            assert self.inner_done == -1
            self._update(s, dt, forcing, R, self.nz - R)
            self.inner_done = s
        else:
            assert self.inner_done == s
            self._update(s, dt, forcing, 0, R)
            self._update(s, dt, forcing, self.nz - R, self.nz)
            self._finish(s)

    def ac_store_state(self):
        return self.buf[self.cur][:, R:-R].reshape(7, self.nz, 1, 1).copy()

    def ac_reduce_raw(self):
        assert self.halo_fresh, "reductions need current z ghost planes (B = curl A reads them)"
        u = self.buf[self.cur]
        g = u[:, 2 * R:] - u[:, :-2 * R]              # something that reads the ghost planes
        return (float((u[:, R:-R] ** 2).sum()), float((u[:, R:-R] ** 2).max()), float((g ** 2).sum()),
                float((g ** 2).max()), float(u[0, R:-R].min()), float(u[0, R:-R].max()))

    def ac_diag_combine(self, raws):
        return {"su": sum(r[0] for r in raws), "mu": max(r[1] for r in raws), "sb": sum(r[2] for r in raws),
                "mb": max(r[3] for r in raws), "lmin": min(r[4] for r in raws), "lmax": max(r[5] for r in raws)}

    def ac_free(self):
        pass


NZ, LEN, DT = 64, (1.0, 1.0, 2 * math.pi), 0.05
FORCINGS = [None, (3.0, 0.4), (1.0, -1.1)]


def _initial():
    rng = np.random.default_rng(3)
    return rng.normal(size=(7, NZ, 1, 1))


def _single_domain():
    ctx = ToyContext((NZ, 1, 1), LEN, binding.AC_F64)
    ctx.ac_load_state(_initial())
    for f in FORCINGS:
        for s in range(3):
            ctx.ac_substep(s, DT, f)
    raw = ctx.ac_reduce_raw()
    return ctx.ac_store_state(), ctx.ac_diag_combine([raw])


def test_schedule_in_process_equals_single_domain():
    want, dwant = _single_domain()
    for world in (2, 4):
        for overlap in (True, False):
            grp = slab.SlabGroupInProcess((NZ, 1, 1), LEN, world, binding.AC_F64, overlap=overlap,
                                          context_factory=ToyContext)
            grp.load_state(_initial())
            for f in FORCINGS:
                grp.step(DT, f)
            d = grp.reduce()
            assert np.array_equal(grp.store_state(), want), (world, overlap)
            assert d["mu"] == dwant["mu"] and d["mb"] == dwant["mb"] and d["lmin"] == dwant["lmin"]
            assert abs(d["su"] - dwant["su"]) <= 1e-12 * dwant["su"] and abs(d["sb"] - dwant["sb"]) <= 1e-12 * dwant["sb"]


def _rank_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # 1. the transport alone
    n = 7 * R * 8
    mk = lambda tag: torch.full((n,), 10 * rank + tag, dtype=torch.uint8)
    recv_lo, recv_hi = torch.zeros(n, dtype=torch.uint8), torch.zeros(n, dtype=torch.uint8)
    slab.ring_transfer(mk(1), mk(2), recv_lo, recv_hi, dist, rank, world)
    ring = (int(recv_lo[0]), int(recv_lo[-1]), int(recv_hi[0]), int(recv_hi[-1]))
    # 2. the schedule, one process per rank
    rk = slab.SlabRank((NZ, 1, 1), LEN, dist, binding.AC_F64, device="cpu", overlap=rank % 2 == 0,
                       context_factory=ToyContext)
    rk.load_state(_initial())
    for f in FORCINGS:
        rk.step(DT, f)
    d = rk.reduce()
    out[rank] = (ring, rk.slab.ctx.ac_store_state(), d)
    dist.barrier()
    dist.destroy_process_group()


def _run_ranks(world, port):
    want, dwant = _single_domain()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_rank_worker, args=(world, port, out), nprocs=world, join=True)
    got = np.concatenate([out[r][1] for r in range(world)], axis=1)
    assert np.array_equal(got, want)
    for r in range(world):
        below, above = (r - 1) % world, (r + 1) % world
        assert out[r][0] == (10 * below + 2, 10 * below + 2, 10 * above + 1, 10 * above + 1)
        d = out[r][2]
        assert d["mu"] == dwant["mu"] and d["lmax"] == dwant["lmax"]
        assert abs(d["sb"] - dwant["sb"]) <= 1e-12 * dwant["sb"]


def test_schedule_and_ring_transfer_world2():
    _run_ranks(2, 29541)


def test_schedule_and_ring_transfer_world4():
    _run_ranks(4, 29543)


def test_local_lengths():
    assert slab.local_lengths((1.0, 2.0, 6.0), 3) == (1.0, 2.0, 2.0)
