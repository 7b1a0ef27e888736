"""z-slab decomposition of the box over several ranks: host-side orchestration only.

Every rank owns nz / p planes and runs the ordinary single-GPU context on them (its ac_grid has nz = nz_local and
lz = L_z / p).  After every substep the 3 ghost planes per side of all 7 fields are replaced by the neighbour ranks'
boundary planes; in the padded device layout those are contiguous blocks, so the exchange is plain copies: peer
sends/receives through torch.distributed (one process per GPU, NCCL) or, for several slabs held by one process on one
GPU (the test set-up), device-to-device copies.  No kernel waits on another rank.  The reductions are combined from
the ranks' raw sums.  Only layouts without packed fp32 pairs can be exchanged this way: fp64, or fp32 with the direct
kernel variant.
"""
import math

import numpy as np

from . import binding

R = 3


def local_lengths(lengths, world):
    lx, ly, lz = lengths
    return (lx, ly, lz / world)


def rank_forcing(forcing, z0):
    """The forcing of Eq. 4 seen from a slab whose first plane sits at z0: phase + k_z z0."""
    if forcing is None:
        return None
    if isinstance(forcing, binding.AcForcing):
        forcing = (tuple(forcing.k), forcing.phase, tuple(forcing.re), tuple(forcing.im))
    k, phase, re, im = forcing
    return (k, phase + k[2] * z0, re, im)


class Slab:
    """One rank's context plus views of its halo planes."""

    def __init__(self, global_shape, lengths, rank, world, dtype=binding.AC_F64, **kw):
        import torch
        nz, ny, nx = global_shape
        if nz % world != 0 or nz // world < 8:
            raise binding.AcError("nz must split into slabs of at least 8 planes")
        self.rank, self.world, self.nzl = rank, world, nz // world
        self.z0 = rank * self.nzl * (lengths[2] / nz)
        self.ctx = binding.Context((self.nzl, ny, nx), local_lengths(lengths, world), dtype, **kw)
        if dtype == binding.AC_F32:
            self.ctx.ac_set_variant(1)              # plain float layout: ghost planes are plain planes
        info = self.ctx.ac_state_layout()
        if info.packed_pairs:
            raise binding.AcError("packed fp32 pairs cannot be exchanged plane-wise")
        self.info = info
        self.tdtype = torch.float64 if info.elem_bytes == 8 else torch.float32
        self._flat = self.ctx.workspace.view(torch.uint8)

    def _planes(self, q, first):
        """torch view of 3 padded planes of field q of the current state, starting at padded plane `first`."""
        import torch
        base = self.ctx.ac_field_device_ptr(q) - self._flat.data_ptr()
        eb = self.info.elem_bytes
        start = base + first * self.info.plane_elems * eb
        n = R * self.info.plane_elems
        return self._flat[start:start + n * eb].view(self.tdtype)

    def halo(self):
        """(send_up, send_dn, recv_lo, recv_hi): lists of 7 views each."""
        nzl = self.nzl
        return ([self._planes(q, nzl) for q in range(7)], [self._planes(q, R) for q in range(7)],
                [self._planes(q, 0) for q in range(7)], [self._planes(q, nzl + R) for q in range(7)])


def exchange_in_process(slabs):
    """All slabs live in this process on one device: ghost planes <- neighbours' boundary planes."""
    p = len(slabs)
    halos = [s.halo() for s in slabs]
    for r in range(p):
        up, dn = halos[(r - 1) % p][0], halos[(r + 1) % p][1]
        for q in range(7):
            halos[r][2][q].copy_(up[q])
            halos[r][3][q].copy_(dn[q])


def ring_exchange(send_up, send_dn, recv_lo, recv_hi, dist, rank, world):
    """One process per rank: 2 sends and 2 receives of the 7 fields' planes, staged in one buffer each.
    send_up goes to rank + 1 (its lower ghost planes), send_dn to rank - 1 (its upper ghost planes)."""
    import torch
    up, dn = (rank + 1) % world, (rank - 1) % world
    s_up, s_dn = torch.stack(list(send_up)), torch.stack(list(send_dn))
    if s_up.is_cuda and dist.get_backend() != "nccl":
        # gloo moves host memory: stage through the CPU (test set-up: several ranks sharing one GPU)
        s_up, s_dn = s_up.cpu(), s_dn.cpu()
    r_lo, r_hi = torch.empty_like(s_up), torch.empty_like(s_dn)
    ops = [dist.P2POp(dist.isend, s_up, up), dist.P2POp(dist.isend, s_dn, dn),
           dist.P2POp(dist.irecv, r_lo, dn), dist.P2POp(dist.irecv, r_hi, up)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    for q in range(len(recv_lo)):
        recv_lo[q].copy_(r_lo[q])
        recv_hi[q].copy_(r_hi[q])


def combine_raw(raws, ncell_global, h, nu, eta, cs, c_u=0.4, c_nu=0.25):
    """Diagnostics of the whole box from the ranks' ac_reduce_raw tuples (G15, G18)."""
    su = sum(r[0] for r in raws)
    sb = sum(r[2] for r in raws)
    mu = max(r[1] for r in raws)
    mb = max(r[3] for r in raws)
    umax = math.sqrt(mu)
    dt = c_u * h / (umax + cs)
    if max(nu, eta) > 0:
        dt = min(dt, c_nu * h * h / max(nu, eta))
    return {"urms": math.sqrt(su / ncell_global), "umax": umax, "brms": math.sqrt(sb / ncell_global),
            "bmax": math.sqrt(mb), "lnrho_min": min(r[4] for r in raws), "lnrho_max": max(r[5] for r in raws),
            "dt_cfl": dt}


class SlabGroupInProcess:
    """p slabs of one box driven by one process on one GPU: the reference behaviour of the decomposition."""

    def __init__(self, global_shape, lengths, world, dtype=binding.AC_F64, **kw):
        self.shape, self.lengths, self.kw = tuple(global_shape), tuple(lengths), kw
        self.slabs = [Slab(global_shape, lengths, r, world, dtype, **kw) for r in range(world)]

    def load_state(self, state):
        nzl = self.slabs[0].nzl
        for s in self.slabs:
            s.ctx.ac_load_state(np.ascontiguousarray(state[:, s.rank * nzl:(s.rank + 1) * nzl]))
        exchange_in_process(self.slabs)

    def step(self, dt, forcing=None):
        for sub in range(3):
            for s in self.slabs:
                s.ctx.ac_substep(sub, dt, rank_forcing(forcing, s.z0))
            exchange_in_process(self.slabs)

    def store_state(self):
        return np.concatenate([s.ctx.ac_store_state() for s in self.slabs], axis=1)

    def reduce(self):
        nz, ny, nx = self.shape
        h = min(self.lengths[0] / nx, self.lengths[1] / ny, self.lengths[2] / nz)
        return combine_raw([s.ctx.ac_reduce_raw() for s in self.slabs], nz * ny * nx, h, self.kw.get("nu", 0.0),
                           self.kw.get("eta", 0.0), self.kw.get("cs", 1.0))

    def free(self):
        for s in self.slabs:
            s.ctx.ac_free()


class SlabRank:
    """One process per rank (torchrun): this rank's slab of the box, exchanged through torch.distributed."""

    def __init__(self, global_shape, lengths, dist, dtype=binding.AC_F64, device="cuda:0", **kw):
        self.dist, self.rank, self.world = dist, dist.get_rank(), dist.get_world_size()
        self.shape, self.lengths, self.kw = tuple(global_shape), tuple(lengths), kw
        self.slab = Slab(global_shape, lengths, self.rank, self.world, dtype, device=device, **kw)

    def forcing_from_draws(self, u1, u2, u3, dt, f0):
        """Eq. 4-6 for the GLOBAL box (the slab's own context would take its shorter l_z for the box length)."""
        f = binding.ac_forcing_params(self.kw.get("k_f", 3.0), self.kw.get("helicity", 0.0), self.kw.get("cs", 1.0),
                                      self.shape, self.lengths, u1, u2, u3, dt, f0)
        return (tuple(f.k), f.phase, tuple(f.re), tuple(f.im))

    def exchange(self):
        if self.world == 1:
            return                                  # the rank's own periodic images are already right
        self.slab.ctx.synchronize()
        ring_exchange(*self.slab.halo(), self.dist, self.rank, self.world)

    def load_state(self, state):
        """state: the GLOBAL (7, nz, ny, nx) array (every rank generates the same seeded input) or this rank's slab."""
        nzl = self.slab.nzl
        if state.shape[1] != nzl:
            state = state[:, self.rank * nzl:(self.rank + 1) * nzl]
        self.slab.ctx.ac_load_state(np.ascontiguousarray(state))
        self.exchange()

    def step(self, dt, forcing=None):
        f = rank_forcing(forcing, self.slab.z0)
        for sub in range(3):
            self.slab.ctx.ac_substep(sub, dt, f)
            self.exchange()

    def reduce(self):
        import torch
        raw = torch.tensor(self.slab.ctx.ac_reduce_raw(), dtype=torch.float64)
        if self.world > 1:
            allr = [torch.empty_like(raw) for _ in range(self.world)]
            dev = raw.cuda() if self.dist.get_backend() == "nccl" else raw
            allr = [torch.empty_like(dev) for _ in range(self.world)]
            self.dist.all_gather(allr, dev)
            raws = [tuple(t.cpu().tolist()) for t in allr]
        else:
            raws = [tuple(raw.tolist())]
        nz, ny, nx = self.shape
        h = min(self.lengths[0] / nx, self.lengths[1] / ny, self.lengths[2] / nz)
        return combine_raw(raws, nz * ny * nx, h, self.kw.get("nu", 0.0), self.kw.get("eta", 0.0), self.kw.get("cs", 1.0))
