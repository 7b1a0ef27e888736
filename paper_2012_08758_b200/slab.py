"""z-slab decomposition of the box over several ranks: host-side orchestration only, no
arithmetic of the method (the phase shift of the forcing, the halo lanes of packed fp32 pairs and the combination of
the diagnostics all live behind the C ABI: ac_set_slab, ac_halo_pack / ac_halo_unpack, ac_diag_combine).

Every rank owns nz / p planes and runs the ordinary context on them.  A substep follows the paper's schedule
(Fig. 3): the halo of the current state travels on a second stream (pack -> send / receive -> unpack)
WHILE the inner planes are updated on the compute stream; the 3 + 3 boundary planes follow once the halo has landed.
Transport: torch.distributed point-to-point operations on the dense halo buffers (NCCL between GPUs; gloo with host
staging for the multi-process test on one GPU), or device-to-device copies for several slabs held by one process (the
one-GPU emulation).  transport="pull" replaces pack / send / receive / unpack by ONE kernel that reads the neighbours'
boundary planes straight from their state arrays (ac_halo_pull): device pointers inside a process, CUDA IPC mappings
between processes (peer memory over NVLink between GPUs), ordered by events (interprocess events between processes,
whose record / wait calls a host barrier keeps in sequence).  No kernel waits on another rank.
"""
import numpy as np

from . import binding

R = 3


def local_lengths(lengths, world):
    lx, ly, lz = lengths
    return (lx, ly, lz / world)


class _HostStream:
    """Stand-in for a CUDA stream / event when a context lives on the host (the CPU tests of the schedule drive this
    module with a numpy stand-in for binding.Context): every call completes before it returns."""
    cuda_stream = 0

    def wait_event(self, ev):
        pass

    def wait_stream(self, st):
        pass

    def synchronize(self):
        pass

    def record(self, st=None):
        pass


class Slab:
    """One rank's context, its halo buffers and its two streams."""

    def __init__(self, global_shape, lengths, rank, world, dtype=binding.AC_F64, variant=0, context_factory=None,
                 interprocess=False, **kw):
        import torch
        nz, ny, nx = global_shape
        if nz % world != 0 or nz // world < 8:
            raise binding.AcError("nz must split into slabs of at least 8 planes")
        self.rank, self.world, self.nzl = rank, world, nz // world
        make = context_factory or binding.Context
        self.ctx = make((self.nzl, ny, nx), local_lengths(lengths, world), dtype, **kw)
        self.ctx.ac_set_variant(variant)
        self.ctx.ac_set_slab(rank * self.nzl, nz)
        dev = self.ctx.device
        nb = self.ctx.ac_halo_bytes()
        self.send_lo, self.send_hi, self.recv_lo, self.recv_hi = (torch.empty(nb, dtype=torch.uint8, device=dev)
                                                                  for _ in range(4))
        if torch.device(dev).type == "cuda":
            with torch.cuda.device(dev):
                self.comm = torch.cuda.Stream(device=dev)
            self.state_ready = torch.cuda.Event(interprocess=True) if interprocess else torch.cuda.Event()
            self.halo_ready = torch.cuda.Event()
        else:
            self.comm = self.state_ready = self.halo_ready = _HostStream()
        self.halo_valid = False           # do the z ghost planes of the current state hold the neighbours' planes?

    # the three phases of an exchange, all on the communication stream
    def pack(self):
        self.state_ready.record(self.ctx.stream)
        self.comm.wait_event(self.state_ready)
        self.ctx.ac_halo_pack(self.send_lo, self.send_hi, self.comm)

    def unpack(self):
        self.ctx.ac_halo_unpack(self.recv_lo, self.recv_hi, self.comm)
        self.halo_ready.record(self.comm)
        self.halo_valid = True

    def wait_halo(self):
        self.ctx.stream.wait_event(self.halo_ready)

    # the exchange as one kernel over the neighbours' memory
    def mark_state(self):
        self.state_ready.record(self.ctx.stream)

    def pull(self, below_ws, above_ws, below_ready, above_ready):
        """below_ws / above_ws: addresses of the neighbours' workspaces; *_ready: their state_ready events."""
        self.comm.wait_event(self.state_ready)
        self.comm.wait_event(below_ready)
        self.comm.wait_event(above_ready)
        self.ctx.ac_halo_pull(below_ws, above_ws, self.comm)
        self.halo_ready.record(self.comm)
        self.halo_valid = True


def transfer_in_process(slabs):
    """All slabs live in this process on one device: neighbour buffers by device-to-device copies."""
    import torch
    p = len(slabs)
    cuda = slabs[0].send_lo.is_cuda
    for r, s in enumerate(slabs):
        below, above = slabs[(r - 1) % p], slabs[(r + 1) % p]
        s.comm.wait_stream(below.comm)                           # their packs
        s.comm.wait_stream(above.comm)
        with (torch.cuda.stream(s.comm) if cuda else _Null()):
            s.recv_lo.copy_(below.send_hi, non_blocking=True)    # the top planes of the slab below
            s.recv_hi.copy_(above.send_lo, non_blocking=True)    # the bottom planes of the slab above
    for r, s in enumerate(slabs):                                # nobody repacks a buffer a neighbour still reads
        s.comm.wait_stream(slabs[(r - 1) % p].comm)
        s.comm.wait_stream(slabs[(r + 1) % p].comm)


class _Null:
    def __enter__(self):
        return self

    def __exit__(self, *a):
        return False


def ring_transfer(send_lo, send_hi, recv_lo, recv_hi, dist, rank, world, stream=None):
    """One process per rank: send_hi goes to rank + 1 (its recv_lo), send_lo to rank - 1 (its recv_hi); 2 sends and
    2 receives of whole halo buffers.  NCCL: enqueued on `stream`, nothing blocks the host.  gloo: device buffers
    are staged through the host (test set-up: several ranks sharing one GPU); host buffers go as they are."""
    import torch
    up, dn = (rank + 1) % world, (rank - 1) % world
    if dist.get_backend() == "nccl":
        with torch.cuda.stream(stream):
            ops = [dist.P2POp(dist.isend, send_hi, up), dist.P2POp(dist.isend, send_lo, dn),
                   dist.P2POp(dist.irecv, recv_lo, dn), dist.P2POp(dist.irecv, recv_hi, up)]
            for req in dist.batch_isend_irecv(ops):
                req.wait()                                      # stream-ordered for NCCL
        return
    if send_hi.is_cuda:
        stream.synchronize()
        s_hi, s_lo = send_hi.cpu(), send_lo.cpu()
        r_lo, r_hi = torch.empty_like(s_hi), torch.empty_like(s_lo)
    else:
        s_hi, s_lo, r_lo, r_hi = send_hi, send_lo, recv_lo, recv_hi
    ops = [dist.P2POp(dist.isend, s_hi, up), dist.P2POp(dist.isend, s_lo, dn),
           dist.P2POp(dist.irecv, r_lo, dn), dist.P2POp(dist.irecv, r_hi, up)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    if send_hi.is_cuda:
        with torch.cuda.stream(stream):
            recv_lo.copy_(r_lo, non_blocking=False)
            recv_hi.copy_(r_hi, non_blocking=False)


def transfer_distributed(slab, dist):
    ring_transfer(slab.send_lo, slab.send_hi, slab.recv_lo, slab.recv_hi, dist, slab.rank, slab.world, slab.comm)


class SlabGroupInProcess:
    """p slabs of one box driven by one process on one GPU: the reference behaviour of the decomposition."""

    def __init__(self, global_shape, lengths, world, dtype=binding.AC_F64, variant=0, overlap=True, context_factory=None,
                 transport="buffers", **kw):
        self.shape, self.lengths, self.kw, self.overlap = tuple(global_shape), tuple(lengths), kw, overlap
        self.transport = transport
        self.slabs = [Slab(global_shape, lengths, r, world, dtype, variant, context_factory, **kw) for r in range(world)]

    def exchange_begin(self):
        if self.transport == "pull":
            for s in self.slabs:
                s.mark_state()
        else:
            for s in self.slabs:
                s.pack()

    def exchange_end(self):
        p = len(self.slabs)
        if self.transport == "pull":
            for r, s in enumerate(self.slabs):
                below, above = self.slabs[(r - 1) % p], self.slabs[(r + 1) % p]
                s.pull(below.ctx.ac_workspace_ptr(), above.ctx.ac_workspace_ptr(), below.state_ready, above.state_ready)
        else:
            transfer_in_process(self.slabs)
            for s in self.slabs:
                s.unpack()

    def exchange(self):
        self.exchange_begin()
        self.exchange_end()

    def load_state(self, state):
        nzl = self.slabs[0].nzl
        for s in self.slabs:
            s.ctx.ac_load_state(np.ascontiguousarray(state[:, s.rank * nzl:(s.rank + 1) * nzl]))
            s.halo_valid = False

    def step(self, dt, forcing=None):
        """forcing: of the GLOBAL box (every slab shifts the phase itself)."""
        for sub in range(3):
            self.exchange_begin()                             # communication stream, after the previous substep
            if self.overlap:
                for s in self.slabs:
                    s.ctx.ac_substep_part(sub, dt, forcing, binding.AC_PART_INNER)    # runs beside the exchange
            self.exchange_end()
            for s in self.slabs:
                s.wait_halo()
                if self.overlap:
                    s.ctx.ac_substep_part(sub, dt, forcing, binding.AC_PART_OUTER)
                else:
                    s.ctx.ac_substep(sub, dt, forcing)
                s.halo_valid = False

    def make_forcing(self, seed, step, dt, f0):
        return self.slabs[0].ctx.ac_make_forcing(seed, step, dt, f0)

    def store_state(self):
        return np.concatenate([s.ctx.ac_store_state() for s in self.slabs], axis=1)

    def reduce(self):
        if not all(s.halo_valid for s in self.slabs):
            self.exchange()
        for s in self.slabs:
            s.wait_halo()
        return self.slabs[0].ctx.ac_diag_combine([s.ctx.ac_reduce_raw() for s in self.slabs])

    def free(self):
        for s in self.slabs:
            s.ctx.ac_free()


class SlabRank:
    """One process per rank (torchrun): this rank's slab of the box, exchanged through torch.distributed."""

    def __init__(self, global_shape, lengths, dist, dtype=binding.AC_F64, device="cuda:0", variant=0, overlap=True,
                 context_factory=None, transport="buffers", **kw):
        self.dist, self.rank, self.world = dist, dist.get_rank(), dist.get_world_size()
        self.shape, self.lengths, self.kw, self.overlap = tuple(global_shape), tuple(lengths), kw, overlap
        self.transport = transport
        if transport == "pull":
            kw = dict(kw, own_workspace=True)                 # ac_ipc_export needs a workspace the library allocated
        self.slab = Slab(global_shape, lengths, self.rank, self.world, dtype, variant, context_factory,
                         interprocess=transport == "pull", device=device, **kw)
        if transport == "pull":
            self._open_neighbours()

    def _open_neighbours(self):
        """CUDA IPC: map the neighbours' workspaces and import their state_ready events."""
        import torch
        s, dist = self.slab, self.dist
        self.host_group = dist.new_group(backend="gloo") if dist.get_backend() != "gloo" else None
        mine = (s.ctx.ac_ipc_export(), s.state_ready.ipc_handle())
        everyone = [None] * self.world
        dist.all_gather_object(everyone, mine, group=self.host_group)
        self._opened = {}
        self.nb_ws, self.nb_ready = [], []
        for r in ((self.rank - 1) % self.world, (self.rank + 1) % self.world):
            if r == self.rank:
                self.nb_ws.append(s.ctx.ac_workspace_ptr())
                self.nb_ready.append(s.state_ready)
                continue
            if r not in self._opened:
                ws = binding.ac_ipc_open(everyone[r][0])
                ev = torch.cuda.Event.from_ipc_handle(torch.device(s.ctx.device), everyone[r][1])
                self._opened[r] = (ws, ev)
            self.nb_ws.append(self._opened[r][0])
            self.nb_ready.append(self._opened[r][1])


    def forcing_from_draws(self, u1, u2, u3, dt, f0):
        """Eq. 4-6 for the GLOBAL box (a slab context knows the global box, ac_set_slab)."""
        return self.slab.ctx.ac_forcing_from_draws(u1, u2, u3, dt, f0)

    def transfer(self):
        if self.world > 1 or self.dist.get_backend() == "nccl":
            # with one rank NCCL sends to itself (the rank is its own neighbour above and below): the same
            # stream-ordered code path as between GPUs
            transfer_distributed(self.slab, self.dist)
        else:
            transfer_in_process([self.slab])

    def exchange_begin(self):
        if self.transport == "pull":
            self.slab.mark_state()
        else:
            self.slab.pack()

    def exchange_end(self):
        if self.transport == "pull":
            # every rank has issued its record before any rank issues the wait on it (a host barrier: no device sync)
            if self.world > 1:
                self.dist.barrier(group=self.host_group)
            self.slab.pull(self.nb_ws[0], self.nb_ws[1], self.nb_ready[0], self.nb_ready[1])
        else:
            self.transfer()
            self.slab.unpack()

    def exchange(self):
        self.exchange_begin()
        self.exchange_end()

    def free(self):
        if self.transport == "pull":
            self.slab.ctx.synchronize()
            self.slab.comm.synchronize()
            if self.world > 1:
                self.dist.barrier(group=self.host_group)     # nobody unmaps memory a neighbour still reads
            for ws, _ in self._opened.values():
                binding.ac_ipc_close(ws)
            self._opened = {}
            if self.world > 1:
                self.dist.barrier(group=self.host_group)
        self.slab.ctx.ac_free()

    def load_state(self, state):
        """state: the GLOBAL (7, nz, ny, nx) array (every rank generates the same seeded input) or this rank's slab."""
        nzl = self.slab.nzl
        if state.shape[1] != nzl:
            state = state[:, self.rank * nzl:(self.rank + 1) * nzl]
        self.slab.ctx.ac_load_state(np.ascontiguousarray(state))
        self.slab.halo_valid = False

    def step(self, dt, forcing=None):
        s = self.slab
        for sub in range(3):
            self.exchange_begin()                             # communication stream, after the previous substep
            if self.overlap:
                s.ctx.ac_substep_part(sub, dt, forcing, binding.AC_PART_INNER)        # runs beside the exchange
            self.exchange_end()
            s.wait_halo()
            if self.overlap:
                s.ctx.ac_substep_part(sub, dt, forcing, binding.AC_PART_OUTER)
            else:
                s.ctx.ac_substep(sub, dt, forcing)
            s.halo_valid = False

    def reduce(self):
        import torch
        if not self.slab.halo_valid:
            self.exchange()
        self.slab.wait_halo()
        raw = torch.tensor(self.slab.ctx.ac_reduce_raw(), dtype=torch.float64)
        if self.world > 1:
            dev = raw.to(self.slab.ctx.device) if self.dist.get_backend() == "nccl" else raw
            allr = [torch.empty_like(dev) for _ in range(self.world)]
            self.dist.all_gather(allr, dev)
            raws = [tuple(t.cpu().tolist()) for t in allr]
        else:
            raws = [tuple(raw.tolist())]
        return self.slab.ctx.ac_diag_combine(raws)
