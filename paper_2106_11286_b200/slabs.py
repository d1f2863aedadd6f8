"""Slab decomposition of the periodic simple cubic lattice along z.

Every slab is an hb context over planes z0 .. z0 + nz - 1 of the whole lattice plus one ghost plane on each side
(include/hb.h, hb_lattice.slab_Lz).  One sweep of the whole lattice is, on every slab,

    for colour in (0, 1):  hb_slab_pass(colour);  send the two boundary planes of that colour to the z-neighbours
    hb_slab_next_sweep()

i.e. ONE exchange step per colour: 2 faces x 3 components x (Lx Ly / 2) floats per slab.  Philox is keyed by the global
site id, so the slabs together walk the single-context trajectory bit for bit (tests/test_slabs.py).

* `LocalSlabs`: all slabs in this process on ONE device (several devices take one process each: `DistSlab`); faces move with
  `Tensor.copy_` on the contexts' stream (a device-to-device copy), or, with `peer_stores=True`, inside the colour
  kernels themselves: a thread that stores an updated spin of a boundary plane stores it into the neighbour's ghost plane
  too (`hb_slab_set_peer`), so the transfer overlaps the pass and only a barrier remains between two passes.
* `DistSlab`: one slab per rank of a `torch.distributed` group (one process per GPU); faces move with
  `batch_isend_irecv` (NCCL send/recv over NVLink between GPUs), M and E with one all_reduce of 4 doubles.

Host-side orchestration only: every pass and reduction runs in the CUDA library, the copies are library copies.
"""
import numpy as np


def partition(Lz, n_slabs):
    """[(z0, nz)] with every nz even and >= 2, as equal as possible, summing to Lz (Lz even)."""
    if Lz % 2 or n_slabs < 1 or Lz < 2 * n_slabs:
        raise ValueError("partition: Lz must be even and hold at least two planes per slab")
    pairs, extra = divmod(Lz // 2, n_slabs)
    out, z0 = [], 0
    for r in range(n_slabs):
        nz = 2 * (pairs + (1 if r < extra else 0))
        out.append((z0, nz))
        z0 += nz
    return out


def neighbours(rank, world):
    """(rank owning the planes below this slab, rank owning the planes above), periodic."""
    return (rank - 1) % world, (rank + 1) % world


def exchange_local(ctxs, colour):
    """Faces of one colour between slabs that live in this process: slab r's low boundary plane becomes the high ghost
    plane of slab r-1, its high boundary plane the low ghost plane of slab r+1 (periodic; a single slab feeds itself)."""
    G = len(ctxs)
    for r, c in enumerate(ctxs):
        down, up = neighbours(r, G)
        for src, dst in zip(c.slab_face(colour, 0, False), ctxs[down].slab_face(colour, 1, True)):
            dst.copy_(src, non_blocking=True)
        for src, dst in zip(c.slab_face(colour, 1, False), ctxs[up].slab_face(colour, 0, True)):
            dst.copy_(src, non_blocking=True)


def exchange_dist(ctx, colour, rank, world, group=None):
    """The same between ranks.  Sends go out low face first, then high face; a rank's receives are posted in the order
    its neighbours send (the upper neighbour's low face fills the high ghost plane, the lower neighbour's high face the
    low ghost plane), so that with two ranks, where both neighbours are the same peer, messages still pair up."""
    import torch.distributed as dist
    down, up = neighbours(rank, world)
    if world == 1:
        exchange_local([ctx], colour)
        return
    send = ctx.slab_face(colour, 0, False) + ctx.slab_face(colour, 1, False)      # low face down, high face up
    recv = ctx.slab_face(colour, 1, True) + ctx.slab_face(colour, 0, True)        # from up into the high ghost, from down
    peers_s, peers_r = [down] * 3 + [up] * 3, [up] * 3 + [down] * 3
    # NCCL moves device memory directly (NVLink between GPUs); any other backend (gloo in the tests) gets host copies
    staged = send[0].is_cuda and dist.get_backend(group) != "nccl"
    if staged:
        send_b = [t.cpu() for t in send]            # synchronises with the stream the pass ran on
        recv_b = [t.new_empty(t.shape, device="cpu") for t in recv]
    else:
        send_b, recv_b = send, recv
    ops = [dist.P2POp(dist.isend, t, p, group) for t, p in zip(send_b, peers_s)]
    ops += [dist.P2POp(dist.irecv, t, p, group) for t, p in zip(recv_b, peers_r)]
    if staged or not send[0].is_cuda:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    else:
        # NCCL enqueues on torch's current stream: make that the stream of the colour passes, so that the sends queue behind
        # the pass that produced the faces and the next pass behind the receives, whatever stream the caller is in
        import torch
        with torch.cuda.stream(ctx.stream):
            for req in dist.batch_isend_irecv(ops):
                req.wait()
    if staged:
        for dst, src in zip(recv, recv_b):
            dst.copy_(src)


class LocalSlabs:
    """n_slabs slab contexts of one periodic sc lattice in this process."""

    def __init__(self, Lx, Ly, Lz, n_slabs, J=1.0, K=0.0, e=(0.0, 0.0, 1.0), seed=1, device="cuda:0", options=None,
                 peer_stores=False, flags=False, kind="sc"):
        """All slabs live on `device`.  (The library issues every call on the CUDA device that is current, and a process that
        drove contexts on several devices would have to switch it around every call and enable peer access itself: that
        path was never run on a multi-GPU box, so it is not offered -- one process per GPU, `DistSlab`, is.)"""
        from .binding import Context, Lattice
        self.shape = (Lx, Ly, Lz)
        self.parts = partition(Lz, n_slabs)
        # kind "bcc" / "fcc": slabs of conventional cells; the colours are the basis indices, one face exchange per sublattice
        # pass; peer stores and flags exist for the simple cubic kernels only
        self.kind = kind
        self.n_colours = {"sc": 2, "bcc": 2, "fcc": 4}[kind]
        if kind != "sc" and (peer_stores or flags):
            raise ValueError("peer stores and neighbour flags exist for simple cubic slabs")
        self.ctxs = [Context(Lattice(kind, Lx, Ly, nz, slab=(z0, Lz)), J, K, e, seed, device=device)
                     for r, (z0, nz) in enumerate(self.parts)]
        for c in self.ctxs:
            for k, v in (options or {}).items():
                c.set_option(k, v)
        self.n = Lx * Ly * Lz * {"sc": 1, "bcc": 2, "fcc": 4}[kind]
        # peer stores (hb_slab_set_peer): the colour kernels write their boundary planes straight into the neighbours'
        # ghost planes, the exchange step disappears
        self.peer_stores = bool(peer_stores)
        if self.peer_stores:
            for r, c in enumerate(self.ctxs):
                down, up = neighbours(r, n_slabs)
                c.slab_set_peer(0, self.ctxs[down].spins_ptr, self.parts[down][1])
                c.slab_set_peer(1, self.ctxs[up].spins_ptr, self.parts[up][1])
        # neighbour flags (include/hb.h, "slab_flags"): the kernels themselves wait for and signal their z-neighbours.  The
        # contexts of this class share one stream, so a pass finds the flags of the pass before already set: this exercises
        # the protocol's bookkeeping (stamps, boundary counters, flag addresses), not its concurrency.
        self.flags = bool(flags) and self.peer_stores
        if self.flags:
            for c in self.ctxs:
                c.set_option("slab_flags", 1)

    def _sync(self):
        import torch
        for c in self.ctxs:
            torch.cuda.synchronize(c.device)

    def _fill_ghosts(self):
        self._sync()
        for colour in range(self.n_colours):
            exchange_local(self.ctxs, colour)
        self._sync()

    def init_random(self):
        for c in self.ctxs:
            c.init_random()
        self._fill_ghosts()

    def init_aligned(self, direction):
        for c in self.ctxs:
            c.init_aligned(direction)
        self._fill_ghosts()

    def set_spins(self, sx, sy, sz):
        # canonical order of the whole lattice: basis-major, z slowest inside a sublattice; a slab takes, per sublattice, its planes
        plane, nb = self.shape[0] * self.shape[1], self.n // (self.shape[0] * self.shape[1] * self.shape[2])
        nc = plane * self.shape[2]
        for c, (z0, nz) in zip(self.ctxs, self.parts):
            c.set_spins(*[np.concatenate([np.asarray(a, np.float32)[b * nc + z0 * plane:b * nc + (z0 + nz) * plane] for b in range(nb)])
                          for a in (sx, sy, sz)])
        self._fill_ghosts()

    def get_spins(self):
        plane, nb = self.shape[0] * self.shape[1], self.n // (self.shape[0] * self.shape[1] * self.shape[2])
        parts = [c.get_spins() for c in self.ctxs]
        out = []
        for k in range(3):
            out.append(np.concatenate([p[k][b * nz * plane:(b + 1) * nz * plane] for b in range(nb) for p, (z0, nz) in zip(parts, self.parts)]))
        return out

    def sweep(self, T, n_sweeps=1):
        several = len({c.stream.cuda_stream for c in self.ctxs}) > 1
        for _ in range(n_sweeps):
            for colour in range(self.n_colours):
                for c in self.ctxs:
                    c.slab_pass(T, colour)
                if several:          # contexts on one stream are ordered by it; otherwise passes and copies meet here
                    self._sync()
                if not self.peer_stores:
                    exchange_local(self.ctxs, colour)
                    if several:
                        self._sync()
            for c in self.ctxs:
                c.slab_next_sweep()

    def measure(self):
        M, E = np.zeros(3), 0.0
        for c in self.ctxs:
            m, e = c.measure()
            M += m
            E += e
        return M, E

    def close(self):
        for c in self.ctxs:
            c.close()


class DistSlab:
    """This rank's slab of a periodic sc lattice split over the ranks of a torch.distributed group.

    peer_stores=True: every rank maps its two z-neighbours' spins buffers (CUDA IPC; on a multi-GPU node this is peer
    memory over NVLink) and the colour kernels store their boundary planes straight into the neighbours' ghost planes
    (hb_slab_set_peer).  No face is sent after the initial fill; between two colour passes there is only a barrier
    (an all_reduce of one word on the stream under NCCL; a host barrier under gloo)."""

    def __init__(self, Lx, Ly, Lz, J=1.0, K=0.0, e=(0.0, 0.0, 1.0), seed=1, device=None, group=None, options=None,
                 peer_stores=False, flags=False, kind="sc"):
        """flags=True (with peer_stores, one GPU per rank): no barrier between two colour passes; the kernels wait for and
        signal their two z-neighbours through flag words in peer memory (include/hb.h, "slab_flags"), boundary tiles first,
        so that interior tiles hide the wait.  Never with several ranks on ONE GPU: their kernels would wait on one another."""
        import torch
        import torch.distributed as dist
        from .binding import Context, Lattice
        self.group = group
        if dist.is_available() and dist.is_initialized():
            self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        else:                                   # no process group: the whole lattice as one slab
            self.rank, self.world = 0, 1
        self.shape = (Lx, Ly, Lz)
        parts = partition(Lz, self.world)
        self.z0, self.nz = parts[self.rank]
        self.kind = kind
        self.n_colours = {"sc": 2, "bcc": 2, "fcc": 4}[kind]      # bcc / fcc: slabs of conventional cells, one face exchange per sublattice pass
        self.peer_stores = bool(peer_stores) and kind == "sc"      # peer stores and flags: simple cubic kernels only
        flags = bool(flags) and kind == "sc"
        self.ctx = Context(Lattice(kind, Lx, Ly, self.nz, slab=(self.z0, Lz)), J, K, e, seed,
                           device=device or "cuda:0", ipc=self.peer_stores and self.world > 1)
        for k, v in (options or {}).items():
            self.ctx.set_option(k, v)
        self.n = Lx * Ly * Lz * {"sc": 1, "bcc": 2, "fcc": 4}[kind]
        self._mapped = {}
        self.flags = False
        if self.peer_stores:
            down, up = neighbours(self.rank, self.world)
            self._nccl = self.world > 1 and dist.get_backend(group) == "nccl"
            self._flag = torch.zeros(1, dtype=torch.int32, device=self.ctx.device) if self._nccl else None
            if self.world == 1:
                ptrs, ok = {0: self.ctx.spins_ptr}, True
            else:
                handles = [None] * self.world
                dist.all_gather_object(handles, self.ctx.ipc_handle(), group=group)
                ok = True
                try:
                    for r in {down, up}:
                        self._mapped[r] = self.ctx.open_ipc(handles[r])
                except Exception:               # no peer access between the two devices: every rank falls back together
                    ok = False
                ptrs = self._mapped
                agree = torch.tensor([1 if ok else 0], dtype=torch.int32, device=self.ctx.device if self._nccl else "cpu")
                dist.all_reduce(agree, op=dist.ReduceOp.MIN, group=group)
                ok = bool(agree.item())
            if ok:
                self.ctx.slab_set_peer(0, ptrs[down], parts[down][1])
                self.ctx.slab_set_peer(1, ptrs[up], parts[up][1])
                if flags:
                    self.ctx.set_option("slab_flags", 1)
                    self.flags = True
            else:
                import warnings
                warnings.warn("DistSlab: a neighbour's spins buffer could not be mapped; faces are sent after every pass instead")
                for ptr in self._mapped.values():
                    self.ctx.close_ipc(ptr)
                self._mapped = {}
                self.peer_stores = False

    def _pass_barrier(self):
        """No rank starts the next colour before every rank has finished this one."""
        if self.world == 1:
            return                                   # one stream orders the passes
        import torch
        import torch.distributed as dist
        if self._nccl:
            # NCCL orders the collective on torch's CURRENT stream: make that the stream the passes run on, whatever stream
            # the caller is in, so that the next pass queues behind the collective and the collective behind this pass
            with torch.cuda.stream(self.ctx.stream):
                dist.all_reduce(self._flag, group=self.group)
        else:
            torch.cuda.synchronize(self.ctx.device)
            dist.barrier(group=self.group)

    def _fill_ghosts(self):
        for colour in range(self.n_colours):
            exchange_dist(self.ctx, colour, self.rank, self.world, self.group)
        if self.peer_stores:
            self._pass_barrier()

    def init_random(self):
        self.ctx.init_random()
        self._fill_ghosts()

    def init_aligned(self, direction):
        self.ctx.init_aligned(direction)
        self._fill_ghosts()

    def sweep(self, T, n_sweeps=1):
        for _ in range(n_sweeps):
            for colour in range(self.n_colours):
                self.ctx.slab_pass(T, colour)
                if self.peer_stores and self.flags:
                    pass                         # the next pass's boundary tiles wait for the neighbours' flags on the device
                elif self.peer_stores:
                    self._pass_barrier()
                else:
                    exchange_dist(self.ctx, colour, self.rank, self.world, self.group)
            self.ctx.slab_next_sweep()
        if self.peer_stores and self.flags and n_sweeps > 0:
            # Flags order a pass only against the neighbours' NEXT pass.  Nothing on this rank's stream waits for the stores
            # the neighbours' LAST pass makes into this slab's ghost planes, and measure() (boundary bonds) and the next
            # ghost fill read those planes: one barrier per call closes the gap (include/hb.h, hb_slab_set_peer).
            self._pass_barrier()

    def measure(self):
        """M and E of the WHOLE lattice on every rank (one all_reduce of 4 doubles)."""
        import torch
        import torch.distributed as dist
        m, e = self.ctx.measure()
        t = torch.tensor([m[0], m[1], m[2], e], dtype=torch.float64, device=self.ctx.device)
        if self.world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
        t = t.cpu().numpy()
        return t[:3].copy(), float(t[3])

    def get_spins(self):
        """This rank's own planes (canonical order, z slowest)."""
        return self.ctx.get_spins()

    def close(self):
        if self.peer_stores and self.world > 1:
            import torch
            import torch.distributed as dist
            torch.cuda.synchronize(self.ctx.device)
            dist.barrier(group=self.group)           # nobody unmaps or frees while a neighbour may still store
            for ptr in self._mapped.values():
                self.ctx.close_ipc(ptr)
            self._mapped = {}
            dist.barrier(group=self.group)
        self.ctx.close()
