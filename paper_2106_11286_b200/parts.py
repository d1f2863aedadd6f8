"""Decomposition of a neighbour table into parts ("CSR: partition by ... slabs of the
canonical order, halo = boundary vertices").

The table of n sites is cut into ranges of the canonical order.  A part is an hb context (include/hb.h,
hb_lattice.part_n_total) over its own sites, local ids 0 .. n_own-1, followed by its GHOST sites: the sites of other parts
that its rows point to, in ascending global order.  One sweep of the whole table is, on every part,

    for colour in 0 .. C-1:  hb_slab_pass(colour);  send the own sites of that colour that are ghosts elsewhere
    hb_slab_next_sweep()

i.e. one exchange step per colour, as for the slabs of the structured lattices (slabs.py): hb_part_gather packs the
listed spins on the owner, hb_part_scatter stores them into the ghosts of the receiver; between the two sits a
device-to-device hand-over (`LocalParts`: none at all, both run on one stream) or a send / recv between ranks
(`DistParts`: NCCL over NVLink, one process per GPU).  Philox is keyed by the global site id and the colouring is the
whole table's, so the parts together walk the single-context trajectory bit for bit (tests/test_parts.py).

Host-side orchestration only: passes, packing and reductions run in the CUDA library.
"""
import numpy as np


def bounds_equal(n, n_parts):
    """n_parts + 1 range bounds of the canonical order, parts as equal as possible."""
    if n_parts < 1 or n < n_parts:
        raise ValueError("split: at least one site per part")
    return [(k * n) // n_parts for k in range(n_parts + 1)]


def split_table(row_ptr, col_idx, colour, n_parts, bounds=None):
    """Cut a symmetric neighbour table with a proper colouring into parts.  Returns one dict per part:
    first, n_own, ghosts (global ids, ascending), to_global (own then ghosts), row_ptr / col_idx (local ids, ghost rows
    empty), colour (own then ghosts), send[q][c] / recv[q][c]: local ids of the own sites of colour c that part q holds as
    ghosts / of the ghosts of colour c that part q owns -- both in ascending global order, so the two lists pair up."""
    row_ptr = np.asarray(row_ptr, np.int64)
    col_idx = np.asarray(col_idx, np.int64)
    colour = np.asarray(colour, np.int32)
    n = row_ptr.size - 1
    bounds = list(bounds) if bounds is not None else bounds_equal(n, n_parts)
    assert len(bounds) == n_parts + 1 and bounds[0] == 0 and bounds[-1] == n and all(b > a for a, b in zip(bounds, bounds[1:]))
    n_colours = int(colour.max()) + 1 if n else 0
    owner_of = lambda ids: np.searchsorted(np.asarray(bounds[1:]), ids, side="right")
    parts = []
    for r in range(n_parts):
        first, n_own = bounds[r], bounds[r + 1] - bounds[r]
        cols = col_idx[row_ptr[first]:row_ptr[first + n_own]]
        outside = (cols < first) | (cols >= first + n_own)
        ghosts = np.unique(cols[outside])
        local = np.where(outside, n_own + np.searchsorted(ghosts, cols), cols - first)
        rp = np.concatenate([row_ptr[first:first + n_own + 1] - row_ptr[first], np.full(ghosts.size, cols.size, np.int64)])
        to_global = np.concatenate([np.arange(first, first + n_own, dtype=np.int64), ghosts])
        parts.append(dict(first=first, n_own=n_own, ghosts=ghosts, to_global=to_global, row_ptr=rp,
                          col_idx=local.astype(np.int32), colour=colour[to_global], n_colours=n_colours, send={}, recv={}))
    for r, p in enumerate(parts):
        own_of = owner_of(p["ghosts"])
        for q in np.unique(own_of):
            q = int(q)
            g = p["ghosts"][own_of == q]                       # ascending global ids, owned by q
            for c in range(n_colours):
                gc = g[colour[g] == c]
                if gc.size == 0:
                    continue
                p["recv"].setdefault(q, {})[c] = (p["n_own"] + np.searchsorted(p["ghosts"], gc)).astype(np.int32)
                parts[q]["send"].setdefault(r, {})[c] = (gc - parts[q]["first"]).astype(np.int32)
    return parts


def part_lattice(p, n_total, K_site=None, e_site=None):
    """The binding's Lattice of one part; K_site / e_site are the WHOLE table's per-site anisotropy (or None)."""
    from .binding import Lattice
    g = p["to_global"]
    return Lattice("csr", row_ptr=p["row_ptr"], col_idx=p["col_idx"], colour=p["colour"], n_colours=p["n_colours"],
                   K_site=None if K_site is None else np.asarray(K_site, np.float32)[g],
                   e_site=None if e_site is None else np.asarray(e_site, np.float32).reshape(-1, 3)[g],
                   part=(p["first"], p["n_own"], n_total))


class _Lists:
    """Device copies of a part's send / recv lists and the buffers its messages are packed into."""

    def __init__(self, p, device):
        import torch
        self.send = {q: {c: torch.as_tensor(ids, device=device) for c, ids in d.items()} for q, d in p["send"].items()}
        self.recv = {q: {c: torch.as_tensor(ids, device=device) for c, ids in d.items()} for q, d in p["recv"].items()}
        self.out = {q: {c: torch.empty(4 * ids.numel(), dtype=torch.float32, device=device) for c, ids in d.items()} for q, d in self.send.items()}
        self.inn = {q: {c: torch.empty(4 * ids.numel(), dtype=torch.float32, device=device) for c, ids in d.items()} for q, d in self.recv.items()}


def exchange_local(ctxs, lists, colour):
    """One exchange step between parts that live in this process on one stream: the owner packs, the holder of the ghosts
    unpacks the same buffer."""
    for r, (c, l) in enumerate(zip(ctxs, lists)):
        for q, by_colour in l.send.items():
            if colour in by_colour:
                c.part_gather(by_colour[colour], l.out[q][colour])
                ctxs[q].part_scatter(lists[q].recv[r][colour], l.out[q][colour])


def exchange_dist(ctx, l, colour, group=None):
    """The same between ranks: pack, send / recv (all peers at once), unpack.  Messages between a pair of ranks are matched by
    the order of posting, one per direction and colour."""
    import torch
    import torch.distributed as dist
    send = [(q, d[colour]) for q, d in sorted(l.send.items()) if colour in d]
    recv = [(q, d[colour]) for q, d in sorted(l.recv.items()) if colour in d]
    for q, ids in send:
        ctx.part_gather(ids, l.out[q][colour])
    if send or recv:
        cuda = (send or recv)[0][1].is_cuda
        staged = cuda and dist.get_backend(group) != "nccl"     # any other backend (gloo in the tests) gets host copies
        sb = [l.out[q][colour].cpu() if staged else l.out[q][colour] for q, _ in send]   # (.cpu() synchronises with the stream)
        rb = [torch.empty(l.inn[q][colour].shape, dtype=torch.float32) if staged else l.inn[q][colour] for q, _ in recv]
        ops = [dist.P2POp(dist.isend, t, q, group) for t, (q, _) in zip(sb, send)]
        ops += [dist.P2POp(dist.irecv, t, q, group) for t, (q, _) in zip(rb, recv)]
        if cuda and not staged:
            with torch.cuda.stream(ctx.stream):      # NCCL enqueues on torch's current stream: the stream of the passes
                for req in dist.batch_isend_irecv(ops):
                    req.wait()
        else:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
        if staged:
            for t, (q, _) in zip(rb, recv):
                l.inn[q][colour].copy_(t)
    for q, ids in recv:
        ctx.part_scatter(ids, l.inn[q][colour])


class LocalParts:
    """n_parts part contexts of one neighbour table in this process, on one device and one stream."""

    def __init__(self, row_ptr, col_idx, colour, n_parts, J=1.0, K=0.0, e=(0.0, 0.0, 1.0), seed=1, K_site=None, e_site=None,
                 device="cuda:0", options=None, bounds=None):
        from .binding import Context
        self.n = int(np.asarray(row_ptr).size - 1)
        self.parts = split_table(row_ptr, col_idx, colour, n_parts, bounds)
        self.n_colours = self.parts[0]["n_colours"]
        self.ctxs = [Context(part_lattice(p, self.n, K_site, e_site), J, K, e, seed, device=device) for p in self.parts]
        for c in self.ctxs:
            for k, v in (options or {}).items():
                c.set_option(k, v)
        self.lists = [_Lists(p, c.device) for p, c in zip(self.parts, self.ctxs)]

    def _fill_ghosts(self):
        for colour in range(self.n_colours):
            exchange_local(self.ctxs, self.lists, colour)

    def init_random(self):
        for c in self.ctxs:
            c.init_random()
        self._fill_ghosts()

    def init_aligned(self, direction):
        for c in self.ctxs:
            c.init_aligned(direction)

    def set_spins(self, sx, sy, sz):
        """Arrays of the WHOLE table, canonical order: every part takes its own sites and its ghosts."""
        for c, p in zip(self.ctxs, self.parts):
            c.set_spins(*[np.asarray(a, np.float32)[p["to_global"]] for a in (sx, sy, sz)])

    def get_spins(self):
        got = [c.get_spins() for c in self.ctxs]
        return [np.concatenate([g[k][:p["n_own"]] for g, p in zip(got, self.parts)]) for k in range(3)]

    def ghosts_current(self):
        """True if every ghost holds exactly its owner's spin (a check for the tests)."""
        whole = self.get_spins()
        return all(np.array_equal(np.asarray(g[k])[p["n_own"]:].view(np.uint32), whole[k][p["ghosts"]].view(np.uint32))
                   for c, p in zip(self.ctxs, self.parts) for g in [c.get_spins()] for k in range(3))

    def sweep(self, T, n_sweeps=1):
        for _ in range(n_sweeps):
            for colour in range(self.n_colours):
                for c in self.ctxs:
                    c.slab_pass(T, colour)
                exchange_local(self.ctxs, self.lists, colour)
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


class DistParts:
    """This rank's part of a neighbour table split over the ranks of a torch.distributed group (one process per GPU).  Every
    rank passes the WHOLE table (host arrays) and keeps its part of it."""

    def __init__(self, row_ptr, col_idx, colour, J=1.0, K=0.0, e=(0.0, 0.0, 1.0), seed=1, K_site=None, e_site=None,
                 device=None, group=None, options=None, bounds=None):
        import torch.distributed as dist
        from .binding import Context
        self.group = group
        if dist.is_available() and dist.is_initialized():
            self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        else:
            self.rank, self.world = 0, 1
        self.n = int(np.asarray(row_ptr).size - 1)
        self.part = split_table(row_ptr, col_idx, colour, self.world, bounds)[self.rank]
        self.n_colours = self.part["n_colours"]
        self.ctx = Context(part_lattice(self.part, self.n, K_site, e_site), J, K, e, seed, device=device or "cuda:0")
        for k, v in (options or {}).items():
            self.ctx.set_option(k, v)
        self.lists = _Lists(self.part, self.ctx.device)

    def _exchange(self, colour):
        if self.world == 1:
            return                                     # a single part has no ghosts
        exchange_dist(self.ctx, self.lists, colour, self.group)

    def init_random(self):
        self.ctx.init_random()
        for colour in range(self.n_colours):
            self._exchange(colour)

    def init_aligned(self, direction):
        self.ctx.init_aligned(direction)

    def set_spins(self, sx, sy, sz):
        self.ctx.set_spins(*[np.asarray(a, np.float32)[self.part["to_global"]] for a in (sx, sy, sz)])

    def get_spins(self):
        """This rank's own sites (canonical order)."""
        return [np.asarray(a)[:self.part["n_own"]] for a in self.ctx.get_spins()]

    def sweep(self, T, n_sweeps=1):
        for _ in range(n_sweeps):
            for colour in range(self.n_colours):
                self.ctx.slab_pass(T, colour)
                self._exchange(colour)
            self.ctx.slab_next_sweep()

    def measure(self):
        """M and E of the WHOLE table on every rank (one all_reduce of 4 doubles)."""
        import torch
        import torch.distributed as dist
        m, e = self.ctx.measure()
        t = torch.tensor([m[0], m[1], m[2], e], dtype=torch.float64, device=self.ctx.device)
        if self.world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
        t = t.cpu().numpy()
        return t[:3].copy(), float(t[3])

    def close(self):
        self.ctx.close()
