"""Worker of tests/test_parts.py: one rank of a world_size-N gloo job on CPU.

Runs the exchange step of paper_2106_11286_b200.parts (the only cross-rank step of a partitioned neighbour table) on
stand-in parts whose state is a CPU tensor.  A "colour pass" here is an integer recurrence on the site's neighbours (exact
in fp32), NOT the method: there is no CPU path.  Every rank also evolves the whole table alone; the parts must agree with
it after every sweep, which they do only if every ghost is current whenever a pass reads it."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

import numpy as np  # noqa: E402
import torch  # noqa: E402
import torch.distributed as dist  # noqa: E402

from paper_2106_11286_b200 import parts, workloads  # noqa: E402
from test_parts import first_fit  # noqa: E402


def toy_pass(S, row_ptr, col, sites, gid, step):
    """S[i] <- (S[i] + sum of the neighbours' S + global id + step) mod 1021, for the listed sites (one colour: no two adjacent)."""
    new = {}
    for i in sites:
        nb = col[row_ptr[i]:row_ptr[i + 1]]
        new[i] = (S[i, :3] + S[nb, :3].sum(0) + float(gid[i] + step)) % 1021.0
    for i, v in new.items():
        S[i, :3] = v


class FakePart:
    """part_gather / part_scatter / slab_pass of the binding, on a CPU tensor of (x, y, z, 0) records."""

    def __init__(self, p):
        self.p = p
        g = p["to_global"]
        self.S = torch.zeros(g.size, 4)
        self.S[:, 0] = torch.as_tensor(g % 7, dtype=torch.float32)
        self.S[:, 1] = torch.as_tensor(g % 11, dtype=torch.float32)
        self.S[:, 2] = torch.as_tensor(g % 13, dtype=torch.float32)
        self.step = 0

    def part_gather(self, ids, out):
        out.view(-1, 4)[:ids.numel()] = self.S[ids.long()]

    def part_scatter(self, ids, src):
        self.S[ids.long(), :3] = src.view(-1, 4)[:ids.numel(), :3]

    def slab_pass(self, colour):
        own = np.nonzero(self.p["colour"][:self.p["n_own"]] == colour)[0]
        toy_pass(self.S, self.p["row_ptr"], self.p["col_idx"], own, self.p["to_global"], self.step)


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    rp, ci = workloads.random_csr_graph(240, 5.0, seed=11)
    colour = first_fit(rp, ci)
    n, C = rp.size - 1, int(colour.max()) + 1
    p = parts.split_table(rp, ci, colour, world)[rank]
    part, lists = FakePart(p), parts._Lists(p, "cpu")
    whole = FakePart(dict(to_global=np.arange(n), n_own=n, colour=colour, row_ptr=rp, col_idx=ci))
    ok = True
    for sweep in range(3):
        for c in range(C):
            part.slab_pass(c)
            parts.exchange_dist(part, lists, c)
            whole.slab_pass(c)
        part.step += 1
        whole.step += 1
        ok = ok and bool(torch.equal(part.S, whole.S[torch.as_tensor(p["to_global"])]))   # own sites AND ghosts
    t = torch.tensor([float(p["n_own"]), float(p["ghosts"].size)], dtype=torch.float64)
    dist.all_reduce(t)
    oks = [None] * world
    dist.all_gather_object(oks, ok)
    if rank == 0:
        print(json.dumps({"world": world, "ok": oks, "own": t[0].item(), "ghosts": t[1].item(), "n": n, "colours": C}))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
