"""Worker of tests/test_slabs.py: one rank of a world_size-N gloo job on CPU.

Runs the face exchange of paper_2106_11286_b200.slabs (the only cross-rank step of the sharded path) on stand-in
slabs whose faces are CPU tensors: every face element is stamped with (owner rank, colour, side, component), so the
test can tell where each ghost plane came from.  No method arithmetic here: there is no CPU path."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402
import torch.distributed as dist  # noqa: E402

from paper_2106_11286_b200 import slabs  # noqa: E402


def stamp(rank, colour, side, comp):
    return float(1000 * rank + 100 * colour + 10 * side + comp)


class FakeSlab:
    """slab_face() of the binding, on CPU tensors."""

    def __init__(self, rank, count=5):
        self.t = {}
        for colour in (0, 1):
            for side in (0, 1):
                self.t[(colour, side, False)] = [torch.full((count,), stamp(rank, colour, side, k)) for k in range(3)]
                self.t[(colour, side, True)] = [torch.full((count,), -1.0) for _ in range(3)]

    def slab_face(self, colour, side, ghost):
        return self.t[(colour, side, bool(ghost))]


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    s = FakeSlab(rank)
    for colour in (0, 1):
        slabs.exchange_dist(s, colour, rank, world)
    got = {"%d%d%d" % (c, side, k): s.t[(c, side, True)][k].tolist() for c in (0, 1) for side in (0, 1) for k in range(3)}
    # the all_reduce DistSlab.measure does, on CPU
    t = torch.tensor([rank + 1.0, 0.0, 0.0, -2.0 * (rank + 1)], dtype=torch.float64)
    dist.all_reduce(t)
    out = [None] * world
    dist.all_gather_object(out, got)
    if rank == 0:
        print(json.dumps({"world": world, "ghosts": out, "sum": t.tolist(), "parts": slabs.partition(20, world)}))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
