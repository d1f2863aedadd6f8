"""Worker of tests/test_slabs.py (-m gpu): one rank of a world_size-2 job whose ranks share cuda:0.

Each rank owns one slab (DistSlab); with peer stores the ranks map each other's spins buffers through CUDA IPC and the
colour kernels write the neighbour's ghost planes directly.  The process group is gloo (NCCL refuses two ranks on one
device); kernels of different ranks never wait on one another: the only cross-rank wait is the host barrier between passes.
Rank 0 gathers the slabs and prints them for the parent test to compare with the oracle."""
import base64
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402
import torch.distributed as dist  # noqa: E402

from paper_2106_11286_b200 import slabs  # noqa: E402


def main():
    peer = sys.argv[1] == "peer"
    shape = tuple(int(x) for x in sys.argv[2:5])
    dist.init_process_group("gloo")
    d = slabs.DistSlab(*shape, J=1.0, K=0.05, e=(0.0, 0.6, 0.8), seed=4242, device="cuda:0", peer_stores=peer)
    d.init_random()
    d.sweep(1.44, 3)
    d.sweep(0.4, 2)
    M, E = d.measure()
    mine = [base64.b64encode(np.ascontiguousarray(a).tobytes()).decode() for a in d.get_spins()]
    parts = [None] * d.world
    dist.all_gather_object(parts, mine)
    if d.rank == 0:
        print(json.dumps({"world": d.world, "M": list(M), "E": E, "spins": parts}))
    d.close()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
