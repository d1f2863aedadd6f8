"""Worker of tests/test_parts.py (-m gpu): one rank of a world_size-2 job whose ranks share cuda:0.

Each rank owns one part of the fcc sphere's neighbour table (DistParts); after every colour pass the ranks exchange the
spins of that colour that are ghosts on the other side (gather kernel, gloo send / recv through host copies, scatter kernel).
Kernels of different ranks never wait on one another.  Rank 0 gathers the parts and prints them for the parent test to
compare with the oracle."""
import base64
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402
import torch.distributed as dist  # noqa: E402

import paper_2106_11286_b200 as hb  # noqa: E402
from paper_2106_11286_b200 import parts  # noqa: E402


def main():
    R = int(sys.argv[1])
    dist.init_process_group("gloo")
    lat = hb.Lattice.fcc_sphere(R, 0.05, (0.0, 0.0, 1.0), 0.5, "greedy")
    d = parts.DistParts(lat.row_ptr, lat.col_idx, lat.colour, J=1.0, K=0.05, e=(0.0, 0.0, 1.0), seed=77,
                        K_site=lat.K_site, e_site=lat.e_site, device="cuda:0")
    d.init_random()
    d.sweep(2.5, 3)
    d.sweep(0.7, 2)
    M, E = d.measure()
    mine = [base64.b64encode(np.ascontiguousarray(a).tobytes()).decode() for a in d.get_spins()]
    got = [None] * d.world
    dist.all_gather_object(got, mine)
    if d.rank == 0:
        print(json.dumps({"world": d.world, "M": list(M), "E": E, "spins": got}))
    d.close()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
