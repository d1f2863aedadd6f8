"""B200-native Metropolis colour sweeps for the classical anisotropic Heisenberg model
(the data-parallel hot path of arXiv 2106.11286).

    from paper_2106_11286_b200 import Lattice, Context
    ctx = Context(Lattice("sc", 464), J=1.0, K=0.01, e=(0, 0, 1), seed=1)
    ctx.init_random(); ctx.sweep(1.44, 200); M, E = ctx.measure()

The work happens in libhb.so (C ABI: include/hb.h; CUDA kernels: csrc/).  Importing the
package does not load the library; constructing a Context does, and raises if the
library is not built or no CUDA device is present -- there is no CPU path.
"""
from .binding import Context, HbError, Lattice, device_math, load_library, measure_sc_noalloc, probe_alu, probe_pipe, sizes  # noqa: F401
from . import workloads  # noqa: F401
