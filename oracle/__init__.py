"""CPU oracle for the Metropolis sweep of arXiv 2106.11286 -- TEST INFRASTRUCTURE.

Only tests/, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl
reference`` legs of ``bench.py`` may import this package.  It never imports the
CUDA package and the CUDA package never imports it.
"""
from .hb_oracle import (  # noqa: F401
    Lattice, State32, State64, build, lib, philox4x32_10, philox_site, u01,
    sincos_spec, sincos_spec_batch, exp_spec, exp_spec_batch, sphere, sphere_batch,
    mt19937_64, total_energy64,
)
