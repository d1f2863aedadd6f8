"""Temperature scans with the protocols of the workloads (reading A13): one state carried through the
scan, `equil` discarded sweeps then `sweeps` measured sweeps per temperature, M and E taken after every measured sweep.

    python -m paper_2106_11286_b200.scan c2          # prints T, <|M|>, <E>/N, chi, C per temperature

Host-side bookkeeping only: every sweep and every reduction runs in the CUDA library.
"""
import sys

import numpy as np

from . import workloads
from .binding import Context, Lattice


def make_context(cfg, device="cuda:0", seed=None):
    if cfg["kind"] == "sphere":
        lat = Lattice.fcc_sphere(cfg["R"], cfg["K"], cfg["e"], cfg["K_surf"], cfg.get("colouring", "greedy"))
    else:
        lat = Lattice(cfg["kind"], cfg["L"])
    ctx = Context(lat, cfg["J"], cfg["K"], cfg["e"], cfg["seed"] if seed is None else seed, device=device)
    if cfg["start"] == "random":
        ctx.init_random()
    else:
        ctx.init_aligned(cfg["e"])
    return ctx


def run_scan(ctx, temperatures, sweeps, equil=0):
    """Returns a dict of arrays over the temperatures: T, absM = <|M|>, E = <E>/N, chi = N (<M^2> - <|M|>^2) / T,
    C = (<E^2> - <E>^2) / (N T^2)."""
    n = ctx.n
    out = {k: [] for k in ("T", "absM", "E", "chi", "C")}
    for T in temperatures:
        if equil:
            ctx.sweep(T, equil)
        M, E = ctx.sweep_series(T, sweeps)
        m = np.linalg.norm(M, axis=1)
        out["T"].append(T)
        out["absM"].append(m.mean())
        out["E"].append(E.mean() / n)
        out["chi"].append(n * ((m * m).mean() - m.mean() ** 2) / T)
        out["C"].append((np.mean(E * E) - E.mean() ** 2) / (n * T * T))
    return {k: np.array(v) for k, v in out.items()}


def main(argv):
    name = argv[1] if len(argv) > 1 else "c2"
    cfg = workloads.CONFIGS[name]
    ctx = make_context(cfg)
    res = run_scan(ctx, cfg["T"], cfg["sweeps"], cfg.get("equil", 0))
    print("# %s: %s, N = %d" % (name, cfg["kind"], ctx.n))
    print("# T  <|M|>  <E>/N  chi  C")
    for i in range(len(res["T"])):
        print("%.4f  %.6f  %.6f  %.4f  %.4f" % tuple(res[k][i] for k in ("T", "absM", "E", "chi", "C")))
    ctx.close()


if __name__ == "__main__":
    main(sys.argv)
