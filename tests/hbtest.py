"""Test helpers: build the CUDA context and the oracle state for one workload description.

The two sides are constructed independently (each with its own lattice builder and its own
colouring); only the description (paper_2106_11286_b200.workloads) is shared.
"""
import numpy as np

import oracle
import paper_2106_11286_b200 as hb


def make_gpu(cfg, **kw):
    kind = cfg["kind"]
    if kind == "sphere":
        lat = hb.Lattice.fcc_sphere(cfg["R"], cfg["K"], cfg["e"], cfg["K_surf"], cfg.get("colouring", "greedy"))
    elif kind == "csr":
        lat = hb.Lattice("csr", row_ptr=cfg["row_ptr"], col_idx=cfg["col_idx"], colour=cfg.get("colour"),
                         n_colours=cfg.get("n_colours", 0), K_site=cfg.get("K_site"), e_site=cfg.get("e_site"))
    else:
        L = cfg["L"]
        Lx, Ly, Lz = (L, L, L) if isinstance(L, int) else L
        lat = hb.Lattice(kind, Lx, Ly, Lz, K_site=cfg.get("K_site"), e_site=cfg.get("e_site"))
    ctx = hb.Context(lat, cfg["J"], cfg["K"], cfg["e"], cfg["seed"], **kw)
    return ctx


def make_oracle(cfg):
    kind = cfg["kind"]
    if kind == "sphere":
        lat = oracle.Lattice.fcc_sphere(cfg["R"], cfg["K"], cfg["e"], cfg["K_surf"], cfg.get("colouring", "greedy"))
    elif kind == "csr":
        lat = oracle.Lattice.csr(cfg["row_ptr"], cfg["col_idx"], cfg.get("colour"), cfg.get("n_colours", 0))
        if cfg.get("K_site") is not None:
            lat.set_site_anisotropy(cfg["K_site"], cfg["e_site"])
        else:
            lat.set_uniform_anisotropy(cfg["K"], cfg["e"])
    else:
        L = cfg["L"]
        Lx, Ly, Lz = (L, L, L) if isinstance(L, int) else L
        lat = getattr(oracle.Lattice, kind)(Lx, Ly, Lz)
        if cfg.get("K_site") is not None:
            lat.set_site_anisotropy(cfg["K_site"], cfg["e_site"])
        else:
            lat.set_uniform_anisotropy(cfg["K"], cfg["e"])
    st = oracle.State32(lat, cfg["J"], cfg["seed"])
    return lat, st


def start(cfg, ctx, st):
    if cfg["start"] == "random":
        ctx.init_random()
        st.init_random()
    else:
        ctx.init_aligned(cfg["e"])
        st.init_aligned(cfg["e"])


def spins_equal(a, b):
    return all(np.array_equal(x.view(np.uint32), y.view(np.uint32)) for x, y in zip(a, b))


def compare_trajectory(cfg, ctx, st, T, n_sweeps, record=True):
    """Run n_sweeps on both sides; returns (attempts, decision mismatches, max |dS| on agreeing sites,
    sites whose spins differ bitwise at the end)."""
    n = ctx.n
    attempts = mism = 0
    max_ds = 0.0
    for s in range(n_sweeps):
        acc_o = st.sweep(T, 1, record=True)[0]
        if record:
            acc_g = ctx.sweep_record(T)
            assert acc_g.max() <= 1, "a site was not attempted"
            bad = acc_g != acc_o
            mism += int(bad.sum())
        else:
            ctx.sweep(T, 1)
            bad = np.zeros(n, bool)
        attempts += n
        g, o = ctx.get_spins(), st.get_spins()
        ok = ~bad
        for x, y in zip(g, o):
            if ok.any():
                max_ds = max(max_ds, float(np.max(np.abs(x[ok].astype(np.float64) - y[ok].astype(np.float64)))))
    g, o = ctx.get_spins(), st.get_spins()
    differ = int(np.sum((g[0].view(np.uint32) != o[0].view(np.uint32)) | (g[1].view(np.uint32) != o[1].view(np.uint32)) |
                        (g[2].view(np.uint32) != o[2].view(np.uint32))))
    return attempts, mism, max_ds, differ
