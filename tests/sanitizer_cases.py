"""Small cases of every engine for compute-sanitizer ("race detection").

    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py

The paper's own scheme tolerates concurrent updates of neighbouring spins ("loss of continuity"); the
colour sweeps here claim to have no race at all, so the code most at risk for that claim runs under the tools: the
mbarrier rings of the warp-specialised kernels (sc variants 2 / 4 / 5, bcc, fcc), their fused launches with progress
words, the cooperative and one-block persistent kernels, replicas, the graph-replay path, slabs with peer stores, the
table engines, parts of a table.  Every case is also checked against the oracle (the tools slow a kernel down, they do not change it).
Not collected by pytest (no test_ prefix): a plain script, so that the tool wraps ONE python process.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

import oracle  # noqa: E402
import paper_2106_11286_b200 as hb  # noqa: E402
from paper_2106_11286_b200 import slabs, workloads as W  # noqa: E402
from hbtest import make_gpu, make_oracle, spins_equal, start  # noqa: E402


def run(name, cfg, opts, sweeps=(1, 3), T=1.44):
    ctx = make_gpu(cfg)
    for k, v in opts:
        ctx.set_option(k, v)
    lat, st = make_oracle(cfg)
    start(cfg, ctx, st)
    for k in sweeps:
        ctx.sweep(T, k)
        st.sweep(T, k)
    ok = spins_equal(ctx.get_spins(), st.get_spins())
    Mg, Eg = ctx.measure()
    Mo, Eo, _ = st.measure()
    ok = ok and np.max(np.abs(Mg - Mo)) <= 1e-7 and abs(Eg - Eo) <= 1e-6 * lat.n
    ctx.close()
    print("%-44s %s" % (name, "ok" if ok else "MISMATCH"), flush=True)
    return ok


def main():
    sc = dict(W.SMALL["c4"], L=(64, 12, 10))
    good = True
    for v in (2, 4, 5):
        good &= run("sc ws variant %d" % v, sc, [("sc_coop", 0), ("graph", 0), ("sc_kernel", 1), ("sc_ws_variant", v)])
    good &= run("sc ws fused launches", sc, [("sc_coop", 0), ("graph", 0), ("sc_ws_variant", 4), ("sc_kernel", 2), ("sc_fused_zt", 2),
                                           ("sc_fused_lag", 3), ("sc_fused_sweeps", 2)], sweeps=(1, 5))
    good &= run("sc direct + graph replay", dict(W.SMALL["c4"], L=(24, 10, 8)), [("sc_coop", 0), ("graph", 1)], sweeps=(1, 18))
    good &= run("sc cooperative grid", dict(W.SMALL["c4"], L=(40, 12, 10)), [("sc_coop", 2)], sweeps=(1, 2))
    good &= run("sc one-block persistent", W.SMALL["c1"], [], sweeps=(1, 3), T=1.2)
    good &= run("bcc direct", W.SMALL["c2"], [("graph", 0)], T=1.8)
    good &= run("bcc ws", dict(W.SMALL["c2"], L=(16, 9, 6)), [("br_kernel", 1), ("graph", 0)], T=1.8)
    good &= run("bcc ws fused", dict(W.SMALL["c2"], L=(16, 9, 6)), [("br_kernel", 2), ("br_zt", 2), ("sc_fused_lag", 3), ("sc_fused_sweeps", 2)],
                sweeps=(1, 5), T=1.8)
    good &= run("fcc direct", dict(W.SMALL["c3"], start="random"), [("graph", 0)], T=3.0)
    good &= run("fcc ws fused", dict(W.SMALL["c3"], L=(8, 5, 6), start="random"), [("br_kernel", 2), ("br_zt", 2), ("sc_fused_sweeps", 2)],
                sweeps=(1, 5), T=3.0)
    good &= run("table engine, ELL (sphere R = 3)", dict(W.SMALL["c5"], R=3), [("graph", 0)], T=2.5)
    rp, ci = W.random_csr_graph(600, 6.0, seed=8)
    good &= run("table engine, CSR (random graph)", dict(kind="csr", row_ptr=rp, col_idx=ci, J=1.0, K=0.2, e=(0, 0, 1), seed=3, start="random",
                                                       T=[1.0]), [("graph", 0)], T=1.0)
    # replicas: one launch, one block per replica
    R = 4
    ctx = hb.Context(hb.Lattice("sc", 8, 8, 8, n_replicas=R), 1.0, 0.01, (0, 0, 1), seed=7)
    ctx.init_random()
    ctx.sweep_each([0.8, 1.2, 1.6, 2.4], 3)
    olat = oracle.Lattice.sc(8)
    olat.set_uniform_anisotropy(0.01, (0, 0, 1))
    ok = True
    for r, T in enumerate([0.8, 1.2, 1.6, 2.4]):
        st = oracle.State32(olat, 1.0, 7 + r)
        st.init_random()
        st.sweep(T, 3)
        ctx.select_replica(r)
        ok &= spins_equal(ctx.get_spins(), st.get_spins())
    ctx.close()
    print("%-44s %s" % ("sc replicas", "ok" if ok else "MISMATCH"), flush=True)
    good &= ok
    # slabs of one process with peer stores (the kernels write the neighbours' ghost planes)
    for kern in (0, 1):
        cfg = dict(W.SMALL["c4"], L=(64, 8, 12))
        sl = slabs.LocalSlabs(64, 8, 12, 3, cfg["J"], cfg["K"], cfg["e"], cfg["seed"], options={"sc_kernel": kern}, peer_stores=True)
        lat, st = make_oracle(cfg)
        sl.init_random()
        st.init_random()
        sl.sweep(1.44, 3)
        st.sweep(1.44, 3)
        ok = spins_equal(sl.get_spins(), st.get_spins())
        sl.close()
        print("%-44s %s" % ("3 slabs, peer stores, sc_kernel %d" % kern, "ok" if ok else "MISMATCH"), flush=True)
        good &= ok
    # parts of a neighbour table: gather / scatter kernels between three contexts (ELL engine)
    from paper_2106_11286_b200 import parts
    plat = hb.Lattice.fcc_sphere(4, 0.05, (0, 0, 1), 0.5, "greedy")
    P = parts.LocalParts(plat.row_ptr, plat.col_idx, plat.colour, 3, 1.0, 0.05, (0, 0, 1), 5, K_site=plat.K_site, e_site=plat.e_site)
    st = oracle.State32(oracle.Lattice.fcc_sphere(4, 0.05, (0, 0, 1), 0.5, "greedy"), 1.0, 5)
    P.init_random()
    st.init_random()
    P.sweep(2.0, 3)
    st.sweep(2.0, 3)
    ok = spins_equal(P.get_spins(), st.get_spins())
    P.close()
    print("%-44s %s" % ("3 parts of the sphere's table", "ok" if ok else "MISMATCH"), flush=True)
    good &= ok
    print("ALL OK" if good else "FAILED", flush=True)
    return 0 if good else 1


if __name__ == "__main__":
    sys.exit(main())
