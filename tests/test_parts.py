"""Parts of a neighbour table (SURVEY 8(e) "CSR: partition by ... slabs of the canonical order"): host
logic on CPU (the cut, the ghost lists, the exchange between ranks under gloo), and on the GPU the partitioned trajectory
against the oracle's trajectory of the whole table."""
import os

import numpy as np
import pytest

from paper_2106_11286_b200 import parts, workloads
from test_multiproc import json_lines, torchrun


def first_fit(row_ptr, col_idx):
    """Greedy first-fit colouring in site order (a stand-in colouring for the host-logic tests)."""
    n = row_ptr.size - 1
    colour = np.full(n, -1, np.int32)
    for i in range(n):
        used = {int(colour[j]) for j in col_idx[row_ptr[i]:row_ptr[i + 1]] if colour[j] >= 0}
        c = 0
        while c in used:
            c += 1
        colour[i] = c
    return colour


@pytest.mark.parametrize("n,deg,n_parts", [(60, 3.0, 1), (200, 6.0, 2), (200, 6.0, 3), (333, 4.0, 7)])
def test_split_table_host_logic(n, deg, n_parts):
    rp, ci = workloads.random_csr_graph(n, deg, seed=n + n_parts)
    colour = first_fit(rp, ci)
    ps = parts.split_table(rp, ci, colour, n_parts)
    assert [p["first"] for p in ps] == parts.bounds_equal(n, n_parts)[:-1] and sum(p["n_own"] for p in ps) == n
    for r, p in enumerate(ps):
        g, n_own = p["to_global"], p["n_own"]
        assert np.array_equal(g[:n_own], np.arange(p["first"], p["first"] + n_own))
        assert np.all(np.diff(p["ghosts"]) > 0) and not np.any((p["ghosts"] >= p["first"]) & (p["ghosts"] < p["first"] + n_own))
        assert np.array_equal(p["colour"], colour[g])
        # every own row is the whole table's row, entry by entry, in local ids; ghost rows are empty
        for i in range(n_own):
            assert np.array_equal(g[p["col_idx"][p["row_ptr"][i]:p["row_ptr"][i + 1]]], ci[rp[p["first"] + i]:rp[p["first"] + i + 1]])
        assert np.all(np.diff(p["row_ptr"][n_own:]) == 0) and p["row_ptr"].size == g.size + 1
        # the ghosts are exactly the outside neighbours of the own rows
        cols = ci[rp[p["first"]]:rp[p["first"] + n_own]]
        assert set(p["ghosts"].tolist()) == {int(j) for j in cols if not p["first"] <= j < p["first"] + n_own}
        # what q sends to r (q's own sites) is, colour by colour and in the same order, what r receives from q (r's ghosts)
        seen = set()
        for q, by_colour in p["recv"].items():
            assert q != r
            for c, ids in by_colour.items():
                assert np.all(ids >= n_own) and np.all(colour[g[ids]] == c)
                assert np.array_equal(g[ids], ps[q]["to_global"][ps[q]["send"][r][c]]) and np.all(ps[q]["send"][r][c] < ps[q]["n_own"])
                seen.update(g[ids].tolist())
        assert seen == set(p["ghosts"].tolist())
        for q, by_colour in p["send"].items():
            assert all(c in ps[q]["recv"][r] for c in by_colour)
    with pytest.raises(ValueError):
        parts.bounds_equal(3, 4)


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_between_ranks_gloo(world):
    res = torchrun([os.path.join("tests", "gloo_parts_worker.py")], nproc=world)
    assert res.returncode == 0, res.stderr[-2000:]
    (r,) = json_lines(res.stdout)
    assert r["world"] == world and r["ok"] == [True] * world and r["own"] == r["n"] and r["ghosts"] > 0


# ---- GPU: the parts together walk the oracle's trajectory of the whole table ---------------------------------------------
def _sphere(R, colouring):
    import oracle
    import paper_2106_11286_b200 as hb
    lat = hb.Lattice.fcc_sphere(R, 0.05, (0.0, 0.0, 1.0), 0.5, colouring)
    olat = oracle.Lattice.fcc_sphere(R, 0.05, (0.0, 0.0, 1.0), 0.5, colouring)
    kw = dict(row_ptr=lat.row_ptr, col_idx=lat.col_idx, colour=lat.colour, K_site=lat.K_site, e_site=lat.e_site)
    return kw, olat


def _graph(n, deg, seed, per_site):
    import oracle
    rp, ci = workloads.random_csr_graph(n, deg, seed)
    colour = first_fit(rp, ci)
    olat = oracle.Lattice.csr(rp, ci, colour, int(colour.max()) + 1)
    kw = dict(row_ptr=rp, col_idx=ci, colour=colour)
    if per_site:
        kw["K_site"] = np.linspace(-0.3, 0.4, n).astype(np.float32)
        kw["e_site"] = workloads.random_unit_vectors(n, seed + 1)
        olat.set_site_anisotropy(kw["K_site"], kw["e_site"])
    else:
        olat.set_uniform_anisotropy(0.2, (0.0, 0.6, 0.8))
    return kw, olat


@pytest.mark.gpu
@pytest.mark.parametrize("case,n_parts", [
    ("sphere5", 1), ("sphere5", 2), ("sphere5", 4), ("sphere4_parity", 3),      # ELL engine, per-site anisotropy
    ("graph", 3), ("graph_persite", 2), ("hub", 2),                              # CSR engine
    ("sphere60", 3),                                                             # config 5 at full size (3.6 M sites)
])
def test_parts_walk_the_single_table_trajectory(case, n_parts):
    import oracle
    from hbtest import spins_equal
    if case.startswith("sphere"):
        kw, olat = _sphere({"sphere5": 5, "sphere4_parity": 4, "sphere60": 60}[case], "parity" if case.endswith("parity") else "greedy")
        K, e, T = 0.05, (0.0, 0.0, 1.0), 2.5
    elif case == "hub":
        # one site tied to 150 others on top of a sparse graph: padding every row would cost too much, so the CSR engine runs
        n = 600
        rp0, ci0 = workloads.random_csr_graph(n, 3.0, seed=5)
        adj = [set(ci0[rp0[i]:rp0[i + 1]].tolist()) for i in range(n)]
        for j in range(1, 151):
            adj[0].add(2 * j); adj[2 * j].add(0)
        rp = np.concatenate([[0], np.cumsum([len(a) for a in adj])]).astype(np.int64)
        ci = np.concatenate([sorted(a) for a in adj]).astype(np.int32)
        colour = first_fit(rp, ci)
        olat = oracle.Lattice.csr(rp, ci, colour, int(colour.max()) + 1)
        olat.set_uniform_anisotropy(0.2, (0.0, 0.6, 0.8))
        kw, K, e, T = dict(row_ptr=rp, col_idx=ci, colour=colour), 0.2, (0.0, 0.6, 0.8), 1.0
    else:
        kw, olat = _graph(700, 6.0, 21, case.endswith("persite"))
        K, e, T = 0.2, (0.0, 0.6, 0.8), 1.0
    st = oracle.State32(olat, 1.0, 99)
    P = parts.LocalParts(n_parts=n_parts, J=1.0, K=K, e=e, seed=99, **kw)
    assert (n_parts == 1) == all(p["ghosts"].size == 0 for p in P.parts)
    if case.startswith("sphere"):
        assert all(c.get_option("ell") == 1 for c in P.ctxs)
    if case == "hub":      # the part with the hub runs the CSR engine, the other one the ELL engine: the exchange does not care
        assert [c.get_option("ell") for c in P.ctxs] == [0, 1]
    P.init_random()
    st.init_random()
    assert spins_equal(P.get_spins(), st.get_spins()) and P.ghosts_current()
    for T_k, k in ((T, 3), (0.4 * T, 2)):
        P.sweep(T_k, k)
        st.sweep(T_k, k)
        assert spins_equal(P.get_spins(), st.get_spins()) and P.ghosts_current()
    M, E = P.measure()
    Mo, Eo = st.measure()[:2]
    assert np.max(np.abs(M - np.asarray(Mo))) <= 1e-7 and abs(E - Eo) <= 1e-6 * olat.n
    # a state handed in from the host (every part takes its own sites and its ghosts), then more sweeps
    rng = np.random.default_rng(3)
    v = rng.normal(size=(olat.n, 3))
    v = (v / np.linalg.norm(v, axis=1, keepdims=True)).astype(np.float32)
    P.set_spins(v[:, 0], v[:, 1], v[:, 2])
    st.set_spins(v[:, 0], v[:, 1], v[:, 2])
    P.sweep(T, 2)
    st.sweep(T, 2)
    assert spins_equal(P.get_spins(), st.get_spins()) and P.ghosts_current()
    P.close()


@pytest.mark.gpu
def test_part_contexts_refuse_whole_table_calls():
    import paper_2106_11286_b200 as hb
    rp, ci = workloads.random_csr_graph(100, 4.0, seed=2)
    colour = first_fit(rp, ci)
    p = parts.split_table(rp, ci, colour, 2)[1]
    ctx = hb.Context(parts.part_lattice(p, 100), 1.0, 0.0, (0, 0, 1), 1)
    ctx.init_random()
    assert ctx.n == p["to_global"].size
    for call in (lambda: ctx.sweep(1.0, 1), lambda: ctx.sweep_series(1.0, 2), lambda: ctx.sweep_record(1.0),
                 lambda: ctx.slab_pass(1.0, int(colour.max()) + 1)):
        with pytest.raises(hb.HbError):
            call()
    ctx.close()
    bad_row = p["row_ptr"].copy()
    bad_row[-1] += 1                                                  # a ghost row that is not empty
    for lat in [hb.Lattice("csr", row_ptr=p["row_ptr"], col_idx=p["col_idx"], part=(p["first"], p["n_own"], 100)),          # no colouring
                hb.Lattice("csr", row_ptr=p["row_ptr"], col_idx=p["col_idx"], colour=p["colour"], n_colours=p["n_colours"], part=(60, p["n_own"], 100)),
                hb.Lattice("csr", row_ptr=bad_row, col_idx=np.append(p["col_idx"], 0).astype(np.int32), colour=p["colour"], n_colours=p["n_colours"],
                           part=(p["first"], p["n_own"], 100)),
                hb.Lattice("sc", 4, 4, 4, part=(0, 32, 64))]:
        with pytest.raises(hb.HbError):
            hb.Context(lat, 1.0, 0.0, (0, 0, 1), 1)
    whole = hb.Context(hb.Lattice("csr", row_ptr=rp, col_idx=ci), 1.0, 0.0, (0, 0, 1), 1)
    with pytest.raises(hb.HbError):
        whole.slab_pass(1.0, 0)
    whole.close()


@pytest.mark.gpu
def test_two_processes_one_part_each():
    import base64
    import oracle
    from hbtest import spins_equal
    R = 4
    res = torchrun([os.path.join("tests", "gloo_parts_gpu_worker.py"), str(R)], nproc=2, timeout=600)
    assert res.returncode == 0, res.stderr[-3000:]
    (r,) = json_lines(res.stdout)
    olat = oracle.Lattice.fcc_sphere(R, 0.05, (0.0, 0.0, 1.0), 0.5, "greedy")
    st = oracle.State32(olat, 1.0, 77)
    st.init_random()
    st.sweep(2.5, 3)
    st.sweep(0.7, 2)
    got = [np.concatenate([np.frombuffer(base64.b64decode(part[k]), np.float32) for part in r["spins"]]) for k in range(3)]
    assert spins_equal(got, st.get_spins())
    Mo, Eo = st.measure()[:2]
    assert np.max(np.abs(np.asarray(r["M"]) - np.asarray(Mo))) <= 1e-7 and abs(r["E"] - Eo) <= 1e-6 * olat.n
