"""Slab decomposition along z: host logic on CPU (partition, neighbour ranks, the face exchange
between ranks under gloo), and on the GPU the sharded trajectory against the oracle's single-lattice trajectory."""
import os

import numpy as np
import pytest

from paper_2106_11286_b200 import slabs
from test_multiproc import json_lines, torchrun


def test_partition_even_planes_cover_the_lattice():
    assert slabs.partition(464, 1) == [(0, 464)]
    assert slabs.partition(464, 8) == [(58 * r, 58) for r in range(8)]
    assert slabs.partition(20, 4) == [(0, 6), (6, 6), (12, 4), (16, 4)]
    for Lz in (2, 4, 10, 16, 30, 464):
        for G in range(1, Lz // 2 + 1):
            p = slabs.partition(Lz, G)
            assert p[0][0] == 0 and all(nz >= 2 and nz % 2 == 0 and z0 % 2 == 0 for z0, nz in p)
            assert all(p[r][0] + p[r][1] == p[r + 1][0] for r in range(G - 1)) and p[-1][0] + p[-1][1] == Lz
            assert max(nz for _, nz in p) - min(nz for _, nz in p) <= 2
    with pytest.raises(ValueError):
        slabs.partition(6, 4)
    with pytest.raises(ValueError):
        slabs.partition(7, 1)
    assert slabs.neighbours(0, 4) == (3, 1) and slabs.neighbours(3, 4) == (2, 0) and slabs.neighbours(0, 1) == (0, 0)


@pytest.mark.parametrize("world", [2, 3])
def test_face_exchange_between_ranks_gloo(world):
    res = torchrun([os.path.join("tests", "gloo_slab_worker.py")], nproc=world)
    assert res.returncode == 0, res.stderr[-2000:]
    (r,) = json_lines(res.stdout)
    assert r["world"] == world and r["sum"] == [sum(range(1, world + 1)), 0.0, 0.0, -2.0 * sum(range(1, world + 1))]
    for rank, ghosts in enumerate(r["ghosts"]):
        down, up = (rank - 1) % world, (rank + 1) % world
        for colour in (0, 1):
            for k in range(3):
                # low ghost plane <- the lower neighbour's high boundary plane; high ghost <- the upper neighbour's low one
                assert set(ghosts["%d0%d" % (colour, k)]) == {1000.0 * down + 100 * colour + 10 * 1 + k}
                assert set(ghosts["%d1%d" % (colour, k)]) == {1000.0 * up + 100 * colour + 10 * 0 + k}


# ---- GPU: the slabs together walk the oracle's trajectory of the whole lattice -----------------------------------------
def _oracle(shape, K, e, seed):
    import oracle
    lat = oracle.Lattice.sc(*shape)
    lat.set_uniform_anisotropy(K, e)
    return lat, oracle.State32(lat, 1.0, seed)


@pytest.mark.gpu
@pytest.mark.parametrize("shape,n_slabs,K,e,options", [
    ((16, 12, 16), 2, 0.0, (0.0, 0.0, 1.0), {}),
    ((16, 12, 20), 4, 0.05, (0.0, 0.0, 1.0), {}),                 # unequal slabs 6, 6, 4, 4
    ((8, 4, 4), 2, 0.3, (0.6, 0.0, 0.8), {}),                     # two-plane slabs: every plane is a boundary plane
    ((16, 12, 12), 1, 0.05, (0.0, 0.0, 1.0), {}),                 # one slab feeding its own ghost planes
    ((40, 14, 24), 3, 0.01, (0.0, 0.0, 1.0), {"sc_kernel": 1}),   # warp-specialised kernel, ragged tiles
    ((464, 8, 8), 2, 0.01, (0.0, 0.0, 1.0), {"sc_kernel": 1}),    # config 4's rows (7-row tiles)
])
def test_slabs_walk_the_single_lattice_trajectory(shape, n_slabs, K, e, options):
    from hbtest import spins_equal
    seed = 12345
    lat, st = _oracle(shape, K, e, seed)
    sl = slabs.LocalSlabs(*shape, n_slabs, J=1.0, K=K, e=e, seed=seed, options=options)
    st.init_random()
    sl.init_random()                       # Philox draw 1 keyed by the global site id
    assert spins_equal(sl.get_spins(), st.get_spins())
    for T, k in ((1.44, 1), (1.44, 3), (0.5, 2)):
        sl.sweep(T, k)
        st.sweep(T, k)
        assert spins_equal(sl.get_spins(), st.get_spins()), (shape, n_slabs, T)
        Mg, Eg = sl.measure()
        Mo, Eo = st.measure()[:2]
        assert np.max(np.abs(Mg - np.asarray(Mo))) <= 1e-7 and abs(Eg - Eo) <= 1e-6 * lat.n
    # a state handed in from the host, and the checkpointed sweep counter, continue the same trajectory
    sx, sy, sz = st.get_spins()
    sl2 = slabs.LocalSlabs(*shape, n_slabs, J=1.0, K=K, e=e, seed=seed, options=options)
    sl2.set_spins(sx, sy, sz)
    for c in sl2.ctxs:
        c.sweep_count = st.sweep_count
    sl2.sweep(1.2, 2)
    st.sweep(1.2, 2)
    assert spins_equal(sl2.get_spins(), st.get_spins())
    sl.close()
    sl2.close()


@pytest.mark.gpu
@pytest.mark.parametrize("shape,n_slabs,options", [
    ((16, 12, 16), 2, {}), ((16, 12, 20), 4, {}), ((8, 4, 4), 2, {}), ((16, 12, 12), 1, {}),
    ((40, 14, 24), 3, {"sc_kernel": 1}), ((464, 8, 8), 2, {"sc_kernel": 1}), ((64, 20, 12), 2, {"sc_kernel": 1, "sc_ws_variant": 2}),
])
def test_peer_stores_replace_the_exchange_step(shape, n_slabs, options):
    # hb_slab_set_peer: the colour kernels store their boundary planes into the neighbours' ghost planes themselves; after
    # the initial fill no face is ever copied, and the slabs still walk the oracle's trajectory of the whole lattice
    from hbtest import spins_equal
    K, e, seed = 0.05, (0.0, 0.6, 0.8), 99
    lat, st = _oracle(shape, K, e, seed)
    sl = slabs.LocalSlabs(*shape, n_slabs, J=1.0, K=K, e=e, seed=seed, options=options, peer_stores=True)
    st.init_random()
    sl.init_random()
    for T, k in ((1.44, 1), (1.44, 5), (0.3, 3), (50.0, 2)):     # low and high acceptance: few / all boundary stores
        sl.sweep(T, k)
        st.sweep(T, k)
        assert spins_equal(sl.get_spins(), st.get_spins()), (shape, n_slabs, T)
        Mg, Eg = sl.measure()
        Mo, Eo = st.measure()[:2]
        assert np.max(np.abs(Mg - np.asarray(Mo))) <= 1e-7 and abs(Eg - Eo) <= 1e-6 * lat.n
    # the ghost planes hold exactly the neighbours' boundary planes (what a face exchange would have written)
    for colour in (0, 1):
        for r, c in enumerate(sl.ctxs):
            down, up = slabs.neighbours(r, n_slabs)
            for mine, theirs in zip(c.slab_face(colour, 0, True), sl.ctxs[down].slab_face(colour, 1, False)):
                assert bool((mine == theirs).all())
            for mine, theirs in zip(c.slab_face(colour, 1, True), sl.ctxs[up].slab_face(colour, 0, False)):
                assert bool((mine == theirs).all())
    sl.close()


@pytest.mark.gpu
@pytest.mark.parametrize("shape,n_slabs,options", [
    ((40, 14, 24), 3, {"sc_kernel": 1}), ((464, 8, 8), 2, {}), ((64, 20, 12), 2, {"sc_kernel": 1, "sc_ws_variant": 2}),
    ((64, 16, 40), 1, {"sc_ws_variant": 4}), ((64, 16, 44), 4, {"sc_ws_variant": 5, "sc_ws_zt": 3}),
])
def test_neighbour_flags_replace_the_barrier(shape, n_slabs, options):
    # hb_set_option("slab_flags", 1): boundary chunks first, a boundary tile waits for its neighbour's flag of the pass before,
    # the last warp of a boundary chunk sets the neighbour's flag.  On one stream every flag is already set when it is waited
    # for: the test covers the bookkeeping (stamps, counters, flag words behind the spins, chunk order), bit for bit against
    # the oracle, and that every slab has published every pass.
    import torch
    from hbtest import spins_equal
    K, e, seed = 0.05, (0.0, 0.6, 0.8), 99
    lat, st = _oracle(shape, K, e, seed)
    sl = slabs.LocalSlabs(*shape, n_slabs, J=1.0, K=K, e=e, seed=seed, options=options, peer_stores=True, flags=True)
    assert all(c.get_option("slab_flags") == 1 and c.get_option("sc_kernel") == 1 for c in sl.ctxs)
    st.init_random()
    sl.init_random()
    passes = 0
    for T, k in ((1.44, 1), (1.44, 4), (0.3, 2)):
        sl.sweep(T, k)
        st.sweep(T, k)
        passes += 2 * k
        assert spins_equal(sl.get_spins(), st.get_spins()), (shape, n_slabs, T)
        for c, (z0, nz) in zip(sl.ctxs, sl.parts):      # both flag words of every slab (behind its spins) carry the number of the last pass
            at = 12 * shape[0] * shape[1] * (nz + 2)
            words = c._spins[at:at + 8].view(torch.int32).cpu().numpy()
            assert list(words) == [passes, passes], (words, passes)
    Mg, Eg = sl.measure()
    Mo, Eo = st.measure()[:2]
    assert np.max(np.abs(Mg - np.asarray(Mo))) <= 1e-7 and abs(Eg - Eo) <= 1e-6 * lat.n
    sl.close()


@pytest.mark.gpu
def test_slab_contexts_refuse_whole_lattice_calls():
    import paper_2106_11286_b200 as hb
    ctx = hb.Context(hb.Lattice("sc", 8, 4, 4, slab=(4, 12)), 1.0, 0.0, (0, 0, 1), 1)
    ctx.init_random()
    assert ctx.n == 8 * 4 * 4
    with pytest.raises(hb.HbError):
        ctx.sweep(1.0, 1)
    with pytest.raises(hb.HbError):
        ctx.sweep_series(1.0, 2)
    with pytest.raises(hb.HbError):
        ctx.slab_pass(1.0, 2)
    ctx.close()
    for bad in [dict(slab=(3, 12)), dict(slab=(4, 6)), dict(slab=(0, 11))]:
        with pytest.raises(hb.HbError):
            hb.Context(hb.Lattice("sc", 8, 4, 4, **bad), 1.0, 0.0, (0, 0, 1), 1)
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("bcc", 4, 4, 4, slab=(6, 8)), 1.0, 0.0, (0, 0, 1), 1)     # 6 + 4 planes do not fit into 8
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("sc", 8, 4, 4, slab=(4, 12), n_replicas=2), 1.0, 0.0, (0, 0, 1), 1)
    whole = hb.Context(hb.Lattice("sc", 8, 4, 4), 1.0, 0.0, (0, 0, 1), 1)
    with pytest.raises(hb.HbError):
        whole.slab_pass(1.0, 0)
    whole.close()


@pytest.mark.gpu
def test_dist_slab_single_rank():
    # world_size 1: the rank's slab is the whole lattice and feeds its own ghost planes; all_reduce is skipped
    import torch.distributed as dist
    from hbtest import spins_equal
    from test_multiproc import free_port
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % free_port(), rank=0, world_size=1)
    try:
        lat, st = _oracle((16, 8, 8), 0.05, (0.0, 0.0, 1.0), 7)
        d = slabs.DistSlab(16, 8, 8, 1.0, 0.05, (0.0, 0.0, 1.0), 7)
        d.init_random()
        st.init_random()
        d.sweep(1.3, 4)
        st.sweep(1.3, 4)
        assert spins_equal(d.get_spins(), st.get_spins())
        M, E = d.measure()
        Mo, Eo = st.measure()[:2]
        assert np.max(np.abs(M - np.asarray(Mo))) <= 1e-7 and abs(E - Eo) <= 1e-6 * lat.n
        d.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
@pytest.mark.skipif(os.environ.get("HB_TEST_HUGE") != "1", reason="70 GB of device memory, outside SURVEY 8: set HB_TEST_HUGE=1 to run it")
def test_more_than_2_31_sites_whole_lattice_equals_its_slabs():
    # 1600 x 1600 x 840 = 2,150,400,000 sites (> 2^31; 25.8 GB of spins): a property that holds at any size -- the whole
    # lattice in one context and the same lattice as two slabs (1.08e9 sites each, other index ranges in every kernel)
    # walk the same trajectory, so M and E agree to the rounding of the final fp64 sums.  The paper stops at 512^3
    # ("1024^3 ... each array would occupy 4.3 GB"); site ids are 32-bit Philox counter words, so the
    # limit here is 2^32 - 1 sites.
    import torch
    import paper_2106_11286_b200 as hb
    if torch.cuda.mem_get_info()[1] < 100e9:
        pytest.skip("needs ~70 GB of device memory")
    shape, T = (1600, 1600, 840), 1.44
    ctx = hb.Context(hb.Lattice("sc", *shape), 1.0, 0.01, (0.0, 0.0, 1.0), 1)
    ctx.init_random()
    ctx.sweep(T, 2)
    M, E = ctx.measure()
    n = ctx.n
    ctx.close()
    del ctx
    torch.cuda.empty_cache()
    assert n == 2150400000 and np.linalg.norm(M) < 1e-3 and -1.0 < E / n < -0.3   # two sweeps after a random start
    sl = slabs.LocalSlabs(*shape, 2, J=1.0, K=0.01, e=(0.0, 0.0, 1.0), seed=1)
    sl.init_random()
    sl.sweep(T, 2)
    Ms, Es = sl.measure()
    sl.close()
    del sl
    torch.cuda.empty_cache()
    assert np.max(np.abs(Ms - M)) <= 1e-12 and abs(Es - E) <= 1e-12 * abs(E)


def test_order_parameter_fit_recovers_a_power_law():
    # host logic of `scan --sc L --fit`: log-log least squares with T_C scanned (the form fitted in the paper's Fig. 3 inset)
    from paper_2106_11286_b200.scan import fit_order_parameter
    T = np.linspace(1.2, 1.5, 61)
    Tc, beta, A = 1.443, 0.3645, 1.05
    m = np.where(T < Tc, A * np.clip(1.0 - T / Tc, 1e-12, None) ** beta, 1e-3)
    got = fit_order_parameter(T, m, 0.01, 0.1)
    assert abs(got[0] - Tc) <= 6e-4 and abs(got[1] - beta) <= 5e-3 and abs(got[2] - A) <= 2e-2 and got[3] < 2e-3


@pytest.mark.gpu
@pytest.mark.parametrize("mode", ["copies", "peer"])
def test_two_processes_one_slab_each(mode):
    # one process per slab (torchrun, gloo, both ranks on cuda:0): faces by send/recv, or -- "peer" -- no faces at all:
    # each rank maps the other's spins buffer through CUDA IPC and the colour kernels store into its ghost planes
    import base64
    from hbtest import spins_equal
    shape = (16, 12, 16)
    res = torchrun([os.path.join("tests", "gloo_slab_gpu_worker.py"), mode] + [str(x) for x in shape], nproc=2, timeout=600)
    assert res.returncode == 0, res.stderr[-3000:]
    (r,) = json_lines(res.stdout)
    lat, st = _oracle(shape, 0.05, (0.0, 0.6, 0.8), 4242)
    st.init_random()
    st.sweep(1.44, 3)
    st.sweep(0.4, 2)
    got = [np.concatenate([np.frombuffer(base64.b64decode(part[k]), np.float32) for part in r["spins"]]) for k in range(3)]
    assert spins_equal(got, st.get_spins())
    Mo, Eo = st.measure()[:2]
    assert np.max(np.abs(np.asarray(r["M"]) - np.asarray(Mo))) <= 1e-7 and abs(r["E"] - Eo) <= 1e-6 * lat.n


def test_slab_lattice_sizes_host_logic():
    # hb_sizes runs no device code: a slab reports its own sites and a buffer that also holds the two ghost planes
    import paper_2106_11286_b200 as hb
    n, spins, ws = hb.sizes(hb.Lattice("sc", 8, 4, 4, slab=(4, 12)))
    n_whole, spins_whole, _ = hb.sizes(hb.Lattice("sc", 8, 4, 6))
    assert n == 8 * 4 * 4 and spins == spins_whole + 256 and spins_whole >= 3 * 4 * 8 * 4 * 6   # + the neighbour flag words behind the spins
    for bad in [dict(slab=(3, 12)), dict(slab=(4, 6)), dict(slab=(0, 11)), dict(slab=(-2, 12))]:
        with pytest.raises(hb.HbError):
            hb.sizes(hb.Lattice("sc", 8, 4, 4, **bad))
    assert hb.sizes(hb.Lattice("fcc", 4, 4, 3, slab=(1, 8)))[0] == 4 * 4 * 4 * 3       # bcc / fcc slabs: any offset, own sites of all sublattices
    with pytest.raises(hb.HbError):
        hb.sizes(hb.Lattice("fcc", 4, 4, 4, slab=(6, 8)))
    # implicit lattices go up to 2^32 - 1 sites; the table engine is bounded by its 32-bit neighbour offsets
    assert hb.sizes(hb.Lattice("sc", 1600, 1600, 1600))[0] == 4096000000
    with pytest.raises(hb.HbError):
        hb.sizes(hb.Lattice("sc", 1626, 1626, 1626))


@pytest.mark.gpu
@pytest.mark.parametrize("kind,shape,n_slabs,K,e", [
    ("bcc", (8, 6, 8), 2, 0.1, (0.0, 0.0, 1.0)), ("bcc", (12, 5, 12), 3, 0.3, (0.6, 0.0, 0.8)), ("bcc", (4, 4, 4), 1, 0.0, (0.0, 0.0, 1.0)),
    ("fcc", (8, 6, 8), 2, 0.05, (0.0, 0.6, 0.8)), ("fcc", (4, 3, 12), 4, 0.0, (0.0, 0.0, 1.0)), ("fcc", (16, 4, 6), 3, 0.2, (0.0, 0.0, 1.0)),
])
def test_bcc_and_fcc_slabs_walk_the_single_lattice_trajectory(kind, shape, n_slabs, K, e):
    # SURVEY 8(e) for the lattices with a basis: slabs of conventional cells, one ghost cell plane per side and sublattice, one
    # face exchange per sublattice pass; Philox keyed by the global site id b * Ncell + cell, so the slabs together walk the
    # oracle's trajectory of the whole lattice bit for bit, from init_random, from a state handed in, and in M and E
    import oracle
    from hbtest import spins_equal
    lat = getattr(oracle.Lattice, kind)(*shape)
    lat.set_uniform_anisotropy(K, e)
    st = oracle.State32(lat, 1.0, 31)
    sl = slabs.LocalSlabs(*shape, n_slabs, J=1.0, K=K, e=e, seed=31, kind=kind)
    assert sl.n == lat.n
    st.init_random()
    sl.init_random()
    assert spins_equal(sl.get_spins(), st.get_spins())
    for T, k in ((2.0, 1), (2.0, 4), (0.4, 3)):
        sl.sweep(T, k)
        st.sweep(T, k)
        assert spins_equal(sl.get_spins(), st.get_spins()), (kind, shape, n_slabs, T)
        Mg, Eg = sl.measure()
        Mo, Eo = st.measure()[:2]
        assert np.max(np.abs(Mg - np.asarray(Mo))) <= 1e-7 and abs(Eg - Eo) <= 1e-6 * lat.n
    sl2 = slabs.LocalSlabs(*shape, n_slabs, J=1.0, K=K, e=e, seed=31, kind=kind)      # checkpoint: state + counter handed in
    sl2.set_spins(*st.get_spins())
    for c in sl2.ctxs:
        c.sweep_count = st.sweep_count
    sl2.sweep(1.5, 2)
    st.sweep(1.5, 2)
    assert spins_equal(sl2.get_spins(), st.get_spins())
    sl.close()
    sl2.close()


def test_flagged_sweeps_end_with_one_barrier_before_anything_reads_the_ghost_planes():
    """Host logic only: with neighbour flags a pass is ordered against the neighbours' NEXT pass, so the stores
    their LAST pass makes into this slab's ghost planes are ordered by nothing unless sweep() ends with a barrier.  A stub
    context records the call order; no device, no process group."""
    calls = []

    class Ctx:
        def slab_pass(self, T, colour):
            calls.append(("pass", colour))

        def slab_next_sweep(self):
            calls.append(("next",))

    for flags, want in ((True, [("pass", 0), ("pass", 1), ("next",)] * 3 + [("barrier",)]),
                        (False, [("pass", 0), ("barrier",), ("pass", 1), ("barrier",), ("next",)] * 3)):
        d = slabs.DistSlab.__new__(slabs.DistSlab)
        d.ctx, d.n_colours, d.peer_stores, d.flags, d.world = Ctx(), 2, True, flags, 2
        d._pass_barrier = lambda: calls.append(("barrier",))
        del calls[:]
        d.sweep(1.0, 3)
        assert calls == want
        del calls[:]
        d.sweep(1.0, 0)
        assert calls == []
