"""GPU-vs-oracle parity through the C ABI.

Bar (BASELINE.json north_star): identical accept/reject decisions on >= 99.9999 % of the
attempts of the first 10 sweeps, max |dS_component| <= 1e-5 on agreeing sites.  With the
arithmetic contract of DESIGN.md section 4 the expected result is 100 % and 0.0; the
small cases assert exactly that, the full-size cases assert the bar and print the counts.
"""
import math

import numpy as np
import pytest

import oracle
import paper_2106_11286_b200 as hb
from paper_2106_11286_b200 import workloads as W

from hbtest import compare_trajectory, make_gpu, make_oracle, spins_equal, start

pytestmark = pytest.mark.gpu


def _bar(attempts, mism, max_ds):
    assert mism <= 1e-6 * attempts, (attempts, mism)
    assert max_ds <= 1e-5, max_ds


def _measure_close(ctx, st, n):
    Mg, Eg = ctx.measure()
    Mo, Eo32, Eo64 = st.measure()
    assert np.max(np.abs(Mg - Mo)) <= 1e-7                      # P2
    assert abs(Eg - Eo32) <= 1e-6 * n and abs(Eg - Eo64) <= 1e-6 * n


SMALL_CASES = {
    "sc16_c1": W.SMALL["c1"],
    "sc24_K": W.SMALL["c4"],
    "sc_v2_ragged": dict(W.SMALL["c4"], L=(12, 10, 6), K=0.3, e=(0.6, 0.0, 0.8)),
    "sc_v1": dict(W.SMALL["c4"], L=(6, 4, 2), K=-0.2, e=(0.0, 1.0, 0.0)),
    "sc_L2": dict(W.SMALL["c4"], L=2, K=0.2),
    "sc_wide": dict(W.SMALL["c4"], L=(528, 6, 4)),
    "bcc8": W.SMALL["c2"],
    "bcc_ragged": dict(W.SMALL["c2"], L=(3, 4, 5)),
    "fcc6": W.SMALL["c3"],
    "fcc_ragged": dict(W.SMALL["c3"], L=(5, 3, 4), start="random"),
    "sphere5": W.SMALL["c5"],
    "sphere5_parity": dict(W.SMALL["c5"], colouring="parity"),
    "sphere2": dict(W.SMALL["c5"], R=2),
    # per-site anisotropy on the periodic kinds runs on the table engine (ELL, maxdeg 6 / 8 / 12)
    "sc_persite": dict(W.SMALL["c4"], L=(6, 4, 8), K_site=np.linspace(-0.4, 0.6, 192).astype(np.float32),
                       e_site=W.random_unit_vectors(192, 21)),
    "bcc_persite": dict(W.SMALL["c2"], L=(4, 3, 5), K_site=np.linspace(0.5, -0.3, 120).astype(np.float32),
                        e_site=W.random_unit_vectors(120, 22)),
    "fcc_persite": dict(W.SMALL["c3"], L=(3, 4, 2), start="random", K_site=np.linspace(0.0, 0.8, 96).astype(np.float32),
                        e_site=W.random_unit_vectors(96, 23)),
}


@pytest.mark.parametrize("name", sorted(SMALL_CASES))
def test_small_trajectories_bit_exact(name):
    cfg = SMALL_CASES[name]
    ctx = make_gpu(cfg)
    lat, st = make_oracle(cfg)
    assert ctx.n == lat.n
    col, nc = ctx.colouring()
    assert nc == lat.n_colours and np.array_equal(col, lat.colour)
    start(cfg, ctx, st)
    assert spins_equal(ctx.get_spins(), st.get_spins())          # a3: same initial state
    for T in (cfg["T"][0], 0.3):
        attempts, mism, max_ds, differ = compare_trajectory(cfg, ctx, st, T, 5)
        assert attempts == 5 * lat.n and mism == 0 and max_ds == 0.0 and differ == 0
        _measure_close(ctx, st, lat.n)
    assert ctx.sweep_count == st.sweep_count == 10
    # the production kernels (no recording) walk the same trajectory: one launch per colour, and for the sc
    # engine the persistent cooperative multi-sweep kernel that small lattices use by default
    sc_engine = cfg["kind"] == "sc" and cfg.get("K_site") is None
    if sc_engine:
        ctx.set_option("sc_coop", 0)
    ctx.sweep(1.0, 3)
    if sc_engine:
        ctx.set_option("sc_coop", 1)
    ctx.sweep(1.0, 4)
    st.sweep(1.0, 7)
    assert spins_equal(ctx.get_spins(), st.get_spins())
    _measure_close(ctx, st, lat.n)
    ctx.close()


def test_sc_tile_shapes_do_not_change_the_result():
    cfg = dict(W.SMALL["c4"], L=(40, 12, 10))
    lat, st = make_oracle(cfg)
    st.init_random()
    st.sweep(1.44, 3)
    want = st.get_spins()
    for v, jx, ty, zt, coop in [(4, 5, 12, 10, 0), (4, 3, 5, 3, 0), (4, 1, 1, 1, 0), (2, 10, 7, 4, 0), (1, 20, 12, 2, 0),
                                (4, 5, 51, 10, 0), (4, 5, 12, 10, 2), (4, 3, 5, 3, 2), (4, 2, 7, 4, 2), (4, 5, 51, 10, 2),
                                (4, 5, 12, 10, 1), (4, 5, 60, 10, 0), (4, 5, 200, 5, 0)]:   # the last two: 512- and 1024-thread blocks
        ctx = make_gpu(cfg)
        ctx.set_option("sc_coop", coop)
        ctx.set_option("sc_v", v)
        ctx.set_option("sc_jx", jx)
        ctx.set_option("sc_ty", ty)
        ctx.set_option("sc_zt", zt)
        ctx.init_random()
        ctx.sweep(1.44, 3)
        assert spins_equal(ctx.get_spins(), want), (v, jx, ty, zt, coop)
        ctx.close()


def test_random_graph_greedy_colouring_and_per_site_anisotropy():
    n = 5000
    rp, ci = W.random_csr_graph(n, 7.0, seed=3)
    rng = np.random.default_rng(4)
    cfg = dict(kind="csr", row_ptr=rp, col_idx=ci, J=0.8, K=0.0, e=(0, 0, 1), seed=77, start="random",
               K_site=rng.uniform(-0.5, 0.5, n).astype(np.float32), e_site=W.random_unit_vectors(n, 5))
    ctx = make_gpu(cfg)
    lat, st = make_oracle(cfg)
    col, nc = ctx.colouring()                                    # both sides ran first-fit on their own
    assert nc == lat.n_colours and np.array_equal(col, lat.colour)
    assert ctx.get_option("ell") == 0                            # irregular degrees: the plain CSR kernel
    sph = make_gpu(W.SMALL["c5"])
    assert sph.get_option("ell") == 1                            # a cut-out of a regular lattice: the ELL kernel
    sph.close()
    start(cfg, ctx, st)
    attempts, mism, max_ds, differ = compare_trajectory(cfg, ctx, st, 0.9, 6)
    assert mism == 0 and max_ds == 0.0 and differ == 0
    _measure_close(ctx, st, n)
    # isolated sites and an empty colour are legal
    rp2 = np.zeros(11, np.int64)
    cfg2 = dict(kind="csr", row_ptr=rp2, col_idx=np.zeros(0, np.int32), colour=np.full(10, 2, np.int32), n_colours=4,
                J=1.0, K=0.7, e=(0, 0, 1), seed=5, start="random")
    c2 = make_gpu(cfg2)
    l2, s2 = make_oracle(cfg2)
    start(cfg2, c2, s2)
    assert compare_trajectory(cfg2, c2, s2, 0.5, 4)[1:] == (0, 0.0, 0)


def test_set_get_spins_and_checkpoint_identity():
    cfg = W.SMALL["c4"]
    lat, st = make_oracle(cfg)
    S = W.random_unit_vectors(lat.n, 9)
    a = make_gpu(cfg)
    a.set_spins(S[:, 0], S[:, 1], S[:, 2])
    back = a.get_spins()
    assert all(np.array_equal(back[k], S[:, k]) for k in range(3))     # layout round trip
    st.set_spins(S[:, 0], S[:, 1], S[:, 2])
    _measure_close(a, st, lat.n)
    a.sweep(1.44, 6)
    b = make_gpu(cfg)
    b.set_spins(S[:, 0], S[:, 1], S[:, 2])
    b.sweep(1.44, 3)
    c = make_gpu(cfg)                                                   # K12: resume from (spins, counter)
    c.set_spins(*b.get_spins())
    c.sweep_count = b.sweep_count
    c.sweep(1.44, 3)
    assert spins_equal(a.get_spins(), c.get_spins())
    st.sweep(1.44, 6)
    assert spins_equal(a.get_spins(), st.get_spins())


def test_c1_full_series():
    # config 1 as specified: sc 16^3, K=0, T=1.2, 1000 sweeps, M and E every sweep
    cfg = W.CONFIGS["c1"]
    ctx = make_gpu(cfg)
    lat, st = make_oracle(cfg)
    start(cfg, ctx, st)
    Mg, Eg = ctx.sweep_series(1.2, 1000)
    Mo, Eo = st.series(1.2, 1000)
    assert spins_equal(ctx.get_spins(), st.get_spins())
    assert np.max(np.abs(Mg - Mo)) <= 1e-7
    assert np.max(np.abs(Eg - Eo)) <= 1e-6 * lat.n
    nrm = sum(x.astype(np.float64) ** 2 for x in ctx.get_spins())
    assert np.max(np.abs(nrm - 1.0)) <= 5e-7                            # K3
    launches, attempts = ctx.counters()
    assert attempts == 1000 * lat.n and launches >= 1
    # the same series from one launch per colour (the persistent kernel off)
    ctx2 = make_gpu(cfg)
    ctx2.set_option("sc_coop", 0)
    ctx2.init_random()
    M2, E2 = ctx2.sweep_series(1.2, 1000)
    assert spins_equal(ctx2.get_spins(), st.get_spins())
    assert np.max(np.abs(M2 - Mo)) <= 1e-7 and np.max(np.abs(E2 - Eo)) <= 1e-6 * lat.n
    assert ctx2.counters()[0] >= 2000


def test_limits_on_device():
    cfg = dict(W.SMALL["c4"], L=16)
    ctx = make_gpu(cfg)
    ctx.init_aligned((0, 0, 1))
    acc = ctx.sweep_record(float("inf"))                                # K8: T = inf accepts everything
    assert acc.min() == 1 and acc.max() == 1
    M, _ = ctx.sweep_series(float("inf"), 100)
    absM = np.linalg.norm(M, axis=1)
    assert abs(absM.mean() - math.sqrt(8 / (3 * math.pi * ctx.n))) < 4 * absM.std(ddof=1) / 10
    ctx.init_aligned((0, 0, 1))
    ctx.sweep(0.01, 20)                                                 # K9: T -> 0 stays ordered
    M, E = ctx.measure()
    assert np.linalg.norm(M) > 0.99 and E / ctx.n < -2.98


def test_error_paths():
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("sc", 15))                                # odd L
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("sc", 8), e=(0, 0, 2))                    # non-unit axis
    rp = np.array([0, 1, 1], np.int64)
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("csr", row_ptr=rp, col_idx=np.array([1], np.int32)))   # asymmetric
    rp = np.array([0, 1, 2], np.int64)
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("csr", row_ptr=rp, col_idx=np.array([1, 0], np.int32),
                              colour=np.zeros(2, np.int32), n_colours=1))             # improper colouring
    ctx = hb.Context(hb.Lattice("sc", 8))
    with pytest.raises(hb.HbError):
        ctx.sweep(1.0, 1)                                               # before init
    ctx.init_random()
    for T in (0.0, -1.0, float("nan")):
        with pytest.raises(hb.HbError):
            ctx.sweep(T, 1)
    ctx.sweep(1.0, 0)                                                   # no-op
    assert ctx.sweep_count == 0


# ---- full-size configs: first 10 sweeps, every attempt ------------------------------------------
@pytest.mark.parametrize("name", ["c2", "c3", "c5", "c4"])
def test_full_size_first_10_sweeps(name):
    cfg = W.CONFIGS[name]
    ctx = make_gpu(cfg)
    lat, st = make_oracle(cfg)
    start(cfg, ctx, st)
    T = cfg["T"][0]
    attempts, mism, max_ds, differ = compare_trajectory(cfg, ctx, st, T, 10)
    print("%s: N=%d attempts=%d decision mismatches=%d max|dS|=%g differing sites=%d"
          % (name, lat.n, attempts, mism, max_ds, differ))
    assert attempts == 10 * lat.n
    _bar(attempts, mism, max_ds)
    if mism == 0:
        assert differ == 0
    _measure_close(ctx, st, lat.n)
    # the timed launch configuration (hb_sweep, no recording) continues the same trajectory
    ctx.sweep(T, 2)
    st.sweep(T, 2)
    if mism == 0:
        assert spins_equal(ctx.get_spins(), st.get_spins())
    if name == "c4":
        # the warp-specialised persistent kernel (TMA-staged neighbour planes) continues the same trajectory
        ctx.set_option("sc_kernel", 1)
        ctx.sweep(T, 1)
        st.sweep(T, 1)
        if mism == 0:
            assert spins_equal(ctx.get_spins(), st.get_spins())
        _measure_close(ctx, st, lat.n)
        # and so do its fused launches (sc_kernel = 2, NEXT-1): three sweeps = one launch of two sweeps (four colour passes
        # chained by progress words over 296 CTAs) + the measured sweep; then the traffic-minimal setting of
        # profiles/r02_c4_fused_full.md (4-plane chunks, lag 3, one sweep per launch)
        ctx.set_option("sc_kernel", 2)
        ctx.sweep(T, 3)
        st.sweep(T, 3)
        if mism == 0:
            assert spins_equal(ctx.get_spins(), st.get_spins())
        _measure_close(ctx, st, lat.n)
        for k, v in (("sc_fused_zt", 4), ("sc_fused_lag", 3), ("sc_fused_sweeps", 1)):
            ctx.set_option(k, v)
        ctx.sweep(T, 2)
        st.sweep(T, 2)
        if mism == 0:
            assert spins_equal(ctx.get_spins(), st.get_spins())
        _measure_close(ctx, st, lat.n)
    if name in ("c2", "c3"):
        # the warp-specialised bcc / fcc kernel (not the default at these sizes) continues the same trajectory, plain and fused
        for kern in (1, 2):
            ctx.set_option("br_kernel", kern)
            ctx.sweep(T, 3)
            st.sweep(T, 3)
            if mism == 0:
                assert spins_equal(ctx.get_spins(), st.get_spins())
            _measure_close(ctx, st, lat.n)


# ---- P3: long-run statistics against the fp64 random-site oracle (BASELINE.json north_star) ----------
# <|M|> and <E>/N of the CUDA path must lie within 3 standard errors of O64.  Standard errors come from
# R independent replicas on each side (replica means, Welch), not from one autocorrelated series
# (SURVEY.md 8(c) P3).  c1 runs at full size; the other kinds at the reduced shapes the oracle finishes
# in seconds, one temperature of their scan each.
P3_CASES = {
    "c1": (W.CONFIGS["c1"], 1.2, 500, 500),
    "bcc8": (W.SMALL["c2"], 1.6, 300, 500),
    "fcc6": (dict(W.SMALL["c3"], start="random"), 2.6, 300, 500),
    "sphere5": (W.SMALL["c5"], 1.5, 300, 500),
}


@pytest.mark.parametrize("name", sorted(P3_CASES))
def test_long_run_statistics_within_3_standard_errors_of_o64(name):
    cfg, T, equil, meas = P3_CASES[name]
    reps = 16
    lat, _ = make_oracle(cfg)
    g_m, g_e, o_m, o_e = [], [], [], []
    for r in range(reps):
        ctx = make_gpu(dict(cfg, seed=1000 + r))
        ctx.init_random()
        ctx.sweep(T, equil)
        M, E = ctx.sweep_series(T, meas)
        g_m.append(np.linalg.norm(M, axis=1).mean())
        g_e.append(E.mean() / lat.n)
        ctx.close()
        st = oracle.State64(lat, cfg["J"], 2000 + r)
        st.init_random()
        st.sweep(T, equil)
        m, e, _ = st.series(T, meas)
        o_m.append(m.mean())
        o_e.append(e.mean() / lat.n)
    for what, x, y in (("|M|", g_m, o_m), ("E/N", g_e, o_e)):
        x, y = np.array(x), np.array(y)
        se = math.sqrt(x.var(ddof=1) / reps + y.var(ddof=1) / reps)
        print("%s %s: gpu %.6f  o64 %.6f  diff %.2e  se %.2e" % (name, what, x.mean(), y.mean(), x.mean() - y.mean(), se))
        assert abs(x.mean() - y.mean()) < 3 * se, (name, what, x.mean(), y.mean(), se)


def test_fused_measurement_equals_the_separate_pass():
    # hb_sweep's last sweep also reduces M and E (SURVEY 8(a) note on fusing a5 into a4); hb_measure then
    # returns those.  Same P2 tolerances against the oracle, and against the separate pass on the same state.
    for cfg, opts in ((W.SMALL["c4"], {}), (W.SMALL["c1"], {}),
                      (dict(W.SMALL["c4"], L=(40, 12, 10), K=0.3, e=(0.6, 0.0, 0.8)), {"sc_jx": 3, "sc_ty": 5, "sc_zt": 3}),
                      (dict(W.SMALL["c4"], L=(64, 8, 6)), {"sc_linear": 96}),
                      (dict(W.SMALL["c4"], L=(40, 12, 10)), {"sc_jx": 5, "sc_ty": 60}), (dict(W.SMALL["c4"], L=(40, 12, 10)), {"sc_jx": 5, "sc_ty": 200}),
                      # bcc / fcc: every colour charges its bonds to the lower colours (already final in the sweep)
                      (dict(W.SMALL["c2"], start="random"), {}), (dict(W.SMALL["c2"], L=(12, 5, 7), start="random"), {"sc_jx": 2, "sc_ty": 3, "sc_zt": 2}),
                      (dict(W.SMALL["c3"], L=8, start="random"), {}), (dict(W.SMALL["c3"], L=(8, 3, 5), start="random"), {"sc_jx": 1, "sc_ty": 2})):
        lat, st = make_oracle(cfg)
        fused, plain = make_gpu(cfg), make_gpu(cfg)
        plain.set_option("fused_measure", 0)
        fused.set_option("sc_coop", 0)                                # this test is about the per-colour launches
        for k, v in opts.items():
            fused.set_option(k, v)
        start(cfg, fused, st)
        plain.init_random() if cfg["start"] == "random" else plain.init_aligned(cfg["e"])
        for T, k in ((1.44, 3), (0.4, 2)):
            fused.sweep(T, k)
            plain.sweep(T, k)
            st.sweep(T, k)
            l0, _ = fused.counters()
            Mf, Ef = fused.measure()
            l1, _ = fused.counters()
            assert l1 == l0                                           # no extra pass was launched
            Mp, Ep = plain.measure()
            Mo, Eo32, Eo64 = st.measure()
            assert np.max(np.abs(Mf - Mo)) <= 1e-7 and np.max(np.abs(Mf - Mp)) <= 1e-7
            assert abs(Ef - Eo32) <= 1e-6 * lat.n and abs(Ef - Eo64) <= 1e-6 * lat.n and abs(Ef - Ep) <= 1e-6 * lat.n
        assert spins_equal(fused.get_spins(), st.get_spins())
        # a state change invalidates the cached measurement
        S = W.random_unit_vectors(lat.n, 11)
        fused.set_spins(S[:, 0], S[:, 1], S[:, 2])
        st.set_spins(S[:, 0], S[:, 1], S[:, 2])
        _measure_close(fused, st, lat.n)


def test_persistent_kernels_match_the_oracle():
    # hb_sweep on a small sc lattice runs all its sweeps in ONE launch: a single block when a colour pass fits 1024
    # threads (the default for N <= 8192, barrier = __syncthreads), or, when forced, a cooperative grid with a
    # grid-wide barrier between colours.  The measurement of the last sweep (or of every sweep, for the series) is
    # reduced inside the launch.
    cases = [(W.SMALL["c1"], -1, 1), (dict(W.SMALL["c4"], L=(8, 6, 4), K=0.3, e=(0.6, 0.0, 0.8)), -1, 1),
             (dict(W.SMALL["c4"], L=(16, 16, 32)), -1, 1), (W.SMALL["c4"], 1, 1), (W.SMALL["c1"], 2, 1),
             (dict(W.SMALL["c4"], L=(40, 12, 10), K=0.3, e=(0.6, 0.0, 0.8)), 2, 1), (dict(W.SMALL["c4"], L=64), 1, 1),
             (W.SMALL["c4"], -1, 0)]
    for cfg, coop, active in cases:
        lat, st = make_oracle(cfg)
        ctx = make_gpu(cfg)
        ctx.set_option("sc_coop", coop)
        assert ctx.get_option("coop_active") == active, (cfg["L"], coop)
        if not active:
            continue
        start(cfg, ctx, st)
        for T, k in ((1.44, 1), (1.44, 6), (0.5, 3)):
            l0, _ = ctx.counters()
            ctx.sweep(T, k)
            l1, _ = ctx.counters()
            assert l1 - l0 == 1                                       # one launch, whatever k
            st.sweep(T, k)
            _measure_close(ctx, st, lat.n)                            # the fused measurement of the last sweep
        assert spins_equal(ctx.get_spins(), st.get_spins())
        Mg, Eg = ctx.sweep_series(1.2, 37)
        Mo, Eo = st.series(1.2, 37)
        assert spins_equal(ctx.get_spins(), st.get_spins())
        assert np.max(np.abs(Mg - Mo)) <= 1e-7 and np.max(np.abs(Eg - Eo)) <= 1e-6 * lat.n
        assert ctx.sweep_count == st.sweep_count
        ctx.close()


def test_warp_specialised_kernel_matches_the_oracle():
    # sc_kernel = 1: producer warp + bulk asynchronous copies into rings of plane slots, consumer warps read LDS,
    # persistent CTAs walking (y-tile, z-chunk) tiles.  Ragged tiles in y and z, a single row, the widest row (Lx = 512),
    # fewer CTAs than tiles (rings running across tile boundaries), both variants, fused measurement.
    cases = [(W.SMALL["c4"], {}), (W.SMALL["c1"], {}),
             (dict(W.SMALL["c4"], L=(40, 12, 10), K=0.3, e=(0.6, 0.0, 0.8)), {"sc_ws_zt": 3}),
             (dict(W.SMALL["c4"], L=(64, 20, 6)), {"sc_ws_zt": 4, "sc_ws_ctas": 2}),
             (dict(W.SMALL["c4"], L=(8, 2, 2)), {}), (dict(W.SMALL["c4"], L=(512, 10, 4)), {"sc_ws_zt": 2}),
             (W.SMALL["c4"], {"sc_ws_variant": 2}), (W.SMALL["c4"], {"sc_ws_variant": 1}), (dict(W.SMALL["c4"], L=(40, 14, 10)), {"sc_ws_variant": 1, "sc_ws_zt": 3}),
             (dict(W.SMALL["c4"], L=(40, 14, 10)), {"sc_ws_variant": 0, "sc_ws_zt": 10, "sc_ws_ctas": 1}),
             # 16-row tiles (one CTA of up to 31 consumer warps per SM): a ragged single tile, three tiles with a ragged
             # last one and balanced z-chunks (sc_ws_zt = 0), the widest row this variant takes (Lx = 496)
             (dict(W.SMALL["c4"], L=(40, 14, 10)), {"sc_ws_variant": 3, "sc_ws_zt": 3}),
             (dict(W.SMALL["c4"], L=(64, 36, 10)), {"sc_ws_variant": 3, "sc_ws_zt": 0, "sc_ws_ctas": 2}),
             (dict(W.SMALL["c4"], L=(496, 34, 6), K=0.3, e=(0.6, 0.0, 0.8)), {"sc_ws_variant": 3}),
             # 7-row tiles, two CTAs per SM (the default for config 4's rows of 232 floats): ragged tiles, full-width rows
             (dict(W.SMALL["c4"], L=(40, 14, 10)), {"sc_ws_variant": 4, "sc_ws_zt": 3}),
             (dict(W.SMALL["c4"], L=(464, 16, 6), K=0.3, e=(0.6, 0.0, 0.8)), {"sc_ws_variant": 4}),
             (dict(W.SMALL["c4"], L=(472, 30, 4)), {"sc_ws_variant": 4, "sc_ws_ctas": 3}),
             # 8-row tiles at a 512-byte row pitch, three CTAs per SM (rows of up to 128 floats): full-width and short rows
             (dict(W.SMALL["c4"], L=(256, 20, 6)), {"sc_ws_variant": 5}),
             (dict(W.SMALL["c4"], L=(40, 14, 10), K=0.3, e=(0.6, 0.0, 0.8)), {"sc_ws_variant": 5, "sc_ws_zt": 3, "sc_ws_ctas": 1})]
    for cfg, opts in cases:
        lat, st = make_oracle(cfg)
        ctx = make_gpu(cfg)
        ctx.set_option("sc_kernel", 1)
        for k, v in opts.items():
            ctx.set_option(k, v)
        start(cfg, ctx, st)
        for T, k in ((1.44, 1), (1.44, 4), (0.4, 2)):
            ctx.sweep(T, k)
            st.sweep(T, k)
            assert spins_equal(ctx.get_spins(), st.get_spins()), (cfg["L"], opts)
            _measure_close(ctx, st, lat.n)
        Mg, Eg = ctx.sweep_series(1.2, 9)
        Mo, Eo = st.series(1.2, 9)
        assert np.max(np.abs(Mg - Mo)) <= 1e-7 and np.max(np.abs(Eg - Eo)) <= 1e-6 * lat.n
        acc_o = st.sweep(1.0, 1, record=True)[0]                     # the recording path falls back to the direct kernel
        assert np.array_equal(ctx.sweep_record(1.0), acc_o)
        ctx.close()
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("sc", 6)).set_option("sc_kernel", 1)   # rows of 3 floats: not a multiple of 4
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("sc", 512, 4, 4)).set_option("sc_ws_variant", 3)   # 16 rows of 64 vectors: more than 1024 threads
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("sc", 480, 4, 4)).set_option("sc_ws_variant", 4)   # 7 rows of 60 vectors: more than 13 warps
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("sc", 264, 4, 4)).set_option("sc_ws_variant", 5)   # rows of 132 floats: longer than the 512-byte pitch


def test_replayed_launches_match_the_oracle():
    # lattices up to 2^23 sites replay a CUDA graph of 8 sweeps inside hb_sweep; the Philox sweep counter of a replayed
    # launch comes from a device counter.  Every engine, several call lengths, a temperature change (graph rebuilt),
    # an option change (graph rebuilt), a checkpointed counter beyond 2^32.
    n = 3000
    rp, ci = W.random_csr_graph(n, 6.0, seed=8)
    cases = [dict(W.SMALL["c4"]), dict(W.SMALL["c4"], L=(40, 12, 10), K=0.3, e=(0.6, 0.0, 0.8)), dict(W.SMALL["c2"], start="random"),
             dict(W.SMALL["c3"], start="random"), W.SMALL["c5"],
             dict(kind="csr", row_ptr=rp, col_idx=ci, J=1.0, K=0.2, e=(0, 0, 1), seed=3, start="random")]
    for cfg in cases:
        lat, st = make_oracle(cfg)
        ctx = make_gpu(cfg)
        ctx.set_option("sc_coop", 0)
        assert ctx.get_option("graph_active") == 1
        start(cfg, ctx, st)
        ctx.sweep_count = st.sweep_count = (1 << 32) - 5            # the counter crosses 2^32 inside a graph
        for T, k in ((1.44, 1), (1.44, 9), (1.44, 8), (0.7, 30), (0.7, 17)):
            l0, a0 = ctx.counters()
            ctx.sweep(T, k)
            l1, a1 = ctx.counters()
            assert a1 - a0 == k * lat.n
            st.sweep(T, k)
            assert spins_equal(ctx.get_spins(), st.get_spins()), (cfg.get("L"), T, k)
            _measure_close(ctx, st, lat.n)
        if cfg["kind"] in ("sc", "bcc", "fcc"):
            ctx.set_option("sc_zt", 1)                               # a launch-shape change invalidates the cached graph
        ctx.sweep(0.7, 20)
        st.sweep(0.7, 20)
        assert spins_equal(ctx.get_spins(), st.get_spins())
        assert ctx.sweep_count == st.sweep_count
        # measured sweeps are replayed too where the measurement is fused (sc, bcc, fcc): 4 graphs + 5 single sweeps
        Mg, Eg = ctx.sweep_series(1.2, 37)
        Mo, Eo = st.series(1.2, 37)
        assert spins_equal(ctx.get_spins(), st.get_spins())
        assert np.max(np.abs(Mg - Mo)) <= 1e-7 and np.max(np.abs(Eg - Eo)) <= 1e-6 * lat.n
        off = make_gpu(cfg)                                          # and with the graph off: same trajectory
        off.set_option("graph", 0)
        off.set_option("sc_coop", 0)
        off.set_spins(*ctx.get_spins())
        off.sweep_count = ctx.sweep_count
        off.sweep(1.0, 12)
        ctx.sweep(1.0, 12)
        assert spins_equal(ctx.get_spins(), off.get_spins())
        ctx.close()
        off.close()


def test_binder_crossing_brackets_the_critical_temperature_on_the_device():
    # Physics of the CUDA path at sizes the oracle does not reach in seconds (paper: T_C/J = 1.445
    # for the simple cubic lattice): the Binder cumulants U_L = 1 - <M^4> / (3 <M^2>^2) of L = 16
    # and L = 32 (K = 0) cross at T_C up to small finite-size corrections; below it the larger lattice is the more
    # ordered one, above it the less ordered one.
    Ts = np.linspace(1.36, 1.52, 9)
    U = {}
    for L in (16, 32):
        u = []
        for T in Ts:
            m2 = m4 = 0.0
            reps = 4
            for r in range(reps):
                ctx = hb.Context(hb.Lattice("sc", L), 1.0, 0.0, (0.0, 0.0, 1.0), seed=500 + r)
                ctx.init_aligned((0.0, 0.0, 1.0))
                ctx.sweep(float(T), 1500)
                M, _ = ctx.sweep_series(float(T), 6000)
                q = np.sum(M * M, axis=1)
                m2 += q.mean() / reps
                m4 += (q * q).mean() / reps
                ctx.close()
            u.append(1.0 - m4 / (3.0 * m2 * m2))
        U[L] = np.array(u)
    d = U[32] - U[16]
    print("T:", Ts, "U16:", U[16], "U32:", U[32])
    assert d[0] > 0 and d[1] > 0 and d[-1] < 0 and d[-2] < 0          # ordered side / disordered side
    k = int(np.argmax(d < 0))                                         # first temperature above the crossing
    Tx = Ts[k - 1] + (Ts[k] - Ts[k - 1]) * d[k - 1] / (d[k - 1] - d[k])
    print("Binder crossing of L = 16, 32 at T = %.4f" % Tx)
    assert abs(Tx - 1.443) < 0.03


@pytest.mark.parametrize("name", ["c2", "c3", "c5"])
def test_full_protocol_scans(name):
    # configs 2, 3, 5 exactly as BASELINE.json states them (full size, every temperature, every sweep), on the device:
    # M(T) falls monotonically with T, is large on the cold side and small on the hot side, and the energy rises
    # with T (full-size scans are sanity-checked for a monotone M(T) and the K8/K9 limits).
    from paper_2106_11286_b200 import scan
    cfg = W.CONFIGS[name]
    ctx = scan.make_context(cfg)
    res = scan.run_scan(ctx, cfg["T"], cfg["sweeps"], cfg.get("equil", 0))
    order = np.argsort(res["T"])
    T, m, e = res["T"][order], res["absM"][order], res["E"][order]
    print(name, "T", T, "|M|", m, "E/N", e)
    assert np.all(np.diff(m) < 0.01)                                  # monotone up to noise on the disordered side
    assert np.all(np.diff(e) > 0)
    cold, hot = {"c2": (0.85, 0.03), "c3": (0.65, 0.03), "c5": (0.30, 0.15)}[name]   # c5 starts random BELOW T_c (2.5 < 3.18): it coarsens, domains freeze in
    assert m[0] > cold and m[-1] < hot
    launches, attempts = ctx.counters()
    per_T = cfg["sweeps"] + cfg.get("equil", 0)
    assert attempts == ctx.n * per_T * len(cfg["T"])
    ctx.close()


def test_kernel_variants_agree_on_random_shapes():
    # 30 seeded random simple cubic shapes (ragged tiles, single rows, wide rows): the direct kernel with a random tile,
    # the warp-specialised kernel with random tile depth / CTA count / variant, replayed launches and the persistent
    # kernels must all leave the same bits behind.  (The oracle pins the first of them in the tests above.)
    rng = np.random.default_rng(20240611)
    for it in range(30):
        Lx = int(rng.choice([8, 16, 24, 40, 64, 120, 232, 512]))
        Ly, Lz = int(2 * rng.integers(1, 12)), int(2 * rng.integers(1, 9))
        K, e = (0.0, (0, 0, 1)) if it % 3 == 0 else ((0.05, (0, 0, 1)) if it % 3 == 1 else (0.2, (0.6, 0.0, 0.8)))
        seed = int(rng.integers(1, 1 << 40))

        def run(opts):
            ctx = hb.Context(hb.Lattice("sc", Lx, Ly, Lz), 1.0, K, e, seed=seed)
            for k, v in opts.items():
                ctx.set_option(k, v)
            ctx.init_random()
            ctx.sweep(1.3, 11)
            out = ctx.get_spins(), ctx.measure()
            ctx.close()
            return out

        H = Lx // 2
        ref, (Mr, Er) = run({"graph": 0, "sc_coop": 0})
        variants = [{"graph": 0, "sc_coop": 0, "sc_jx": int(rng.integers(1, H // 4 + 1)), "sc_ty": int(rng.integers(1, 9)),
                     "sc_zt": int(rng.integers(1, Lz + 1)), "pdl": it % 2},
                    {"graph": 1, "sc_coop": 0, "pdl": (it + 1) % 2},
                    {"graph": 0, "sc_coop": 2},
                    {"graph": int(rng.integers(0, 2)), "sc_kernel": 1, "sc_ws_zt": int(rng.integers(0, Lz + 1)),
                     "sc_ws_ctas": int(rng.integers(1, 5)),
                     "sc_ws_variant": int(rng.choice([0, 1, 2] + ([3] if H <= 248 else []) + ([4] if H <= 236 else []) + ([5] if H <= 128 else [])))}]
        # fused launches (sc_kernel = 2): random chunk size, lag, sweeps per launch and CTA count; the variant first, then the kernel
        fv = int(rng.choice([2] + ([4] if H <= 236 else []) + ([5] if H <= 128 else [])))
        variants.append({"graph": 0, "sc_coop": 0, "sc_ws_variant": fv, "sc_kernel": 2, "sc_fused_zt": int(rng.integers(1, Lz + 1)),
                         "sc_fused_lag": int(rng.integers(3, 9)), "sc_fused_sweeps": int(rng.integers(1, 17)), "sc_ws_ctas": int(rng.integers(1, 5))})
        for opts in variants:
            got, (Mg, Eg) = run(opts)
            assert spins_equal(got, ref), (Lx, Ly, Lz, opts)
            assert np.max(np.abs(Mg - Mr)) <= 1e-7 and abs(Eg - Er) <= 1e-6 * Lx * Ly * Lz, (Lx, Ly, Lz, opts)


def test_replicas_match_independent_oracle_runs():
    # hb_lattice.n_replicas = R: replica r is the system with seed + r; one launch sweeps all of them, each in its own
    # thread block at its own temperature.  Every replica must walk the trajectory the oracle walks
    # for (seed + r, T_r), and its measurements and series must be the oracle's.
    for cfg, R in ((W.SMALL["c1"], 5), (dict(W.SMALL["c4"], L=(8, 6, 4), K=0.3, e=(0.6, 0.0, 0.8)), 37),
                   (dict(W.SMALL["c4"], L=(16, 16, 32)), 3)):
        L = cfg["L"]
        Lx, Ly, Lz = (L, L, L) if isinstance(L, int) else L
        ctx = hb.Context(hb.Lattice("sc", Lx, Ly, Lz, n_replicas=R), cfg["J"], cfg["K"], cfg["e"], cfg["seed"])
        Ts = np.linspace(0.6, 2.4, R).astype(np.float32)
        states = []
        for r in range(R):
            lat, st = make_oracle(dict(cfg, seed=cfg["seed"] + r))
            st.init_random()
            states.append(st)
        ctx.init_random()
        l0, _ = ctx.counters()
        ctx.sweep_each(Ts, 7)
        l1, a1 = ctx.counters()
        assert l1 - l0 == 1 and a1 == 7 * lat.n * R                   # one launch for all replicas
        for r, st in enumerate(states):
            st.sweep(float(Ts[r]), 7)
        M, E = ctx.measure_each()                                     # reduced inside that launch
        for r, st in enumerate(states):
            Mo, Eo32, Eo64 = st.measure()
            assert np.max(np.abs(M[r] - Mo)) <= 1e-7 and abs(E[r] - Eo32) <= 1e-6 * lat.n
            ctx.select_replica(r)
            assert spins_equal(ctx.get_spins(), st.get_spins()), (cfg["L"], r)
            Ms, Es = ctx.measure()
            assert np.max(np.abs(Ms - Mo)) <= 1e-7 and abs(Es - Eo32) <= 1e-6 * lat.n
        Mser, Eser = ctx.sweep_series_each(Ts, 9)
        ctx.sweep(1.1, 2)                                             # one temperature for all
        for r, st in enumerate(states):
            Mo, Eo = st.series(float(Ts[r]), 9)
            assert np.max(np.abs(Mser[r] - Mo)) <= 1e-7 and np.max(np.abs(Eser[r] - Eo)) <= 1e-6 * lat.n
            st.sweep(1.1, 2)
            ctx.select_replica(r)
            assert spins_equal(ctx.get_spins(), st.get_spins())
        # a replica's state can be replaced; measuring then takes the separate pass
        S = W.random_unit_vectors(lat.n, 5)
        ctx.select_replica(1)
        ctx.set_spins(S[:, 0], S[:, 1], S[:, 2])
        states[1].set_spins(S[:, 0], S[:, 1], S[:, 2])
        M, E = ctx.measure_each()
        for r in (0, 1, R - 1):
            Mo, Eo32, _ = states[r].measure()
            assert np.max(np.abs(M[r] - Mo)) <= 1e-7 and abs(E[r] - Eo32) <= 1e-6 * lat.n
        with pytest.raises(hb.HbError):
            ctx.sweep_record(1.0)
        ctx.close()
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("sc", 32, n_replicas=2))                # 32768 sites: a colour pass does not fit one block
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("bcc", 4, n_replicas=2))


def test_alu_probe_reports_a_plausible_ceiling():
    # hb_probe_alu: the attempt arithmetic alone; any colour kernel must stay below it, and it cannot exceed the issue
    # bound of 20 IMAD.WIDE per attempt (one per 4 clocks per SM sub-partition: 592 x 32 lanes x 1.965 GHz / 80)
    rate = hb.probe_alu(0.2)
    assert 2e10 < rate < 592 * 32 * 1.965e9 / 80
    with pytest.raises(hb.HbError):
        hb.probe_alu(0.0)


def test_programmatic_launches_match_the_oracle():
    # option pdl = 1: colour kernels launched with programmatic stream serialisation (their blocks become resident while the
    # previous colour drains and wait in griddepcontrol.wait before they read anything).  Every engine, with plain
    # launches and with replayed graphs, many short launches back to back: the trajectory must be the oracle's.
    for name in ("c1", "c2", "c3", "c5"):
        cfg = W.SMALL[name]
        for graph in (0, 1):
            lat, st = make_oracle(cfg)
            ctx = make_gpu(cfg)
            ctx.set_option("pdl", 1)
            ctx.set_option("graph", graph)
            if cfg["kind"] == "sc":
                ctx.set_option("sc_coop", 0)
            assert ctx.get_option("pdl") == 1
            start(cfg, ctx, st)
            for T, k in ((1.5, 20), (0.7, 13)):
                ctx.sweep(T, k)
                st.sweep(T, k)
                assert spins_equal(ctx.get_spins(), st.get_spins()), (name, graph)
                _measure_close(ctx, st, lat.n)
            ctx.close()


@pytest.mark.parametrize("name", ["sc16_c1", "sc24_K", "sc_wide", "sc_v2_ragged", "bcc8", "fcc6", "sphere5", "sc_persite"])
def test_stats_count_the_accepted_moves_like_the_oracle(name):
    # hb_stats (rule (iii) [P:20] defines an accepted move): the device counts, inside the measuring passes,
    # exactly the moves the oracle accepts
    cfg = SMALL_CASES[name]
    ctx = make_gpu(cfg)
    lat, st = make_oracle(cfg)
    start(cfg, ctx, st)
    n = lat.n
    assert ctx.stats() == (0, 0)
    for T in (cfg["T"][0], 0.4):
        for _ in range(3):                      # one-sweep calls: every sweep is the last of its call, so every sweep counts
            ctx.sweep(T, 1)
            st.sweep(T, 1)
    assert ctx.stats() == st.stats() == (6 * n, st.stats()[1])
    ctx.sweep_series(1.1, 5)                    # every sweep of a series counts
    st.sweep(1.1, 5)
    assert ctx.stats() == st.stats()
    before = ctx.stats()
    ctx.sweep(0.9, 19)                          # a longer call counts its last sweep only (graph replay + a measured tail)
    acc = st.sweep(0.9, 19, record=True)
    after = ctx.stats()
    assert after[0] - before[0] == n and after[1] - before[1] == int(acc[-1].sum())
    got = ctx.sweep_record(0.9)                 # a recorded sweep counts what it records
    assert ctx.stats()[1] - after[1] == int(got.sum()) and ctx.stats()[0] - after[0] == n
    assert spins_equal(ctx.get_spins(), (st.sweep(0.9, 1), st.get_spins())[1])
    ctx.close()


def test_stats_on_the_warp_specialised_kernel_and_on_replicas():
    cfg = dict(W.SMALL["c4"], L=(64, 12, 10))
    ctx = make_gpu(cfg)
    ctx.set_option("sc_coop", 0)
    ctx.set_option("sc_kernel", 1)
    lat, st = make_oracle(cfg)
    start(cfg, ctx, st)
    for _ in range(4):
        ctx.sweep(1.44, 1)
        st.sweep(1.44, 1)
    assert ctx.stats() == st.stats()
    ctx.close()
    # replicas: the counter sums over all of them
    R, T = 5, [0.8, 1.2, 1.44, 2.0, 3.0]
    lat_g = hb.Lattice("sc", 8, 8, 8, n_replicas=R)
    ctx = hb.Context(lat_g, 1.0, 0.01, (0, 0, 1), seed=7)
    ctx.init_random()
    want_att = want_acc = 0
    olat = oracle.Lattice.sc(8)
    olat.set_uniform_anisotropy(0.01, (0, 0, 1))
    sts = [oracle.State32(olat, 1.0, 7 + r) for r in range(R)]
    for s in sts:
        s.init_random()
    for _ in range(3):
        ctx.sweep_each(T, 1)
        for r, s in enumerate(sts):
            s.sweep(T[r], 1)
    for s in sts:
        a, b = s.stats()
        want_att += a
        want_acc += b
    assert ctx.stats() == (want_att, want_acc)
    ctx.close()


def test_fused_launches_match_the_oracle():
    # sc_kernel = 2 (DESIGN 6.9): all colour passes of several sweeps in ONE launch, tiles ordered in rounds with
    # dependencies between the passes instead of a launch boundary per colour.  Same trajectory, bit for bit, for every
    # chunk size / lag / sweeps per launch, ragged tiles in y and z, fewer chunks than the dependency window, general anisotropy,
    # the fused measurement, the series, hb_stats and a sweep counter that crosses 2^32 inside a launch.
    cases = [(dict(W.SMALL["c4"], L=(64, 30, 22)), [dict(sc_ws_variant=2), dict(sc_ws_variant=4, sc_fused_zt=3, sc_fused_lag=3, sc_fused_sweeps=3),
                                                     dict(sc_ws_variant=5, sc_fused_zt=1, sc_fused_lag=5, sc_fused_sweeps=16),
                                                     dict(sc_ws_variant=4, sc_fused_zt=22, sc_fused_sweeps=2),          # one chunk
                                                     dict(sc_ws_variant=2, sc_fused_zt=11, sc_fused_lag=7, sc_fused_sweeps=5)]),   # two chunks
             (dict(W.SMALL["c4"], L=(464, 16, 12), K=0.3, e=(0.6, 0.0, 0.8)), [dict(sc_ws_variant=4, sc_fused_zt=2, sc_fused_sweeps=4),
                                                                             dict(sc_ws_variant=2, sc_fused_zt=5, sc_fused_lag=3)]),
             (dict(W.SMALL["c4"], L=(240, 44, 40), K=0.0), [dict(sc_ws_variant=5, sc_fused_zt=4, sc_fused_sweeps=6, sc_ws_ctas=3),   # few CTAs: deep queues
                                                            dict(sc_ws_variant=4, sc_fused_zt=8, sc_fused_sweeps=2)])]
    for cfg, variants in cases:
        lat, st0 = make_oracle(cfg)
        for opts in variants:
            lat, st = make_oracle(cfg)
            ctx = make_gpu(cfg)
            ctx.set_option("sc_coop", 0)
            ctx.set_option("graph", 0)
            for k, v in opts.items():
                if k == "sc_ws_variant":
                    ctx.set_option(k, v)
            ctx.set_option("sc_kernel", 2)
            for k, v in opts.items():
                ctx.set_option(k, v)
            assert ctx.get_option("sc_kernel") == 2
            start(cfg, ctx, st)
            ctx.sweep_count = st.sweep_count = (1 << 32) - 3
            for T, k in ((1.44, 1), (1.44, 2), (1.44, 11), (0.4, 7)):
                l0, a0 = ctx.counters()
                ctx.sweep(T, k)
                l1, a1 = ctx.counters()
                assert a1 - a0 == k * lat.n
                S = opts.get("sc_fused_sweeps", 8)
                assert l1 - l0 == -(-(k - 1) // S) + 2                  # ceil((k-1)/S) launches + the measured sweep + its reduction
                st.sweep(T, k)
                assert spins_equal(ctx.get_spins(), st.get_spins()), (cfg["L"], opts, T, k)
                _measure_close(ctx, st, lat.n)
            Mg, Eg = ctx.sweep_series(1.2, 5)
            Mo, Eo = st.series(1.2, 5)
            assert np.max(np.abs(Mg - Mo)) <= 1e-7 and np.max(np.abs(Eg - Eo)) <= 1e-6 * lat.n
            assert ctx.sweep_count == st.sweep_count
            ctx.close()
        # hb_stats through the fused measuring launch
        lat, st = make_oracle(cfg)
        ctx = make_gpu(cfg)
        ctx.set_option("sc_coop", 0)
        ctx.set_option("graph", 0)
        ctx.set_option("sc_ws_variant", 2)
        ctx.set_option("sc_kernel", 2)
        start(cfg, ctx, st)
        for _ in range(3):
            ctx.sweep(1.0, 1)
            st.sweep(1.0, 1)
        assert ctx.stats() == st.stats()
        ctx.close()
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("sc", 6)).set_option("sc_kernel", 2)


def test_l2_fold_probe_reports_a_rate_and_invalidates_the_state():
    # hb_probe_sc_l2: the sc colour kernel with plane addresses folded onto 16 L2-resident planes (DESIGN 6.9): a rate, not a
    # trajectory; the spins are undefined afterwards
    ctx = hb.Context(hb.Lattice("sc", 232, 64, 64), 1.0, 0.01, (0, 0, 1), seed=1)
    ctx.init_random()
    rate = ctx.probe_sc_l2(1.44, 10, 16)
    assert 1e9 < rate < 400e9
    with pytest.raises(hb.HbError):
        ctx.sweep(1.44, 1)                      # HB_ESTATE until the spins are initialised again
    ctx.init_random()
    ctx.sweep(1.44, 1)
    with pytest.raises(hb.HbError):
        ctx.probe_sc_l2(1.44, 10, 12)           # planes must be a power of two
    ctx.close()


def test_bravais_warp_specialised_kernel_matches_the_oracle():
    # br_kernel = 1 / 2 (DESIGN 6.10): bcc and fcc colour passes with TMA-staged neighbour groups; 2 = all colour passes of
    # several sweeps in one launch.  Every launch shape (rows of up to 64 / 128 / 256 cells), ragged tiles in y and z, every
    # anisotropy case, the fused measurement, series, stats, a sweep counter crossing 2^32.
    cases = [dict(W.SMALL["c2"]), dict(W.SMALL["c2"], L=(12, 5, 7), K=0.0), dict(W.SMALL["c2"], L=(68, 11, 6), K=0.3, e=(0.6, 0.0, 0.8)),
             dict(W.SMALL["c2"], L=(132, 6, 5)), dict(W.SMALL["c3"], L=(8, 6, 6), start="random"),
             dict(W.SMALL["c3"], L=(4, 3, 5), start="random", K=0.0), dict(W.SMALL["c3"], L=(72, 9, 4), start="random", K=0.2, e=(0.0, 0.0, 1.0)),
             dict(W.SMALL["c3"], L=(132, 5, 3), start="random"), dict(W.SMALL["c3"], L=(64, 16, 24), start="aligned")]
    for cfg in cases:
        for opts in (dict(br_kernel=1), dict(br_kernel=2), dict(br_kernel=2, br_zt=1, sc_fused_lag=3, sc_fused_sweeps=3),
                     dict(br_kernel=2, br_zt=2, sc_fused_lag=5, sc_fused_sweeps=16, sc_ws_ctas=2), dict(br_kernel=1, br_zt=3, graph=0)):
            lat, st = make_oracle(cfg)
            ctx = make_gpu(cfg)
            for k, v in opts.items():
                ctx.set_option(k, v)
            start(cfg, ctx, st)
            ctx.sweep_count = st.sweep_count = (1 << 32) - 4
            for T, k in ((cfg["T"][0], 1), (cfg["T"][0], 2), (1.5, 13), (0.4, 6)):
                ctx.sweep(T, k)
                st.sweep(T, k)
                assert spins_equal(ctx.get_spins(), st.get_spins()), (cfg["kind"], cfg["L"], opts, T, k)
                _measure_close(ctx, st, lat.n)
            Mg, Eg = ctx.sweep_series(1.2, 5)
            Mo, Eo = st.series(1.2, 5)
            assert np.max(np.abs(Mg - Mo)) <= 1e-7 and np.max(np.abs(Eg - Eo)) <= 1e-6 * lat.n
            acc_o = st.sweep(1.0, 1, record=True)[0]                 # the recording path stays on the direct kernel
            assert np.array_equal(ctx.sweep_record(1.0), acc_o)
            assert ctx.sweep_count == st.sweep_count
            ctx.close()
        lat, st = make_oracle(cfg)
        ctx = make_gpu(cfg)
        ctx.set_option("br_kernel", 2)
        start(cfg, ctx, st)
        for _ in range(3):
            ctx.sweep(1.0, 1)
            st.sweep(1.0, 1)
        assert ctx.stats() == st.stats()
        ctx.close()
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("bcc", 6)).set_option("br_kernel", 1)      # rows of 6 cells: not a multiple of 4


def test_large_bcc_runs_the_warp_specialised_kernel_by_default():
    # lattices of 2^24 sites and more: bcc defaults to br_kernel = 1 (DESIGN 6.10); first sweeps against the oracle, bit for bit
    cfg = dict(W.SMALL["c2"], L=(256, 128, 256))
    ctx = make_gpu(cfg)
    assert ctx.get_option("br_kernel") == 1 and ctx.get_option("graph_active") == 0
    lat, st = make_oracle(cfg)
    start(cfg, ctx, st)
    ctx.sweep(1.8, 2)
    st.sweep(1.8, 2)
    assert spins_equal(ctx.get_spins(), st.get_spins())
    _measure_close(ctx, st, lat.n)
    ctx.close()


def test_fig3_protocol_shortened():
    # The paper's accuracy experiment [P:52-58, Fig. 3] shortened (2000 + 2000 sweeps per temperature instead of 10^4 + 10^4;
    # the full scans and their fits: profiles/fig3/): sc 128^3 and 256^3, aligned start, heating.  K = 0: the fitted critical
    # temperature is the literature value 1.443 (the paper prints 1.445).  K = 0.01 (the paper's): the two sizes give the same
    # <|M|>(T) to 1e-3 below the transition ("numerical stability ... up to 10^8 spins" [P:54]).
    from paper_2106_11286_b200 import scan
    def curve(L, K, Ts, sweeps=2000):
        ctx = scan.make_context(dict(kind="sc", L=L, J=1.0, K=K, e=(0.0, 0.0, 1.0), seed=1, start="aligned"))
        res = scan.run_scan(ctx, Ts, sweeps, sweeps)
        ctx.close()
        return res
    Ts = [float(t) for t in np.arange(1.30, 1.4351, 0.0075)]
    r128 = curve(128, 0.0, Ts)
    Tc, beta = scan.fit_order_parameter(r128["T"], r128["absM"], 0.01, 0.1)[:2]
    assert abs(Tc - 1.443) <= 0.005, (Tc, beta)
    assert 0.32 <= beta <= 0.38, (Tc, beta)
    assert np.all(np.diff(r128["absM"]) < 0)                      # M(T) falls monotonically towards T_C
    Tk = [1.30, 1.32, 1.34, 1.36, 1.38, 1.40]
    a, b = curve(128, 0.01, Tk, 5000), curve(256, 0.01, Tk, 5000)
    assert np.max(np.abs(a["absM"] - b["absM"])) <= 1e-3, (a["absM"], b["absM"])
    assert np.max(np.abs(a["E"] - b["E"])) <= 1e-3


@pytest.mark.parametrize("name", ["c2", "c3", "c5"])
def test_scan_statistics_over_the_full_temperature_lists(name):
    # SURVEY 8(c) P3 at the reduced shapes over the FULL temperature lists of configs 2, 3 and 5, with their protocol (DESIGN
    # A13: one state carried through the scan, cooling from a random start, heating from an aligned one): 16 replicas on each
    # side, replica means per temperature, Welch.  With 2 observables x 10-20 temperatures the bar is the 3 standard errors of
    # BASELINE.json for all but at most two of the comparisons, and 4.2 for every one of them (P < 1e-3 for the whole table).
    cfg = W.SMALL[name]
    Ts = W.CONFIGS[name]["T"]
    equil, meas, reps = 150, 250, 16
    lat, _ = make_oracle(cfg)
    g = np.zeros((reps, len(Ts), 2))
    o = np.zeros((reps, len(Ts), 2))
    for r in range(reps):
        ctx = make_gpu(dict(cfg, seed=3000 + r))
        st = oracle.State64(lat, cfg["J"], 4000 + r)
        if cfg["start"] == "random":
            ctx.init_random()
            st.init_random()
        else:
            ctx.init_aligned(cfg["e"])
            st.init_aligned(cfg["e"])
        for k, T in enumerate(Ts):
            ctx.sweep(T, equil)
            M, E = ctx.sweep_series(T, meas)
            g[r, k] = np.linalg.norm(M, axis=1).mean(), E.mean() / lat.n
            st.sweep(T, equil)
            m, e, _ = st.series(T, meas)
            o[r, k] = m.mean(), e.mean() / lat.n
        ctx.close()
    se = np.sqrt(g.var(axis=0, ddof=1) / reps + o.var(axis=0, ddof=1) / reps)
    z = (g.mean(axis=0) - o.mean(axis=0)) / se
    for k, T in enumerate(Ts):
        print("%s T %.3f  |M| gpu %.5f o64 %.5f z %+.2f   E/N gpu %.5f o64 %.5f z %+.2f" %
              (name, T, g[:, k, 0].mean(), o[:, k, 0].mean(), z[k, 0], g[:, k, 1].mean(), o[:, k, 1].mean(), z[k, 1]))
    assert np.max(np.abs(z)) < 4.2, z
    assert int(np.sum(np.abs(z) > 3.0)) <= 2, z
    m = g[:, :, 0].mean(axis=0)                                # the transition lies inside the window: ordered at one end, not at the other
    assert max(m[0], m[-1]) > 1.5 * min(m[0], m[-1])


def test_paper_scheme_emulation_statistics():
    # the paper's own block scheme [P:30-32] (N / n blocks of n spins, one random spin per block and step, racy),
    # emulated by hb_sweep_paper_scheme.  It has no trajectory to compare; its statistics are compared with the fp64 random-site
    # oracle (the same steps (i)-(iii) of [P:20], sequentially).  With the paper's n = 8 the two agree to a few 1e-3 on a 16^3
    # lattice below T_C; n = 1 (every spin updated at once against its neighbours' old values) is the limit in which the
    # "loss of continuity" [P:32] is complete.  Counters: N attempts per MCS, all of them counted by hb_stats.
    cfg = W.CONFIGS["c1"]
    lat, _ = make_oracle(cfg)
    T, equil, meas, reps = 1.2, 300, 400, 12
    def gpu(n_per_block):
        m_all, e_all = [], []
        for r in range(reps):
            ctx = make_gpu(dict(cfg, seed=500 + r))
            ctx.init_random()
            ctx.sweep_paper_scheme(T, equil, n_per_block)
            ms, es = [], []
            for _ in range(meas):
                ctx.sweep_paper_scheme(T, 1, n_per_block)
                M, E = ctx.measure()
                ms.append(np.linalg.norm(M)); es.append(E / lat.n)
            m_all.append(np.mean(ms)); e_all.append(np.mean(es))
            if r == 0:
                att, acc = ctx.stats()
                assert att == (equil + meas) * lat.n and 0 < acc < att
                assert ctx.sweep_count == equil + meas
            ctx.close()
        return np.array(m_all), np.array(e_all)
    o_m, o_e = [], []
    for r in range(reps):
        st = oracle.State64(lat, cfg["J"], 700 + r)
        st.init_random()
        st.sweep(T, equil)
        m, e, _ = st.series(T, meas)
        o_m.append(m.mean()); o_e.append(e.mean() / lat.n)
    o_m, o_e = np.array(o_m), np.array(o_e)
    for n_per_block in (8, 64, 1):
        g_m, g_e = gpu(n_per_block)
        dm, de = g_m.mean() - o_m.mean(), g_e.mean() - o_e.mean()
        se_m = math.sqrt(g_m.var(ddof=1) / reps + o_m.var(ddof=1) / reps)
        se_e = math.sqrt(g_e.var(ddof=1) / reps + o_e.var(ddof=1) / reps)
        print("paper scheme n = %d: |M| %.5f (o64 %.5f, diff %+.1e, se %.1e)  E/N %.5f (o64 %.5f, diff %+.1e, se %.1e)" %
              (n_per_block, g_m.mean(), o_m.mean(), dm, se_m, g_e.mean(), o_e.mean(), de, se_e))
        if n_per_block >= 8:
            # The emulation is racy by the paper's own account [P:32], so its bias is a property of the scheme, not a parity
            # figure; the bound is the bias measured on B200s (n = 8: +6.4e-3 in E/N, +2e-3 in |M|; n = 64: +3e-3 +- 3e-3, taken as 1e-3;
            # DESIGN.md 4b) plus 4 standard errors of THIS run's two replica sets (se ~ 2.5e-3 each): ~0.016, where the
            # n = 1 limit sits at +0.17.  A materially worse emulation (a scheme that lets more neighbours move at once)
            # lands between the two and fails.
            bias_e, bias_m = (6e-3, 2e-3) if n_per_block == 8 else (1e-3, 1e-3)
            assert abs(de) <= bias_e + 4.0 * se_e and abs(dm) <= bias_m + 4.0 * se_m, (n_per_block, dm, se_m, de, se_e)
        else:                     # n = 1: every spin moves against stale neighbours: the bias is an order of magnitude larger
            assert de > 0.05, (n_per_block, de)
    with pytest.raises(hb.HbError):
        hb.Context(hb.Lattice("sc", 6)).sweep_paper_scheme(1.0, 1, 8)     # before init; and 216 sites are not a multiple of 8


@pytest.mark.parametrize("name", ["sc24_K", "sc16_c1", "bcc8", "sphere5"])
def test_staged_upload_equals_set_spins(name):
    # hb_stage_spins / hb_commit_spins: the upload in two halves (the copy overlaps earlier sweeps); the committed state is the
    # one hb_set_spins would have set, in stream order with the sweeps around it
    import torch
    cfg = SMALL_CASES[name]
    ctx = make_gpu(cfg)
    lat, st = make_oracle(cfg)
    start(cfg, ctx, st)
    st.sweep(1.3, 2)
    target = st.get_spins()
    host = [torch.from_numpy(a.copy()).pin_memory() for a in target]
    with pytest.raises(hb.HbError):
        ctx.commit_spins()                         # nothing staged
    ctx.sweep(1.3, 5)                              # work in flight while the copy runs
    ctx.stage_spins(*host)
    with pytest.raises(hb.HbError) as second:      # one staged state at a time: the area and the first host arrays are still in use
        ctx.stage_spins(*host)
    assert second.value.status == -4               # HB_ESTATE
    ctx.sweep(1.3, 3)
    ctx.commit_spins()
    assert spins_equal(ctx.get_spins(), target)
    ctx.sweep_count = st.sweep_count
    for k in (1, 4):                               # and twice in a row: the second upload waits for the first commit's reads
        ctx.sweep(1.3, k)
        st.sweep(1.3, k)
        assert spins_equal(ctx.get_spins(), st.get_spins())
        _measure_close(ctx, st, lat.n)
        host2 = [torch.from_numpy(a.copy()).pin_memory() for a in st.get_spins()]
        ctx.stage_spins(*host2)
        ctx.commit_spins()
        assert spins_equal(ctx.get_spins(), st.get_spins())
    ctx.close()


def test_long_fcc_lattice_runs_on_its_default_kernel_choice():
    # hb_create picks the all-passes launch (br_kernel 2, 8 sweeps per launch) for fcc with Lx > 128 and
    # >= 2^24 sites without checking its progress-word bound; a long thin lattice (31 * ceil(Lz / 16) > 16384 words) then
    # failed in hb_sweep with HB_ECUDA.  The choice is clamped at create time now (one sweep per launch): the default
    # context sweeps, and walks the trajectory of the direct kernel bit for bit.
    cfg = dict(W.SMALL["c3"], L=(132, 4, 8452), start="random")
    a, b = make_gpu(cfg), make_gpu(cfg)
    assert a.get_option("br_kernel") == 2 and a.get_option("sc_fused_sweeps") == 1
    b.set_option("br_kernel", 0)
    for c in (a, b):
        c.init_random()
        c.sweep(1.1, 3)
    assert spins_equal(a.get_spins(), b.get_spins())
    Ma, Ea = a.measure()
    Mb, Eb = b.measure()
    assert np.max(np.abs(Ma - Mb)) <= 1e-7 and abs(Ea - Eb) <= 1e-6 * a.n
    a.close()
    b.close()


def test_many_ctas_of_the_bcc_fcc_ws_kernel_do_not_overrun_the_block_partials():
    # with sc_ws_ctas = 4096 a colour launch of the warp-specialised fcc kernel can have 12288 blocks; four
    # colours of block partials side by side would overrun the buffer (32768 blocks) into the series / counter area.  Such
    # grids now measure in the separate pass: M, E and the acceptance counters stay those of the default grid.
    cfg = dict(W.SMALL["c3"], L=(64, 256, 260), start="random")    # 32 row groups x 260 one-plane chunks = 8320 blocks per colour
    a, b = make_gpu(cfg), make_gpu(cfg)
    for c, ctas in ((a, 4096), (b, 0)):
        c.set_option("br_kernel", 1)
        c.set_option("br_zt", 1)
        if ctas:
            c.set_option("sc_ws_ctas", ctas)
        c.init_random()
        c.sweep(1.1, 3)
    Ma, Ea = a.measure()
    Mb, Eb = b.measure()
    assert spins_equal(a.get_spins(), b.get_spins())
    assert np.max(np.abs(Ma - Mb)) <= 1e-7 and abs(Ea - Eb) <= 1e-6 * a.n
    assert a.stats() == b.stats()
    a.close()
    b.close()
