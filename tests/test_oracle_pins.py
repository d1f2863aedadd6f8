"""Pins of the CPU oracle's building blocks against what the paper and the
mathematics fix.  CPU only."""
import math
import os

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


# ---- K1: Philox4x32-10 known answers ------------------------------------------
def test_philox_known_answers():
    for r in _rows("philox4x32_10_kat.txt"):
        w = [int(x, 16) for x in r]
        out = oracle.philox4x32_10(w[0:4], w[4:6])
        assert [int(x) for x in out] == w[6:10]


def _philox_bigint(ctr, key):
    # second, independent statement with Python integers (128-bit view of the rounds)
    c, k = list(ctr), list(key)
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return c


def test_philox_random_counters_and_site_keying():
    rng = np.random.default_rng(7)
    for _ in range(200):
        ctr = [int(x) for x in rng.integers(0, 2**32, 4)]
        key = [int(x) for x in rng.integers(0, 2**32, 2)]
        assert [int(x) for x in oracle.philox4x32_10(ctr, key)] == _philox_bigint(ctr, key)
    # counter = (site, draw, sweep_lo, sweep_hi), key = (seed_lo, seed_hi)
    seed, site, draw, sweep = 0x1234567890ABCDEF, 77, 1, (5 << 32) | 9
    assert [int(x) for x in oracle.philox_site(seed, site, draw, sweep)] == _philox_bigint(
        [site, draw, 9, 5], [seed & 0xFFFFFFFF, seed >> 32])


def test_mt19937_64_known_answers():
    for seed, idx, val in _rows("mt19937_64_kat.txt"):
        assert int(oracle.mt19937_64(int(seed), int(idx))[-1]) == int(val)


# ---- the (0,1) map --------------------------------------------------------------
def test_u01_is_exact_open_and_symmetric():
    assert float(oracle.u01(0)) == 2.0**-24
    assert float(oracle.u01(0xFFFFFFFF)) == 1.0 - 2.0**-24
    rng = np.random.default_rng(3)
    for r in rng.integers(0, 2**32, 500):
        r = int(r)
        u = float(oracle.u01(r))
        assert u == (2 * (r >> 9) + 1) / 2.0**24            # exact rational
        assert 0.0 < u < 1.0
        assert u + float(oracle.u01(r ^ 0xFFFFFFFF)) == 1.0  # symmetric about 1/2


# ---- K5: spec sincos / exp against libm in double --------------------------------
def test_sincos_spec_exhaustive():
    # every odd k in [1, 2^24-1]: phi = 2*pi*k/2^24
    count = 1 << 23
    s, c = oracle.sincos_spec_batch(1, 2, count)
    k = 1 + 2 * np.arange(count, dtype=np.float64)
    phi = k * (2.0 * math.pi / 2.0**24)
    assert np.max(np.abs(s.astype(np.float64) - np.sin(phi))) <= 8e-8
    assert np.max(np.abs(c.astype(np.float64) - np.cos(phi))) <= 8e-8
    s64, c64 = s.astype(np.float64), c.astype(np.float64)
    assert np.max(np.abs(s64 * s64 + c64 * c64 - 1.0)) <= 2e-7
    # the quadrants: cos>0 for phi near 0, sin>0 in (0,pi) ...
    assert c[0] > 0.999999 and abs(s[0]) < 1e-6
    assert abs(c[count // 4]) < 1e-6 and s[count // 4] > 0.999999       # phi ~ pi/2
    assert c[count // 2] < -0.999999 and abs(s[count // 2]) < 1e-6      # phi ~ pi
    assert abs(c[3 * count // 4]) < 1e-6 and s[3 * count // 4] < -0.999999


def test_exp_spec_against_libm():
    x = np.concatenate([np.linspace(-17.0, 0.0, 2_000_001), -np.logspace(-8, 1.2, 200_001)])
    x = x[(x >= -17.0) & (x <= 0.0)].astype(np.float32)
    got = oracle.exp_spec_batch(x).astype(np.float64)
    ref = np.exp(x.astype(np.float64))
    ulp = np.spacing(ref.astype(np.float32)).astype(np.float64)
    assert np.max(np.abs(got - ref) / ulp) <= 1.5
    assert float(oracle.exp_spec(0.0)) == 1.0 and float(oracle.exp_spec(-0.0)) == 1.0
    # the cut-off: exp(-17) < 2^-24 = the smallest u, so "x < -17 => reject" loses nothing
    assert math.exp(-17.0) < 2.0**-24 < math.exp(-16.0)
    # constants: Cody-Waite split of ln 2
    assert abs((0.693359375 - float(np.float32(2.12194442e-04))) - math.log(2.0)) < 2e-11


# ---- K2/K3: the sphere map ---------------------------------------------------------
def test_sphere_closed_form_and_unit_norm():
    rng = np.random.default_rng(11)
    r0 = rng.integers(0, 2**32, 200_000, dtype=np.uint64).astype(np.uint32)
    r1 = rng.integers(0, 2**32, 200_000, dtype=np.uint64).astype(np.uint32)
    s = oracle.sphere_batch(r0, r1).astype(np.float64)
    u1 = (2.0 * (r0 >> 9).astype(np.float64) + 1.0) / 2.0**24
    u2 = (2.0 * (r1 >> 9).astype(np.float64) + 1.0) / 2.0**24
    z = 1.0 - 2.0 * u1
    rr = np.sqrt(1.0 - z * z)
    ref = np.stack([rr * np.cos(2 * np.pi * u2), rr * np.sin(2 * np.pi * u2), z], axis=1)
    assert np.max(np.abs(s - ref)) <= 2e-7
    assert np.all(s[:, 2] == z)                                  # z is exact
    assert np.max(np.abs(np.sum(s * s, axis=1) - 1.0)) <= 5e-7   # |S| = 1 [P:40]


def test_worked_attempt_seed1_site5_sweep3():
    # SURVEY.md 8(c) K2, recomputed here in double from the definitions
    r = [int(x) for x in oracle.philox_site(1, 5, 0, 3)]
    assert r == _philox_bigint([5, 0, 3, 0], [1, 0])
    u = [(2 * (x >> 9) + 1) / 2.0**24 for x in r[:3]]
    assert [float(oracle.u01(x)) for x in r[:3]] == u
    z = 1 - 2 * u[0]
    rr = math.sqrt(1 - z * z)
    ref = [rr * math.cos(2 * math.pi * u[1]), rr * math.sin(2 * math.pi * u[1]), z]
    assert np.max(np.abs(oracle.sphere(r[0], r[1]).astype(np.float64) - ref)) <= 2e-7
    k = 2 * (r[1] >> 9) + 1
    q = (k + (1 << 21)) >> 22
    assert 0 <= q <= 4 and abs(k - q * (1 << 22)) <= (1 << 21)


def test_sphere_map_is_uniform():
    # z uniform on [-1,1], phi uniform on [0,2pi): Kolmogorov-Smirnov on a Philox stream
    from scipy import stats
    n = 100_000
    r = np.array([oracle.philox_site(2024, i, 0, 0) for i in range(n)], dtype=np.uint32)
    s = oracle.sphere_batch(r[:, 0], r[:, 1]).astype(np.float64)
    assert stats.kstest((s[:, 2] + 1) / 2, "uniform").pvalue > 1e-3
    phi = np.mod(np.arctan2(s[:, 1], s[:, 0]), 2 * np.pi) / (2 * np.pi)
    assert stats.kstest(phi, "uniform").pvalue > 1e-3
    assert abs(np.mean(s[:, 2] ** 2) - 1 / 3) < 4 * math.sqrt(4 / 45 / n)     # <z^2> = 1/3
    assert abs(np.corrcoef(s[:, 2], phi)[0, 1]) < 4 / math.sqrt(n)


# ---- K11: lattices against independent constructions ------------------------------
def _adj(lat):
    rp, col = lat.row_ptr, lat.col
    return [list(col[rp[i]:rp[i + 1]]) for i in range(lat.n)]


def _check_structure(lat, z=None):
    rp, col, colour = lat.row_ptr, lat.col, lat.colour
    n = lat.n
    assert rp[0] == 0 and rp[-1] == lat.nnz == col.size
    row = np.repeat(np.arange(n), np.diff(rp))
    assert np.all(col != row)                                    # no self loops
    assert np.all(colour[row] != colour[col])                    # proper colouring
    assert colour.min() == 0 and colour.max() == lat.n_colours - 1
    a = np.sort(row.astype(np.int64) * n + col)                  # symmetric with multiplicity
    b = np.sort(col.astype(np.int64) * n + row)
    assert np.array_equal(a, b)
    if z is not None:
        assert np.all(np.diff(rp) == z)


def test_sc_neighbours_order_and_colour():
    Lx, Ly, Lz = 4, 6, 2
    lat = oracle.Lattice.sc(Lx, Ly, Lz)
    _check_structure(lat, 6)
    ids = np.arange(Lx * Ly * Lz).reshape(Lz, Ly, Lx)            # id = (z*Ly + y)*Lx + x
    want = np.stack([np.roll(ids, 1, 2), np.roll(ids, -1, 2), np.roll(ids, 1, 1),
                     np.roll(ids, -1, 1), np.roll(ids, 1, 0), np.roll(ids, -1, 0)], axis=-1)
    assert np.array_equal(lat.col.reshape(-1, 6), want.reshape(-1, 6))   # -x,+x,-y,+y,-z,+z
    zz, yy, xx = np.meshgrid(np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    assert np.array_equal(lat.colour, ((xx + yy + zz) & 1).ravel())


def _min_image_d2(pa, pb, box):
    d = np.abs(pa - pb)
    d = np.minimum(d, box - d)
    return np.sum(d * d, axis=-1)


@pytest.mark.parametrize("kind,z,d2", [("bcc", 8, 3), ("fcc", 12, 2)])
def test_bravais_geometry(kind, z, d2):
    # positions in doubled integer units; every listed neighbour sits at the nearest-
    # neighbour distance under the minimum image, and all z of them are distinct
    L = (3, 4, 5)
    lat = getattr(oracle.Lattice, kind)(*L)
    _check_structure(lat, z)
    nc = L[0] * L[1] * L[2]
    basis = {"bcc": [(0, 0, 0), (1, 1, 1)], "fcc": [(0, 0, 0), (0, 1, 1), (1, 0, 1), (1, 1, 0)]}[kind]
    pos = np.zeros((lat.n, 3), np.int64)
    for b, off in enumerate(basis):
        cz, cy, cx = np.meshgrid(np.arange(L[2]), np.arange(L[1]), np.arange(L[0]), indexing="ij")
        pos[b * nc:(b + 1) * nc] = np.stack([2 * cx.ravel() + off[0], 2 * cy.ravel() + off[1], 2 * cz.ravel() + off[2]], 1)
    assert np.array_equal(lat.colour, np.repeat(np.arange(len(basis)), nc))
    box = 2 * np.array(L)
    col = lat.col.reshape(lat.n, z)
    for k in range(z):
        assert np.all(_min_image_d2(pos, pos[col[:, k]], box) == d2)
    assert all(len(set(r)) == z for r in col)
    # brute force: the set of sites at that distance is exactly the list
    for i in (0, nc - 1, nc, lat.n - 1):
        near = np.nonzero(_min_image_d2(pos[i], pos, box) == d2)[0]
        assert sorted(near) == sorted(col[i])
    if kind == "fcc":   # the canonical offset order of [D:A16]
        off = np.array([(1, 1, 0), (1, -1, 0), (-1, 1, 0), (-1, -1, 0), (1, 0, 1), (1, 0, -1),
                        (-1, 0, 1), (-1, 0, -1), (0, 1, 1), (0, 1, -1), (0, -1, 1), (0, -1, -1)])
        for k in range(12):
            assert np.all(np.mod(pos + off[k], box) == pos[col[:, k]])
    else:               # corner: centres of cells (x-1|x, y-1|y, z-1|z), x fastest; centre: (x|x+1,...)
        k = 0
        for dz in (-1, 0):
            for dy in (-1, 0):
                for dx in (-1, 0):
                    want = np.mod(pos[:nc] + 2 * np.array([dx, dy, dz]) + 1, box)
                    assert np.all(want == pos[col[:nc, k]])
                    want = np.mod(pos[nc:] - 1 + 2 * np.array([dx + 1, dy + 1, dz + 1]), box)
                    assert np.all(want == pos[col[nc:, k]])
                    k += 1


def test_small_periodic_lattices_keep_multi_edges():
    # [D:A17] L = 2: a neighbour reached through both faces is listed twice
    lat = oracle.Lattice.sc(2)
    _check_structure(lat, 6)
    assert all(sorted(r)[0::2] == sorted(r)[1::2] for r in _adj(lat))
    for kind, z in (("bcc", 8), ("fcc", 12)):
        _check_structure(getattr(oracle.Lattice, kind)(2), z)


def _sphere_brute(R):
    D = 2 * R
    ax = np.arange(-D, D + 1)
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    inside = (((X + Y + Z) & 1) == 0) & (X * X + Y * Y + Z * Z <= D * D)
    pad = np.pad(inside, 1)
    deg = np.zeros(inside.shape, np.int32)
    for o in [(1, 1, 0), (1, -1, 0), (-1, 1, 0), (-1, -1, 0), (1, 0, 1), (1, 0, -1),
              (-1, 0, 1), (-1, 0, -1), (0, 1, 1), (0, 1, -1), (0, -1, 1), (0, -1, -1)]:
        deg += pad[1 + o[2]:1 + o[2] + inside.shape[0], 1 + o[1]:1 + o[1] + inside.shape[1],
                   1 + o[0]:1 + o[0] + inside.shape[2]]
    return inside, deg[inside], np.stack([X[inside], Y[inside], Z[inside]], 1)


@pytest.mark.parametrize("R,n_expect", [(2, 141), (5, 2123)])
def test_fcc_sphere_small(R, n_expect):
    lat = oracle.Lattice.fcc_sphere(R, 0.05, (0, 0, 1), 0.5)
    inside, deg, xyz = _sphere_brute(R)
    assert lat.n == n_expect == int(inside.sum())
    assert np.array_equal(lat.xyz, xyz)                          # ascending (Z,Y,X)
    assert np.array_equal(np.diff(lat.row_ptr), deg)
    _check_structure(lat)
    # every listed neighbour is at doubled distance^2 = 2
    row = np.repeat(np.arange(lat.n), np.diff(lat.row_ptr))
    d = lat.xyz[row] - lat.xyz[lat.col]
    assert np.all(np.sum(d * d, 1) == 2)
    # [D:A11] core sites K=0.05 along z, surface sites K=0.5 along the radial direction
    K, e = lat.K, lat.e
    core = deg == 12
    assert np.all(K[core] == np.float32(0.05)) and np.all(e[core] == np.array([0, 0, 1], np.float32))
    assert np.all(K[~core] == np.float32(0.5))
    r = xyz[~core].astype(np.float64)
    assert np.array_equal(e[~core], (r / np.linalg.norm(r, axis=1, keepdims=True)).astype(np.float32))


def test_fcc_sphere_R60_counts():
    # config 5: N and nnz by brute force over the integer grid
    inside, deg, _ = _sphere_brute(60)
    lat = oracle.Lattice.fcc_sphere(60, 0.05, (0, 0, 1), 0.5)
    assert lat.n == int(inside.sum()) == 3_618_393
    assert lat.nnz == int(deg.sum()) == 43_037_280
    assert np.array_equal(np.diff(lat.row_ptr), deg)
    hist = np.bincount(deg, minlength=13)
    assert hist[12] == 3_502_959 and int(hist[:12].sum()) == 115_434
    _check_structure(lat)
    assert lat.n_colours == 7                                    # first-fit in (Z,Y,X) order [D:A12]
    par = oracle.Lattice.fcc_sphere(60, colouring="parity")
    _check_structure(par)
    assert par.n_colours == 4


def test_greedy_colouring_is_first_fit():
    # path 0-1-2-3 plus triangle 4-5-6: first fit gives 0,1,0,1 and 0,1,2
    edges = [(0, 1), (1, 2), (2, 3), (4, 5), (5, 6), (4, 6)]
    n = 7
    nb = [[] for _ in range(n)]
    for a, b in edges:
        nb[a].append(b)
        nb[b].append(a)
    rp = np.cumsum([0] + [len(x) for x in nb])
    lat = oracle.Lattice.csr(rp, np.concatenate(nb))
    assert list(lat.colour) == [0, 1, 0, 1, 0, 1, 2] and lat.n_colours == 3


# ---- K4: local dH equals the brute-force difference of the total energy --------------
def _total_energy_numpy(lat, J, S):
    rp, col = lat.row_ptr, lat.col
    row = np.repeat(np.arange(lat.n), np.diff(rp))
    ex = np.sum(S[row] * S[col])                                 # every bond twice
    a = np.sum(S * lat.e.astype(np.float64), axis=1)
    return -0.5 * J * ex - np.sum(lat.K.astype(np.float64) * a * a)


def _random_units(rng, n):
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


@pytest.mark.parametrize("make", [
    lambda: oracle.Lattice.sc(2), lambda: oracle.Lattice.sc(4), lambda: oracle.Lattice.sc(4, 2, 6),
    lambda: oracle.Lattice.bcc(2), lambda: oracle.Lattice.bcc(3), lambda: oracle.Lattice.fcc(2),
    lambda: oracle.Lattice.fcc(3), lambda: oracle.Lattice.fcc_sphere(2)])
def test_delta_h_equals_bruteforce_energy_difference(make):
    rng = np.random.default_rng(5)
    lat = make()
    n = lat.n
    lat.set_site_anisotropy(rng.uniform(-0.7, 0.7, n), _random_units(rng, n))
    J = 1.25   # exact in fp32
    S = _random_units(rng, n)
    S32 = S.astype(np.float32)
    st64 = oracle.State64(lat, J, 1)
    st64.set_spins(S[:, 0], S[:, 1], S[:, 2])
    st32 = oracle.State32(lat, J, 1)
    st32.set_spins(S32[:, 0], S32[:, 1], S32[:, 2])
    E0 = _total_energy_numpy(lat, J, S)
    assert abs(oracle.total_energy64(lat, J, S[:, 0], S[:, 1], S[:, 2]) - E0) <= 1e-10
    E0_32 = _total_energy_numpy(lat, J, S32.astype(np.float64))
    for i in rng.integers(0, n, 40):
        i = int(i)
        new = _random_units(rng, 1)[0]
        S2 = S.copy()
        S2[i] = new
        assert abs(st64.delta_h(i, new) - (_total_energy_numpy(lat, J, S2) - E0)) <= 1e-12 * 50
        new32 = new.astype(np.float32)
        T2 = S32.astype(np.float64).copy()
        T2[i] = new32
        assert abs(float(st32.delta_h(i, new32)) - (_total_energy_numpy(lat, J, T2) - E0_32)) <= 1e-5
    # the measured energy is the same total
    m32, e32, e64 = st32.measure()
    assert abs(e64 - E0_32) <= 1e-9 and abs(e32 - E0_32) <= 2e-6 * n
    # eq. (2) [P:22] by component, sign included: a permuted or negated component of O32's M fails here
    want_m = S32.astype(np.float64).mean(0)
    assert np.max(np.abs(np.asarray(m32, np.float64) - want_m)) <= 1e-7
    assert np.max(np.abs(want_m)) > 1e-3 and len({round(abs(float(v)), 6) for v in want_m}) == 3   # the pin can tell components apart
    M, E = st64.measure()
    assert abs(E - E0) <= 1e-10 and np.allclose(M, S.mean(0), atol=1e-14)


@pytest.mark.parametrize("make", [lambda: oracle.Lattice.sc(4), lambda: oracle.Lattice.bcc(3), lambda: oracle.Lattice.fcc(2),
                                  lambda: oracle.Lattice.fcc_sphere(2)])
def test_o32_magnetisation_by_component(make):
    # eq. (2) [P:22]: M = (1/N) sum_i S_i as a VECTOR.  A state whose three component sums are distinct, of mixed sign and
    # known in closed form: S_i = (0.6, 0, -0.8) on even sites, (0, 1, 0) on odd ones.
    lat = make()
    lat.set_uniform_anisotropy(0.0, (0, 0, 1))
    n = lat.n
    even = (np.arange(n) % 2 == 0)
    sx = np.where(even, np.float32(0.6), np.float32(0.0)).astype(np.float32)
    sy = np.where(even, np.float32(0.0), np.float32(1.0)).astype(np.float32)
    sz = np.where(even, np.float32(-0.8), np.float32(0.0)).astype(np.float32)
    st = oracle.State32(lat, 1.0, 1)
    st.set_spins(sx, sy, sz)
    M = np.asarray(st.measure()[0], np.float64)
    ne = int(even.sum())
    want = np.array([float(np.float32(0.6)) * ne / n, (n - ne) / n, float(np.float32(-0.8)) * ne / n])
    assert np.max(np.abs(M - want)) <= 1e-12
    assert M[0] > 0 > M[2] and M[1] > M[0]


# ---- K12/K13: invariants of the counter-based stream ----------------------------------
def test_checkpoint_and_order_invariance():
    lat = oracle.Lattice.bcc(4)
    lat.set_uniform_anisotropy(0.1, (0, 0, 1))
    a = oracle.State32(lat, 1.0, 42)
    a.init_random()
    a.sweep(1.5, 6)
    b = oracle.State32(lat, 1.0, 42)
    b.init_random()
    b.sweep(1.5, 3)
    c = oracle.State32(lat, 1.0, 42)                             # resume from (spins, counter)
    c.set_spins(*b.get_spins())
    c.sweep_count = b.sweep_count
    c.sweep(1.5, 3)
    assert all(np.array_equal(x, y) for x, y in zip(a.get_spins(), c.get_spins()))
    d = oracle.State32(lat, 1.0, 42)                             # descending site order within a colour
    d.init_random()
    d.sweep(1.5, 6, order=1)
    assert all(np.array_equal(x, y) for x, y in zip(a.get_spins(), d.get_spins()))
    e = oracle.State32(lat, 1.0, 43)                             # another seed is another trajectory
    e.init_random()
    assert not np.array_equal(a.get_spins()[0], e.get_spins()[0])


def test_accept_rule_and_norm_preserved():
    # K3 + rule (iii): recompute every decision of one sweep from the proposal and dH
    lat = oracle.Lattice.sc(6)
    lat.set_uniform_anisotropy(0.3, (0.6, 0.0, 0.8))
    st = oracle.State32(lat, 1.0, 9)
    st.init_random()
    st.sweep(0.7, 3)
    T = 0.7
    colour = lat.colour
    ref = oracle.State32(lat, 1.0, 9)
    ref.set_spins(*st.get_spins())
    ref.sweep_count = st.sweep_count
    acc = st.sweep(T, 1, record=True)[0]
    for c in range(2):
        for i in np.nonzero(colour == c)[0]:
            s_new, u3 = ref.proposal(int(i))
            dH = float(ref.delta_h(int(i), s_new))
            want = dH <= 0 or (u3 <= math.exp(-dH / T) * (1 + 4e-7) and -dH / T >= -17.0)
            near = dH > 0 and abs(float(u3) - math.exp(-dH / T)) < 1e-6
            if not near:
                assert bool(acc[i]) == want
            if acc[i]:
                sx, sy, sz = ref.get_spins()
                sx[i], sy[i], sz[i] = s_new
                ref.set_spins(sx, sy, sz)
    got, want = st.get_spins(), ref.get_spins()
    assert all(np.array_equal(x, y) for x, y in zip(got, want))
    nrm = sum(x.astype(np.float64) ** 2 for x in got)
    assert np.max(np.abs(nrm - 1.0)) <= 5e-7
    att, ok = st.stats()
    assert att == 4 * lat.n and 0 < ok < att
