"""The device's arithmetic contract, element by element, against the CPU oracle.

`hb_device_math` (include/hb.h) evaluates the building blocks of one attempt exactly as the colour kernels do -- the scalar
functions and the packed fp32x2 copies -- and these tests compare them BIT FOR BIT with `oracle.*_batch` over every
argument that can occur: all 2^23 values of r >> 9 (u, z = 1 - 2u, the square root), all 2^23 odd k (sincos), and for
exp a dense sweep of [-17, 0] plus the cut-off.  The trajectory tests only visit the arguments a run happens to draw.
"""
import numpy as np
import pytest

import oracle
import paper_2106_11286_b200 as hb

pytestmark = pytest.mark.gpu

N23 = 1 << 23


def _bits(a):
    return np.ascontiguousarray(a, np.float32).view(np.uint32)


def test_u01_every_mantissa():
    r = (np.arange(N23, dtype=np.uint64) << 9).astype(np.uint32)
    r |= np.random.default_rng(0).integers(0, 512, N23, dtype=np.uint32)          # the low 9 bits must not matter
    got = hb.device_math("u01", r)
    want = ((2.0 * (r >> 9).astype(np.float64) + 1.0) * 2.0 ** -24).astype(np.float32)   # the definition, exact in fp32
    assert np.array_equal(_bits(got[:, 0]), _bits(want)) and np.array_equal(_bits(got[:, 1]), _bits(want))
    assert got.min() > 0.0 and got.max() < 1.0
    assert float(oracle.u01(int(r[12345]))) == float(want[12345])


def test_sincos_every_angle_bitwise():
    # k = (r1 >> 8) | 1 runs over all 2^23 odd values in [1, 2^24 - 1]
    r1 = (np.arange(N23, dtype=np.uint64) << 9).astype(np.uint32)
    got = hb.device_math("sincos", r1)
    s, c = oracle.sincos_spec_batch(1, 2, N23)
    assert np.array_equal(_bits(got[:, 0]), _bits(s))
    assert np.array_equal(_bits(got[:, 1]), _bits(c))


def test_sqrt_is_correctly_rounded_on_every_reachable_argument():
    r0 = (np.arange(N23, dtype=np.uint64) << 9).astype(np.uint32)
    got = hb.device_math("sqrt", r0)
    assert np.array_equal(_bits(got[:, 0]), _bits(got[:, 1]))                     # rsqrt + Newton == __fsqrt_rn
    u = ((2.0 * (r0 >> 9).astype(np.float64) + 1.0) * 2.0 ** -24)
    z = (1.0 - 2.0 * u).astype(np.float32).astype(np.float64)                     # exact
    w = (1.0 - z * z).astype(np.float32)                                          # one rounding, like fma(-z, z, 1)
    assert np.array_equal(_bits(got[:, 1]), _bits(np.sqrt(w)))                    # numpy's fp32 sqrt is IEEE


def test_sphere_every_z_and_every_angle_bitwise():
    rng = np.random.default_rng(1)
    # every r0 >> 9 once with random angles, then every angle once with random z: scalar and packed paths
    for r0, r1 in (((np.arange(N23, dtype=np.uint64) << 9).astype(np.uint32), rng.integers(0, 1 << 32, N23, dtype=np.uint64).astype(np.uint32)),
                   (rng.integers(0, 1 << 32, N23, dtype=np.uint64).astype(np.uint32), (np.arange(N23, dtype=np.uint64) << 9).astype(np.uint32))):
        got = hb.device_math("sphere", r0, r1)
        want = oracle.sphere_batch(r0, r1)
        assert np.array_equal(_bits(got[:, 0:3]), _bits(want))
        assert np.array_equal(_bits(got[:, 3:6]), _bits(want))
    # an odd count: the last element has no partner in its pair
    got = hb.device_math("sphere", r0[:1001], r1[:1001])
    assert np.array_equal(_bits(got[:, 3:6]), _bits(oracle.sphere_batch(r0[:1001], r1[:1001])))


def test_exp_dense_and_cutoff_bitwise():
    rng = np.random.default_rng(2)
    x = np.concatenate([
        -np.linspace(0.0, 17.0, 3_000_001),
        -rng.uniform(0.0, 17.0, 1_000_000),
        -np.ldexp(rng.uniform(0.5, 1.0, 200_000), rng.integers(-40, 5, 200_000)),           # tiny and mid magnitudes
        (np.arange(-25, 1)[:, None] * np.log(2.0) + np.linspace(-1e-5, 1e-5, 2001)[None, :]).ravel(),   # around n ln 2
        (np.arange(-24.5, 0.0)[:, None] * np.log(2.0) + np.linspace(-1e-5, 1e-5, 2001)[None, :]).ravel(),   # rounding ties of n
        np.array([0.0, -0.0, -17.0, np.nextafter(np.float32(-17.0), np.float32(0.0)), -16.635532, -1e-30, -1e-45]),
    ]).astype(np.float32)
    x = x[(x <= 0.0) & (x >= -17.0)]
    assert x.size > 4_000_000
    got = hb.device_math("exp", x.view(np.uint32))
    want = oracle.exp_spec_batch(x)
    assert np.array_equal(_bits(got[:, 0]), _bits(want))
    assert np.array_equal(_bits(got[:, 1]), _bits(want))


def test_whole_attempts_match_the_oracle_on_random_inputs():
    # the fused packed attempt (Philox -> proposal -> dH -> acceptance) on arbitrary old spins and fields,
    # against the oracle's attempt on a 2-site dimer whose only neighbour carries the field
    rng = np.random.default_rng(3)
    n = 4000
    site = np.zeros(n, np.uint32)                       # the dimer's site 0
    J, K, T = np.float32(0.75), np.float32(-0.3), np.float32(0.9)
    e = np.array([0.6, 0.0, 0.8], np.float32)
    beta = np.float32(1.0) / T
    v = rng.normal(size=(n, 3)); s_old = (v / np.linalg.norm(v, axis=1, keepdims=True)).astype(np.float32)
    v = rng.normal(size=(n, 3)); h = (v / np.linalg.norm(v, axis=1, keepdims=True)).astype(np.float32)   # one unit neighbour
    sweeps = rng.integers(0, 1 << 40, n, dtype=np.uint64)
    seed = 12345
    words = np.zeros((n, 16), np.uint32)
    words[:, 0] = (sweeps & 0xFFFFFFFF).astype(np.uint32); words[:, 1] = (sweeps >> 32).astype(np.uint32)
    words[:, 2] = seed; words[:, 3] = 0
    for k, val in enumerate((J, K, beta, e[0], e[1], e[2])):
        words[:, 4 + k] = np.float32(val).view(np.uint32)
    words[:, 10:13] = h.view(np.uint32)
    words[:, 13:16] = s_old.view(np.uint32)
    got = hb.device_math("attempt", site, words)
    lat = oracle.Lattice.csr(np.array([0, 1, 2], np.int64), np.array([1, 0], np.int32), np.array([0, 1], np.int32), 2)
    lat.set_uniform_anisotropy(float(K), e)
    acc_total = 0
    for i in range(n):
        st = oracle.State32(lat, float(J), seed)
        st.set_spins(np.array([s_old[i, 0], h[i, 0]], np.float32), np.array([s_old[i, 1], h[i, 1]], np.float32),
                     np.array([s_old[i, 2], h[i, 2]], np.float32))
        st.sweep_count = int(sweeps[i])
        acc = st.sweep(float(T), 1, record=True)[0]
        sx, sy, sz = st.get_spins()
        want = np.array([sx[0], sy[0], sz[0]], np.float32)
        assert np.array_equal(_bits(got[i, 0:3]), _bits(want)), i
        assert int(got[i, 3]) == int(acc[0]), i
        acc_total += int(acc[0])
    assert 0.2 * n < acc_total < 0.95 * n               # both branches of rule (iii) were exercised
