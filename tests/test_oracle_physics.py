"""Statistical pins of the CPU oracle (both O32 and O64) against closed forms and
the value the paper prints.  CPU only.

All seeds are fixed, so every run gives the same numbers; the sigma-based
tolerances document how far from the closed form a correct program lands.
"""
import math

import numpy as np
import pytest
from scipy import integrate

import oracle


def _isolated(n, K, e):
    lat = oracle.Lattice.csr(np.zeros(n + 1, np.int64), np.zeros(0, np.int32), np.zeros(n, np.int32), 1)
    lat.set_uniform_anisotropy(K, e)
    return lat


def _a2_exact(kappa):
    num = integrate.quad(lambda x: x * x * math.exp(kappa * (x * x - 1)), -1, 1, epsabs=1e-13)[0]
    den = integrate.quad(lambda x: math.exp(kappa * (x * x - 1)), -1, 1, epsabs=1e-13)[0]
    return num / den


def _blocked_sem(x, nblock=20):
    b = np.array_split(np.asarray(x), nblock)
    m = np.array([v.mean() for v in b])
    return m.mean(), m.std(ddof=1) / math.sqrt(nblock)


# ---- K6: one spin, anisotropy only: <(S.e)^2> = int x^2 e^{kx^2} / int e^{kx^2} ----------
@pytest.mark.parametrize("kappa", [-5.0, -1.0, 0.1, 1.0, 5.0])
def test_single_spin_anisotropy_closed_form(kappa):
    T, n = 0.5, 2048
    K = kappa * T
    e = np.array([0.48, -0.6, 0.64])                       # a unit vector, exact-ish in fp32
    exact = _a2_exact(kappa)
    if abs(kappa) == 1.0:                                   # the values listed in SURVEY 8(c) K6
        assert abs(exact - {1.0: 0.4292307, -1.0: 0.2537041}[kappa]) < 1e-6
    lat = _isolated(n, K, e)
    e32 = lat.e.astype(np.float64)
    st = oracle.State32(lat, 1.0, 17)
    st.init_random()
    st.sweep(T, 50)
    vals = []
    for _ in range(300):
        st.sweep(T, 1)
        s = np.stack(st.get_spins(), 1).astype(np.float64)
        vals.append(np.mean(np.sum(s * e32, 1) ** 2))
    m, sem = _blocked_sem(vals)
    assert abs(m - exact) < 4 * sem + 1e-4, (m, exact, sem)
    st64 = oracle.State64(lat, 1.0, 99)
    st64.init_random()
    st64.sweep(T, 50)
    _, _, a2 = st64.series(T, 300)
    m, sem = _blocked_sem(a2)
    assert abs(m - exact) < 4 * sem + 1e-4, (m, exact, sem)


# ---- K7: open Heisenberg chain: <S_i.S_{i+r}> = L(J/T)^r, L(x) = coth x - 1/x --------------
def _chains(n_chain, length):
    nb = [[] for _ in range(n_chain * length)]
    for c in range(n_chain):
        for k in range(length - 1):
            a = c * length + k
            nb[a].append(a + 1)
            nb[a + 1].append(a)
    for r in nb:
        r.sort()
    rp = np.cumsum([0] + [len(x) for x in nb])
    colour = np.tile(np.arange(length) & 1, n_chain).astype(np.int32)
    return oracle.Lattice.csr(rp, np.concatenate(nb), colour, 2)


@pytest.mark.parametrize("x", [0.5, 2.0])
def test_open_chain_closed_form(x):
    J, length, n_chain = 1.0, 8, 256
    T = J / x
    lang = 1.0 / math.tanh(x) - 1.0 / x
    if x == 2.0:
        assert abs(lang - 0.5373147) < 1e-6
    lat = _chains(n_chain, length)
    for which in ("O32", "O64"):
        st = oracle.State32(lat, J, 5) if which == "O32" else oracle.State64(lat, J, 5)
        st.init_random()
        st.sweep(T, 200)
        nn, r3, en = [], [], []
        for _ in range(400):
            st.sweep(T, 1)
            s = np.stack(st.get_spins(), 1).astype(np.float64).reshape(n_chain, length, 3)
            nn.append(np.mean(np.sum(s[:, :-1] * s[:, 1:], -1)))
            r3.append(np.mean(np.sum(s[:, :-3] * s[:, 3:], -1)))
            en.append(st.measure()[-1] / n_chain)
        m, sem = _blocked_sem(nn)
        assert abs(m - lang) < 4 * sem + 1e-4, (which, m, lang, sem)
        m, sem = _blocked_sem(r3)
        assert abs(m - lang**3) < 4 * sem + 1e-4, (which, m, lang**3, sem)
        m, sem = _blocked_sem(en)                           # <E> = -(n-1) J L per chain (bond once [D:A1])
        assert abs(m + (length - 1) * J * lang) < 4 * sem + 1e-3, (which, m, sem)


# ---- K8: T = infinity ---------------------------------------------------------------------
def test_infinite_temperature():
    lat = oracle.Lattice.sc(16)
    lat.set_uniform_anisotropy(0.3, (0, 0, 1))
    st = oracle.State32(lat, 1.0, 1)
    st.init_aligned((0, 0, 1))
    M, E = st.series(float("inf"), 200)
    att, acc = st.stats()
    assert att == acc == 200 * 4096                          # every move accepted
    absM = np.linalg.norm(M, axis=1)
    expect = math.sqrt(8 / (3 * math.pi * 4096))             # <|M|> of N i.i.d. unit vectors
    assert abs(expect - 0.0143956) < 1e-7
    assert abs(absM.mean() - expect) < 4 * absM.std(ddof=1) / math.sqrt(200)
    assert abs(np.mean(absM**2) - 1 / 4096) < 4 * np.std(absM**2, ddof=1) / math.sqrt(200)
    # <E> = -K N <z^2> = -K N / 3 ; exchange part averages to 0
    assert abs(E.mean() + 0.3 * 4096 / 3) < 4 * E.std(ddof=1) / math.sqrt(200)
    st64 = oracle.State64(lat, 1.0, 8)
    st64.init_aligned((0, 0, 1))
    m, e, _ = st64.series(1e300, 200)
    att, acc = st64.stats()
    assert att == acc
    assert abs(m.mean() - expect) < 4 * m.std(ddof=1) / math.sqrt(200)


# ---- K9: T -> 0 and the low-temperature expansion --------------------------------------------
def test_low_temperature_limits():
    lat = oracle.Lattice.sc(16)
    st = oracle.State32(lat, 1.0, 1)
    st.init_aligned((0, 0, 1))
    M, E = st.series(0.01, 50)
    att, acc = st.stats()
    assert np.linalg.norm(M[-1]) > 0.99 and acc / att < 0.01
    assert E[-1] / 4096 < -2.98
    # classical spin-wave, first order: E/N = -3J + T (1 - 1/N);  M = 1 - T W_L / (6J)
    kx = 2 * np.pi * np.arange(16) / 16
    g = (np.cos(kx)[:, None, None] + np.cos(kx)[None, :, None] + np.cos(kx)[None, None, :]) / 3
    w = 1.0 / (1.0 - g.ravel()[1:])
    W = w.sum() / 4096
    assert abs(W - 1.43178) < 1e-4
    T = 0.1
    for which in ("O32", "O64"):
        if which == "O32":
            s = oracle.State32(lat, 1.0, 2)
            s.init_aligned((0, 0, 1))
            s.sweep(T, 500)
            M, E = s.series(T, 1500)
            absM = np.linalg.norm(M, axis=1)
        else:
            s = oracle.State64(lat, 1.0, 2)
            s.init_aligned((0, 0, 1))
            s.sweep(T, 500)
            absM, E, _ = s.series(T, 1500)
        assert abs(absM.mean() - (1 - T * W / 6)) < 0.005 * (1 - T * W / 6), (which, absM.mean())
        assert abs(E.mean() / 4096 - (-3 + T * (1 - 1 / 4096))) < 0.005 * 3, (which, E.mean() / 4096)


# ---- K10 / [D:A1]: the sc transition sits where the paper says ------------------------------
def _binder(L, T, seed, therm, meas):
    lat = oracle.Lattice.sc(L)
    st = oracle.State32(lat, 1.0, seed)
    st.init_aligned((0, 0, 1))
    st.sweep(T, therm)
    M, _ = st.series(T, meas)
    m2 = np.sum(M * M, 1)
    return 1.0 - np.mean(m2 * m2) / (3.0 * np.mean(m2) ** 2), math.sqrt(np.mean(m2))


def test_sc_critical_temperature_bracket():
    # paper: T_C/J = 1.445 (tests/golden/paper_values.txt, [P:52]).  Binder cumulants of
    # L = 6 and L = 12 cross at T_c: below it the larger lattice has the larger U, above
    # it the smaller.  Bonds counted twice would put T_c near 2.89 and fail the upper side.
    Tc = 1.445
    lo, hi = Tc - 0.10, Tc + 0.10
    u6_lo, _ = _binder(6, lo, 3, 2000, 12000)
    u12_lo, m_lo = _binder(12, lo, 4, 2000, 12000)
    u6_hi, _ = _binder(6, hi, 5, 2000, 12000)
    u12_hi, m_hi = _binder(12, hi, 6, 2000, 12000)
    assert u12_lo > u6_lo + 0.005, (u6_lo, u12_lo)
    assert u12_hi < u6_hi - 0.005, (u6_hi, u12_hi)
    assert m_lo > 0.30 > m_hi                                 # order parameter drops across T_c
    # far sides: ordered at 0.5 T_c, disordered at 2 T_c (where a double-counted model is still ordered)
    _, m_cold = _binder(8, 0.5 * Tc, 7, 300, 700)
    _, m_hot = _binder(8, 2.0 * Tc, 8, 300, 700)
    assert m_cold > 0.75 and m_hot < 0.12


# ---- S3: the two oracles agree statistically (colour-ordered fp32 vs random-site fp64) --------
def test_o32_and_o64_agree():
    lat = oracle.Lattice.sc(8)
    lat.set_uniform_anisotropy(0.1, (0, 0, 1))
    T, reps = 1.2, 12
    a_m, a_e, b_m, b_e = [], [], [], []
    for r in range(reps):
        a = oracle.State32(lat, 1.0, 100 + r)
        a.init_random()
        a.sweep(T, 400)
        M, E = a.series(T, 800)
        a_m.append(np.linalg.norm(M, axis=1).mean())
        a_e.append(E.mean() / lat.n)
        b = oracle.State64(lat, 1.0, 200 + r)
        b.init_random()
        b.sweep(T, 400)
        m, e, _ = b.series(T, 800)
        b_m.append(m.mean())
        b_e.append(e.mean() / lat.n)
    for x, y in ((a_m, b_m), (a_e, b_e)):
        x, y = np.array(x), np.array(y)
        se = math.sqrt(x.var(ddof=1) / reps + y.var(ddof=1) / reps)
        assert abs(x.mean() - y.mean()) < 3 * se, (x.mean(), y.mean(), se)
