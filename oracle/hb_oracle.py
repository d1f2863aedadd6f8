"""ctypes front end of oracle/hb_oracle.cpp -- TEST INFRASTRUCTURE, not the product.

Argument marshalling only; every number comes from the C++ translation unit,
which states the passages of the paper it follows.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hb_oracle.cpp")
_SO = os.path.join(_HERE, "libhb_oracle.so")
_lib = None


def build(force=False):
    """Compile the oracle with g++ (no fast-math, no fp contraction)."""
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(_SRC):
        return _SO
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]
    try:  # fmaf() as one instruction where the CPU has it; the result is the same either way
        with open("/proc/cpuinfo") as f:
            if " fma " in f.read():
                cmd.append("-mfma")
    except OSError:
        pass
    tmp = _SO + ".tmp%d" % os.getpid()
    subprocess.run(cmd + ["-o", tmp, _SRC], check=True)
    os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(build())
    vp, i32, i64, u32, u64, f32, f64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_uint64, C.c_float, C.c_double
    sig = {
        "orc_philox4x32_10": (None, [vp, vp, vp]),
        "orc_philox_site": (None, [u64, u32, u32, u64, vp]),
        "orc_u01": (f32, [u32]),
        "orc_sincos_spec": (None, [u32, vp, vp]),
        "orc_sincos_spec_batch": (None, [u32, u32, i64, vp, vp]),
        "orc_exp_spec": (f32, [f32]),
        "orc_exp_spec_batch": (None, [vp, i64, vp]),
        "orc_sphere": (None, [u32, u32, vp]),
        "orc_sphere_batch": (None, [vp, vp, i64, vp]),
        "orc_mt19937_64": (None, [u64, i64, vp]),
        "orc_lattice_sc": (vp, [i32, i32, i32]),
        "orc_lattice_bcc": (vp, [i32, i32, i32]),
        "orc_lattice_fcc": (vp, [i32, i32, i32]),
        "orc_lattice_fcc_sphere": (vp, [i32]),
        "orc_lattice_csr": (vp, [i64, vp, vp, vp, i32]),
        "orc_lattice_free": (None, [vp]),
        "orc_lattice_greedy_colour": (None, [vp]),
        "orc_lattice_set_colour": (None, [vp, vp, i32]),
        "orc_lattice_set_uniform_anisotropy": (None, [vp, f32, vp]),
        "orc_lattice_set_site_anisotropy": (None, [vp, vp, vp]),
        "orc_lattice_sphere_anisotropy": (None, [vp, f32, vp, f32]),
        "orc_lattice_n": (i64, [vp]),
        "orc_lattice_nnz": (i64, [vp]),
        "orc_lattice_n_colours": (i32, [vp]),
        "orc_lattice_get": (None, [vp, vp, vp, vp, vp, vp, vp]),
        "orc_state32_create": (vp, [vp, f32, u64]),
        "orc_state32_free": (None, [vp]),
        "orc_state32_init_random": (None, [vp]),
        "orc_state32_init_aligned": (None, [vp, vp]),
        "orc_state32_set": (None, [vp, vp, vp, vp]),
        "orc_state32_get": (None, [vp, vp, vp, vp]),
        "orc_state32_sweep_count": (u64, [vp]),
        "orc_state32_set_sweep_count": (None, [vp, u64]),
        "orc_state32_stats": (None, [vp, vp, vp]),
        "orc_state32_sweep": (None, [vp, f32, i64, C.c_int, vp]),
        "orc_state32_measure": (None, [vp, vp, vp, vp]),
        "orc_state32_series": (None, [vp, f32, i64, vp, vp]),
        "orc_state32_delta_h": (f32, [vp, i64, vp]),
        "orc_state32_proposal": (None, [vp, i64, vp, vp]),
        "orc_state64_create": (vp, [vp, f64, u64]),
        "orc_state64_free": (None, [vp]),
        "orc_state64_init_random": (None, [vp]),
        "orc_state64_init_aligned": (None, [vp, vp]),
        "orc_state64_set": (None, [vp, vp, vp, vp]),
        "orc_state64_get": (None, [vp, vp, vp, vp]),
        "orc_state64_sweep": (None, [vp, f64, i64]),
        "orc_state64_stats": (None, [vp, vp, vp]),
        "orc_state64_measure": (None, [vp, vp, vp]),
        "orc_state64_series": (None, [vp, f64, i64, vp, vp, vp]),
        "orc_total_energy64": (f64, [vp, f64, vp, vp, vp]),
        "orc_state64_delta_h": (f64, [vp, i64, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _arr(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


# ---- scalar pieces of the arithmetic contract --------------------------------
def philox4x32_10(ctr, key):
    c, k, o = _arr(ctr, np.uint32), _arr(key, np.uint32), np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(o))
    return o


def philox_site(seed, site, draw, sweep):
    o = np.zeros(4, np.uint32)
    lib().orc_philox_site(seed, site, draw, sweep, _p(o))
    return o


def u01(r):
    return np.float32(lib().orc_u01(int(r)))


def sincos_spec(k):
    s, c = np.zeros(1, np.float32), np.zeros(1, np.float32)
    lib().orc_sincos_spec(int(k), _p(s), _p(c))
    return s[0], c[0]


def sincos_spec_batch(k0, step, count):
    s, c = np.zeros(count, np.float32), np.zeros(count, np.float32)
    lib().orc_sincos_spec_batch(int(k0), int(step), int(count), _p(s), _p(c))
    return s, c


def exp_spec(x):
    return np.float32(lib().orc_exp_spec(float(np.float32(x))))


def exp_spec_batch(x):
    x = _arr(x, np.float32)
    o = np.zeros_like(x)
    lib().orc_exp_spec_batch(_p(x), x.size, _p(o))
    return o


def sphere(r0, r1):
    o = np.zeros(3, np.float32)
    lib().orc_sphere(int(r0), int(r1), _p(o))
    return o


def sphere_batch(r0, r1):
    r0, r1 = _arr(r0, np.uint32), _arr(r1, np.uint32)
    o = np.zeros((r0.size, 3), np.float32)
    lib().orc_sphere_batch(_p(r0), _p(r1), r0.size, _p(o))
    return o


def mt19937_64(seed, count):
    o = np.zeros(count, np.uint64)
    lib().orc_mt19937_64(int(seed), int(count), _p(o))
    return o


# ---- lattice -------------------------------------------------------------------
class Lattice:
    """Explicit neighbour lists in canonical order, colours, per-site (K_i, e_i)."""

    def __init__(self, handle, kind):
        self.h, self.kind = handle, kind

    @classmethod
    def sc(cls, Lx, Ly=None, Lz=None):
        Ly, Lz = Ly or Lx, Lz or Lx
        return cls(lib().orc_lattice_sc(Lx, Ly, Lz), "sc")

    @classmethod
    def bcc(cls, Lx, Ly=None, Lz=None):
        Ly, Lz = Ly or Lx, Lz or Lx
        return cls(lib().orc_lattice_bcc(Lx, Ly, Lz), "bcc")

    @classmethod
    def fcc(cls, Lx, Ly=None, Lz=None):
        Ly, Lz = Ly or Lx, Lz or Lx
        return cls(lib().orc_lattice_fcc(Lx, Ly, Lz), "fcc")

    @classmethod
    def fcc_sphere(cls, R, K_core=0.0, e_core=(0, 0, 1), K_surf=0.0, colouring="greedy"):
        lat = cls(lib().orc_lattice_fcc_sphere(R), "sphere")
        lat.sphere_anisotropy(K_core, e_core, K_surf)
        if colouring == "greedy":
            lat.greedy_colour()
        elif colouring == "parity":  # [D:A12] the four parity classes of (X mod 2, Y mod 2)
            xyz = lat.xyz
            lat.set_colour(((xyz[:, 0] & 1) * 2 + (xyz[:, 1] & 1)).astype(np.int32), 4)
        else:
            raise ValueError(colouring)
        return lat

    @classmethod
    def csr(cls, row_ptr, col, colour=None, n_colours=0):
        rp, ci = _arr(row_ptr, np.int64), _arr(col, np.int32)
        cc = _arr(colour, np.int32) if colour is not None else None
        return cls(lib().orc_lattice_csr(rp.size - 1, _p(rp), _p(ci), _p(cc), n_colours), "csr")

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.orc_lattice_free(self.h)
            self.h = None

    @property
    def n(self):
        return lib().orc_lattice_n(self.h)

    @property
    def nnz(self):
        return lib().orc_lattice_nnz(self.h)

    @property
    def n_colours(self):
        return lib().orc_lattice_n_colours(self.h)

    def _get(self, which):
        n, nnz = self.n, self.nnz
        bufs = {"row_ptr": np.zeros(n + 1, np.int64), "col": np.zeros(nnz, np.int32), "colour": np.zeros(n, np.int32),
                "K": np.zeros(n, np.float32), "e": np.zeros((n, 3), np.float32), "xyz": np.zeros((n, 3), np.int32)}
        order = ["row_ptr", "col", "colour", "K", "e", "xyz"]
        lib().orc_lattice_get(self.h, *[_p(bufs[k]) if k == which else None for k in order])
        return bufs[which]

    row_ptr = property(lambda s: s._get("row_ptr"))
    col = property(lambda s: s._get("col"))
    colour = property(lambda s: s._get("colour"))
    K = property(lambda s: s._get("K"))
    e = property(lambda s: s._get("e"))
    xyz = property(lambda s: s._get("xyz"))

    def greedy_colour(self):
        lib().orc_lattice_greedy_colour(self.h)

    def set_colour(self, colour, n_colours):
        c = _arr(colour, np.int32)
        lib().orc_lattice_set_colour(self.h, _p(c), n_colours)

    def set_uniform_anisotropy(self, K, e):
        ee = _arr(e, np.float32)
        lib().orc_lattice_set_uniform_anisotropy(self.h, K, _p(ee))

    def set_site_anisotropy(self, K, e):
        kk, ee = _arr(K, np.float32), _arr(e, np.float32)
        lib().orc_lattice_set_site_anisotropy(self.h, _p(kk), _p(ee))

    def sphere_anisotropy(self, K_core, e_core, K_surf):
        ee = _arr(e_core, np.float32)
        lib().orc_lattice_sphere_anisotropy(self.h, K_core, _p(ee), K_surf)


# ---- O32 -----------------------------------------------------------------------
class State32:
    """fp32 colour-ordered sweep, Philox stream (trajectory oracle)."""

    def __init__(self, lat, J, seed):
        self.lat, self.h = lat, lib().orc_state32_create(lat.h, J, seed)

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.orc_state32_free(self.h)
            self.h = None

    def init_random(self):
        lib().orc_state32_init_random(self.h)

    def init_aligned(self, d):
        dd = _arr(d, np.float32)
        lib().orc_state32_init_aligned(self.h, _p(dd))

    def set_spins(self, sx, sy, sz):
        a, b, c = _arr(sx, np.float32), _arr(sy, np.float32), _arr(sz, np.float32)
        lib().orc_state32_set(self.h, _p(a), _p(b), _p(c))

    def get_spins(self):
        n = self.lat.n
        a, b, c = np.zeros(n, np.float32), np.zeros(n, np.float32), np.zeros(n, np.float32)
        lib().orc_state32_get(self.h, _p(a), _p(b), _p(c))
        return a, b, c

    @property
    def sweep_count(self):
        return lib().orc_state32_sweep_count(self.h)

    @sweep_count.setter
    def sweep_count(self, s):
        lib().orc_state32_set_sweep_count(self.h, s)

    def stats(self):
        a, b = C.c_uint64(), C.c_uint64()
        lib().orc_state32_stats(self.h, C.byref(a), C.byref(b))
        return a.value, b.value

    def sweep(self, T, n_sweeps=1, order=0, record=False):
        acc = np.zeros((n_sweeps, self.lat.n), np.uint8) if record else None
        lib().orc_state32_sweep(self.h, T, n_sweeps, order, _p(acc))
        return acc

    def measure(self):
        M = np.zeros(3, np.float64)
        e32, e64 = C.c_double(), C.c_double()
        lib().orc_state32_measure(self.h, _p(M), C.byref(e32), C.byref(e64))
        return M, e32.value, e64.value

    def series(self, T, n_sweeps):
        M, E = np.zeros((n_sweeps, 3), np.float64), np.zeros(n_sweeps, np.float64)
        lib().orc_state32_series(self.h, T, n_sweeps, _p(M), _p(E))
        return M, E

    def delta_h(self, site, s_new):
        s = _arr(s_new, np.float32)
        return np.float32(lib().orc_state32_delta_h(self.h, site, _p(s)))

    def proposal(self, site):
        s, u = np.zeros(3, np.float32), np.zeros(1, np.float32)
        lib().orc_state32_proposal(self.h, site, _p(s), _p(u))
        return s, u[0]


# ---- O64 -----------------------------------------------------------------------
class State64:
    """fp64 random-site Metropolis, the paper's steps (i)-(iii) (statistics oracle)."""

    def __init__(self, lat, J, mt_seed):
        self.lat, self.h = lat, lib().orc_state64_create(lat.h, J, mt_seed)

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.orc_state64_free(self.h)
            self.h = None

    def init_random(self):
        lib().orc_state64_init_random(self.h)

    def init_aligned(self, d):
        dd = _arr(d, np.float64)
        lib().orc_state64_init_aligned(self.h, _p(dd))

    def set_spins(self, sx, sy, sz):
        a, b, c = _arr(sx, np.float64), _arr(sy, np.float64), _arr(sz, np.float64)
        lib().orc_state64_set(self.h, _p(a), _p(b), _p(c))

    def get_spins(self):
        n = self.lat.n
        a, b, c = np.zeros(n), np.zeros(n), np.zeros(n)
        lib().orc_state64_get(self.h, _p(a), _p(b), _p(c))
        return a, b, c

    def sweep(self, T, n_sweeps=1):
        lib().orc_state64_sweep(self.h, T, n_sweeps)

    def stats(self):
        a, b = C.c_uint64(), C.c_uint64()
        lib().orc_state64_stats(self.h, C.byref(a), C.byref(b))
        return a.value, b.value

    def measure(self):
        M, E = np.zeros(3), C.c_double()
        lib().orc_state64_measure(self.h, _p(M), C.byref(E))
        return M, E.value

    def series(self, T, n_sweeps):
        m, e, a2 = np.zeros(n_sweeps), np.zeros(n_sweeps), np.zeros(n_sweeps)
        lib().orc_state64_series(self.h, T, n_sweeps, _p(m), _p(e), _p(a2))
        return m, e, a2

    def delta_h(self, site, s_new):
        s = _arr(s_new, np.float64)
        return lib().orc_state64_delta_h(self.h, site, _p(s))


def total_energy64(lat, J, sx, sy, sz):
    a, b, c = _arr(sx, np.float64), _arr(sy, np.float64), _arr(sz, np.float64)
    return lib().orc_total_energy64(lat.h, J, _p(a), _p(b), _p(c))
