"""The C-ABI boundary without a GPU: libhb.so loads, exports every symbol include/hb.h declares,
the binding names the same set, and the host-only entry points (sizes, validation, the sphere
builder, error strings) behave as the header says.  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2106_11286_b200 as hb
from paper_2106_11286_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    """Every function declared in include/*.h (comments stripped)."""
    names = []
    inc = os.path.join(ROOT, "include")
    for fn in sorted(os.listdir(inc)):
        if not fn.endswith(".h"):
            continue
        text = open(os.path.join(inc, fn)).read()
        text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)
        text = re.sub(r"//[^\n]*", " ", text)
        names += re.findall(r"\b(hb_[a-z0-9_]+)\s*\(", text)
    return sorted(set(names))


def test_header_declares_the_three_north_star_calls():
    names = declared_functions()
    for must in ("hb_create", "hb_sweep", "hb_measure"):
        assert must in names


def test_library_exports_every_declared_symbol():
    lib = hb.load_library()
    names = declared_functions()
    assert len(names) >= 20
    for name in names:
        assert hasattr(lib, name), "libhb.so does not export %s" % name
    # the binding marshals exactly the declared set
    assert sorted(binding.EXPORTS) == names


def test_library_has_sm100a_code_only():
    """The kernels are built for sm_100a (no PTX-only or multi-arch fallback)."""
    import shutil
    import subprocess
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(exe):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([exe, "-lelf", binding.library_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_packed_multiplies_are_not_contracted_into_fused_multiply_adds():
    """The arithmetic contract spells out every fused multiply-add.  ptxas 12.9 contracts
    mul.rn.f32x2 + add.rn.f32x2 into one FFMA2 although both carry .rn (hb_device.cuh, add2_prod): one rounding where
    the oracle has two.  Guard: the arithmetic probe holds exactly two packed ANISO_Z attempts per iteration, each with
    13 packed multiplications that must survive as FMUL2, and 24 written fused multiply-adds plus the one fma(prod, 1, c)
    of exp_spec2 that stands for an addition; the warp-specialised and direct sc kernels hold the same two attempts."""
    import shutil
    import subprocess
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(exe):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([exe, "-sass", binding.library_path()], capture_output=True, text=True).stdout
    funcs = {}
    name = None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            funcs[name] = []
        elif name is not None:
            funcs[name].append(line)
    def mix(substr):
        hit = [k for k in funcs if substr in k]
        assert len(hit) == 1, (substr, hit)
        text = "\n".join(funcs[hit[0]])
        return len(re.findall(r"\bFMUL2\b", text)), len(re.findall(r"\bFFMA2\b", text))
    for kernel in ("k_probe_alu", "k_sweep_sc_wsILi7ELi1024ELi4ELi2ELi1ELb0ELb0ELb0ELb0EE", "k_sweep_sc_wsILi7ELi1024ELi4ELi2ELi1ELb0ELb0ELb1ELb0EE", "k_sweep_scILi4ELi1ELb0ELi1ELi256ELb0ELb0E"):
        assert mix(kernel) == (26, 50), (kernel, mix(kernel))


def test_strerror_and_null_arguments():
    lib = hb.load_library()
    assert lib.hb_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4):
        assert lib.hb_strerror(code) not in (b"", b"ok", b"unknown status")
    assert lib.hb_strerror(-99) == b"unknown status"
    assert lib.hb_sizes(None, None, None, None) == -1            # HB_EINVAL
    assert lib.hb_create(None, None, 1.0, 0.0, None, 0, None) == -1
    assert lib.hb_destroy(None) == 0
    assert lib.hb_lattice_free(None) == 0
    assert lib.hb_error_detail(None) == b""


@pytest.mark.parametrize("kind,L,n", [("sc", 16, 4096), ("bcc", 64, 524288), ("fcc", 128, 8388608), ("sc", 464, 99897344)])
def test_sizes_of_the_baseline_configs(kind, L, n):
    got, spins_bytes, ws_bytes = hb.sizes(hb.Lattice(kind, L))
    assert got == n
    assert spins_bytes >= 12 * n and spins_bytes % 256 == 0
    assert ws_bytes > 0 and ws_bytes % 256 == 0


def test_sizes_rejects_bad_lattices():
    for lat in (hb.Lattice("sc", 15), hb.Lattice("sc", 16, 16, 7), hb.Lattice("bcc", 0), hb.Lattice(7, 4)):
        with pytest.raises(hb.HbError) as e:
            hb.sizes(lat)
        assert e.value.status == -1
    # more than 2^32-1 sites cannot be keyed by a 32-bit Philox counter word
    with pytest.raises(hb.HbError):
        hb.sizes(hb.Lattice("fcc", 1100))


def test_table_validation_happens_before_anything_is_sized_or_allocated():
    # a caller-supplied colouring with an absurd colour count, a row_ptr that decreases or does not start at 0
    # must be rejected by hb_sizes / hb_create before any table is sized from them
    rp = np.array([0, 1, 2], np.int64)
    ci = np.array([1, 0], np.int32)
    ok = hb.Lattice("csr", row_ptr=rp, col_idx=ci, colour=np.array([0, 1], np.int32), n_colours=2)
    assert hb.sizes(ok)[0] == 2
    for bad in (hb.Lattice("csr", row_ptr=rp, col_idx=ci, colour=np.array([0, 1], np.int32), n_colours=200),
                hb.Lattice("csr", row_ptr=rp, col_idx=ci, colour=np.array([0, 1], np.int32), n_colours=1 << 30),
                hb.Lattice("csr", row_ptr=rp, col_idx=ci, colour=np.array([0, 1], np.int32), n_colours=0),
                hb.Lattice("csr", row_ptr=np.array([0, 2, 1], np.int64), col_idx=ci),
                hb.Lattice("csr", row_ptr=np.array([1, 2, 3], np.int64), col_idx=ci)):
        with pytest.raises(hb.HbError) as e:
            hb.sizes(bad)
        assert e.value.status == -1


def _create_status(lat):
    """hb_create with library-owned memory, straight through ctypes (no device is needed to be refused)."""
    lib = hb.load_library()
    h = C.c_void_p()
    s = lat.struct()
    rc = lib.hb_create(C.byref(h), C.byref(s), 1.0, 0.0, (C.c_float * 3)(0, 0, 1), 1, None)
    detail = lib.hb_error_detail(h).decode() if h else ""
    lib.hb_destroy(h)
    return rc, detail


def test_symmetry_check_of_hub_graphs():
    # a star with 200 leaves: rows longer than 64 entries take the sort-based symmetry check of validate_csr
    n = 201
    rp = np.concatenate([[0, 200], 200 + np.arange(1, 201)]).astype(np.int64)
    ci = np.concatenate([np.arange(1, 201), np.zeros(200)]).astype(np.int32)
    rc, detail = _create_status(hb.Lattice("csr", row_ptr=rp, col_idx=ci))
    assert rc != -1 or "symmetric" not in detail          # valid table: whatever stops it on a box without a GPU, it is not the table
    bad = ci.copy()
    bad[-1] = 5                                            # leaf 200 points at leaf 5 instead of the hub
    rc, detail = _create_status(hb.Lattice("csr", row_ptr=rp, col_idx=bad))
    assert rc == -1 and "symmetric" in detail


def test_memory_plan_of_table_engines_and_replicas():
    # host logic of hb_sizes: neighbour tables of near-uniform degree take the colour-major ELL layout with AoS float4
    # spins (16 B per site), irregular graphs the plain CSR layout (12 B per site); replicas multiply the state
    from paper_2106_11286_b200 import workloads as W
    sph = hb.Lattice.fcc_sphere(5, 0.05, (0, 0, 1), 0.5)
    n, spins_bytes, _ = hb.sizes(sph)
    assert n == 2123 and spins_bytes == -(-16 * n // 256) * 256
    rp, ci = W.random_csr_graph(5000, 7.0, seed=3)
    n, spins_bytes, _ = hb.sizes(hb.Lattice("csr", row_ptr=rp, col_idx=ci))
    assert n == 5000 and spins_bytes == -(-12 * n // 256) * 256
    per_site = hb.Lattice("bcc", 4, K_site=np.zeros(128, np.float32), e_site=np.tile(np.float32([0, 0, 1]), (128, 1)))
    assert hb.sizes(per_site)[1] == -(-16 * 128 // 256) * 256           # regular degree 8: ELL
    n, one, ws1 = hb.sizes(hb.Lattice("sc", 16))
    n_r, many, ws37 = hb.sizes(hb.Lattice("sc", 16, n_replicas=37))
    assert n_r == n == 4096 and many == 37 * one and ws37 > ws1         # n_sites is per replica
    for bad in (hb.Lattice("sc", 32, n_replicas=2), hb.Lattice("bcc", 4, n_replicas=2), hb.Lattice("sc", 12, n_replicas=2),
                hb.Lattice("sc", 8, n_replicas=5000)):
        with pytest.raises(hb.HbError):
            hb.sizes(bad)


def test_sphere_builder_matches_the_oracles_independent_builder():
    """Host logic of rows a1/a2: the library's fcc-sphere table, anisotropy classes and greedy
    colouring against the oracle's own construction (the two share no code)."""
    import oracle
    for R, colouring in ((2, "greedy"), (5, "greedy"), (5, "parity"), (0, "greedy")):
        g = hb.Lattice.fcc_sphere(R, 0.05, (0, 0, 1), 0.5, colouring)
        o = oracle.Lattice.fcc_sphere(R, 0.05, (0, 0, 1), 0.5, colouring)
        assert g.row_ptr.size - 1 == o.n
        assert np.array_equal(g.row_ptr, o.row_ptr)
        assert np.array_equal(g.col_idx, o.col)
        assert g.n_colours == o.n_colours
        assert np.array_equal(g.colour, o.colour)
        assert np.array_equal(g.K_site.view(np.uint32), o.K.view(np.uint32))
        assert np.array_equal(g.e_site.view(np.uint32).ravel(), o.e.view(np.uint32).ravel())
        assert np.array_equal(g.xyz, o.xyz)


def test_no_cpu_path():
    """Without a CUDA device the product refuses to construct a context (no fallback)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError):
        hb.Context(hb.Lattice("sc", 4))


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2106_11286_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cpp", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), fn
                assert "hb_oracle" not in text, fn
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for fn in files:
            if fn.endswith((".py", ".cpp", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(import|from)\s+paper_2106_11286_b200\b", text, flags=re.M), fn
                assert not re.search(r"#\s*include\s*[\"<][^\">]*(hb\.h|hb_internal\.h|hb_device\.cuh)", text), fn
                assert "libhb.so" not in text, fn


def test_absurd_table_size_is_refused_before_the_table_is_read():
    """A CSR description of 2^40 sites: HB_EINVAL from hb_sizes and hb_create, without walking row_ptr past the caller's array."""
    lib = hb.load_library()
    rp = np.zeros(4, np.int64)
    lat = binding.hb_lattice()
    lat.kind, lat.n_sites = binding.HB_CSR, 2 ** 40
    lat.row_ptr = rp.ctypes.data_as(C.c_void_p)
    n, a, b = C.c_int64(), C.c_size_t(), C.c_size_t()
    assert lib.hb_sizes(C.byref(lat), C.byref(n), C.byref(a), C.byref(b)) == -1
    h = C.c_void_p()
    assert lib.hb_create(C.byref(h), C.byref(lat), 1.0, 0.0, (C.c_float * 3)(0, 0, 1), 1, None) == -1
    assert b"2^32" in lib.hb_error_detail(h)
    lib.hb_destroy(h)


def test_a_failed_host_allocation_comes_back_as_a_status_not_as_an_abort():
    """include/hb.h: nothing throws or aborts.  The host side builds tables in std::vector; with the address space of a child
    process capped, the sphere builder at its largest radius (1.3 x 10^8 sites, gigabytes of tables) runs out of memory and
    must return HB_ENOMEM -- before the entry points caught at the boundary this ended in std::terminate (SIGABRT)."""
    import subprocess
    import sys
    code = (
        "import ctypes as C, resource, sys\n"
        "lib = C.CDLL(%r)\n"
        "resource.setrlimit(resource.RLIMIT_AS, (3 << 29, 3 << 29))\n"       # 1.5 GiB
        "class L(C.Structure):\n"
        "    _fields_ = [('b', C.c_char * 256)]\n"
        "out, xyz = L(), C.c_void_p()\n"
        "lib.hb_lattice_fcc_sphere.argtypes = [C.c_int32, C.c_float, C.POINTER(C.c_float), C.c_float, C.c_int32, C.c_void_p, C.c_void_p]\n"
        "rc = lib.hb_lattice_fcc_sphere(200, 0.0, (C.c_float * 3)(0, 0, 1), 0.0, 1, C.byref(out), C.byref(xyz))\n"
        "print('rc', rc)\n" % binding.library_path())
    res = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, (res.returncode, res.stderr[-400:])
    assert "rc -2" in res.stdout, res.stdout
