"""hb_measure_sc_noalloc (include/hb_noalloc.h): the measurement call for programs that cannot allocate.

Some users of this library are not allowed a cudaMalloc at the point where they need M and E: their process has given
all device memory to one pool and a guest library's allocation would fail or break the budget; or they sit in a loop
where the device-wide stall of cudaMalloc / cudaFree is not acceptable; or they are plug-in code that receives input and
output pointers and has nowhere to keep a context.  For them the library keeps the scratch memory of one measurement
kernel (the block partial sums) in a 256 KiB array compiled into libhb.so, and this file checks that the entry point
built on it returns what the ordinary path (hb_create + hb_measure, scratch in the context's workspace) returns.

What is checked, and why in this shape:
  * the same state measured by both paths agrees within the bars the parity tests use for a measurement
    (|dM| <= 1e-7, |dE| <= 1e-6 N): both compute the same fp32 per-site terms and differ only in the order of the fp64
    additions;
  * TWO calls in a row, the second on a much smaller lattice and then again on the first one after more sweeps: the array
    is shared by all calls and still holds the previous call's partial sums, so a call that read one entry too many, or
    relied on zeros, would show here;
  * the size limit is refused with a message that names the limit (no GPU needed: the check comes before any CUDA call).

The file name sorts last on purpose: `pytest -x` stops at the first failure, so a fault here cannot hide the results of
the parity tests.  It keeps no state between tests and passes alone in a fresh process as well as after all the others.
"""
import ctypes as C

import numpy as np
import pytest

import paper_2106_11286_b200 as hb
from paper_2106_11286_b200 import binding

M_TOL, E_TOL_PER_SITE = 1e-7, 1e-6      # the P2 bars of tests/test_gpu_parity.py::_measure_close


def _both_paths(ctx, dims, J, K, e, out):
    """(M, E) of the context's current state from hb_measure and from the no-alloc call."""
    import torch
    M_ctx, E_ctx = ctx.measure()
    planes = [torch.from_numpy(a).to(out.device) for a in ctx.get_spins()]      # canonical order, on the device
    out.fill_(float("nan"))                                                     # nothing of an earlier result may survive
    hb.measure_sc_noalloc(planes[0], planes[1], planes[2], dims[0], dims[1], dims[2], J, K, e, out)
    torch.cuda.synchronize(out.device)
    got = out.cpu().numpy()
    return M_ctx, E_ctx, got[:3].copy(), float(got[3])


def _assert_same(M_ctx, E_ctx, M_new, E_new, n):
    assert np.all(np.isfinite(M_new)) and np.isfinite(E_new)
    assert np.max(np.abs(M_new - M_ctx)) <= M_TOL, (M_new, M_ctx)
    assert abs(E_new - E_ctx) <= E_TOL_PER_SITE * n, (E_new, E_ctx)


@pytest.mark.gpu
def test_no_alloc_measurement_equals_hb_measure_on_calls_in_a_row():
    import torch
    dev = torch.device("cuda:0")
    J, K, e = 1.0, 0.3, (0.6, 0.0, 0.8)
    big, small = (48, 40, 36), (6, 4, 2)          # 69,120 sites = 16 full blocks of 4096 + a ragged one; 48 sites = part of one block
    out = torch.empty(4, dtype=torch.float64, device=dev)
    ctx_big = hb.Context(hb.Lattice("sc", *big), J, K, e, seed=7, device="cuda:0")
    ctx_small = hb.Context(hb.Lattice("sc", *small), J, K, e, seed=8, device="cuda:0")
    try:
        ctx_big.init_random()
        ctx_big.sweep(0.9, 5)                     # partly ordered: M and E are far from zero
        ctx_small.init_aligned(e)
        ctx_small.sweep(2.5, 3)
        n_big, n_small = ctx_big.n, ctx_small.n
        # call 1: the large lattice fills 17 entries of the shared array
        _assert_same(*_both_paths(ctx_big, big, J, K, e, out), n_big)
        # call 2, straight after: one block; the 16 stale entries behind it must not leak into the sums
        r = _both_paths(ctx_small, small, J, K, e, out)
        _assert_same(*r, n_small)
        assert abs(r[3]) <= 4.0 * n_small           # |E| <= (3 J + |K|) N: a leaked partial of the big lattice would be ~1e5
        # call 3: the large lattice again in a different state
        ctx_big.sweep(0.9, 4)
        r1 = _both_paths(ctx_big, big, J, K, e, out)
        _assert_same(*r1, n_big)
        # and the same state twice gives the same bits (the call has no hidden state)
        r2 = _both_paths(ctx_big, big, J, K, e, out)
        assert np.array_equal(r1[2], r2[2]) and r1[3] == r2[3]
    finally:
        ctx_big.close()
        ctx_small.close()


@pytest.mark.gpu
def test_no_alloc_measurement_on_odd_sizes_against_the_definition():
    """Odd periodic sizes have no context to compare with (the colour sweeps need even ones): eq. 1 and eq. 2 in fp64."""
    import torch
    dev = torch.device("cuda:0")
    Lx, Ly, Lz, J, K = 7, 5, 3, 1.0, -0.2
    e = np.array([0.0, 0.6, 0.8])
    rng = np.random.default_rng(11)
    s = rng.normal(size=(3, Lz, Ly, Lx))
    s = (s / np.linalg.norm(s, axis=0)).astype(np.float32)
    s64 = s.astype(np.float64)
    h = sum(np.roll(s64, sh, axis=ax) for ax in (1, 2, 3) for sh in (1, -1))
    E_def = float(np.sum(-0.5 * J * np.sum(s64 * h, axis=0) - K * np.tensordot(e, s64, axes=1) ** 2))
    M_def = s64.reshape(3, -1).mean(axis=1)
    planes = [torch.from_numpy(np.ascontiguousarray(s[c]).ravel()).to(dev) for c in range(3)]
    out = torch.full((4,), float("nan"), dtype=torch.float64, device=dev)
    hb.measure_sc_noalloc(planes[0], planes[1], planes[2], Lx, Ly, Lz, J, K, e, out)
    torch.cuda.synchronize(dev)
    got = out.cpu().numpy()
    n = Lx * Ly * Lz
    assert np.max(np.abs(got[:3] - M_def)) <= M_TOL
    assert abs(got[3] - E_def) <= E_TOL_PER_SITE * n * 10      # fp32 per-site terms against fp64 ones: a few ulp of 3 J per site


def test_no_alloc_entry_point_refuses_sizes_beyond_its_static_array():
    """Argument checks precede every CUDA call, so this runs without a device: nothing is launched after HB_EINVAL, the
    dummy addresses are never dereferenced."""
    lib = hb.load_library()
    assert binding.NOALLOC_MAX_SITES == 4096 * 8192
    fake = C.c_void_p(256)
    e = (C.c_float * 3)(0.0, 0.0, 1.0)
    err = C.create_string_buffer(512)

    def call(Lx, Ly, Lz, axis=e, buf=err):
        return lib.hb_measure_sc_noalloc(fake, fake, fake, Lx, Ly, Lz, 1.0, 0.0, axis, fake, None, buf, len(buf) if buf else 0)

    assert call(324, 324, 324) == -1                       # HB_EINVAL: 34,012,224 sites > 33,554,432 (322^3 would fit)
    msg = err.value.decode()
    assert "33554432" in msg and "324 x 324 x 324" in msg, msg
    assert call(2 ** 31 - 1, 2 ** 31 - 1, 2 ** 31 - 1) == -1 and "33554432" in err.value.decode()   # no int64 overflow
    assert call(4096, 4096, 3) == -1 and "33554432" in err.value.decode()
    assert call(0, 4, 4) == -1 and ">= 1" in err.value.decode()
    assert call(4, 4, 4, axis=(C.c_float * 3)(0.0, 0.0, 0.5)) == -1 and "unit vector" in err.value.decode()
    assert call(324, 324, 324, buf=None) == -1             # the message buffer is optional
    assert lib.hb_measure_sc_noalloc(None, fake, fake, 4, 4, 4, 1.0, 0.0, e, fake, None, err, len(err)) == -1
    assert "NULL" in err.value.decode()
