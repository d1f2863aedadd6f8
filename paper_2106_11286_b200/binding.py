"""Thin ctypes binding of libhb.so (include/hb.h; diagnostics and options: include/hb_diag.h; the call that never
allocates: include/hb_noalloc.h): argument marshalling only.

Every step of the hot path runs inside the CUDA library.  PyTorch supplies device
memory and the stream.  There is no CPU fallback: if the library is missing or no
CUDA device is present, construction raises.
"""
import ctypes as C
import os

import numpy as np

HB_SC, HB_BCC, HB_FCC, HB_CSR = 0, 1, 2, 3
_KINDS = {"sc": HB_SC, "bcc": HB_BCC, "fcc": HB_FCC, "csr": HB_CSR}

EXPORTS = [
    "hb_sizes", "hb_create", "hb_destroy", "hb_init_random", "hb_init_aligned", "hb_set_spins", "hb_get_spins",
    "hb_stage_spins", "hb_commit_spins",
    "hb_sweep", "hb_measure", "hb_sweep_series", "hb_sweep_record", "hb_sweep_count", "hb_set_sweep_count",
    "hb_sweep_each", "hb_measure_each", "hb_sweep_series_each", "hb_select_replica",
    "hb_slab_pass", "hb_slab_next_sweep", "hb_slab_face", "hb_slab_set_peer", "hb_part_gather", "hb_part_scatter", "hb_probe_alu",
    "hb_device_alloc", "hb_device_free", "hb_ipc_export", "hb_ipc_open", "hb_ipc_close",
    "hb_get_colouring", "hb_counters", "hb_stats", "hb_device_math", "hb_probe_sc_l2", "hb_probe_pipe", "hb_sweep_paper_scheme", "hb_set_option", "hb_get_option", "hb_lattice_fcc_sphere", "hb_lattice_free",
    "hb_strerror", "hb_error_detail",
    "hb_measure_sc_noalloc",     # include/hb_noalloc.h
]


class hb_lattice(C.Structure):
    _fields_ = [("kind", C.c_int32), ("Lx", C.c_int32), ("Ly", C.c_int32), ("Lz", C.c_int32),
                ("n_sites", C.c_int64), ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p),
                ("n_colours", C.c_int32), ("colour", C.c_void_p), ("K_site", C.c_void_p), ("e_site", C.c_void_p),
                ("n_replicas", C.c_int32), ("slab_Lz", C.c_int32), ("slab_z0", C.c_int32),
                ("part_n_total", C.c_int64), ("part_first", C.c_int64), ("part_n_own", C.c_int64)]


class hb_buffers(C.Structure):
    _fields_ = [("spins", C.c_void_p), ("spins_bytes", C.c_size_t), ("workspace", C.c_void_p),
                ("workspace_bytes", C.c_size_t), ("cuda_stream", C.c_void_p)]


class HbError(RuntimeError):
    def __init__(self, status, what, detail=""):
        super().__init__("%s: %s%s" % (what, status, (" (" + detail + ")") if detail else ""))
        self.status = status


_lib = None


def library_path():
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "libhb.so")


def load_library():
    """dlopen libhb.so and declare the prototypes of include/*.h.  Fails loudly if it is not built."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path):
        raise ImportError("libhb.so is not built: run `python -m paper_2106_11286_b200.build` (needs nvcc)")
    L = C.CDLL(path)
    vp, i32, i64, u64, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64, C.c_float
    P = C.POINTER
    protos = {
        "hb_sizes": [P(hb_lattice), P(i64), P(C.c_size_t), P(C.c_size_t)],
        "hb_create": [P(vp), P(hb_lattice), f32, f32, P(f32), u64, P(hb_buffers)],
        "hb_destroy": [vp],
        "hb_init_random": [vp],
        "hb_init_aligned": [vp, P(f32)],
        "hb_set_spins": [vp, vp, vp, vp],
        "hb_get_spins": [vp, vp, vp, vp],
        "hb_stage_spins": [vp, vp, vp, vp],
        "hb_commit_spins": [vp],
        "hb_sweep": [vp, f32, i64],
        "hb_measure": [vp, P(C.c_double), P(C.c_double)],
        "hb_sweep_series": [vp, f32, i64, vp, vp],
        "hb_sweep_record": [vp, f32, vp],
        "hb_sweep_each": [vp, vp, i64],
        "hb_measure_each": [vp, vp, vp],
        "hb_sweep_series_each": [vp, vp, i64, vp, vp],
        "hb_select_replica": [vp, i32],
        "hb_slab_pass": [vp, f32, i32],
        "hb_slab_next_sweep": [vp],
        "hb_slab_face": [vp, i32, i32, i32, P(C.c_size_t), P(C.c_size_t)],
        "hb_slab_set_peer": [vp, i32, vp, i32],
        "hb_part_gather": [vp, vp, i64, vp],
        "hb_part_scatter": [vp, vp, i64, vp],
        "hb_probe_alu": [vp, C.c_double, P(C.c_double)],
        "hb_device_alloc": [C.c_size_t, P(vp)],
        "hb_device_free": [vp],
        "hb_ipc_export": [vp, vp],
        "hb_ipc_open": [vp, P(vp)],
        "hb_ipc_close": [vp],
        "hb_sweep_count": [vp, P(u64)],
        "hb_set_sweep_count": [vp, u64],
        "hb_get_colouring": [vp, vp, P(i32)],
        "hb_counters": [vp, P(u64), P(u64)],
        "hb_stats": [vp, P(u64), P(u64)],
        "hb_device_math": [i32, i64, vp, vp, vp],
        "hb_probe_sc_l2": [vp, f32, i64, i32, P(C.c_double)],
        "hb_probe_pipe": [vp, i32, P(C.c_double)],
        "hb_sweep_paper_scheme": [vp, f32, i64, i32],
        "hb_set_option": [vp, C.c_char_p, i64],
        "hb_get_option": [vp, C.c_char_p, P(i64)],
        "hb_lattice_fcc_sphere": [i32, f32, P(f32), f32, i32, P(hb_lattice), P(vp)],
        "hb_lattice_free": [P(hb_lattice)],
        "hb_measure_sc_noalloc": [vp, vp, vp, i32, i32, i32, f32, f32, P(f32), vp, vp, C.c_char_p, C.c_size_t],
    }
    for name, args in protos.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = C.c_int, args
    L.hb_strerror.restype, L.hb_strerror.argtypes = C.c_char_p, [C.c_int]
    L.hb_error_detail.restype, L.hb_error_detail.argtypes = C.c_char_p, [vp]
    _lib = L
    return L


def _vec3(v):
    return (C.c_float * 3)(*[float(x) for x in v])


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


class Lattice:
    """Host description of a lattice (the hb_lattice struct plus the arrays it points to)."""

    def __init__(self, kind, Lx=0, Ly=0, Lz=0, row_ptr=None, col_idx=None, colour=None, n_colours=0,
                 K_site=None, e_site=None, xyz=None, n_replicas=1, slab=None, part=None):
        self.kind = _KINDS[kind] if isinstance(kind, str) else int(kind)
        self.Lx, self.Ly, self.Lz = int(Lx), int(Ly or Lx), int(Lz or Lx)
        self.row_ptr = _np(row_ptr, np.int64) if row_ptr is not None else None
        self.col_idx = _np(col_idx, np.int32) if col_idx is not None else None
        self.colour = _np(colour, np.int32) if colour is not None else None
        self.n_colours = int(n_colours)
        self.K_site = _np(K_site, np.float32) if K_site is not None else None
        self.e_site = _np(e_site, np.float32) if e_site is not None else None
        self.xyz = xyz
        self.n_replicas = int(n_replicas)
        # slab = (z0, Lz_global): this lattice is planes z0 .. z0 + Lz - 1 of a periodic sc lattice Lx x Ly x Lz_global
        self.slab = (int(slab[0]), int(slab[1])) if slab is not None else None
        # part = (first, n_own, n_total): local sites 0 .. n_own-1 are sites first .. of a table of n_total sites, the rest ghosts
        self.part = tuple(int(v) for v in part) if part is not None else None

    @classmethod
    def fcc_sphere(cls, R, K_core=0.0, e_core=(0, 0, 1), K_surf=0.0, colouring="greedy"):
        """hb_lattice_fcc_sphere: the library's own builder (A10-A12)."""
        L = load_library()
        out, xyz = hb_lattice(), C.c_void_p()
        rc = L.hb_lattice_fcc_sphere(R, K_core, _vec3(e_core), K_surf, {"greedy": 0, "parity": 1}[colouring],
                                     C.byref(out), C.byref(xyz))
        if rc != 0:
            raise HbError(rc, "hb_lattice_fcc_sphere", L.hb_strerror(rc).decode())
        n = out.n_sites

        def take(ptr, count, ctype, dt):
            return np.ctypeslib.as_array(C.cast(ptr, C.POINTER(ctype)), shape=(count,)).astype(dt, copy=True)

        rp = take(out.row_ptr, n + 1, C.c_int64, np.int64)
        lat = cls("csr", row_ptr=rp, col_idx=take(out.col_idx, max(int(rp[-1]), 1), C.c_int32, np.int32)[:int(rp[-1])],
                  colour=take(out.colour, n, C.c_int32, np.int32), n_colours=out.n_colours,
                  K_site=take(out.K_site, n, C.c_float, np.float32),
                  e_site=take(out.e_site, 3 * n, C.c_float, np.float32).reshape(n, 3),
                  xyz=take(xyz, 3 * n, C.c_int32, np.int32).reshape(n, 3))
        L.hb_lattice_free(C.byref(out))
        C.CDLL(None).free(xyz)
        return lat

    def struct(self):
        s = hb_lattice()
        s.kind, s.Lx, s.Ly, s.Lz = self.kind, self.Lx, self.Ly, self.Lz
        s.n_replicas = self.n_replicas
        if self.slab is not None:
            s.slab_z0, s.slab_Lz = self.slab
        if self.part is not None:
            s.part_first, s.part_n_own, s.part_n_total = self.part
        if self.row_ptr is not None:
            s.n_sites = self.row_ptr.size - 1
            s.row_ptr = _ptr(self.row_ptr)
            s.col_idx = _ptr(self.col_idx) if self.col_idx is not None and self.col_idx.size else None
        if self.colour is not None:
            s.colour, s.n_colours = _ptr(self.colour), self.n_colours
        if self.K_site is not None:
            s.K_site, s.e_site = _ptr(self.K_site), _ptr(self.e_site)
        return s


def probe_alu(seconds=0.5, device="cuda:0"):
    """hb_probe_alu: attempted updates per second of the attempt arithmetic alone (no memory traffic) on `device`."""
    import torch
    L = load_library()
    torch.cuda.set_device(torch.device(device))
    v = C.c_double()
    rc = L.hb_probe_alu(torch.cuda.current_stream(torch.device(device)).cuda_stream, float(seconds), C.byref(v))
    if rc != 0:
        raise HbError(rc, "hb_probe_alu", L.hb_strerror(rc).decode())
    return v.value


MATH_OPS = {"u01": (0, 2, 0), "sincos": (1, 2, 0), "sphere": (2, 6, 1), "exp": (3, 2, 0), "sqrt": (4, 2, 0), "attempt": (5, 4, 16)}


def device_math(op, in0, in1=None, device="cuda:0"):
    """hb_device_math: the device's building blocks of an attempt, element by element (include/hb_diag.h).
    Returns a float32 array of shape (count, floats per element)."""
    import torch
    L = load_library()
    torch.cuda.set_device(torch.device(device))
    code, per_out, per_in1 = MATH_OPS[op]
    a = _np(in0, np.uint32).ravel()
    b = _np(in1, np.uint32).ravel() if in1 is not None else None
    assert (b is None) == (per_in1 == 0) and (b is None or b.size == per_in1 * a.size)
    out = np.zeros((a.size, per_out), np.float32)
    rc = L.hb_device_math(code, a.size, _ptr(a), _ptr(b) if b is not None else None, _ptr(out))
    if rc != 0:
        raise HbError(rc, "hb_device_math", L.hb_strerror(rc).decode())
    return out


PIPE_KINDS = ["FFMA", "FFMA2", "IMAD", "IMAD.WIDE", "LOP3", "IMAD.WIDE+LOP3", "FFMA+IMAD.WIDE+LOP3", "FFMA2+IMAD.WIDE+LOP3"]


def probe_pipe(kind, device="cuda:0"):
    """hb_probe_pipe: warp-instructions per clock per SM of one instruction kind or mix (index into PIPE_KINDS)."""
    import torch
    L = load_library()
    torch.cuda.set_device(torch.device(device))
    v = C.c_double()
    rc = L.hb_probe_pipe(torch.cuda.current_stream(torch.device(device)).cuda_stream, int(kind), C.byref(v))
    if rc != 0:
        raise HbError(rc, "hb_probe_pipe", L.hb_strerror(rc).decode())
    return v.value


NOALLOC_MAX_SITES = 4096 * 8192     # HB_NOALLOC_MAX_SITES of include/hb_noalloc.h


def measure_sc_noalloc(sx, sy, sz, Lx, Ly, Lz, J, K, e, out, stream=None):
    """hb_measure_sc_noalloc (include/hb_noalloc.h): M and E of a periodic simple cubic lattice from three CUDA float32
    tensors in canonical site order, written into `out`, a CUDA float64 tensor of 4 elements (Mx, My, Mz, E), on `stream`
    (default: torch's current stream of that device), without synchronising.

    This is the call for code that must not allocate device memory where it runs: the library side neither calls
    cudaMalloc nor needs a Context or a workspace, because its partial sums live in a 256 KiB array built into
    libhb.so.  The wrapper keeps to that too: it allocates no tensor, the caller brings `out`.  The first call on
    a device looks up that array's address, so make it during start-up.  All calls on one GPU share the array: keep
    them on one stream.  Lattices of more than NOALLOC_MAX_SITES sites raise HbError with the limit in the message."""
    import torch
    L = load_library()
    n = int(Lx) * int(Ly) * int(Lz)
    for t in (sx, sy, sz):
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.numel() == n and t.device == out.device
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 4
    if stream is None:
        stream = torch.cuda.current_stream(out.device)
    err = C.create_string_buffer(512)
    with torch.cuda.device(out.device):
        rc = L.hb_measure_sc_noalloc(sx.data_ptr(), sy.data_ptr(), sz.data_ptr(), int(Lx), int(Ly), int(Lz), float(J), float(K),
                                     _vec3(e), out.data_ptr(), stream.cuda_stream, err, len(err))
    if rc != 0:
        raise HbError(rc, "hb_measure_sc_noalloc", err.value.decode() or L.hb_strerror(rc).decode())
    return out


def sizes(lat):
    """hb_sizes -> (n_sites, spins_bytes, workspace_bytes)."""
    L = load_library()
    n, a, b = C.c_int64(), C.c_size_t(), C.c_size_t()
    s = lat.struct()
    rc = L.hb_sizes(C.byref(s), C.byref(n), C.byref(a), C.byref(b))
    if rc != 0:
        raise HbError(rc, "hb_sizes", L.hb_strerror(rc).decode())
    return n.value, a.value, b.value


class Context:
    """hb_ctx with torch-owned device memory.  Method names follow include/hb.h."""

    def __init__(self, lat, J=1.0, K=0.0, e=(0.0, 0.0, 1.0), seed=1, device="cuda:0", stream=None, ipc=False):
        """ipc=True: the spins buffer comes from hb_device_alloc (a plain cudaMalloc) instead of torch's caching allocator, so
        that another process can map it (ipc_handle / open_ipc; peer stores between slabs of different processes)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2106_11286_b200 needs a CUDA device; there is no CPU path")
        self._L = load_library()
        self.lat = lat
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.n, spins_bytes, ws_bytes = sizes(lat)      # n: sites of ONE replica
        self.n_replicas = max(1, lat.n_replicas)
        self._raw = None
        if ipc:
            raw = C.c_void_p()
            rc = self._L.hb_device_alloc(spins_bytes, C.byref(raw))
            if rc != 0:
                raise HbError(rc, "hb_device_alloc", self._L.hb_strerror(rc).decode())
            self._raw = raw

            class _View:      # torch maps foreign device memory through the CUDA array interface, without a copy
                __cuda_array_interface__ = {"shape": (spins_bytes,), "typestr": "|u1", "data": (raw.value, False), "version": 2}
            self._spins = torch.as_tensor(_View(), device=self.device)
        else:
            self._spins = torch.empty(spins_bytes, dtype=torch.uint8, device=self.device)
        self._ws = torch.empty(ws_bytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        bufs = hb_buffers(self._spins.data_ptr(), spins_bytes, self._ws.data_ptr(), ws_bytes, self.stream.cuda_stream)
        s = lat.struct()
        h = C.c_void_p()
        rc = self._L.hb_create(C.byref(h), C.byref(s), J, K, _vec3(e), seed, C.byref(bufs))
        self._h = h
        if rc != 0:
            detail = self._L.hb_error_detail(h).decode() if h else ""
            self._L.hb_destroy(h)
            self._h = None
            raise HbError(rc, "hb_create", detail or self._L.hb_strerror(rc).decode())

    def _check(self, rc, what):
        if rc != 0:
            raise HbError(rc, what, self._L.hb_error_detail(self._h).decode() or self._L.hb_strerror(rc).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.hb_destroy(self._h)
            self._h = None
        if getattr(self, "_raw", None):
            import torch
            torch.cuda.synchronize(self.device)
            self._spins = None
            self._L.hb_device_free(self._raw)
            self._raw = None

    def ipc_handle(self):
        """64-byte CUDA IPC handle of the spins buffer (Context(..., ipc=True))."""
        if not self._raw:
            raise RuntimeError("ipc_handle needs Context(..., ipc=True)")
        h = (C.c_ubyte * 64)()
        self._check(self._L.hb_ipc_export(self._raw, h), "hb_ipc_export")
        return bytes(h)

    def open_ipc(self, handle):
        """Map another process's spins buffer; returns its device address here (for slab_set_peer)."""
        h = (C.c_ubyte * 64).from_buffer_copy(handle)
        p = C.c_void_p()
        self._check(self._L.hb_ipc_open(h, C.byref(p)), "hb_ipc_open")
        return p.value

    def close_ipc(self, ptr):
        self._L.hb_ipc_close(C.c_void_p(ptr))

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init_random(self):
        self._check(self._L.hb_init_random(self._h), "hb_init_random")

    def init_aligned(self, direction):
        self._check(self._L.hb_init_aligned(self._h, _vec3(direction)), "hb_init_aligned")

    def set_spins(self, sx, sy, sz):
        """Host arrays (numpy, or pinned torch CPU tensors) of n floats, canonical order."""
        p = [self._host_ptr(a) for a in (sx, sy, sz)]
        self._check(self._L.hb_set_spins(self._h, p[0][0], p[1][0], p[2][0]), "hb_set_spins")

    def stage_spins(self, sx, sy, sz):
        """hb_stage_spins: start the upload of the next state (pinned torch CPU tensors) while the stream computes."""
        p = [self._host_ptr(a) for a in (sx, sy, sz)]
        self._check(self._L.hb_stage_spins(self._h, p[0][0], p[1][0], p[2][0]), "hb_stage_spins")   # HB_ESTATE if one is pending
        self._staged = [q[1] for q in p]          # keep the host arrays alive until the commit

    def commit_spins(self):
        self._check(self._L.hb_commit_spins(self._h), "hb_commit_spins")
        self._staged = None

    def _host_ptr(self, a):
        if isinstance(a, np.ndarray):
            b = _np(a, np.float32)
            assert b.size == self.n
            return C.c_void_p(b.ctypes.data), b
        assert a.device.type == "cpu" and a.is_contiguous() and a.numel() == self.n and a.element_size() == 4
        return C.c_void_p(a.data_ptr()), a

    def get_spins(self, out=None):
        if out is None:
            out = [np.empty(self.n, np.float32) for _ in range(3)]
        p = [self._host_ptr(a) for a in out]
        self._check(self._L.hb_get_spins(self._h, p[0][0], p[1][0], p[2][0]), "hb_get_spins")
        return out

    def sweep(self, T, n_sweeps=1):
        self._check(self._L.hb_sweep(self._h, T, n_sweeps), "hb_sweep")

    def measure(self):
        M, E = (C.c_double * 3)(), C.c_double()
        self._check(self._L.hb_measure(self._h, M, C.byref(E)), "hb_measure")
        return np.array(M[:]), E.value

    def sweep_series(self, T, n_sweeps):
        M, E = np.zeros((n_sweeps, 3)), np.zeros(n_sweeps)
        self._check(self._L.hb_sweep_series(self._h, T, n_sweeps, _ptr(M), _ptr(E)), "hb_sweep_series")
        return M, E

    # ---- replicas (Lattice(..., n_replicas=R)): one launch runs all of them, each at its own temperature ----------
    def select_replica(self, r):
        self._check(self._L.hb_select_replica(self._h, int(r)), "hb_select_replica")

    def sweep_each(self, T, n_sweeps=1):
        t = _np(T, np.float32)
        assert t.size == self.n_replicas
        self._check(self._L.hb_sweep_each(self._h, _ptr(t), n_sweeps), "hb_sweep_each")

    def measure_each(self):
        M, E = np.zeros((self.n_replicas, 3)), np.zeros(self.n_replicas)
        self._check(self._L.hb_measure_each(self._h, _ptr(M), _ptr(E)), "hb_measure_each")
        return M, E

    def sweep_series_each(self, T, n_sweeps):
        t = _np(T, np.float32)
        assert t.size == self.n_replicas
        M, E = np.zeros((self.n_replicas, n_sweeps, 3)), np.zeros((self.n_replicas, n_sweeps))
        self._check(self._L.hb_sweep_series_each(self._h, _ptr(t), n_sweeps, _ptr(M), _ptr(E)), "hb_sweep_series_each")
        return M, E

    # ---- slabs (Lattice("sc", Lx, Ly, Lz, slab=(z0, Lz_global))); paper_2106_11286_b200.slabs drives them --------
    def slab_pass(self, T, colour):
        self._check(self._L.hb_slab_pass(self._h, T, int(colour)), "hb_slab_pass")

    def slab_next_sweep(self):
        self._check(self._L.hb_slab_next_sweep(self._h), "hb_slab_next_sweep")

    def slab_face(self, colour, side, ghost):
        """The three component runs (torch float32 views of the spins buffer) of one face of one colour: side 0 = low z,
        1 = high z; ghost False = the slab's own boundary plane, True = the ghost plane beyond it."""
        import torch
        off, cnt = (C.c_size_t * 3)(), C.c_size_t()
        self._check(self._L.hb_slab_face(self._h, int(colour), int(side), int(bool(ghost)), off, C.byref(cnt)), "hb_slab_face")
        f = self._spins.view(torch.float32)
        return [f[off[k]:off[k] + cnt.value] for k in range(3)]

    def slab_set_peer(self, side, peer_spins_ptr, peer_Lz):
        """Peer stores for one side (include/hb.h): peer_spins_ptr = device address of the z-neighbour's spins buffer."""
        self._check(self._L.hb_slab_set_peer(self._h, int(side), C.c_void_p(peer_spins_ptr), int(peer_Lz)), "hb_slab_set_peer")

    # ---- parts of a neighbour table (Lattice("csr", ..., part=(first, n_own, n_total))); paper_2106_11286_b200.parts drives them ----
    def part_gather(self, ids, out):
        """hb_part_gather: spins of the local sites ids (torch int32, device) -> out (torch float32, device, 4 floats per site)."""
        assert ids.is_cuda and out.is_cuda and out.numel() >= 4 * ids.numel()
        self._check(self._L.hb_part_gather(self._h, C.c_void_p(ids.data_ptr()), ids.numel(), C.c_void_p(out.data_ptr())), "hb_part_gather")

    def part_scatter(self, ids, src):
        """hb_part_scatter: src (4 floats per site) -> spins of the local sites ids."""
        assert ids.is_cuda and src.is_cuda and src.numel() >= 4 * ids.numel()
        self._check(self._L.hb_part_scatter(self._h, C.c_void_p(ids.data_ptr()), ids.numel(), C.c_void_p(src.data_ptr())), "hb_part_scatter")

    @property
    def spins_ptr(self):
        return self._spins.data_ptr()

    def sweep_record(self, T):
        acc = np.zeros(self.n, np.uint8)
        self._check(self._L.hb_sweep_record(self._h, T, _ptr(acc)), "hb_sweep_record")
        return acc

    @property
    def sweep_count(self):
        v = C.c_uint64()
        self._check(self._L.hb_sweep_count(self._h, C.byref(v)), "hb_sweep_count")
        return v.value

    @sweep_count.setter
    def sweep_count(self, value):
        self._check(self._L.hb_set_sweep_count(self._h, value), "hb_set_sweep_count")

    def colouring(self):
        col, nc = np.zeros(self.n, np.int32), C.c_int32()
        self._check(self._L.hb_get_colouring(self._h, _ptr(col), C.byref(nc)), "hb_get_colouring")
        return col, nc.value

    def counters(self):
        a, b = C.c_uint64(), C.c_uint64()
        self._check(self._L.hb_counters(self._h, C.byref(a), C.byref(b)), "hb_counters")
        return a.value, b.value

    def stats(self):
        """hb_stats -> (attempts, accepts) of the counted sweeps (include/hb.h)."""
        a, b = C.c_uint64(), C.c_uint64()
        self._check(self._L.hb_stats(self._h, C.byref(a), C.byref(b)), "hb_stats")
        return a.value, b.value

    def sweep_paper_scheme(self, T, n_mcs=1, n_per_block=8):
        """hb_sweep_paper_scheme: the paper's own racy block scheme, emulated (context only; include/hb_diag.h)."""
        self._check(self._L.hb_sweep_paper_scheme(self._h, T, int(n_mcs), int(n_per_block)), "hb_sweep_paper_scheme")

    def probe_sc_l2(self, T, n_sweeps=50, planes=16):
        """hb_probe_sc_l2: updates per second of the sc colour kernel with its HBM traffic folded into L2 (destroys the state)."""
        v = C.c_double()
        self._check(self._L.hb_probe_sc_l2(self._h, T, int(n_sweeps), int(planes), C.byref(v)), "hb_probe_sc_l2")
        return v.value

    def set_option(self, name, value):
        self._check(self._L.hb_set_option(self._h, name.encode(), int(value)), "hb_set_option(%s)" % name)

    def get_option(self, name):
        v = C.c_int64()
        self._check(self._L.hb_get_option(self._h, name.encode(), C.byref(v)), "hb_get_option(%s)" % name)
        return v.value
