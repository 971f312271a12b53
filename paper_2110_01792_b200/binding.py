"""Thin ctypes binding of libqk.so (include/qk.h): same names, argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used here to hold the
device allocation (qk_bind_storage) and the stream (qk_set_stream).  There is no CPU path: if
the library is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqk.so")

NG = 4
FIELDS = ["rho", "mx", "my", "mz", "E", "Er", "Fx", "Fy", "Fz", "kappaP", "kappaR", "src"]
QK_OK, QK_EINVAL, QK_ENOMEM, QK_ECUDA, QK_ENEWTON, QK_ESTATE = range(6)
QK_BC_PERIODIC, QK_BC_OUTFLOW, QK_BC_REFLECTING, QK_BC_FIXED = 0, 1, 2, 3
QK_FLAG_TAU_CORR, QK_FLAG_STATIC_MATTER, QK_FLAG_NEWTON_LITERAL = 1, 2, 4
QK_FLAG_PLM, QK_FLAG_EDDINGTON, QK_FLAG_MINERBO = 8, 16, 32
QK_FILL_HYDRO, QK_FILL_RAD, QK_FILL_OPACITY, QK_FILL_ALL = 1, 2, 4, 7

EXPORTS = [
    "qk_init", "qk_free", "qk_state_bytes", "qk_bind_storage", "qk_set_stream", "qk_set_constants",
    "qk_set_params", "qk_set_state", "qk_get_state", "qk_set_raw", "qk_get_raw", "qk_fill_boundary",
    "qk_cfl_dt", "qk_hydro_step", "qk_rad_transport", "qk_exchange", "qk_rad_step", "qk_rhd_step",
    "qk_nsub_for", "qk_last_info", "qk_launch_count", "qk_set_profiling", "qk_set_flatten_path",
    "qk_kernel_class_count", "qk_kernel_class_name", "qk_kernel_times", "qk_version", "qk_fp64_probe",
    "qk_selftest_divsqrt", "qk_set_eos", "qk_set_opacity_law", "qk_set_opacity_law_T", "qk_set_face_boundaries",
    "qk_hydro_step_cfl", "qk_rhd_step_cfl", "qk_last_dt", "qk_set_halo_exchange", "qk_halo_doubles", "qk_halo_pack",
    "qk_halo_unpack", "qk_set_state_all", "qk_get_state_all", "qk_wait_copies", "qk_halo_export", "qk_set_halo_peers",
    "qk_noalloc_setup", "qk_noalloc_max_cells", "qk_cfl_dt_noalloc",
    "qk_graph_capture", "qk_graph_launch", "qk_graph_free",
]


class qk_info(C.Structure):
    _fields_ = [("nsub", C.c_int), ("newton_max_iters", C.c_int), ("newton_fail_cells", C.c_longlong),
                ("newton_total_iters", C.c_longlong), ("bad_state_cells", C.c_longlong),
                ("fallback_states", C.c_longlong), ("guard_faces", C.c_longlong), ("status", C.c_int)]


class qk_halo_handle(C.Structure):
    _fields_ = [("ipc", C.c_ubyte * 64), ("base", C.c_ulonglong), ("offset", C.c_ulonglong), ("pid", C.c_longlong),
                ("device", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("has_ipc", C.c_int)]


QK_FACE_ZLO, QK_FACE_ZHI = 1, 2
QK_EOS_IDEAL, QK_EOS_ALPHA_T3 = 0, 1
QK_GRAPH_HYDRO, QK_GRAPH_RHD = 0, 1
HALO_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int)


class QkError(RuntimeError):
    pass


_lib = None


def lib():
    """Load libqk.so (built in-tree by paper_2110_01792_b200.build).  Raises if it is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise QkError("libqk.so is not built: run `python -m paper_2110_01792_b200.build` "
                      "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    i, d, p, u, ll = C.c_int, C.c_double, C.c_void_p, C.c_uint, C.c_longlong
    sig = {
        "qk_init": (i, [i, i, i, d, d, d, d, i, C.POINTER(p)]),
        "qk_free": (i, [p]),
        "qk_state_bytes": (C.c_size_t, [i, i, i]),
        "qk_bind_storage": (i, [p, p, C.c_size_t]),
        "qk_set_stream": (i, [p, p]),
        "qk_set_constants": (i, [p, d, d]),
        "qk_set_params": (i, [p, d, d, i, i, u]),
        "qk_set_eos": (i, [p, i, d]),
        "qk_set_opacity_law": (i, [p, d, d, d, i]),
        "qk_set_opacity_law_T": (i, [p, d, d, d, i, d, i]),
        "qk_set_face_boundaries": (i, [p, C.POINTER(C.c_int)]),
        "qk_set_state": (i, [p, i, p]),
        "qk_get_state": (i, [p, i, p]),
        "qk_set_state_all": (i, [p, i, C.POINTER(i), C.POINTER(p)]),
        "qk_get_state_all": (i, [p, i, C.POINTER(i), C.POINTER(p)]),
        "qk_wait_copies": (i, [p]),
        "qk_set_raw": (i, [p, i, p]),
        "qk_get_raw": (i, [p, i, p]),
        "qk_fill_boundary": (i, [p, i]),
        "qk_cfl_dt": (d, [p]),
        "qk_hydro_step": (i, [p, d]),
        "qk_hydro_step_cfl": (i, [p]),
        "qk_rhd_step_cfl": (i, [p, i]),
        "qk_last_dt": (i, [p, C.POINTER(d)]),
        "qk_graph_capture": (i, [p, i, i]),
        "qk_graph_launch": (i, [p, i]),
        "qk_graph_free": (i, [p]),
        "qk_rad_transport": (i, [p, d]),
        "qk_exchange": (i, [p, d]),
        "qk_rad_step": (i, [p, d]),
        "qk_rhd_step": (i, [p, d]),
        "qk_nsub_for": (i, [p, d]),
        "qk_last_info": (i, [p, C.POINTER(qk_info)]),
        "qk_launch_count": (ll, [p]),
        "qk_set_profiling": (i, [p, i]),
        "qk_set_flatten_path": (i, [p, i]),
        "qk_kernel_class_count": (i, []),
        "qk_kernel_class_name": (C.c_char_p, [i]),
        "qk_kernel_times": (i, [p, C.POINTER(d), C.POINTER(ll)]),
        "qk_version": (C.c_char_p, []),
        "qk_fp64_probe": (i, [i, i, p, C.POINTER(d)]),
        "qk_noalloc_setup": (i, []),
        "qk_noalloc_max_cells": (ll, []),
        "qk_cfl_dt_noalloc": (i, [p, p, p, p, p, ll, d, d, d, p, p]),
        "qk_selftest_divsqrt": (i, [ll, C.c_ulonglong, i, p, C.POINTER(ll)]),
        "qk_set_halo_exchange": (i, [p, u, HALO_FN, p]),
        "qk_halo_doubles": (C.c_size_t, [p]),
        "qk_halo_pack": (i, [p, i, p]),
        "qk_halo_unpack": (i, [p, i, p]),
        "qk_halo_export": (i, [p, C.POINTER(qk_halo_handle)]),
        "qk_set_halo_peers": (i, [p, C.POINTER(qk_halo_handle), C.POINTER(qk_halo_handle)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


def qk_fp64_probe(kind=0, iters=20000):
    """fp64 instructions x lanes per second of the fp64 pipe (see include/qk.h)."""
    import torch
    out = C.c_double()
    _check(lib().qk_fp64_probe(kind, iters, C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(out)),
           "qk_fp64_probe")
    return float(out.value)


def qk_noalloc_setup():
    _check(lib().qk_noalloc_setup(), "qk_noalloc_setup")


def qk_noalloc_max_cells():
    return int(lib().qk_noalloc_max_cells())


def qk_cfl_dt_noalloc(rho, mx, my, mz, E, ncells, gamma, cfl, dx, dt_out, stream=None):
    """Allocation-free eq 21 timestep (include/qk.h).  rho..E, dt_out: DEVICE addresses (ints); dt_out receives one
    double.  Asynchronous on `stream` (a raw cudaStream_t; default: torch's current stream)."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    rc = lib().qk_cfl_dt_noalloc(C.c_void_p(rho), C.c_void_p(mx), C.c_void_p(my), C.c_void_p(mz), C.c_void_p(E),
                                 int(ncells), float(gamma), float(cfl), float(dx), C.c_void_p(stream), C.c_void_p(dt_out))
    if rc == QK_ENOMEM:
        raise QkError("qk_cfl_dt_noalloc: %d cells exceed the fixed scratch's limit of %d" % (ncells, qk_noalloc_max_cells()))
    _check(rc, "qk_cfl_dt_noalloc")


def qk_selftest_divsqrt(n, seed=1, exponent_span=2046):
    """(div accepted, div mismatches, sqrt accepted, sqrt mismatches) -- see include/qk.h."""
    import torch
    out = (C.c_longlong * 4)()
    _check(lib().qk_selftest_divsqrt(n, seed, exponent_span, C.c_void_p(torch.cuda.current_stream().cuda_stream), out),
           "qk_selftest_divsqrt")
    return tuple(int(v) for v in out)


def _check(rc, what):
    if rc != QK_OK:
        names = {1: "QK_EINVAL", 2: "QK_ENOMEM", 3: "QK_ECUDA", 4: "QK_ENEWTON", 5: "QK_ESTATE"}
        raise QkError("%s failed: %s" % (what, names.get(rc, rc)))


def _ptr(a):
    """Address of a numpy array (host) or torch tensor (host or device), C-contiguous float64."""
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
        return C.c_void_p(a.ctypes.data)
    assert a.dtype.is_floating_point and a.element_size() == 8 and a.is_contiguous()
    return C.c_void_p(a.data_ptr())


class Context:
    """One box on the current CUDA device.  Methods are the C entry points, name for name."""

    def __init__(self, nx, ny, nz, dx, gamma, c_hat=0.0, c=0.0, boundary=QK_BC_PERIODIC, device="cuda:0",
                 torch_storage=True):
        import torch
        if not torch.cuda.is_available():
            raise QkError("no CUDA device: this library has no CPU path")
        self.L = lib()
        self.nx, self.ny, self.nz = nx, ny, nz
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        h = C.c_void_p()
        _check(self.L.qk_init(nx, ny, nz, dx, gamma, c_hat, c, boundary, C.byref(h)), "qk_init")
        self.h = h
        self.storage = None
        if torch_storage:   # PyTorch owns the device memory
            nbytes = self.L.qk_state_bytes(nx, ny, nz)
            self.storage = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.storage.data_ptr()
            aligned = (base + 255) // 256 * 256
            _check(self.L.qk_bind_storage(self.h, C.c_void_p(aligned), nbytes), "qk_bind_storage")
        self.qk_set_stream(torch.cuda.current_stream(self.device).cuda_stream)

    def close(self):
        if getattr(self, "h", None):
            self.L.qk_free(self.h)
            self.h = None
            self.storage = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # ---- one method per C entry point -----------------------------------------------------------
    def qk_set_stream(self, cuda_stream):
        _check(self.L.qk_set_stream(self.h, C.c_void_p(cuda_stream)), "qk_set_stream")
        self.stream_ptr = int(cuda_stream)

    def qk_set_constants(self, a_rad, kB_over_mu_mH):
        _check(self.L.qk_set_constants(self.h, a_rad, kB_over_mu_mH), "qk_set_constants")

    def qk_set_params(self, cfl=0.3, newton_tol=1e-10, newton_maxit=400, nsub_max=10, flags=0):
        _check(self.L.qk_set_params(self.h, cfl, newton_tol, newton_maxit, nsub_max, flags), "qk_set_params")

    def qk_set_face_boundaries(self, bc6):
        arr = (C.c_int * 6)(*[int(b) for b in bc6])
        _check(self.L.qk_set_face_boundaries(self.h, arr), "qk_set_face_boundaries")

    def qk_set_opacity_law(self, kappaP0, kappaR0, rho0, exponent):
        _check(self.L.qk_set_opacity_law(self.h, kappaP0, kappaR0, rho0, exponent), "qk_set_opacity_law")

    def qk_set_eos(self, eos, alpha=0.0):
        _check(self.L.qk_set_eos(self.h, eos, alpha), "qk_set_eos")

    def qk_set_opacity_law_T(self, kappaP0, kappaR0, rho0, exponent, T0, texp2):
        _check(self.L.qk_set_opacity_law_T(self.h, kappaP0, kappaR0, rho0, exponent, T0, texp2), "qk_set_opacity_law_T")

    def qk_set_state(self, field, a):
        assert tuple(a.shape) == (self.nz, self.ny, self.nx), tuple(a.shape)
        _check(self.L.qk_set_state(self.h, field, _ptr(a)), "qk_set_state")

    def qk_get_state(self, field, out=None):
        if out is None:
            out = np.empty((self.nz, self.ny, self.nx), dtype=np.float64)
        assert tuple(out.shape) == (self.nz, self.ny, self.nx)
        _check(self.L.qk_get_state(self.h, field, _ptr(out)), "qk_get_state")
        return out

    def _field_list(self, fields, arrays):
        n = len(fields)
        for a in arrays:
            assert tuple(a.shape) == (self.nz, self.ny, self.nx), tuple(a.shape)
        return n, (C.c_int * n)(*[int(f) for f in fields]), (C.c_void_p * n)(*[_ptr(a) for a in arrays])

    def qk_set_state_all(self, fields, arrays):
        """Asynchronous upload of several fields (see include/qk.h); keep `arrays` alive until qk_wait_copies."""
        n, f, p = self._field_list(fields, arrays)
        _check(self.L.qk_set_state_all(self.h, n, f, p), "qk_set_state_all")

    def qk_get_state_all(self, fields, arrays):
        n, f, p = self._field_list(fields, arrays)
        _check(self.L.qk_get_state_all(self.h, n, f, p), "qk_get_state_all")

    def qk_wait_copies(self):
        _check(self.L.qk_wait_copies(self.h), "qk_wait_copies")

    def qk_set_raw(self, field, a):
        assert tuple(a.shape) == (self.nz + 2 * NG, self.ny + 2 * NG, self.nx + 2 * NG)
        _check(self.L.qk_set_raw(self.h, field, _ptr(a)), "qk_set_raw")

    def qk_get_raw(self, field, out=None):
        if out is None:
            out = np.empty((self.nz + 2 * NG, self.ny + 2 * NG, self.nx + 2 * NG), dtype=np.float64)
        _check(self.L.qk_get_raw(self.h, field, _ptr(out)), "qk_get_raw")
        return out

    def qk_set_halo_exchange(self, faces, fn):
        """fn(nfields) is called before every ghost fill (see include/qk.h); None switches it off."""
        if fn is None or not faces:
            self._halo_cb = None
            _check(self.L.qk_set_halo_exchange(self.h, 0, C.cast(None, HALO_FN), None), "qk_set_halo_exchange")
            return
        def thunk(user, nfields):          # the callback's status aborts the step (a Python exception counts as failure)
            try:
                rc = fn(nfields)
                return 0 if rc is None else int(rc)
            except Exception as e:         # ctypes cannot propagate it through C: remember it for the caller
                self._halo_error = e
                return 1
        self._halo_error = None
        self._halo_cb = HALO_FN(thunk)     # keep the thunk alive
        _check(self.L.qk_set_halo_exchange(self.h, faces, self._halo_cb, None), "qk_set_halo_exchange")

    def qk_halo_export(self):
        """This context's storage as bytes (a qk_halo_handle): picklable, so it can cross ranks by all_gather_object."""
        h = qk_halo_handle()
        _check(self.L.qk_halo_export(self.h, C.byref(h)), "qk_halo_export")
        return bytes(h)

    def qk_set_halo_peers(self, lo, hi):
        """lo / hi: handle bytes of the neighbour below / above in z, or None at a physical boundary."""
        hl = qk_halo_handle.from_buffer_copy(lo) if lo is not None else None
        hh = qk_halo_handle.from_buffer_copy(hi) if hi is not None else None
        _check(self.L.qk_set_halo_peers(self.h, C.byref(hl) if hl is not None else None,
                                        C.byref(hh) if hh is not None else None), "qk_set_halo_peers")

    def new_buffer(self, ndoubles):
        """Device buffer for halo planes (PyTorch owns the memory)."""
        import torch
        return torch.empty(ndoubles, dtype=torch.float64, device=self.device)

    def qk_halo_doubles(self):
        return int(self.L.qk_halo_doubles(self.h))

    def qk_halo_pack(self, face, buf):
        _check(self.L.qk_halo_pack(self.h, face, _ptr(buf)), "qk_halo_pack")

    def qk_halo_unpack(self, face, buf):
        _check(self.L.qk_halo_unpack(self.h, face, _ptr(buf)), "qk_halo_unpack")

    def qk_fill_boundary(self, which=QK_FILL_ALL):
        _check(self.L.qk_fill_boundary(self.h, which), "qk_fill_boundary")

    def qk_cfl_dt(self):
        return float(self.L.qk_cfl_dt(self.h))

    def qk_hydro_step(self, dt):
        _check(self.L.qk_hydro_step(self.h, dt), "qk_hydro_step")

    def qk_hydro_step_cfl(self):
        _check(self.L.qk_hydro_step_cfl(self.h), "qk_hydro_step_cfl")

    def qk_rhd_step_cfl(self, nsub):
        _check(self.L.qk_rhd_step_cfl(self.h, nsub), "qk_rhd_step_cfl")

    def qk_graph_capture(self, kind, nsub=0):
        _check(self.L.qk_graph_capture(self.h, kind, nsub), "qk_graph_capture")

    def qk_graph_launch(self, nsteps=1):
        _check(self.L.qk_graph_launch(self.h, nsteps), "qk_graph_launch")

    def qk_graph_free(self):
        _check(self.L.qk_graph_free(self.h), "qk_graph_free")

    def qk_last_dt(self):
        out = C.c_double()
        _check(self.L.qk_last_dt(self.h, C.byref(out)), "qk_last_dt")
        return float(out.value)

    def qk_rad_transport(self, dt):
        _check(self.L.qk_rad_transport(self.h, dt), "qk_rad_transport")

    def qk_exchange(self, dt):
        _check(self.L.qk_exchange(self.h, dt), "qk_exchange")

    def qk_rad_step(self, dt):
        _check(self.L.qk_rad_step(self.h, dt), "qk_rad_step")

    def qk_rhd_step(self, dt):
        _check(self.L.qk_rhd_step(self.h, dt), "qk_rhd_step")

    def qk_nsub_for(self, dt):
        return int(self.L.qk_nsub_for(self.h, dt))

    def qk_last_info(self):
        info = qk_info()
        _check(self.L.qk_last_info(self.h, C.byref(info)), "qk_last_info")
        return {name: int(getattr(info, name)) for name, _ in qk_info._fields_}

    def qk_launch_count(self):
        return int(self.L.qk_launch_count(self.h))

    def qk_set_profiling(self, on):
        _check(self.L.qk_set_profiling(self.h, int(on)), "qk_set_profiling")

    def qk_set_flatten_path(self, path):
        _check(self.L.qk_set_flatten_path(self.h, int(path)), "qk_set_flatten_path")

    def qk_kernel_times(self):
        n = self.L.qk_kernel_class_count()
        ms = (C.c_double * n)()
        cnt = (C.c_longlong * n)()
        _check(self.L.qk_kernel_times(self.h, ms, cnt), "qk_kernel_times")
        return {self.L.qk_kernel_class_name(k).decode(): (float(ms[k]), int(cnt[k])) for k in range(n) if cnt[k]}

    # ---- marshalling helpers (no arithmetic) -------------------------------------------------------
    def set_all(self, fields: dict):
        for name, a in fields.items():
            self.qk_set_state(FIELDS.index(name), np.ascontiguousarray(a, dtype=np.float64))

    def get_all(self, names=None):
        return {n: self.qk_get_state(FIELDS.index(n)) for n in (names or FIELDS)}


def from_params(params: dict, fields: dict | None = None, **kw) -> Context:
    """Context from an inputs.py (params, fields) pair."""
    ctx = Context(params["nx"], params["ny"], params["nz"], params["dx"], params["gamma"],
                  params.get("c_hat", 0.0), params.get("c", 0.0), params.get("bc", QK_BC_PERIODIC), **kw)
    if "a_rad" in params:
        ctx.qk_set_constants(params["a_rad"], params["kB_mu"])
    ctx.qk_set_params(cfl=params.get("cfl", 0.3), flags=params.get("flags", 0))
    if fields is not None:
        ctx.set_all(fields)
    return ctx
