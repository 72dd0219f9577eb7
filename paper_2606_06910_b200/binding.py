"""Thin ctypes binding over the C ABI of include/fdtd_b200.h — argument marshalling only.

Same names as the C entry points (fdtd_create, fdtd_set_model, fdtd_step, fdtd_get_field, fdtd_destroy, ...)
plus a small `Fdtd` convenience class that owns the device workspace as a torch uint8 tensor (PyTorch is used
for device memory and streams only).  There is no CPU path: if the CUDA library is missing this module raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfdtd_b200.so")

FDTD_P, FDTD_VX, FDTD_VY, FDTD_VZ = 0, 1, 2, 3
FDTD_PSI_VX, FDTD_PSI_VY, FDTD_PSI_VZ, FDTD_PSI_PX, FDTD_PSI_PY, FDTD_PSI_PZ = range(6)
FDTD_WALL, FDTD_PERIODIC = 0, 1
FDTD_KERNEL_AUTO, FDTD_KERNEL_REF, FDTD_KERNEL_FUSED = 0, 1, 2
FDTD_DENSITY_UNIFORM, FDTD_DENSITY_ARRAY = 0, 1
FDTD_MEDIUM_ARRAY, FDTD_MEDIUM_UNIFORM = 0, 1
FDTD_PRECISION_FP32, FDTD_PRECISION_FP64 = 0, 1
FDTD_OK, FDTD_EINVAL, FDTD_EWORKSPACE, FDTD_ECUDA, FDTD_EUNSUPPORTED = 0, -1, -2, -3, -4

# every symbol include/fdtd_b200.h declares
EXPORTS = [
    "fdtd_workspace_bytes", "fdtd_create", "fdtd_set_model", "fdtd_set_sources", "fdtd_step", "fdtd_step_profiled", "fdtd_get_field",
    "fdtd_get_field_box", "fdtd_set_field", "fdtd_get_field_f64", "fdtd_set_field_f64", "fdtd_get_psi_f64", "fdtd_fill_hash", "fdtd_get_psi", "fdtd_field_absmax", "fdtd_cpml_table",
    "fdtd_coeffs", "fdtd_absmax_noalloc", "fdtd_time_block_stats", "fdtd_kernel_in_use", "fdtd_launch_count", "fdtd_dims", "fdtd_destroy", "fdtd_last_error",
]


class fdtd_params(C.Structure):
    _fields_ = [
        ("n_interior", C.c_int32 * 3),
        ("cpml", C.c_int32 * 6),
        ("dx", C.c_double),
        ("dt", C.c_double),
        ("cpml_order", C.c_int32),
        ("boundary", C.c_int32),
        ("cpml_R0", C.c_double),
        ("cpml_kappa_max", C.c_double),
        ("cpml_alpha_max", C.c_double),
        ("cpml_c_ref", C.c_double),
        ("decomp", C.c_int32 * 3),
        ("ghost", C.c_int32),
        ("substeps_per_exchange", C.c_int32),
        ("kernel", C.c_int32),
        ("density", C.c_int32),
        ("medium", C.c_int32),
        ("precision", C.c_int32),
        ("time_block", C.c_int32),
        ("time_block_planes", C.c_int32),
        ("device", C.c_int32),
        ("stream", C.c_void_p),
        ("workspace", C.c_void_p),
        ("workspace_bytes", C.c_uint64),
    ]


class FdtdError(RuntimeError):
    pass


def _load():
    if not os.path.exists(LIB_PATH):
        raise FdtdError("CUDA library %s is missing: build it with `python -m paper_2606_06910_b200.build` "
                        "(there is no CPU fallback)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, i32, u64, f64 = C.c_void_p, C.c_int32, C.c_uint64, C.c_double
    L.fdtd_workspace_bytes.restype = u64
    L.fdtd_workspace_bytes.argtypes = [C.POINTER(fdtd_params)]
    L.fdtd_create.restype = vp
    L.fdtd_create.argtypes = [C.POINTER(fdtd_params)]
    L.fdtd_set_model.argtypes = [vp, vp, vp]
    L.fdtd_set_sources.argtypes = [vp, i32, vp, vp, i32]
    L.fdtd_absmax_noalloc.argtypes = [vp, u64, vp, vp]
    L.fdtd_step.argtypes = [vp, i32]
    L.fdtd_step_profiled.argtypes = [vp, i32, vp]
    L.fdtd_get_field.argtypes = [vp, i32, vp]
    L.fdtd_get_field_box.argtypes = [vp, i32, vp, vp, vp]
    L.fdtd_set_field.argtypes = [vp, i32, vp]
    L.fdtd_get_field_f64.argtypes = [vp, i32, vp]
    L.fdtd_set_field_f64.argtypes = [vp, i32, vp]
    L.fdtd_get_psi_f64.argtypes = [vp, i32, vp]
    L.fdtd_fill_hash.argtypes = [vp, i32, u64, f64]
    L.fdtd_get_psi.argtypes = [vp, i32, vp]
    L.fdtd_field_absmax.argtypes = [vp, i32, vp, vp, vp]
    L.fdtd_cpml_table.argtypes = [vp, i32, i32, vp, vp, vp]
    L.fdtd_coeffs.argtypes = [vp]
    L.fdtd_launch_count.restype = C.c_int64
    L.fdtd_launch_count.argtypes = [vp]
    L.fdtd_dims.argtypes = [vp, vp]
    L.fdtd_kernel_in_use.argtypes = [vp]
    L.fdtd_time_block_stats.argtypes = [vp, vp]
    L.fdtd_destroy.argtypes = [vp]
    L.fdtd_last_error.restype = C.c_char_p
    return L


lib = _load()


def last_error():
    return (lib.fdtd_last_error() or b"").decode()


def _check(rc, what):
    if rc != 0:
        raise FdtdError("%s failed (%d): %s" % (what, rc, last_error()))


FDTD_NOALLOC_MAX_ELEMS = 1 << 30


def fdtd_absmax_noalloc(in_dev_ptr, n, out_dev_ptr, stream_ptr=0):
    """max |f| of n fp32 values at device address in_dev_ptr into the device float at out_dev_ptr, on the current device,
    asynchronous on the stream; allocates nothing (static device scratch, n <= FDTD_NOALLOC_MAX_ELEMS)."""
    _check(lib.fdtd_absmax_noalloc(C.c_void_p(int(in_dev_ptr)), C.c_uint64(int(n)), C.c_void_p(int(out_dev_ptr)), C.c_void_p(int(stream_ptr))),
           "fdtd_absmax_noalloc")


def fdtd_coeffs():
    out = np.zeros(4, np.float32)
    _check(lib.fdtd_coeffs(out.ctypes.data), "fdtd_coeffs")
    return out


def make_params(n_interior, cpml=(0,) * 6, dx=1.0, dt=0.4, cpml_order=2, cpml_R0=1e-5, cpml_kappa_max=1.0,
                cpml_alpha_max=0.0, cpml_c_ref=1.0, boundary=FDTD_WALL, decomp=(1, 1, 1), ghost=0, substeps=0,
                kernel=FDTD_KERNEL_AUTO, density=FDTD_DENSITY_UNIFORM, medium=FDTD_MEDIUM_ARRAY, precision=FDTD_PRECISION_FP32, time_block=0, time_block_planes=0, device=0):
    p = fdtd_params()
    p.n_interior[:] = [int(v) for v in n_interior]
    p.cpml[:] = [int(v) for v in cpml]
    p.dx, p.dt = float(dx), float(dt)
    p.cpml_order, p.boundary = int(cpml_order), int(boundary)
    p.cpml_R0, p.cpml_kappa_max = float(cpml_R0), float(cpml_kappa_max)
    p.cpml_alpha_max, p.cpml_c_ref = float(cpml_alpha_max), float(cpml_c_ref)
    p.decomp[:] = [int(v) for v in decomp]
    p.ghost, p.substeps_per_exchange = int(ghost), int(substeps)
    p.kernel, p.density, p.medium, p.precision, p.device = int(kernel), int(density), int(medium), int(precision), int(device)
    p.time_block, p.time_block_planes = int(time_block), int(time_block_planes)
    return p


def fdtd_workspace_bytes(params):
    return int(lib.fdtd_workspace_bytes(C.byref(params)))


class Fdtd:
    """One simulation context.  Host arrays in and out are float32 numpy arrays of shape (Nz, Ny, Nx)."""

    def __init__(self, n_interior, cpml=(0,) * 6, stream=None, **kw):
        import torch

        if not torch.cuda.is_available():
            raise FdtdError("no CUDA device: the FDTD path has no CPU fallback")
        self.params = make_params(n_interior, cpml, **kw)
        nbytes = fdtd_workspace_bytes(self.params)
        if nbytes == 0:
            raise FdtdError("invalid parameters: " + last_error())
        dev = torch.device("cuda", self.params.device)
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)       # owned here, outlives the context
        ptr = (self._ws.data_ptr() + 255) // 256 * 256
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        self.stream = st
        self.params.stream = C.c_void_p(st.cuda_stream)
        self.params.workspace = C.c_void_p(ptr)
        self.params.workspace_bytes = nbytes
        self.workspace_bytes = nbytes
        self._h = lib.fdtd_create(C.byref(self.params))
        if not self._h:
            raise FdtdError("fdtd_create failed: " + last_error())
        d = (C.c_int32 * 3)()
        _check(lib.fdtd_dims(self._h, d), "fdtd_dims")
        self.nx, self.ny, self.nz = int(d[0]), int(d[1]), int(d[2])
        self.shape = (self.nz, self.ny, self.nx)

    # --- the C ABI, one method per entry point -----------------------------------------------------------
    def set_model(self, c=None, rho=None):
        ca = None if c is None else np.ascontiguousarray(c, np.float32).reshape(self.shape)
        ra = None if rho is None else np.ascontiguousarray(rho, np.float32).reshape(self.shape)
        _check(lib.fdtd_set_model(self._h, None if ca is None else ca.ctypes.data, None if ra is None else ra.ctypes.data),
               "fdtd_set_model")

    def set_sources(self, ijk, wavelets):
        ijk = np.ascontiguousarray(ijk, np.int32).reshape(-1, 3)
        w = np.ascontiguousarray(wavelets, np.float32).reshape(ijk.shape[0], -1)
        _check(lib.fdtd_set_sources(self._h, ijk.shape[0], ijk.ctypes.data, w.ctypes.data, w.shape[1]), "fdtd_set_sources")

    def step(self, n=1):
        _check(lib.fdtd_step(self._h, int(n)), "fdtd_step")

    def step_profiled(self, n=1):
        """-> dict of milliseconds per launch group over the n steps (CUDA events on the launching stream)."""
        out = np.zeros(4, np.float64)
        _check(lib.fdtd_step_profiled(self._h, int(n), out.ctypes.data), "fdtd_step_profiled")
        return dict(update_v=float(out[0]), update_p=float(out[1]), inject=float(out[2]), exchange=float(out[3]))

    @property
    def fp64(self):
        return self.params.precision == FDTD_PRECISION_FP64

    def get_field(self, which, out=None):
        """float32 array, or float64 for a context created with precision=FDTD_PRECISION_FP64."""
        if self.fp64:
            out = np.empty(self.shape, np.float64) if out is None else out
            _check(lib.fdtd_get_field_f64(self._h, int(which), out.ctypes.data), "fdtd_get_field_f64")
            return out
        if out is None:
            out = np.empty(self.shape, np.float32)
        _check(lib.fdtd_get_field(self._h, int(which), out.ctypes.data), "fdtd_get_field")
        return out

    def get_field_into(self, which, host_ptr):
        """Raw-pointer variant (e.g. a pinned torch tensor's data_ptr())."""
        _check(lib.fdtd_get_field(self._h, int(which), C.c_void_p(host_ptr)), "fdtd_get_field")

    def set_model_from(self, c_ptr):
        _check(lib.fdtd_set_model(self._h, C.c_void_p(c_ptr), None), "fdtd_set_model")

    def get_field_box(self, which, lo, size):
        lo_a = np.asarray(lo, np.int32)
        sz_a = np.asarray(size, np.int32)
        out = np.empty((int(sz_a[2]), int(sz_a[1]), int(sz_a[0])), np.float32)
        _check(lib.fdtd_get_field_box(self._h, int(which), lo_a.ctypes.data, sz_a.ctypes.data, out.ctypes.data), "fdtd_get_field_box")
        return out

    def set_field(self, which, arr):
        if self.fp64:
            a = np.ascontiguousarray(arr, np.float64).reshape(self.shape)
            _check(lib.fdtd_set_field_f64(self._h, int(which), a.ctypes.data), "fdtd_set_field_f64")
            return
        a = np.ascontiguousarray(arr, np.float32).reshape(self.shape)
        _check(lib.fdtd_set_field(self._h, int(which), a.ctypes.data), "fdtd_set_field")

    def fill_hash(self, which, seed, scale=1.0):
        _check(lib.fdtd_fill_hash(self._h, int(which), C.c_uint64(int(seed)), float(scale)), "fdtd_fill_hash")

    def get_psi(self, which):
        if self.fp64:
            out = np.empty(self.shape, np.float64)
            _check(lib.fdtd_get_psi_f64(self._h, int(which), out.ctypes.data), "fdtd_get_psi_f64")
            return out
        out = np.empty(self.shape, np.float32)
        _check(lib.fdtd_get_psi(self._h, int(which), out.ctypes.data), "fdtd_get_psi")
        return out

    def field_absmax(self, which, lo=(0, 0, 0), size=None):
        lo_a = np.asarray(lo, np.int32)
        sz_a = np.asarray(size if size is not None else (self.nx, self.ny, self.nz), np.int32)
        out = np.zeros(1, np.float32)
        _check(lib.fdtd_field_absmax(self._h, int(which), lo_a.ctypes.data, sz_a.ctypes.data, out.ctypes.data), "fdtd_field_absmax")
        return float(out[0])

    def cpml_table(self, axis, half):
        n = (self.nx, self.ny, self.nz)[axis]
        a, b, ik = (np.zeros(n, np.float32) for _ in range(3))
        _check(lib.fdtd_cpml_table(self._h, int(axis), int(half), a.ctypes.data, b.ctypes.data, ik.ctypes.data), "fdtd_cpml_table")
        return a, b, ik

    def time_block_stats(self):
        """-> (plane-steps computed, plane-steps owned) of the time-blocked mode."""
        out = np.zeros(2, np.int64)
        _check(lib.fdtd_time_block_stats(self._h, out.ctypes.data), "fdtd_time_block_stats")
        return int(out[0]), int(out[1])

    def kernel_in_use(self):
        return int(lib.fdtd_kernel_in_use(self._h))

    def launch_count(self):
        return int(lib.fdtd_launch_count(self._h))

    def destroy(self):
        if getattr(self, "_h", None):
            rc = lib.fdtd_destroy(self._h)
            self._h = None
            big = self.workspace_bytes > (1 << 30)
            self._ws = None                      # the context is gone: give the workspace back
            if big:                              # ... to the driver too, so the next large context is one contiguous block
                import torch
                torch.cuda.empty_cache()
            _check(rc, "fdtd_destroy")

    close = destroy

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def from_workload(w, **kw):
    """Context + model + sources for an inputs.Workload."""
    kw.setdefault("medium", FDTD_MEDIUM_ARRAY if w.c is not None else FDTD_MEDIUM_UNIFORM)
    sim = Fdtd(w.n_interior, w.cpml, decomp=kw.pop("decomp", w.decomp), ghost=kw.pop("ghost", w.ghost),
               substeps=kw.pop("substeps", w.substeps), **w.cpml_kwargs(), **kw)
    if w.c is not None:
        sim.set_model(w.c)
    sim.set_sources(w.sources, w.wavelets)
    return sim
