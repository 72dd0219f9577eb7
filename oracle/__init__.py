"""ORACLE — test infrastructure only (see fdtd_oracle.cpp header).

ctypes wrapper around the plain C++ CPU implementation of the FDTD+CPML time
step.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package; the product
package paper_2606_06910_b200 never does.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fdtd_oracle.cpp")
_LIB = os.path.join(_HERE, "libfdtd_oracle.so")

P, VX, VY, VZ = 0, 1, 2, 3
PSI_VX, PSI_VY, PSI_VZ, PSI_PX, PSI_PY, PSI_PZ = 4, 5, 6, 7, 8, 9


def build(force=False):
    """Compile the oracle with gcc: -O2, no FMA contraction (reading R25), OpenMP over z planes."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", _SRC, "-o", _LIB]
        subprocess.check_call(cmd)
    return _LIB


class Params(C.Structure):
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
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(Params), C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_dims.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_max_threads.restype = C.c_int
        L.orc_set_ftz.argtypes = [C.c_void_p, C.c_int]
        L.orc_track_energy.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_model.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_set_sources.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int]
        L.orc_step.argtypes = [C.c_void_p, C.c_int]
        L.orc_substep_v.argtypes = [C.c_void_p]
        L.orc_substep_p.argtypes = [C.c_void_p]
        L.orc_energy.restype = C.c_double
        L.orc_energy.argtypes = [C.c_void_p]
        L.orc_get_field.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.orc_set_field.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.orc_fill_hash.argtypes = [C.c_void_p, C.c_int, C.c_uint64, C.c_void_p, C.c_void_p, C.c_double]
        L.orc_cpml_table.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_coeffs.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def coeffs():
    out = np.zeros(4, np.float32)
    lib().orc_coeffs(out.ctypes.data)
    return out


class Oracle:
    """One simulation.  Fields are exchanged as float64 numpy arrays of shape (Nz, Ny, Nx)."""

    def __init__(self, n_interior, cpml=(0,) * 6, dx=1.0, dt=0.4, cpml_order=2, cpml_R0=1e-5,
                 cpml_kappa_max=1.0, cpml_alpha_max=0.0, cpml_c_ref=1.0, boundary=0, fp64=False):
        p = Params()
        p.n_interior[:] = list(n_interior)
        p.cpml[:] = list(cpml)
        p.dx, p.dt = float(dx), float(dt)
        p.cpml_order, p.boundary = int(cpml_order), int(boundary)
        p.cpml_R0, p.cpml_kappa_max = float(cpml_R0), float(cpml_kappa_max)
        p.cpml_alpha_max, p.cpml_c_ref = float(cpml_alpha_max), float(cpml_c_ref)
        self.params = p
        self.fp64 = bool(fp64)
        self._h = lib().orc_create(C.byref(p), int(fp64))
        d = (C.c_int32 * 3)()
        lib().orc_dims(self._h, d)
        self.nx, self.ny, self.nz = int(d[0]), int(d[1]), int(d[2])
        self.shape = (self.nz, self.ny, self.nx)

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_model(self, c=None, rho=None):
        ca = None if c is None else np.ascontiguousarray(c, np.float32).reshape(self.shape)
        ra = None if rho is None else np.ascontiguousarray(rho, np.float32).reshape(self.shape)
        lib().orc_set_model(self._h, None if ca is None else ca.ctypes.data, None if ra is None else ra.ctypes.data)

    def set_sources(self, ijk, wavelets):
        ijk = np.ascontiguousarray(ijk, np.int32).reshape(-1, 3)
        w = np.ascontiguousarray(wavelets, np.float32).reshape(ijk.shape[0], -1)
        lib().orc_set_sources(self._h, ijk.shape[0], ijk.ctypes.data, w.ctypes.data, w.shape[1])

    def step(self, n=1):
        lib().orc_step(self._h, int(n))

    def substep_v(self):
        lib().orc_substep_v(self._h)

    def substep_p(self):
        lib().orc_substep_p(self._h)

    def set_ftz(self, on=True):
        lib().orc_set_ftz(self._h, int(on))

    def track_energy(self, on=True):
        lib().orc_track_energy(self._h, int(on))

    def energy(self):
        return float(lib().orc_energy(self._h))

    def get(self, which):
        out = np.empty(self.shape, np.float64)
        lib().orc_get_field(self._h, int(which), out.ctypes.data)
        return out

    def set(self, which, arr):
        a = np.ascontiguousarray(arr, np.float64).reshape(self.shape)
        lib().orc_set_field(self._h, int(which), a.ctypes.data)

    def fill_hash(self, which, seed, gdim=None, off=(0, 0, 0), scale=1.0):
        g = np.asarray(gdim if gdim is not None else (self.nx, self.ny, self.nz), np.int64)
        o = np.asarray(off, np.int64)
        lib().orc_fill_hash(self._h, int(which), C.c_uint64(int(seed)), g.ctypes.data, o.ctypes.data, float(scale))

    def cpml_table(self, axis, half):
        n = (self.nx, self.ny, self.nz)[axis]
        a, b, ik = (np.zeros(n, np.float32) for _ in range(3))
        inn = np.zeros(n, np.uint8)
        lib().orc_cpml_table(self._h, axis, int(half), a.ctypes.data, b.ctypes.data, ik.ctypes.data, inn.ctypes.data)
        return a, b, ik, inn


def set_threads(n):
    lib().orc_set_threads(int(n))


def max_threads():
    return int(lib().orc_max_threads())
