"""ctypes wrapper around oracle/liboracle.so (TEST INFRASTRUCTURE, NOT PRODUCT CODE).

Argument marshalling only; every number comes from oracle/fts_oracle.cpp.
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None


class OracleParams(C.Structure):
    _fields_ = [("model", C.c_int), ("fA", C.c_double), ("chiN", C.c_double), ("B", C.c_double), ("C", C.c_double),
                ("lambda_plus", C.c_double), ("lambda_minus", C.c_double), ("noise_scale", C.c_double),
                ("store_both", C.c_int)]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp, ip, dp = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double)
        L.oracle_create.argtypes = [ip, dp, C.c_int, C.POINTER(OracleParams), C.c_int, C.POINTER(vp)]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_destroy.restype = None
        L.oracle_set_fields.argtypes = [vp, vp, vp]
        L.oracle_get_fields.argtypes = [vp, vp, vp]
        L.oracle_propagate.argtypes = [vp]
        L.oracle_propagate_steps.argtypes = [vp, C.c_int]
        L.oracle_density_operators.argtypes = [vp, vp, vp, dp]
        L.oracle_set_blocks.argtypes = [vp, C.c_int, ip, ip]
        L.oracle_get_slice.argtypes = [vp, C.c_int, C.c_int, vp]
        L.oracle_scft_step.argtypes = [vp, C.c_double, C.c_double, C.c_int, dp, dp]
        L.oracle_cl_step.argtypes = [vp, C.c_double, C.c_int, C.c_uint64, C.c_uint64]
        L.oracle_operators.argtypes = [vp, dp, dp, dp]
        L.oracle_fft1d.argtypes = [vp, C.c_int, C.c_int]
        L.oracle_fft1d.restype = None
        L.oracle_dft1d_direct.argtypes = [vp, C.c_int, C.c_int]
        L.oracle_dft1d_direct.restype = None
        L.oracle_rqm4_step.argtypes = [ip, dp, C.c_double, vp, vp, vp]
        L.oracle_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.oracle_philox4x32_10.restype = None
        L.oracle_normal.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint64]
        L.oracle_normal.restype = C.c_double
        L.oracle_debye.argtypes = [C.c_double]
        L.oracle_debye.restype = C.c_double
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c2(x):
    return complex(x[0], x[1])


class Oracle:
    """Same call names as the product's Python binding, on host (numpy) arrays."""

    def __init__(self, grid, cell, Ns, model, precision="f64", fA=0.5, chiN=10.0, B=1.0, Cc=1.0,
                 lambda_plus=1.0, lambda_minus=1.0, noise_scale=1.0):
        self.grid = tuple(int(g) for g in grid)
        self.M = int(np.prod(self.grid))
        self.model = {"external": 0, "edwards": 1, "diblock": 2}.get(model, model)
        self.cdtype = np.complex128 if precision in ("f64", 0) else np.complex64
        p = OracleParams(self.model, fA, chiN, B, Cc, lambda_plus, lambda_minus, noise_scale, 1)
        h = C.c_void_p()
        g = (C.c_int * 3)(*self.grid)
        c = (C.c_double * 3)(*[float(x) for x in cell])
        rc = lib().oracle_create(g, c, int(Ns), C.byref(p), 0 if self.cdtype == np.complex128 else 1, C.byref(h))
        if rc:
            raise ValueError(f"oracle_create failed with status {rc}")
        self.h, self.Ns = h, int(Ns)

    def __del__(self):
        if getattr(self, "h", None):
            lib().oracle_destroy(self.h)
            self.h = None

    def _chk(self, rc, what):
        if rc:
            raise RuntimeError(f"{what} failed with status {rc}")

    def set_fields(self, f0, f1=None):
        a = np.ascontiguousarray(f0, dtype=self.cdtype)
        b = None if f1 is None else np.ascontiguousarray(f1, dtype=self.cdtype)
        self._chk(lib().oracle_set_fields(self.h, _ptr(a), _ptr(b)), "oracle_set_fields")

    def get_fields(self):
        a = np.empty(self.grid, self.cdtype)
        b = np.empty(self.grid, self.cdtype) if self.model == 2 else None
        self._chk(lib().oracle_get_fields(self.h, _ptr(a), _ptr(b)), "oracle_get_fields")
        return a, b

    def set_blocks(self, species, steps):
        n = len(species)
        self._chk(lib().oracle_set_blocks(self.h, n, (C.c_int * n)(*species), (C.c_int * n)(*steps)), "oracle_set_blocks")

    def propagate(self, nsteps=None):
        if nsteps is None:
            self._chk(lib().oracle_propagate(self.h), "oracle_propagate")
        else:
            self._chk(lib().oracle_propagate_steps(self.h, int(nsteps)), "oracle_propagate_steps")

    def density_operators(self):
        a = np.empty(self.grid, self.cdtype)
        b = np.empty(self.grid, self.cdtype) if self.model == 2 else None
        Q = (C.c_double * 2)()
        self._chk(lib().oracle_density_operators(self.h, _ptr(a), _ptr(b), Q), "oracle_density_operators")
        return _c2(Q), a, b

    def get_slice(self, which, j):
        a = np.empty(self.grid, self.cdtype)
        self._chk(lib().oracle_get_slice(self.h, int(which), int(j), _ptr(a)), "oracle_get_slice")
        return a

    def scft_step(self, dt_plus, dt_minus, seidel=1):
        H, r = (C.c_double * 2)(), (C.c_double * 2)()
        self._chk(lib().oracle_scft_step(self.h, dt_plus, dt_minus, int(seidel), H, r), "oracle_scft_step")
        return _c2(H), (r[0], r[1])

    def cl_step(self, dt, scheme, seed, step):
        self._chk(lib().oracle_cl_step(self.h, dt, int(scheme), int(seed), int(step)), "oracle_cl_step")

    def operators(self):
        H, mu, Pi = (C.c_double * 2)(), (C.c_double * 2)(), (C.c_double * 2)()
        self._chk(lib().oracle_operators(self.h, H, mu, Pi), "oracle_operators")
        return _c2(H), _c2(mu), _c2(Pi)


def fft1d(x, sign):
    a = np.ascontiguousarray(x, dtype=np.complex128).copy()
    lib().oracle_fft1d(_ptr(a), a.size, sign)
    return a


def dft1d_direct(x, sign):
    a = np.ascontiguousarray(x, dtype=np.complex128).copy()
    lib().oracle_dft1d_direct(_ptr(a), a.size, sign)
    return a


def rqm4_step(grid, cell, ds, w, q):
    g = (C.c_int * 3)(*[int(v) for v in grid])
    c = (C.c_double * 3)(*[float(v) for v in cell])
    wa = np.ascontiguousarray(w, dtype=np.complex128)
    qa = np.ascontiguousarray(q, dtype=np.complex128)
    out = np.empty_like(qa)
    lib().oracle_rqm4_step(g, c, float(ds), _ptr(wa), _ptr(qa), _ptr(out))
    return out


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


def normal(seed, step, field_id, site):
    return lib().oracle_normal(int(seed), int(step), int(field_id), int(site))


def debye(x):
    return lib().oracle_debye(float(x))
