"""Thin Python binding of the C-ABI library (include/fts.h): argument marshalling only.

PyTorch supplies device memory (tensors) and streams; every step of the path runs inside libfts.so.
There is no fallback: if the library cannot be loaded, importing fails loudly.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfts.so")

STATUS = {0: "FTS_OK", 1: "FTS_EINVAL", 2: "FTS_ESTATE", 3: "FTS_EWORKSPACE", 4: "FTS_ECUDA", 5: "FTS_ENONFINITE",
          6: "FTS_EUNSUPPORTED"}
MODELS = {"external": 0, "edwards": 1, "diblock": 2}
EXPORTS = ["fts_workspace_bytes", "fts_create", "fts_destroy", "fts_set_fields", "fts_get_fields", "fts_propagate",
           "fts_propagate_steps", "fts_set_blocks", "fts_density_operators", "fts_get_slice", "fts_scft_step", "fts_cl_step",
           "fts_operators", "fts_set_option", "fts_mean_noalloc", "fts_debug_normals", "fts_debug_philox", "fts_debug_fma_peak", "fts_launch_count", "fts_last_error", "fts_version"]


class FtsParams(C.Structure):
    _fields_ = [("model", C.c_int), ("fA", C.c_double), ("chiN", C.c_double), ("B", C.c_double), ("C", C.c_double),
                ("lambda_plus", C.c_double), ("lambda_minus", C.c_double), ("noise_scale", C.c_double),
                ("store_both", C.c_int)]


class FtsError(RuntimeError):
    def __init__(self, what, status, detail=""):
        self.status = status
        super().__init__(f"{what}: {STATUS.get(status, status)} {detail}".strip())


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1204_5434_b200.build` (no CPU fallback exists)")
        L = C.CDLL(LIB_PATH)
        vp, ip, dp = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double)
        pp = C.POINTER(FtsParams)
        L.fts_workspace_bytes.argtypes = [ip, C.c_int, pp, C.c_int, C.POINTER(C.c_size_t)]
        L.fts_create.argtypes = [ip, dp, C.c_int, pp, C.c_int, vp, C.c_size_t, C.POINTER(vp)]
        L.fts_destroy.argtypes = [vp]
        L.fts_set_blocks.argtypes = [vp, C.c_int, ip, ip]
        L.fts_set_fields.argtypes = [vp, vp, vp, vp]
        L.fts_get_fields.argtypes = [vp, vp, vp, vp]
        L.fts_propagate.argtypes = [vp, vp]
        L.fts_propagate_steps.argtypes = [vp, C.c_int, vp]
        L.fts_density_operators.argtypes = [vp, vp, vp, dp, vp]
        L.fts_get_slice.argtypes = [vp, C.c_int, C.c_int, vp, vp]
        L.fts_scft_step.argtypes = [vp, C.c_double, C.c_double, C.c_int, dp, dp, vp]
        L.fts_cl_step.argtypes = [vp, C.c_double, C.c_int, C.c_uint64, C.c_uint64, vp]
        L.fts_operators.argtypes = [vp, dp, dp, dp, vp]
        L.fts_set_option.argtypes = [vp, C.c_char_p, C.c_longlong]
        L.fts_debug_normals.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint64, C.c_size_t, vp, vp]
        L.fts_debug_philox.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint64, C.c_size_t, vp, vp]
        L.fts_debug_fma_peak.argtypes = [C.c_int, C.c_int, vp, C.c_size_t, dp, vp]
        L.fts_mean_noalloc.argtypes = [vp, C.c_size_t, C.c_int, vp, vp, C.c_char_p, C.c_size_t]
        L.fts_launch_count.restype = C.c_uint64
        L.fts_last_error.argtypes = [vp]
        L.fts_last_error.restype = C.c_char_p
        L.fts_version.restype = C.c_char_p
        _lib = L
    return _lib


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _p(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def make_params(model, fA=0.5, chiN=10.0, B=1.0, Cc=1.0, lambda_plus=1.0, lambda_minus=1.0, noise_scale=1.0, store_both=0):
    return FtsParams(MODELS.get(model, model), fA, chiN, B, Cc, lambda_plus, lambda_minus, noise_scale, int(store_both))


def workspace_bytes(grid, Ns, params, precision="f64"):
    n = C.c_size_t()
    g = (C.c_int * 3)(*[int(v) for v in grid])
    rc = lib().fts_workspace_bytes(g, int(Ns), C.byref(params), 0 if precision == "f64" else 1, C.byref(n))
    if rc:
        raise FtsError("fts_workspace_bytes", rc)
    return n.value


class Fts:
    """One simulation context on `device`.  Methods mirror the C calls one to one; each makes the context's device current
    for the duration of the call (the library launches on the current device), so a context on cuda:1 can be driven
    while cuda:0 is the process's current device.  The stream is the current stream OF THAT DEVICE."""

    def __init__(self, grid, cell, Ns, model, precision="f64", device="cuda:0", options=None, **kw):
        self.grid = tuple(int(v) for v in grid)
        self.Ns = int(Ns)
        self.model = MODELS.get(model, model)
        self.precision = precision
        self.cdtype = torch.complex128 if precision == "f64" else torch.complex64
        self.device = torch.device(device)
        self.params = make_params(model, **kw)
        nbytes = workspace_bytes(self.grid, self.Ns, self.params, precision)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)      # caller-owned device memory
        h = C.c_void_p()
        g = (C.c_int * 3)(*self.grid)
        c = (C.c_double * 3)(*[float(v) for v in cell])
        with torch.cuda.device(self.device):
            rc = lib().fts_create(g, c, self.Ns, C.byref(self.params), 0 if precision == "f64" else 1,
                                  _p(self.workspace), nbytes, C.byref(h))
        if rc:
            raise FtsError("fts_create", rc)
        self.h = h
        for k, v in (options or {}).items():
            self.set_option(k, v)

    def set_option(self, key, value):
        with torch.cuda.device(self.device):
            self._chk(lib().fts_set_option(self.h, str(key).encode(), int(value)), f"fts_set_option({key})")

    def set_blocks(self, species, steps):
        n = len(species)
        with torch.cuda.device(self.device):
            self._chk(lib().fts_set_blocks(self.h, n, (C.c_int * n)(*[int(v) for v in species]), (C.c_int * n)(*[int(v) for v in steps])), "fts_set_blocks")

    def close(self):
        if getattr(self, "h", None) and _lib is not None:
            with torch.cuda.device(self.device):
                _lib.fts_destroy(self.h)
        self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:           # interpreter shutdown: module globals may already be gone
            pass

    def _chk(self, rc, what):
        if rc:
            raise FtsError(what, rc, lib().fts_last_error(self.h).decode())

    def _new(self):
        return torch.empty(self.grid, dtype=self.cdtype, device=self.device)

    def set_fields(self, f0, f1=None):
        assert f0.is_cuda and f0.dtype == self.cdtype and f0.is_contiguous() and tuple(f0.shape) == self.grid
        assert f1 is None or (f1.is_cuda and f1.dtype == self.cdtype and f1.is_contiguous())
        with torch.cuda.device(self.device):
            self._chk(lib().fts_set_fields(self.h, _p(f0), _p(f1), _stream()), "fts_set_fields")

    def get_fields(self):
        a = self._new()
        b = self._new() if self.model == 2 else None
        with torch.cuda.device(self.device):
            self._chk(lib().fts_get_fields(self.h, _p(a), _p(b), _stream()), "fts_get_fields")
        return a, b

    def propagate(self, nsteps=None):
        with torch.cuda.device(self.device):
            if nsteps is None:
                self._chk(lib().fts_propagate(self.h, _stream()), "fts_propagate")
            else:
                self._chk(lib().fts_propagate_steps(self.h, int(nsteps), _stream()), "fts_propagate_steps")

    def density_operators(self, phiA=None, phiB=None):
        phiA = self._new() if phiA is None else phiA
        phiB = (self._new() if phiB is None else phiB) if self.model == 2 else None
        Q = (C.c_double * 2)()
        with torch.cuda.device(self.device):
            self._chk(lib().fts_density_operators(self.h, _p(phiA), _p(phiB), Q, _stream()), "fts_density_operators")
        return complex(Q[0], Q[1]), phiA, phiB

    def get_slice(self, which, j, out=None):
        out = self._new() if out is None else out
        with torch.cuda.device(self.device):
            self._chk(lib().fts_get_slice(self.h, int(which), int(j), _p(out), _stream()), "fts_get_slice")
        return out

    def scft_step(self, dt_plus, dt_minus, seidel=1):
        H, r = (C.c_double * 2)(), (C.c_double * 2)()
        with torch.cuda.device(self.device):
            self._chk(lib().fts_scft_step(self.h, dt_plus, dt_minus, int(seidel), H, r, _stream()), "fts_scft_step")
        return complex(H[0], H[1]), (r[0], r[1])

    def cl_step(self, dt, scheme, seed, step):
        with torch.cuda.device(self.device):
            self._chk(lib().fts_cl_step(self.h, dt, int(scheme), int(seed), int(step), _stream()), "fts_cl_step")

    def operators(self, want_pi=True):
        H, mu, Pi = (C.c_double * 2)(), (C.c_double * 2)(), (C.c_double * 2)()
        with torch.cuda.device(self.device):
            self._chk(lib().fts_operators(self.h, H, mu, Pi if want_pi else None, _stream()), "fts_operators")
        return complex(H[0], H[1]), complex(mu[0], mu[1]), complex(Pi[0], Pi[1])


MEAN_NOALLOC_MAX_POINTS = 1 << 24      # FTS_MEAN_NOALLOC_MAX_POINTS of include/fts.h


def mean_noalloc(field, out, npoints=None):
    """fts_mean_noalloc: enqueue mean(field) -> out (2 float64 on the device: re, im) on the current stream of field's
    device.  For callers that own no workspace and may not allocate (see include/fts.h): the library's reduction scratch
    is a fixed array inside libfts.so, so neither this wrapper nor the library allocates anything - `out` is the
    caller's, which is why it is not optional.  Calls that may overlap on one GPU (different streams) race on that array.
    The first call on a device does a one-time address look-up: make it before any stream capture.  npoints overrides
    field.numel() (tests of the size limit).  Returns `out`; nothing is synchronised."""
    assert field.is_cuda and field.is_contiguous() and field.dtype in (torch.complex128, torch.complex64)
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() >= 2 and out.is_contiguous() and out.device == field.device
    n = field.numel() if npoints is None else int(npoints)
    err = C.create_string_buffer(256)
    with torch.cuda.device(field.device):
        rc = lib().fts_mean_noalloc(_p(field), n, 0 if field.dtype == torch.complex128 else 1, _p(out), _stream(), err, len(err))
    if rc:
        raise FtsError("fts_mean_noalloc", rc, err.value.decode())
    return out


def debug_normals(seed, step, field_id, site0, n, device="cuda:0"):
    out = torch.empty(n, dtype=torch.float64, device=device)
    with torch.cuda.device(out.device):
        rc = lib().fts_debug_normals(int(seed), int(step), int(field_id), int(site0), int(n), _p(out), _stream())
    if rc:
        raise FtsError("fts_debug_normals", rc)
    return out


def debug_philox(seed, step, field_id, site0, n, device="cuda:0"):
    """(n, 4) int64 tensor holding the raw 32-bit Philox words of sites site0 .. site0 + n - 1."""
    out = torch.empty((n, 4), dtype=torch.int32, device=device)
    with torch.cuda.device(out.device):
        rc = lib().fts_debug_philox(int(seed), int(step), int(field_id), int(site0), int(n), _p(out), _stream())
    if rc:
        raise FtsError("fts_debug_philox", rc)
    return out.to(torch.int64) & 0xFFFFFFFF


def launch_count():
    return int(lib().fts_launch_count())


def fma_peak_launch(precision, iters, scratch):
    """Enqueue the FMA-chain kernel on the current stream; returns the FMA count of that launch."""
    n = C.c_double()
    with torch.cuda.device(scratch.device):
        rc = lib().fts_debug_fma_peak(0 if precision == "f64" else 1, int(iters), _p(scratch), scratch.numel() * scratch.element_size(),
                                      C.byref(n), _stream())
    if rc:
        raise FtsError("fts_debug_fma_peak", rc)
    return n.value
