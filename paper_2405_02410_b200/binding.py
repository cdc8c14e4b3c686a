"""Thin ctypes binding of libpss.so (include/pss.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch is used for exactly two
things: the device workspace (``torch.empty(..., device="cuda")``) and the CUDA stream handle.
There is no CPU fallback: without the compiled library or a CUDA device this module raises.

Method names mirror the C ABI; operators are dicts
``{"coef": c, "q2_pow": m, "invq_pow": p, "iq_pow": (ax, ay, az)}`` (missing keys: coef 1, powers 0).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

F32, F64 = 0, 1
DEALIAS_PAPER, DEALIAS_TWO_THIRDS, DEALIAS_OFF = 0, 1, 2
OK, EINVAL, EUNSUPPORTED, ESTATE, ECUDA, ETOOBIG = 0, -1, -2, -3, -4, -5
STATIC_NOISE_MAX_MODES = 1024 * 513   # include/pss.h: capacity of the fixed device array behind debug_noise_noalloc

SYMBOLS = ["pss_create", "pss_add_field", "pss_add_linear", "pss_add_aux_def", "pss_add_aux_lhs", "pss_set_frame", "pss_add_aux_term", "pss_add_term",
           "pss_set_noise", "pss_set_dealias", "pss_set_replicas", "pss_select_replica", "pss_replicas", "pss_finalize", "pss_bind", "pss_set_field", "pss_step",
           "pss_get_field", "pss_get_field_fourier", "pss_set_field_fourier", "pss_set_step_count", "pss_debug_noise", "pss_debug_noise_noalloc", "pss_profile_step", "pss_uses_fused_kernel", "pss_launch_count", "pss_hermitian_period",
           "pss_model_bytes_per_step", "pss_step_count", "pss_strerror", "pss_last_cuda_error",
           "pss_destroy"]


class _Op(C.Structure):
    _fields_ = [("coef", C.c_double), ("q2_pow", C.c_int), ("invq_pow", C.c_int), ("iq_pow", C.c_int * 3)]


def _op(d):
    o = _Op()
    o.coef = float(d.get("coef", 1.0))
    o.q2_pow = int(d.get("q2_pow", 0))
    o.invq_pow = int(d.get("invq_pow", 0))
    iq = tuple(d.get("iq_pow", (0, 0, 0))) + (0, 0, 0)
    for j in range(3):
        o.iq_pow[j] = int(iq[j])
    return o


_lib = None


def lib():
    """Load (building if needed) libpss.so and declare every entry point of include/pss.h."""
    global _lib
    if _lib is None:
        path = _build.build()
        if not os.path.exists(path):
            raise RuntimeError("libpss.so is missing and could not be built: the CUDA product has no fallback")
        L = C.CDLL(path)
        P = C.c_void_p
        L.pss_create.argtypes = [C.POINTER(P), C.c_int, C.POINTER(C.c_int64), C.POINTER(C.c_double), C.c_double,
                                 C.c_int, C.c_uint64]
        L.pss_add_field.argtypes = [P, C.c_char_p, C.c_int, C.POINTER(C.c_int)]
        L.pss_add_linear.argtypes = [P, C.c_int, C.POINTER(_Op)]
        L.pss_add_aux_def.argtypes = [P, C.c_int, C.POINTER(_Op), C.c_int]
        L.pss_set_frame.argtypes = [P, C.c_int, C.c_int, C.c_int64, C.c_double, C.c_int64, C.c_double]
        L.pss_add_aux_lhs.argtypes = [P, C.c_int, C.POINTER(_Op)]
        L.pss_add_aux_term.argtypes = [P, C.c_int, C.POINTER(_Op), C.c_int, C.POINTER(C.c_int)]
        L.pss_add_term.argtypes = [P, C.c_int, C.POINTER(_Op), C.c_int, C.POINTER(C.c_int)]
        L.pss_set_noise.argtypes = [P, C.c_int, C.c_double, C.c_int]
        L.pss_set_dealias.argtypes = [P, C.c_int]
        L.pss_set_replicas.argtypes = [P, C.c_int]
        L.pss_select_replica.argtypes = [P, C.c_int]
        L.pss_replicas.argtypes = [P]
        L.pss_finalize.argtypes = [P, C.POINTER(C.c_size_t)]
        L.pss_bind.argtypes = [P, P, C.c_size_t, P]
        L.pss_set_field.argtypes = [P, C.c_int, P, C.c_int]
        L.pss_step.argtypes = [P, C.c_int64]
        L.pss_get_field.argtypes = [P, C.c_int, P, C.c_int]
        L.pss_get_field_fourier.argtypes = [P, C.c_int, P, C.c_int]
        L.pss_set_field_fourier.argtypes = [P, C.c_int, P, C.c_int]
        L.pss_set_step_count.argtypes = [P, C.c_uint64]
        L.pss_debug_noise.argtypes = [P, C.c_int, C.c_uint64, P, P]
        L.pss_debug_noise_noalloc.argtypes = [P, C.c_int, C.c_uint64, P, P]
        L.pss_profile_step.argtypes = [P, C.c_int64, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.pss_uses_fused_kernel.argtypes = [P]
        L.pss_launch_count.argtypes = [P]
        L.pss_hermitian_period.argtypes = [P]
        L.pss_hermitian_period.restype = C.c_int64
        L.pss_launch_count.restype = C.c_uint64
        L.pss_model_bytes_per_step.argtypes = [P, C.c_int]
        L.pss_model_bytes_per_step.restype = C.c_double
        L.pss_step_count.argtypes = [P]
        L.pss_step_count.restype = C.c_uint64
        L.pss_strerror.argtypes = [C.c_int]
        L.pss_strerror.restype = C.c_char_p
        L.pss_last_cuda_error.argtypes = [P]
        L.pss_last_cuda_error.restype = C.c_char_p
        L.pss_destroy.argtypes = [P]
        L.pss_destroy.restype = None
        _lib = L
    return _lib


class PssError(RuntimeError):
    def __init__(self, code, detail=""):
        self.code = code
        msg = lib().pss_strerror(code).decode()
        super().__init__("pss error %d: %s%s" % (code, msg, (" [" + detail + "]") if detail else ""))


def _n3(n):
    n = tuple(int(v) for v in n)
    return (C.c_int64 * 3)(*(n + (1, 1, 1))[:3])


class System:
    """One field system on the GPU.  ``n`` and ``dx`` are given x first: (Nx[, Ny[, Nz]])."""

    def __init__(self, n, dx, dt, prec="f32", seed=0, device="cuda:0", stream=None, replicas=1):
        self.n = tuple(int(v) for v in n)
        self.ndim = len(self.n)
        self.prec = {"f32": F32, "f64": F64, F32: F32, F64: F64}[prec]
        self.rdtype = np.float32 if self.prec == F32 else np.float64
        self.cdtype = np.complex64 if self.prec == F32 else np.complex128
        self.device = device
        self._stream = stream
        self._ws = None
        self._h = C.c_void_p()
        dxs = tuple(float(v) for v in dx)
        rc = lib().pss_create(C.byref(self._h), self.ndim, _n3(self.n),
                              (C.c_double * 3)(*(dxs + (1.0, 1.0, 1.0))[:3]), float(dt), self.prec,
                              C.c_uint64(int(seed)))
        if rc != 0:
            raise PssError(rc)
        if int(replicas) != 1:
            self.set_replicas(replicas)
        self.shape = self.n[::-1]
        self.hshape = self.n[::-1][:-1] + (self.n[0] // 2 + 1,)

    def _chk(self, rc):
        if rc != 0:
            detail = lib().pss_last_cuda_error(self._h).decode() if rc == ECUDA else ""
            raise PssError(rc, detail)

    def __del__(self):
        try:
            if self._h:
                lib().pss_destroy(self._h)
                self._h = C.c_void_p()
        except Exception:
            pass

    # ---- field system ----
    def add_field(self, name, dynamic=True):
        fid = C.c_int(-1)
        self._chk(lib().pss_add_field(self._h, name.encode(), int(bool(dynamic)), C.byref(fid)))
        return fid.value

    def add_linear(self, field, op):
        self._chk(lib().pss_add_linear(self._h, int(field), C.byref(_op(op))))

    def add_aux_def(self, aux, op, src):
        self._chk(lib().pss_add_aux_def(self._h, int(aux), C.byref(_op(op)), int(src)))

    def set_frame(self, field, axis, lo_width, lo_value, hi_width, hi_value):
        self._chk(lib().pss_set_frame(self._h, int(field), int(axis), int(lo_width), float(lo_value), int(hi_width), float(hi_value)))

    def add_aux_lhs(self, aux, op):
        self._chk(lib().pss_add_aux_lhs(self._h, int(aux), C.byref(_op(op))))

    def add_aux_term(self, aux, outer, factors):
        factors = [int(f) for f in factors]
        arr = (C.c_int * max(1, len(factors)))(*factors)
        self._chk(lib().pss_add_aux_term(self._h, int(aux), C.byref(_op(outer)), len(factors), arr))

    def add_term(self, field, outer, factors):
        factors = [int(f) for f in factors]
        arr = (C.c_int * max(1, len(factors)))(*factors)
        self._chk(lib().pss_add_term(self._h, int(field), C.byref(_op(outer)), len(factors), arr))

    def set_noise(self, field, D, q_power):
        self._chk(lib().pss_set_noise(self._h, int(field), float(D), int(q_power)))

    def set_replicas(self, nreplicas):
        """ensemble of independent realisations (replica r = seed + r), stepped together; before finalize"""
        self._chk(lib().pss_set_replicas(self._h, int(nreplicas)))

    def select_replica(self, r):
        self._chk(lib().pss_select_replica(self._h, int(r)))

    @property
    def replicas(self):
        return int(lib().pss_replicas(self._h))

    def set_dealias(self, rule):
        self._chk(lib().pss_set_dealias(self._h, int(rule)))

    def finalize(self, bind=True):
        """pss_finalize, then (by default) allocate the workspace with torch and pss_bind it."""
        ws = C.c_size_t(0)
        self._chk(lib().pss_finalize(self._h, C.byref(ws)))
        self.workspace_bytes = ws.value
        if bind:
            self.bind()
        return ws.value

    def bind(self):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("pss: no CUDA device; the product path has no CPU fallback")
        dev = torch.device(self.device)
        self._ws = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=dev)
        ptr = (self._ws.data_ptr() + 255) // 256 * 256
        with torch.cuda.device(dev):
            st = self._stream if self._stream is not None else torch.cuda.current_stream(dev)
        self._torch_stream = st
        self._chk(lib().pss_bind(self._h, C.c_void_p(ptr), self.workspace_bytes, C.c_void_p(st.cuda_stream)))

    # ---- data in / step / data out ----
    def set_field(self, field, arr):
        """arr: numpy array (host) or torch CUDA tensor (device), shaped n[::-1], of the system precision."""
        if hasattr(arr, "data_ptr"):
            t = arr.contiguous()
            assert t.is_cuda and t.numel() == int(np.prod(self.shape)) and t.element_size() == np.dtype(self.rdtype).itemsize
            self._chk(lib().pss_set_field(self._h, int(field), C.c_void_p(t.data_ptr()), 1))
            return
        a = np.ascontiguousarray(np.asarray(arr), dtype=self.rdtype)
        assert a.size == int(np.prod(self.shape)), (a.shape, self.shape)
        self._chk(lib().pss_set_field(self._h, int(field), a.ctypes.data_as(C.c_void_p), 0))

    def step(self, n=1):
        self._chk(lib().pss_step(self._h, int(n)))

    def get_field(self, field, out=None):
        """Returns a numpy array; or fills ``out`` (numpy host array or torch CUDA tensor) in place."""
        if out is not None and hasattr(out, "data_ptr"):
            assert out.is_cuda and out.is_contiguous() and out.numel() == int(np.prod(self.shape))
            self._chk(lib().pss_get_field(self._h, int(field), C.c_void_p(out.data_ptr()), 1))
            return out
        if out is None:
            out = np.empty(self.shape, dtype=self.rdtype)
        assert out.dtype == self.rdtype and out.flags["C_CONTIGUOUS"]
        self._chk(lib().pss_get_field(self._h, int(field), out.ctypes.data_as(C.c_void_p), 0))
        return out

    def get_field_fourier(self, field):
        out = np.empty(self.hshape, dtype=self.cdtype)
        self._chk(lib().pss_get_field_fourier(self._h, int(field), out.ctypes.data_as(C.c_void_p), 0))
        return out

    def set_field_fourier(self, field, spec):
        """restore a half-spectrum written by get_field_fourier (numpy complex array, logical layout)"""
        a = np.ascontiguousarray(np.asarray(spec), dtype=self.cdtype)
        assert a.shape == tuple(self.hshape), (a.shape, self.hshape)
        self._chk(lib().pss_set_field_fourier(self._h, int(field), a.ctypes.data_as(C.c_void_p), 0))

    def set_step_count(self, step):
        self._chk(lib().pss_set_step_count(self._h, C.c_uint64(int(step))))

    def debug_noise(self, field, step):
        nm = int(np.prod(self.hshape))
        bits = np.empty((nm, 4), dtype=np.uint32)
        z = np.empty(self.hshape, dtype=self.cdtype)
        self._chk(lib().pss_debug_noise(self._h, int(field), C.c_uint64(int(step)),
                                        bits.ctypes.data_as(C.c_void_p), z.ctypes.data_as(C.c_void_p)))
        return bits.reshape(self.hshape + (4,)), z

    def debug_noise_noalloc(self, field, step):
        """``debug_noise`` for processes that must not, or cannot, call cudaMalloc/cudaFree (a framework's memory pool
        owns the GPU, a device-wide synchronisation is unaffordable, or a graph capture is under way elsewhere in the
        process): pss_debug_noise_noalloc stages the values in a fixed 16 MiB device array that is part of libpss.so.
        Same values as ``debug_noise``.  At most STATIC_NOISE_MAX_MODES modes (PssError ETOOBIG beyond); one array per
        GPU, so do not run two of these calls at the same time on one GPU.  Make the first call on each GPU at set-up
        time, before any stream capture."""
        nm = int(np.prod(self.hshape))
        bits = np.empty((nm, 4), dtype=np.uint32)
        z = np.empty(self.hshape, dtype=self.cdtype)
        self._chk(lib().pss_debug_noise_noalloc(self._h, int(field), C.c_uint64(int(step)),
                                                bits.ctypes.data_as(C.c_void_p), z.ctypes.data_as(C.c_void_p)))
        return bits.reshape(self.hshape + (4,)), z

    def profile_step(self, n):
        """n steps with a CUDA-event pair around every launch -> {kernel: (mean ms per launch, launches)}."""
        ms = (C.c_double * 4)()
        cnt = (C.c_int64 * 4)()
        self._chk(lib().pss_profile_step(self._h, int(n), ms, cnt))
        return {k: (ms[i], int(cnt[i])) for i, k in enumerate(("k_rows", "k_update", "k_mid", "k_fused2d"))}

    @property
    def uses_fused_kernel(self):
        return bool(lib().pss_uses_fused_kernel(self._h))

    @property
    def fused_kernel_name(self):
        """None, or the persistent kernel that runs the steps"""
        return {0: None, 1: "k_fused2d", 2: "k_persist2d"}[int(lib().pss_uses_fused_kernel(self._h))]

    def synchronize(self):
        self._torch_stream.synchronize()

    @property
    def step_count(self):
        return int(lib().pss_step_count(self._h))

    @property
    def hermitian_period(self):
        """pss_step projects the planes kx = 0 and kx = n0/2 of the state onto Hermitian symmetry after every step whose
        number is a multiple of this (include/pss.h, pss_hermitian_period)"""
        return int(lib().pss_hermitian_period(self._h))

    @property
    def launch_count(self):
        return int(lib().pss_launch_count(self._h))

    def model_bytes_per_step(self, pruned=True):
        return float(lib().pss_model_bytes_per_step(self._h, int(bool(pruned))))
