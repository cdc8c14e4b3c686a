"""ctypes binding of the CPU oracle (oracle/libopss.so).

TEST INFRASTRUCTURE ONLY: imported by tests/, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of bench.py.  Nothing under
paper_2405_02410_b200/ imports this module, and this module imports nothing from there.

Method names mirror the C ABI (opss.h) and the product binding, so one driver can build the
same field system on both sides.  Operators are plain dicts
``{"coef": c, "q2_pow": m, "invq_pow": p, "iq_pow": (ax, ay, az)}`` (missing keys = 0, coef = 1).
"""
import ctypes as C
import numpy as np

from . import build as _build  # oracle/build.py

F32, F64 = 0, 1
DEALIAS_PAPER, DEALIAS_TWO_THIRDS, DEALIAS_OFF = 0, 1, 2
OK, EINVAL, EUNSUPPORTED, ESTATE = 0, -1, -2, -3


class _Op(C.Structure):
    _fields_ = [("coef", C.c_double), ("q2_pow", C.c_int), ("invq_pow", C.c_int),
                ("iq_pow", C.c_int * 3)]


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
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        P = C.c_void_p
        L.opss_create.argtypes = [C.POINTER(P), C.c_int, C.POINTER(C.c_int64), C.POINTER(C.c_double),
                                  C.c_double, C.c_int, C.c_uint64]
        L.opss_add_field.argtypes = [P, C.c_char_p, C.c_int, C.POINTER(C.c_int)]
        L.opss_add_linear.argtypes = [P, C.c_int, C.POINTER(_Op)]
        L.opss_add_aux_def.argtypes = [P, C.c_int, C.POINTER(_Op), C.c_int]
        L.opss_add_term.argtypes = [P, C.c_int, C.POINTER(_Op), C.c_int, C.POINTER(C.c_int)]
        L.opss_set_frame.argtypes = [P, C.c_int, C.c_int, C.c_int64, C.c_double, C.c_int64, C.c_double]
        L.opss_add_aux_lhs.argtypes = [P, C.c_int, C.POINTER(_Op)]
        L.opss_add_aux_term.argtypes = [P, C.c_int, C.POINTER(_Op), C.c_int, C.POINTER(C.c_int)]
        L.opss_set_noise.argtypes = [P, C.c_int, C.c_double, C.c_int]
        L.opss_set_dealias.argtypes = [P, C.c_int]
        L.opss_finalize.argtypes = [P, C.POINTER(C.c_size_t)]
        L.opss_set_field.argtypes = [P, C.c_int, P]
        L.opss_set_threads.argtypes = [P, C.c_int]
        L.opss_step.argtypes = [P, C.c_int64]
        L.opss_get_field.argtypes = [P, C.c_int, P]
        L.opss_get_field_fourier.argtypes = [P, C.c_int, P]
        L.opss_get_field_fourier_f64.argtypes = [P, C.c_int, P]
        L.opss_debug_noise.argtypes = [P, C.c_int, C.c_uint64, P, P]
        L.opss_step_count.argtypes = [P]
        L.opss_step_count.restype = C.c_uint64
        L.opss_strerror.argtypes = [C.c_int]
        L.opss_strerror.restype = C.c_char_p
        L.opss_destroy.argtypes = [P]
        L.opss_destroy.restype = None
        L.opss_debug_fft_lines.argtypes = [P, C.c_int64, C.c_int64, C.c_int]
        L.opss_debug_r2c.argtypes = [P, P, C.c_int, C.POINTER(C.c_int64)]
        L.opss_debug_c2r.argtypes = [P, P, C.c_int, C.POINTER(C.c_int64)]
        L.opss_debug_op.argtypes = [P, C.POINTER(_Op), C.POINTER(C.c_int64), C.POINTER(C.c_double)]
        L.opss_debug_mask.argtypes = [P, C.c_int, P]
        L.opss_debug_philox.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.opss_debug_philox.restype = None
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code):
        self.code = code
        super().__init__("opss error %d: %s" % (code, lib().opss_strerror(code).decode()))


def _chk(rc):
    if rc != 0:
        raise OracleError(rc)


def _n3(n):
    n = tuple(int(v) for v in n)
    return (C.c_int64 * 3)(*(n + (1, 1, 1))[:3])


class System:
    """One field system on the oracle.  ``n`` and ``dx`` are given x first: (Nx[, Ny[, Nz]])."""

    def __init__(self, n, dx, dt, prec="f32", seed=0):
        self.n = tuple(int(v) for v in n)
        self.ndim = len(self.n)
        self.prec = {"f32": F32, "f64": F64, F32: F32, F64: F64}[prec]
        self.rdtype = np.float32 if self.prec == F32 else np.float64
        self.cdtype = np.complex64 if self.prec == F32 else np.complex128
        self._h = C.c_void_p()
        dxs = tuple(float(v) for v in dx)
        rc = lib().opss_create(C.byref(self._h), self.ndim, _n3(self.n),
                               (C.c_double * 3)(*(dxs + (1.0, 1.0, 1.0))[:3]), float(dt), self.prec,
                               C.c_uint64(int(seed)))
        _chk(rc)
        self.shape = self.n[::-1]
        self.hshape = self.n[::-1][:-1] + (self.n[0] // 2 + 1,)

    def __del__(self):
        try:
            if self._h:
                lib().opss_destroy(self._h)
                self._h = C.c_void_p()
        except Exception:
            pass

    def add_field(self, name, dynamic=True):
        fid = C.c_int(-1)
        _chk(lib().opss_add_field(self._h, name.encode(), int(bool(dynamic)), C.byref(fid)))
        return fid.value

    def add_linear(self, field, op):
        _chk(lib().opss_add_linear(self._h, int(field), C.byref(_op(op))))

    def add_aux_def(self, aux, op, src):
        _chk(lib().opss_add_aux_def(self._h, int(aux), C.byref(_op(op)), int(src)))

    def set_frame(self, field, axis, lo_width, lo_value, hi_width, hi_value):
        _chk(lib().opss_set_frame(self._h, int(field), int(axis), int(lo_width), float(lo_value), int(hi_width), float(hi_value)))

    def add_aux_lhs(self, aux, op):
        _chk(lib().opss_add_aux_lhs(self._h, int(aux), C.byref(_op(op))))

    def add_aux_term(self, aux, outer, factors):
        factors = [int(f) for f in factors]
        arr = (C.c_int * max(1, len(factors)))(*factors)
        _chk(lib().opss_add_aux_term(self._h, int(aux), C.byref(_op(outer)), len(factors), arr))

    def add_term(self, field, outer, factors):
        factors = [int(f) for f in factors]
        arr = (C.c_int * max(1, len(factors)))(*factors)
        _chk(lib().opss_add_term(self._h, int(field), C.byref(_op(outer)), len(factors), arr))

    def set_noise(self, field, D, q_power):
        _chk(lib().opss_set_noise(self._h, int(field), float(D), int(q_power)))

    def set_dealias(self, rule):
        _chk(lib().opss_set_dealias(self._h, int(rule)))

    def finalize(self):
        ws = C.c_size_t(0)
        _chk(lib().opss_finalize(self._h, C.byref(ws)))
        return ws.value

    def set_threads(self, n):
        _chk(lib().opss_set_threads(self._h, int(n)))

    def set_field(self, field, arr):
        a = np.ascontiguousarray(np.asarray(arr), dtype=self.rdtype)
        assert a.size == int(np.prod(self.shape)), (a.shape, self.shape)
        _chk(lib().opss_set_field(self._h, int(field), a.ctypes.data_as(C.c_void_p)))

    def step(self, n=1):
        _chk(lib().opss_step(self._h, int(n)))

    def get_field(self, field):
        out = np.empty(self.shape, dtype=self.rdtype)
        _chk(lib().opss_get_field(self._h, int(field), out.ctypes.data_as(C.c_void_p)))
        return out

    def get_field_fourier(self, field):
        out = np.empty(self.hshape, dtype=self.cdtype)
        _chk(lib().opss_get_field_fourier(self._h, int(field), out.ctypes.data_as(C.c_void_p)))
        return out

    def get_field_fourier_f64(self, field):
        out = np.empty(self.hshape, dtype=np.complex128)
        _chk(lib().opss_get_field_fourier_f64(self._h, int(field), out.ctypes.data_as(C.c_void_p)))
        return out

    def debug_noise(self, field, step):
        nm = int(np.prod(self.hshape))
        bits = np.empty((nm, 4), dtype=np.uint32)
        z = np.empty(self.hshape, dtype=np.complex128)
        _chk(lib().opss_debug_noise(self._h, int(field), C.c_uint64(int(step)),
                                    bits.ctypes.data_as(C.c_void_p), z.ctypes.data_as(C.c_void_p)))
        return bits.reshape(self.hshape + (4,)), z

    def debug_op(self, op, k):
        out = (C.c_double * 2)()
        _chk(lib().opss_debug_op(self._h, C.byref(_op(op)), _n3(tuple(k) + (0, 0, 0)), out))
        return complex(out[0], out[1])

    def debug_mask(self, field):
        m = np.empty(self.hshape, dtype=np.uint8)
        rc = lib().opss_debug_mask(self._h, int(field), m.ctypes.data_as(C.c_void_p))
        if rc == 1:
            return None
        _chk(rc)
        return m

    @property
    def step_count(self):
        return int(lib().opss_step_count(self._h))


def fft_lines(data, sign):
    """complex DFT of each row of a 2-D complex128 array (oracle's own FFT)."""
    a = np.array(data, dtype=np.complex128, order="C", copy=True)
    a2 = a.reshape(-1, a.shape[-1])
    _chk(lib().opss_debug_fft_lines(a2.ctypes.data_as(C.c_void_p), a2.shape[1], a2.shape[0], int(sign)))
    return a


def r2c(real):
    """oracle R2C of a real array shaped (Nz, Ny, Nx) / (Ny, Nx) / (Nx,)."""
    a = np.ascontiguousarray(real, dtype=np.float64)
    n = a.shape[::-1]
    out = np.empty(a.shape[:-1] + (a.shape[-1] // 2 + 1,), dtype=np.complex128)
    _chk(lib().opss_debug_r2c(a.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p), a.ndim, _n3(n)))
    return out


def c2r(half, nx):
    a = np.ascontiguousarray(half, dtype=np.complex128)
    shape = a.shape[:-1] + (int(nx),)
    out = np.empty(shape, dtype=np.float64)
    _chk(lib().opss_debug_c2r(a.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p), a.ndim, _n3(shape[::-1])))
    return out


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) for v in key])
    o = (C.c_uint32 * 4)()
    lib().opss_debug_philox(c, k, o)
    return tuple(int(v) for v in o)
