"""ctypes wrapper around oracle/fdtd_oracle.cpp.

TEST INFRASTRUCTURE — NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It never imports the product package
(paper_2603_24027_b200) and the product never imports it.

Argument marshalling only: every number is computed by the C++ oracle, whose functions cite the
passages of PAPER.md they follow.  Field containers are float64 numpy arrays of shape (6, nx, ny, nz)
(Ex,Ey,Ez,Hx,Hy,Hz; z fastest), also for the float32 oracle (values are exactly representable).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

# store dtype ids (0..3 = the product's; 4 = "native", i.e. an uncompressed copy in the oracle's own
# precision; >= 10 = the paper's unscaled float8 flavours)
F32, F16, BF16, E4M3_SCALED, NATIVE = 0, 1, 2, 3, 4
# 5 = micro-scaled e4m3: blocks of 32 values share a power-of-two scale, stored as one byte X + 127 after the codes
E4M3_MX32 = 5
MX_BLOCK = 32
E4M3B11FNUZ, E5M2FNUZ, E4M3FNUZ, E4M3, E3M4, E4M3FN = 10, 11, 12, 13, 14, 15
STORE_ALL, STORE_TANGENTIAL = 0, 1
LINEAR, CUBIC = 0, 1
# reverse modes: the method / plain definition from store-all snapshots / pure time reversal (P = 0)
METHOD, STORE_ALL, PURE_REVERSAL = 0, 1, 2

# CPML defaults (reading R5; the paper prints none): sigma_factor, kappa_max, alpha_max, grading order
CPML_DEFAULTS = (0.8, 1.0, 0.01, 3.0)

_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(_build.build())
    dp = C.POINTER(C.c_double)
    ip = C.POINTER(C.c_int)
    vp = C.c_void_p
    L.orc_create.restype = vp
    L.orc_create.argtypes = [C.c_int] * 5 + [C.c_double, dp] + [C.c_double] * 4
    L.orc_destroy.argtypes = [vp]
    L.orc_reset.argtypes = [vp]
    L.orc_set_design.argtypes = [vp, ip, ip]
    L.orc_set_store_mode.argtypes = [vp, C.c_int]
    L.orc_set_monitor.argtypes = [vp, ip, ip, C.c_uint]
    L.orc_clear_sources.argtypes = [vp]
    L.orc_add_source.argtypes = [vp, C.c_int, ip, ip, dp, dp, C.c_int]
    L.orc_set_keep_all.argtypes = [vp, C.c_int]
    L.orc_forward.argtypes = [vp, C.c_int, C.c_int, C.c_int]
    L.orc_reverse.argtypes = [vp, dp, dp, C.c_int, C.c_int, dp]
    L.orc_get_fields.argtypes = [vp, dp]
    L.orc_set_fields.argtypes = [vp, dp]
    L.orc_get_adjoint.argtypes = [vp, dp]
    L.orc_get_monitor.argtypes = [vp, dp]
    L.orc_monitor_size.restype = C.c_size_t
    L.orc_monitor_size.argtypes = [vp]
    L.orc_store_bytes.restype = C.c_size_t
    L.orc_store_bytes.argtypes = [vp]
    L.orc_num_slots.argtypes = [vp]
    L.orc_slot_values.restype = C.c_size_t
    L.orc_slot_values.argtypes = [vp]
    L.orc_slot_step.argtypes = [vp, C.c_int]
    L.orc_get_slot.argtypes = [vp, C.c_int, C.c_void_p, C.c_void_p]
    L.orc_slot_bytes.restype = C.c_size_t
    L.orc_slot_bytes.argtypes = [vp, C.c_int]
    L.orc_block_offset.restype = C.c_size_t
    L.orc_block_offset.argtypes = [vp, C.c_int, C.c_int]
    L.orc_encode_mx.argtypes = [C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p]
    L.orc_decode_mx.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
    L.orc_slice_offset.restype = C.c_size_t
    L.orc_slice_offset.argtypes = [vp, C.c_int, C.c_int]
    L.orc_face_size.restype = C.c_size_t
    L.orc_face_size.argtypes = [vp, C.c_int]
    L.orc_fetch.restype = C.c_double
    L.orc_fetch.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_size_t, C.c_int]
    L.orc_fetch_face.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, dp]
    L.orc_get_tables.argtypes = [vp, C.c_int, dp]
    L.orc_apply_step.argtypes = [vp, dp, dp]
    L.orc_apply_step_transpose.argtypes = [vp, dp, dp]
    L.orc_elem_bytes.argtypes = [C.c_int]
    L.orc_encode.argtypes = [C.c_int, C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p]
    L.orc_decode.argtypes = [C.c_int, C.c_void_p, C.c_size_t, C.c_float, C.c_void_p]
    L.orc_decode_code.restype = C.c_double
    L.orc_decode_code.argtypes = [C.c_int, C.c_uint]
    L.orc_encode_value.restype = C.c_uint
    L.orc_encode_value.argtypes = [C.c_int, C.c_double]
    L.orc_format_max.restype = C.c_double
    L.orc_format_max.argtypes = [C.c_int]
    L.orc_lerp.restype = C.c_float
    L.orc_lerp.argtypes = [C.c_float, C.c_float, C.c_int, C.c_int]
    L.orc_cubic.restype = C.c_float
    L.orc_cubic.argtypes = [C.c_float] * 4 + [C.c_int, C.c_int]
    L.orc_lerp64.restype = C.c_double
    L.orc_lerp64.argtypes = [C.c_double, C.c_double, C.c_int, C.c_int]
    L.orc_cubic64.restype = C.c_double
    L.orc_cubic64.argtypes = [C.c_double] * 4 + [C.c_int, C.c_int]
    L.orc_set_threads.argtypes = [C.c_int]
    L.orc_get_threads.restype = C.c_int
    _lib = L
    return L


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _i3(v):
    return (C.c_int * 3)(*[int(x) for x in v])


def courant_number(dx, dt):
    """S = c*dt/dx  (eq. 1 gives dt = C*dx/(c*sqrt(3)), so S = C/sqrt(3))."""
    return 299792458.0 * dt / dx


def cfl_dt(dx, courant_factor=0.99):
    """PAPER.md:39 eq. (1)."""
    return courant_factor * dx / (299792458.0 * np.sqrt(3.0))


def set_threads(n):
    lib().orc_set_threads(int(n))


def get_threads():
    return lib().orc_get_threads()


class OracleSim:
    """One oracle simulation.  prec = 32 or 64 (the arithmetic type of every field update)."""

    def __init__(self, prec, eps, P, S, cpml=CPML_DEFAULTS):
        eps = np.ascontiguousarray(eps, dtype=np.float64)
        assert eps.ndim == 3 and prec in (32, 64)
        self.prec, self.shape, self.P, self.S = prec, eps.shape, int(P), float(S)
        self.N = eps.size
        self._h = lib().orc_create(prec, eps.shape[0], eps.shape[1], eps.shape[2], int(P), float(S), _dp(eps),
                                   *[float(x) for x in cpml])
        self.design = None
        self.monitor = None

    def __del__(self):
        if getattr(self, "_h", None) and lib is not None:   # at interpreter exit the module globals may be gone already
            lib().orc_destroy(self._h)
            self._h = None

    # ---- configuration ----
    def reset(self):
        lib().orc_reset(self._h)

    def set_design(self, lo, hi):
        self.design = (tuple(lo), tuple(hi))
        lib().orc_set_design(self._h, _i3(lo), _i3(hi))

    def set_store_mode(self, mode):
        """STORE_ALL (0, default) or STORE_TANGENTIAL (1): only the two tangential H components on the low faces and the two
        tangential E components on the high faces are stored and injected; the design box must then avoid the shell."""
        self.store_mode = int(mode)
        lib().orc_set_store_mode(self._h, int(mode))

    def set_monitor(self, lo, hi, comp_mask):
        self.monitor = (tuple(lo), tuple(hi), int(comp_mask))
        lib().orc_set_monitor(self._h, _i3(lo), _i3(hi), int(comp_mask))

    def clear_sources(self):
        lib().orc_clear_sources(self._h)

    def add_source(self, comp, lo, hi, amp, wave):
        wave = np.ascontiguousarray(wave, dtype=np.float64)
        a = None if amp is None else np.ascontiguousarray(amp, dtype=np.float64)
        lib().orc_add_source(self._h, int(comp), _i3(lo), _i3(hi), None if a is None else _dp(a), _dp(wave), wave.size)

    def set_keep_all(self, on):
        lib().orc_set_keep_all(self._h, int(bool(on)))

    # ---- runs ----
    def forward(self, nsteps, dtype=F32, k=1):
        self.nsteps = int(nsteps)
        lib().orc_forward(self._h, int(nsteps), int(dtype), int(k))

    def reverse(self, dfinal=None, dmon=None, interp=LINEAR, mode=METHOD):
        """Returns grad_eps over the design box (float64, shape hi-lo), or None without a design box."""
        df = None if dfinal is None else np.ascontiguousarray(dfinal, dtype=np.float64)
        dm = None if dmon is None else np.ascontiguousarray(dmon, dtype=np.float64)
        if df is not None:
            assert df.size == 6 * self.N
        if dm is not None:
            assert dm.size == lib().orc_monitor_size(self._h)
        g = None
        if self.design is not None:
            lo, hi = self.design
            if getattr(self, "store_mode", 0) == STORE_TANGENTIAL and mode == METHOD:
                assert all(lo[a] >= self.P + 1 and hi[a] <= self.shape[a] - self.P - 1 for a in range(3)), \
                    "tangential store: the design box must lie in the inner interior (the shell is not reconstructed)"
            g = np.zeros([hi[a] - lo[a] for a in range(3)], dtype=np.float64)
        lib().orc_reverse(self._h, None if df is None else _dp(df), None if dm is None else _dp(dm), int(interp),
                          int(mode), None if g is None else _dp(g))
        return g

    # ---- state access ----
    def fields(self):
        out = np.empty((6,) + self.shape, dtype=np.float64)
        lib().orc_get_fields(self._h, _dp(out))
        return out

    def set_fields(self, f):
        f = np.ascontiguousarray(f, dtype=np.float64)
        assert f.size == 6 * self.N
        lib().orc_set_fields(self._h, _dp(f))

    def adjoint(self):
        out = np.empty((6,) + self.shape, dtype=np.float64)
        lib().orc_get_adjoint(self._h, _dp(out))
        return out

    def monitor_record(self):
        lo, hi, mask = self.monitor
        ncomp = bin(mask).count("1")
        out = np.empty((self.nsteps, ncomp) + tuple(hi[a] - lo[a] for a in range(3)), dtype=np.float64)
        assert out.size == lib().orc_monitor_size(self._h)
        lib().orc_get_monitor(self._h, _dp(out))
        return out

    # ---- store ----
    def store_bytes(self):
        return lib().orc_store_bytes(self._h)

    def num_slots(self):
        return lib().orc_num_slots(self._h)

    def slot_values(self):
        return lib().orc_slot_values(self._h)

    def slot_step(self, j):
        return lib().orc_slot_step(self._h, j)

    def slot(self, j, dtype):
        """(raw bytes as uint8 array, 36 float32 scales) of stored slot j.  E4M3_MX32: the bytes are the slot_values codes
        followed by the block-scale bytes (block_offset gives a slice's first block)."""
        data = np.empty(lib().orc_slot_bytes(self._h, j), dtype=np.uint8)
        scales = np.empty(36, dtype=np.float32)
        lib().orc_get_slot(self._h, j, data.ctypes.data, scales.ctypes.data)
        return data, scales

    def block_offset(self, face, comp):
        return lib().orc_block_offset(self._h, face, comp)

    def slice_offset(self, face, comp):
        return lib().orc_slice_offset(self._h, face, comp)

    def face_size(self, face):
        return lib().orc_face_size(self._h, face)

    def fetch(self, nstate, face, comp, e, interp=LINEAR):
        return lib().orc_fetch(self._h, nstate, face, comp, e, interp)

    def fetch_face(self, nstate, face, comp, interp=LINEAR):
        out = np.empty(self.face_size(face), dtype=np.float64)
        lib().orc_fetch_face(self._h, nstate, face, comp, interp, _dp(out))
        return out

    def tables(self, axis):
        out = np.empty((6, self.shape[axis]), dtype=np.float64)
        lib().orc_get_tables(self._h, axis, _dp(out))
        return out

    # ---- single-step operators (dot-product test); vector = [E(3N) | H(3N) | psiE(6N) | psiH(6N)] ----
    def apply_step(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        y = np.empty(18 * self.N)
        lib().orc_apply_step(self._h, _dp(x), _dp(y))
        return y

    def apply_step_transpose(self, y):
        y = np.ascontiguousarray(y, dtype=np.float64)
        x = np.empty(18 * self.N)
        lib().orc_apply_step_transpose(self._h, _dp(y), _dp(x))
        return x


# ---- standalone codec ----
def elem_bytes(dtype):
    return lib().orc_elem_bytes(dtype)


def encode(dtype, x):
    """Encode one slice of float32 values; returns (codes as uint8 byte array, float32 scale)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    out = np.empty(x.size * elem_bytes(dtype), dtype=np.uint8)
    sc = np.empty(1, dtype=np.float32)
    lib().orc_encode(dtype, x.ctypes.data, x.size, out.ctypes.data, sc.ctypes.data)
    return out, sc[0]


def decode(dtype, codes, scale=1.0):
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    n = codes.size // elem_bytes(dtype)
    out = np.empty(n, dtype=np.float32)
    lib().orc_decode(dtype, codes.ctypes.data, n, float(scale), out.ctypes.data)
    return out


def encode_mx(x):
    """Micro-scaled e4m3 of one slice: (codes uint8 [n], block-scale bytes uint8 [ceil(n/32)], byte = X + 127)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    codes = np.empty(x.size, dtype=np.uint8)
    bs = np.empty((x.size + MX_BLOCK - 1) // MX_BLOCK, dtype=np.uint8)
    lib().orc_encode_mx(x.ctypes.data, x.size, codes.ctypes.data, bs.ctypes.data)
    return codes, bs


def decode_mx(codes, bscale):
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    bscale = np.ascontiguousarray(bscale, dtype=np.uint8)
    out = np.empty(codes.size, dtype=np.float32)
    lib().orc_decode_mx(codes.ctypes.data, bscale.ctypes.data, codes.size, out.ctypes.data)
    return out


def decode_code(dtype, code):
    return lib().orc_decode_code(dtype, int(code))


def encode_value(dtype, x):
    return lib().orc_encode_value(dtype, float(x))


def format_max(dtype):
    return lib().orc_format_max(dtype)


def lerp(a, b, num, den):
    return lib().orc_lerp(a, b, num, den)


def cubic(vm1, v0, v1, v2, num, den):
    return lib().orc_cubic(vm1, v0, v1, v2, num, den)


def lerp64(a, b, num, den):
    return lib().orc_lerp64(a, b, num, den)


def cubic64(vm1, v0, v1, v2, num, den):
    return lib().orc_cubic64(vm1, v0, v1, v2, num, den)
