"""Thin Python binding of libfdtd_b200.so (include/fdtd.h): argument marshalling only.

PyTorch is used for device memory (the workspace, inputs, outputs) and the CUDA stream; every step of the path
runs in the library's sm_100a kernels.  There is no CPU fallback: a missing library or a missing CUDA device raises.
Function names mirror the C ABI (fdtd_create -> Sim(...), fdtd_forward -> Sim.forward, ...).
"""
import ctypes as C
import os

import numpy as np

F32, F16, BF16, F8E4M3_SCALED = 0, 1, 2, 3
# micro-scaled E4M3: blocks of 32 values share a power-of-two scale byte kept behind the slot's codes (R20)
F8E4M3_MX32 = 5
# the paper's unscaled float8 flavours
F8E4M3B11FNUZ, F8E5M2FNUZ, F8E4M3FNUZ, F8E4M3, F8E3M4 = 10, 11, 12, 13, 14
LINEAR, CUBIC = 0, 1
STORE_ALL, STORE_TANGENTIAL = 0, 1
WS_REVERSE, WS_HOST_IO = 1, 2
NOALLOC_MAX_SLICES = 4096   # FDTD_NOALLOC_MAX_SLICES (include/fdtd.h)
WS_GUARD = 4   # debugging aid (include/fdtd_bench.h): guard bands + 0xFF fill
STATUS = {0: "FDTD_OK", 1: "FDTD_ERR_INVALID_ARG", 2: "FDTD_ERR_OOM", 3: "FDTD_ERR_CUDA", 4: "FDTD_ERR_STATE",
          5: "FDTD_ERR_UNSUPPORTED"}
ELEM_BYTES = {F32: 4, F16: 2, BF16: 2, F8E4M3_SCALED: 1, F8E4M3_MX32: 1, F8E4M3B11FNUZ: 1, F8E5M2FNUZ: 1, F8E4M3FNUZ: 1, F8E4M3: 1,
              F8E3M4: 1}

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libfdtd_b200.so")


class FdtdError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class _Source(C.Structure):
    _fields_ = [("comp", C.c_int), ("lo", C.c_int * 3), ("hi", C.c_int * 3), ("amp", C.c_void_p), ("wave", C.c_void_p)]


class _Cotangent(C.Structure):
    _fields_ = [("lo", C.c_int * 3), ("hi", C.c_int * 3), ("comp_mask", C.c_uint), ("g_dev", C.c_void_p)]


_lib = None


def lib():
    """Load the C-ABI library (built in-tree by paper_2603_24027_b200/build.py).  Fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FdtdError(5, f"{LIB_PATH} is missing: run `python -m paper_2603_24027_b200.build` "
                           "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(LIB_PATH)
    vp, i3 = C.c_void_p, C.POINTER(C.c_int)
    L.fdtd_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, vp, vp]
    L.fdtd_forward.argtypes = [vp, C.c_int, C.POINTER(_Source), C.c_int, C.c_int, C.c_int]
    L.fdtd_reverse.argtypes = [vp, C.POINTER(_Cotangent), vp, C.c_int, vp]
    L.fdtd_store_bytes.restype = C.c_size_t
    L.fdtd_store_bytes.argtypes = [vp]
    L.fdtd_set_cpml.argtypes = [vp] + [C.c_double] * 4
    L.fdtd_set_design.argtypes = [vp, i3, i3]
    L.fdtd_set_monitor.argtypes = [vp, i3, i3, C.c_uint, vp]
    L.fdtd_workspace_bytes.restype = C.c_size_t
    L.fdtd_workspace_bytes.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_uint]
    L.fdtd_set_workspace.argtypes = [vp, vp, C.c_size_t, C.c_int, C.c_int, C.c_int, C.c_uint]
    L.fdtd_set_eps.argtypes = [vp, vp]
    L.fdtd_reset.argtypes = [vp]
    L.fdtd_set_graphs.argtypes = [vp, C.c_int]
    L.fdtd_set_fused.argtypes = [vp, C.c_int, C.c_int]
    L.fdtd_uses_fused.argtypes = [vp, C.c_int]
    L.fdtd_uses_fused_reverse.argtypes = [vp]
    L.fdtd_uses_fused_adjoint.argtypes = [vp]
    L.fdtd_set_rows.argtypes = [vp, C.c_int]
    L.fdtd_set_store_mode.argtypes = [vp, C.c_int]
    L.fdtd_get_fields.argtypes = [vp, vp]
    L.fdtd_get_adjoint.argtypes = [vp, vp]
    L.fdtd_get_box.argtypes = [vp, i3, i3, C.c_uint, vp]
    L.fdtd_num_slots.argtypes = [vp]
    L.fdtd_slot_values.restype = C.c_size_t
    L.fdtd_slot_values.argtypes = [vp]
    L.fdtd_slot_ptr.argtypes = [vp, C.c_int, C.POINTER(vp), C.POINTER(vp)]
    L.fdtd_slot_bytes.restype = C.c_size_t
    L.fdtd_slot_bytes.argtypes = [vp, C.c_int]
    L.fdtd_set_eps_host.argtypes = [vp, vp]
    L.fdtd_forward_host.argtypes = [vp, C.c_int, C.POINTER(_Source), C.c_int, C.c_int, C.c_int, vp]
    L.fdtd_reverse_host.argtypes = [vp, vp, C.c_int, vp]
    L.fdtd_codec_encode.argtypes = [C.c_int, vp, C.c_size_t, vp, vp, vp, vp]
    L.fdtd_codec_fetch.argtypes = [C.c_int, C.c_int, C.POINTER(vp), C.POINTER(C.c_float), C.c_int, C.c_int, C.c_size_t, vp, vp]
    L.fdtd_codec_encode_slices_noalloc.argtypes = [C.c_int, vp, C.c_int, C.c_size_t, vp, vp, vp]
    L.fdtd_noalloc_last_error.restype = C.c_char_p
    L.fdtd_noalloc_last_error.argtypes = []
    L.fdtd_profile_kernel.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.fdtd_sync.argtypes = [vp]
    L.fdtd_last_error.restype = C.c_char_p
    L.fdtd_last_error.argtypes = [vp]
    L.fdtd_destroy.argtypes = [vp]
    L.fdtd_launch_count.restype = C.c_ulonglong
    L.fdtd_launch_count.argtypes = [vp]
    L.fdtd_debug_guard_check.restype = C.c_longlong
    L.fdtd_debug_guard_check.argtypes = [vp]
    _lib = L
    return L


EXPORTED = ["fdtd_create", "fdtd_forward", "fdtd_reverse", "fdtd_store_bytes", "fdtd_set_cpml", "fdtd_set_design",
            "fdtd_set_monitor", "fdtd_workspace_bytes", "fdtd_set_workspace", "fdtd_set_eps", "fdtd_reset",
            "fdtd_set_graphs", "fdtd_set_fused", "fdtd_set_rows", "fdtd_uses_fused", "fdtd_uses_fused_reverse", "fdtd_uses_fused_adjoint", "fdtd_set_store_mode", "fdtd_get_fields", "fdtd_get_box", "fdtd_get_adjoint", "fdtd_num_slots",
            "fdtd_slot_values", "fdtd_slot_ptr", "fdtd_slot_bytes", "fdtd_set_eps_host", "fdtd_forward_host", "fdtd_reverse_host",
            "fdtd_codec_encode", "fdtd_codec_fetch", "fdtd_codec_encode_slices_noalloc", "fdtd_noalloc_last_error", "fdtd_profile_kernel", "fdtd_sync", "fdtd_last_error", "fdtd_destroy",
            "fdtd_launch_count", "fdtd_debug_guard_check"]


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise FdtdError(3, "no CUDA device: the FDTD path runs only in the sm_100a kernels (no CPU fallback)")
    return torch


def _i3(v):
    return (C.c_int * 3)(*[int(x) for x in v])


def _stream_ptr(torch):
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Sim:
    """fdtd_sim handle.  eps: float32 CUDA tensor [nx,ny,nz] (kept alive by this object).

    Stream rule: the library is bound to the CUDA stream that is current when the object is created, and the tensors this
    binding allocates per call (monitor record, gradient, source amplitudes) are ordered against that stream only.  forward,
    reverse, fields, slot ... therefore raise FDTD_ERR_STATE when called under another torch.cuda.stream(...)."""

    def __init__(self, eps, dx, dt, pml_width, design=None, monitor=None, cpml=None, store_mode=STORE_ALL, rows=-1):
        torch = _torch()
        self._torch = torch
        self._L = lib()
        assert eps.is_cuda and eps.dtype == torch.float32 and eps.is_contiguous() and eps.dim() == 3
        self.eps = eps
        self.shape = tuple(eps.shape)
        self.pml = int(pml_width)
        self._h = C.c_void_p()
        self._stream = torch.cuda.current_stream().cuda_stream
        st = self._L.fdtd_create(C.byref(self._h), *self.shape, float(dx), float(dt), int(pml_width), C.c_void_p(eps.data_ptr()),
                                 _stream_ptr(torch))
        if st != 0:
            raise FdtdError(st, "fdtd_create rejected its arguments")
        self.ws = None
        self.ws_key = None
        self.design = None
        self.monitor = None
        self.mon_rec = None
        self._keep = []
        if cpml is not None:
            self._check(self._L.fdtd_set_cpml(self._h, *[float(x) for x in cpml]))
        self.store_mode = int(store_mode)
        if store_mode != STORE_ALL:
            self._check(self._L.fdtd_set_store_mode(self._h, int(store_mode)))
        if rows != -1:
            self._check(self._L.fdtd_set_rows(self._h, int(rows)))
        if design is not None:
            self.design = (tuple(design[0]), tuple(design[1]))
            self._check(self._L.fdtd_set_design(self._h, _i3(design[0]), _i3(design[1])))
        if monitor is not None:
            self.monitor = (tuple(monitor[0]), tuple(monitor[1]), int(monitor[2]))
            self._check(self._L.fdtd_set_monitor(self._h, _i3(monitor[0]), _i3(monitor[1]), int(monitor[2]), None))

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._torch.cuda.synchronize()
            self._L.fdtd_destroy(self._h)
            self._h = C.c_void_p()

    def _check(self, st):
        if st != 0:
            raise FdtdError(st, self._L.fdtd_last_error(self._h).decode())

    def _same_stream(self):
        if self._torch.cuda.current_stream().cuda_stream != self._stream:
            raise FdtdError(4, "called under another CUDA stream than the one the Sim was created on: tensors allocated by this "
                               "call would not be ordered against the library's stream")

    # ---- workspace ----
    def workspace_bytes(self, nsteps, dtype, k, flags=WS_REVERSE):
        return self._L.fdtd_workspace_bytes(self._h, int(nsteps), int(dtype), int(k), int(flags))

    def set_workspace(self, nsteps, dtype, k, flags=WS_REVERSE, bytes_override=None):
        torch = self._torch
        need = self.workspace_bytes(nsteps, dtype, k, flags)
        nbytes = need if bytes_override is None else int(bytes_override)
        self.ws = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=self.eps.device)
        self._check(self._L.fdtd_set_workspace(self._h, C.c_void_p(self.ws.data_ptr()), nbytes, int(nsteps), int(dtype), int(k),
                                               int(flags)))
        self.ws_key = (int(nsteps), int(dtype), int(k), int(flags))

    def _ensure_ws(self, nsteps, dtype, k, flags):
        """Reuse the installed workspace when the requested run fits into it, else allocate a new one."""
        def slots(n, kk):
            return n // kk + 1 + (1 if n % kk else 0)
        if self.ws is not None and self.ws_key is not None:
            n0, d0, k0, f0 = self.ws_key
            if (f0 & flags) == flags and nsteps <= n0 and slots(nsteps, k) <= slots(n0, k0) and \
                    slots(nsteps, k) * self.slot_bytes(dtype) <= slots(n0, k0) * self.slot_bytes(d0):
                return
        self.set_workspace(nsteps, dtype, k, flags)

    def _monitor_shape(self, nsteps):
        lo, hi, mask = self.monitor
        return (int(nsteps), bin(mask).count("1")) + tuple(hi[a] - lo[a] for a in range(3))

    def _sources(self, sources, nsteps, host_amp):
        torch = self._torch
        arr = (_Source * max(len(sources), 1))()
        keep = []
        for i, s in enumerate(sources):
            wave = np.ascontiguousarray(s.wave, dtype=np.float32)
            assert wave.size >= nsteps
            keep.append(wave)
            arr[i].comp = int(s.comp)
            arr[i].lo = _i3(s.lo)
            arr[i].hi = _i3(s.hi)
            arr[i].wave = wave.ctypes.data
            if s.amp is None:
                arr[i].amp = None
            elif host_amp:
                a = np.ascontiguousarray(s.amp, dtype=np.float32)
                keep.append(a)
                arr[i].amp = a.ctypes.data
            else:
                a = torch.as_tensor(np.ascontiguousarray(s.amp, dtype=np.float32)).to(self.eps.device)
                keep.append(a)
                arr[i].amp = a.data_ptr()
        self._keep = keep
        return arr

    # ---- the four calls ----
    def forward(self, nsteps, sources, store_dtype=F32, k=1, flags=WS_REVERSE, reset=True):
        """fdtd_forward from state 0 (reset=True) or from the current state.  Returns the monitor record tensor
        [nsteps][ncomp][box] (or None)."""
        self._same_stream()
        torch = self._torch
        self._ensure_ws(nsteps, store_dtype, k, flags)
        if reset:
            self.reset()
        if self.monitor is not None:
            self.mon_rec = torch.empty(self._monitor_shape(nsteps), dtype=torch.float32, device=self.eps.device)
            lo, hi, mask = self.monitor
            self._check(self._L.fdtd_set_monitor(self._h, _i3(lo), _i3(hi), mask, C.c_void_p(self.mon_rec.data_ptr())))
        arr = self._sources(sources, nsteps, host_amp=False)
        self._check(self._L.fdtd_forward(self._h, int(nsteps), arr, len(sources), int(store_dtype), int(k)))
        self.nsteps = int(nsteps)
        return self.mon_rec

    def reverse(self, dL_dfinal=None, dL_dmon=None, interp=LINEAR):
        """fdtd_reverse.  dL_dfinal = (lo, hi, comp_mask, tensor[ncomp][box]) or None; dL_dmon = tensor like the
        monitor record or None.  Returns grad_eps over the design box (float32 CUDA tensor) or None."""
        self._same_stream()
        torch = self._torch
        cot = None
        if dL_dfinal is not None:
            lo, hi, mask, g = dL_dfinal
            assert g.is_cuda and g.dtype == torch.float32 and g.is_contiguous()
            cot = _Cotangent(_i3(lo), _i3(hi), int(mask), g.data_ptr())
        if dL_dmon is not None:
            assert dL_dmon.is_cuda and dL_dmon.dtype == torch.float32 and dL_dmon.is_contiguous()
            assert tuple(dL_dmon.shape) == self._monitor_shape(self.nsteps)
        grad = None
        if self.design is not None:
            lo, hi = self.design
            grad = torch.empty([hi[a] - lo[a] for a in range(3)], dtype=torch.float32, device=self.eps.device)
        self._check(self._L.fdtd_reverse(self._h, C.byref(cot) if cot is not None else None,
                                         C.c_void_p(dL_dmon.data_ptr()) if dL_dmon is not None else None, int(interp),
                                         C.c_void_p(grad.data_ptr()) if grad is not None else None))
        return grad

    def store_bytes(self):
        return self._L.fdtd_store_bytes(self._h)

    # ---- host-buffer variants (end-to-end path) ----
    def set_eps_host(self, eps_host):
        assert eps_host.dtype == self._torch.float32 and not eps_host.is_cuda and eps_host.is_contiguous()
        self._check(self._L.fdtd_set_eps_host(self._h, C.c_void_p(eps_host.data_ptr())))

    def forward_host(self, nsteps, sources, store_dtype, k, mon_host):
        arr = self._sources(sources, nsteps, host_amp=True)
        self._check(self._L.fdtd_forward_host(self._h, int(nsteps), arr, len(sources), int(store_dtype), int(k),
                                              C.c_void_p(mon_host.data_ptr()) if mon_host is not None else None))
        self.nsteps = int(nsteps)

    def reverse_host(self, dmon_host, interp, grad_host):
        self._check(self._L.fdtd_reverse_host(self._h, C.c_void_p(dmon_host.data_ptr()) if dmon_host is not None else None,
                                              int(interp), C.c_void_p(grad_host.data_ptr()) if grad_host is not None else None))

    # ---- auxiliaries ----
    def set_eps(self, eps):
        assert eps.is_cuda and eps.dtype == self._torch.float32 and eps.is_contiguous() and tuple(eps.shape) == self.shape
        self.eps = eps
        self._check(self._L.fdtd_set_eps(self._h, C.c_void_p(eps.data_ptr())))

    def reset(self):
        self._check(self._L.fdtd_reset(self._h))

    def set_graphs(self, on):
        self._check(self._L.fdtd_set_graphs(self._h, int(bool(on))))

    def set_fused(self, mode, xseg=0):
        self._check(self._L.fdtd_set_fused(self._h, int(mode), int(xseg)))

    def uses_fused(self, nsteps):
        return bool(self._L.fdtd_uses_fused(self._h, int(nsteps)))

    def uses_fused_reverse(self):
        return bool(self._L.fdtd_uses_fused_reverse(self._h))

    def uses_fused_adjoint(self):
        return bool(self._L.fdtd_uses_fused_adjoint(self._h))

    def fields(self):
        self._same_stream()
        out = self._torch.empty((6,) + self.shape, dtype=self._torch.float32, device=self.eps.device)
        self._check(self._L.fdtd_get_fields(self._h, C.c_void_p(out.data_ptr())))
        return out

    def adjoint(self):
        out = self._torch.empty((6,) + self.shape, dtype=self._torch.float32, device=self.eps.device)
        self._check(self._L.fdtd_get_adjoint(self._h, C.c_void_p(out.data_ptr())))
        return out

    def box(self, lo, hi, comp_mask):
        ncomp = bin(comp_mask).count("1")
        out = self._torch.empty((ncomp,) + tuple(hi[a] - lo[a] for a in range(3)), dtype=self._torch.float32, device=self.eps.device)
        self._check(self._L.fdtd_get_box(self._h, _i3(lo), _i3(hi), int(comp_mask), C.c_void_p(out.data_ptr())))
        return out

    def num_slots(self):
        return self._L.fdtd_num_slots(self._h)

    def slot_values(self):
        return self._L.fdtd_slot_values(self._h)

    def slot_bytes(self, dtype):
        return self._L.fdtd_slot_bytes(self._h, int(dtype))

    def slot(self, j, dtype):
        """(raw bytes uint8 CUDA tensor copy, 36 float32 scales) of stored slot j.  F8E4M3_MX32: the bytes are the slot_values
        codes followed by the block-scale bytes."""
        torch = self._torch
        self._same_stream()
        dp, sp = C.c_void_p(), C.c_void_p()
        self._check(self._L.fdtd_slot_ptr(self._h, int(j), C.byref(dp), C.byref(sp)))
        nbytes = self.slot_bytes(dtype)
        off = dp.value - self.ws.data_ptr()
        soff = sp.value - self.ws.data_ptr()
        self.sync()
        data = self.ws[off:off + nbytes].clone()
        scales = self.ws[soff:soff + 144].clone().view(torch.float32)
        return data, scales

    def sync(self):
        self._check(self._L.fdtd_sync(self._h))

    KERNELS = ["fwd_e", "fwd_h", "inv_h", "adj_h", "grad_inv_e", "adj_e", "record", "inject_h", "inject_e",
               "fwd_fused", "fwd_fused_slabs"]   # the last two: the fused forward path (fdtd_fused.cuh), large grids only
    # kernel groups of fdtd_profile_kernel by name; rev_fused / grad: the fused reverse primal (large grids) and the gradient kernel
    KERNEL_IDS = {**{n: i for i, n in enumerate(KERNELS)}, "rev_fused": 19, "grad": 20, "adj_fused": 21, "adj_fused_slabs": 22}

    def profile_kernel(self, kernel_id, warm=5, reps=50):
        """(mean ms per launch, algorithmic bytes per launch) of one kernel timed alone, back to back (fdtd_profile_kernel)."""
        ms, by = C.c_double(), C.c_double()
        self._check(self._L.fdtd_profile_kernel(self._h, int(kernel_id), int(warm), int(reps), C.byref(ms), C.byref(by)))
        return ms.value, by.value

    def launch_count(self):
        return int(self._L.fdtd_launch_count(self._h))

    def guard_check(self):
        """Guard bytes overwritten since fdtd_set_workspace(flags | WS_GUARD); -1 without a guarded workspace."""
        return int(self._L.fdtd_debug_guard_check(self._h))


# ---- stand-alone codec (bit-exactness tests on identical slices) ----
def codec_encode(dtype, x):
    """x: float32 CUDA tensor (one slice).  Returns (codes uint8 CUDA tensor, scale float)."""
    torch = _torch()
    L = lib()
    x = x.contiguous()
    nbytes = x.numel() * ELEM_BYTES[dtype] + ((x.numel() + 31) // 32 if dtype == F8E4M3_MX32 else 0)
    codes = torch.empty(nbytes, dtype=torch.uint8, device=x.device)
    scale = torch.zeros(1, dtype=torch.float32, device=x.device)
    scratch = torch.zeros(1, dtype=torch.int32, device=x.device)
    st = L.fdtd_codec_encode(int(dtype), C.c_void_p(x.data_ptr()), x.numel(), C.c_void_p(codes.data_ptr()),
                             C.c_void_p(scale.data_ptr()), C.c_void_p(scratch.data_ptr()), _stream_ptr(torch))
    if st != 0:
        raise FdtdError(st, "fdtd_codec_encode")
    return codes, float(scale.item())


def codec_fetch(dtype, interp, codes, scales, num, den, n=None):
    """codes: list of 4 uint8 CUDA tensors (or None) for steps -1, 0, 1, 2; scales: 4 floats.  F8E4M3_MX32: each tensor holds
    n codes followed by ceil(n/32) scale bytes, and n must be given."""
    torch = _torch()
    L = lib()
    ref = codes[1]
    if n is None:
        assert dtype != F8E4M3_MX32
        n = ref.numel() // ELEM_BYTES[dtype]
    ptrs = (C.c_void_p * 4)(*[C.c_void_p(c.data_ptr()) if c is not None else None for c in codes])
    sc = (C.c_float * 4)(*[float(s) for s in scales])
    out = torch.empty(n, dtype=torch.float32, device=ref.device)
    st = L.fdtd_codec_fetch(int(dtype), int(interp), ptrs, sc, int(num), int(den), n, C.c_void_p(out.data_ptr()), _stream_ptr(torch))
    if st != 0:
        raise FdtdError(st, "fdtd_codec_fetch")
    return out


def codec_encode_slices_noalloc(dtype, x, codes=None, scales=None):
    """fdtd_codec_encode_slices_noalloc: x float32 CUDA tensor [nslices, slice_len]; codes (uint8 [nslices, slice_len * bytes]) and
    scales (float32 [nslices]) are the caller's output tensors (allocated here only when not given).  The library call itself
    allocates nothing: its reduction scratch is a static device array (at most NOALLOC_MAX_SLICES slices per call)."""
    torch = _torch()
    L = lib()
    assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous() and x.dim() == 2
    nslices, slice_len = x.shape
    if codes is None:
        codes = torch.empty((nslices, slice_len * ELEM_BYTES[dtype]), dtype=torch.uint8, device=x.device)
    if scales is None:
        scales = torch.empty(nslices, dtype=torch.float32, device=x.device)
    st = L.fdtd_codec_encode_slices_noalloc(int(dtype), C.c_void_p(x.data_ptr()), int(nslices), int(slice_len),
                                            C.c_void_p(codes.data_ptr()), C.c_void_p(scales.data_ptr()), _stream_ptr(torch))
    if st != 0:
        raise FdtdError(st, L.fdtd_noalloc_last_error().decode())
    return codes, scales
