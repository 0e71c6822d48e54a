"""Thin ctypes binding of liboptflow.so (include/optflow.h): argument marshalling only.

Every step of the method runs in the CUDA kernels of ``csrc/``.  PyTorch is used for device memory
(``torch.empty(device='cuda')``, ``data_ptr()``) and streams (``torch.cuda.current_stream()``).
There is no CPU fallback: if the library is missing or there is no GPU, calls raise.
"""
from __future__ import annotations

import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liboptflow.so")

OF_WINDOW_BOX, OF_WINDOW_GAUSSIAN = 0, 1
OF_DTYPE_F32, OF_DTYPE_U8, OF_DTYPE_U16 = 0, 1, 2
OF_STREAM_CONSECUTIVE, OF_STREAM_PAIRS = 0, 1
OF_OK = 0
OF_STATIC_MAX_PIXELS = 16777216
OF_ERR_INVALID_ARG, OF_ERR_ALLOC, OF_ERR_CUDA, OF_ERR_STATE = -1, -2, -3, -4

_c = ctypes
_vp, _i = _c.c_void_p, _c.c_int

# name -> (restype, argtypes): exactly the symbols include/optflow.h declares
SIGNATURES = {
    "of_create": (_vp, [_i] * 6),
    "of_compute": (_i, [_vp] * 6),
    "of_destroy": (None, [_vp]),
    "of_compute_u8": (_i, [_vp] * 6),
    "of_compute_u16": (_i, [_vp] * 6),
    "of_compute_dual": (_i, [_vp, _vp, _i] + [_vp] * 9),
    "of_run_solve_dual": (_i, [_vp, _vp, _i, _vp]),
    "of_last_error": (_c.c_char_p, []),
    "of_set_conditioning": (_i, [_vp, _c.c_float, _c.c_float]),
    "of_set_equalisation": (_i, [_vp, _i]),
    "of_set_mask": (_i, [_vp, _vp, _i]),
    "of_set_graph": (_i, [_vp, _i]),
    "of_set_persistent": (_i, [_vp, _i]),
    "of_set_hoist": (_i, [_vp, _i]),
    "of_set_fused": (_i, [_vp, _i]),
    "of_bubble_threshold": (_i, [_vp, _vp, _i, _vp, _vp, _vp]),
    "of_bubble_count_dev": (_i, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "of_stream_result_validity": (_i, [_vp, ctypes.POINTER(ctypes.c_void_p)]),
    "of_solve_timeline": (_i, [_vp, _i, _i, _vp, _i]),
    "of_get_validity": (_i, [_vp, _vp, _vp]),
    "of_level_size": (_i, [_vp, _i, _c.POINTER(_i), _c.POINTER(_i)]),
    "of_last_launch_count": (_i, [_vp]),
    "of_get_debug_plane": (_i, [_vp, _i, _i, _vp, _vp]),
    "of_run_step": (_i, [_vp, _i, _i, _i, _vp]),
    "of_run_solve": (_i, [_vp, _i, _vp]),
    "of_field_accumulate": (_i, [_vp, _vp, _vp, _vp]),
    "of_field_minmax": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "of_bubble_count": (_i, [_vp, _vp, _vp, _c.c_float, _vp, _vp]),
    "of_field_minmax_static": (_i, [_vp, _vp, _c.c_size_t, _vp, _vp]),
    "of_pyramid_down": (_i, [_vp, _i, _i, _vp, _vp]),
    "of_upsample_flow": (_i, [_vp, _vp, _i, _i, _vp, _vp, _i, _i, _vp]),
    "of_stream_open": (_i, [_vp, _i, _i, _i]),
    "of_stream_acquire": (_vp, [_vp]),
    "of_stream_submit": (_i, [_vp]),
    "of_stream_result": (_i, [_vp, _c.POINTER(_vp), _c.POINTER(_vp), _c.POINTER(_i)]),
    "of_stream_close": (_i, [_vp]),
}

_lib = None


class OptflowError(RuntimeError):
    pass


def lib():
    """Load liboptflow.so (built in-tree by ``paper_1306_2461_b200.build``).  Raises if missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise OptflowError(
                "liboptflow.so not found at %s: build it with `python -m paper_1306_2461_b200.build` "
                "(there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def last_error() -> str:
    return lib().of_last_error().decode("utf-8", "replace")


def _check(rc: int):
    if rc != OF_OK:
        raise OptflowError("optflow error %d: %s" % (rc, last_error()))


def _stream_ptr(stream=None):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return _vp(s.cuda_stream)


def field_minmax_static(field, out, valid=None, stream=None):
    """of_field_minmax_static: min / max of `field` over the available vectors into the caller's `out` (2 floats, device).
    No handle and no allocation (static device scratch; at most OF_STATIC_MAX_PIXELS elements; calls must not overlap on the GPU)."""
    _check(lib().of_field_minmax_static(field.data_ptr(), valid.data_ptr() if valid is not None else None,
                                        field.numel(), out.data_ptr(), _stream_ptr(stream)))
    return out


def _dtype_code(t, torch):
    if t == torch.float32:
        return OF_DTYPE_F32
    if t == torch.uint8:
        return OF_DTYPE_U8
    if t in (torch.uint16, torch.int16):
        return OF_DTYPE_U16
    raise OptflowError("unsupported image dtype %s" % t)


def compute_dual(ofa, ofb, I1a, I2a, I1b, I2b, ua=None, va=None, ub=None, vb=None, stream=None):
    """of_compute_dual: pair a with handle `ofa`, pair b with handle `ofb` (two OpticalFlow objects created with the same
    arguments), one launch for both (throughput mode).  Returns (ua, va, ub, vb); same tensors rules as OpticalFlow.compute."""
    import torch
    H, W = ofa.height, ofa.width
    outs = []
    for f in (ua, va, ub, vb):
        if f is None:
            f = torch.empty((H, W), dtype=torch.float32, device=I1a.device)
        assert f.is_cuda and f.is_contiguous() and f.dtype == torch.float32 and tuple(f.shape) == (H, W)
        outs.append(f)
    for t in (I1a, I2a, I1b, I2b):
        assert t.is_cuda and t.is_contiguous() and tuple(t.shape) == (H, W) and t.dtype == I1a.dtype
    _check(lib().of_compute_dual(ofa._h, ofb._h, _dtype_code(I1a.dtype, torch), I1a.data_ptr(), I2a.data_ptr(), outs[0].data_ptr(),
                                 outs[1].data_ptr(), I1b.data_ptr(), I2b.data_ptr(), outs[2].data_ptr(), outs[3].data_ptr(),
                                 _stream_ptr(stream)))
    return tuple(outs)


def run_solve_dual(ofa, ofb, repeat=1, stream=None):
    _check(lib().of_run_solve_dual(ofa._h, ofb._h, repeat, _stream_ptr(stream)))


class OpticalFlow:
    """Handle wrapper: ``of_create`` / ``of_compute*`` / ``of_destroy`` and the extras."""

    def __init__(self, width, height, levels, window_radius, iterations, window_type):
        import torch
        if not torch.cuda.is_available():
            raise OptflowError("no CUDA device: the optical-flow path runs on the GPU only")
        self.width, self.height, self.levels = int(width), int(height), int(levels)
        self.window_radius, self.iterations, self.window_type = int(window_radius), int(iterations), int(window_type)
        self._h = lib().of_create(self.width, self.height, self.levels, self.window_radius,
                                  self.iterations, self.window_type)
        if not self._h:
            raise OptflowError("of_create failed: %s" % last_error())
        self._torch = torch

    # -- lifetime ---------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            lib().of_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- solve ------------------------------------------------------------------------------
    def compute(self, I1, I2, u=None, v=None, stream=None):
        """I1, I2: CUDA tensors (H, W) of dtype float32 / uint8 / uint16 (or int16 holding uint16
        bits).  Returns (u, v) float32 CUDA tensors; asynchronous on the stream."""
        torch = self._torch
        assert I1.is_cuda and I2.is_cuda and I1.is_contiguous() and I2.is_contiguous()
        assert tuple(I1.shape) == (self.height, self.width) == tuple(I2.shape) and I1.dtype == I2.dtype
        if u is None:
            u = torch.empty((self.height, self.width), dtype=torch.float32, device=I1.device)
        if v is None:
            v = torch.empty((self.height, self.width), dtype=torch.float32, device=I1.device)
        for f in (u, v):
            assert f.is_cuda and f.is_contiguous() and f.dtype == torch.float32 and tuple(f.shape) == (self.height, self.width)
        if I1.dtype == torch.float32:
            fn = lib().of_compute
        elif I1.dtype == torch.uint8:
            fn = lib().of_compute_u8
        elif I1.dtype in (torch.uint16, torch.int16):
            fn = lib().of_compute_u16
        else:
            raise OptflowError("unsupported image dtype %s" % I1.dtype)
        _check(fn(self._h, I1.data_ptr(), I2.data_ptr(), u.data_ptr(), v.data_ptr(), _stream_ptr(stream)))
        return u, v

    def set_conditioning(self, eps_rel=1e-3, max_step_px=3.0):
        _check(lib().of_set_conditioning(self._h, eps_rel, max_step_px))

    def set_equalisation(self, radius: int):
        _check(lib().of_set_equalisation(self._h, int(radius)))

    def set_mask(self, mask):
        """Obstacle mask: HxW array, non-zero = fluid; None removes it.  Set-up call (synchronises)."""
        if mask is None:
            _check(lib().of_set_mask(self._h, None, 0))
            return
        import numpy as np
        m = np.ascontiguousarray(np.asarray(mask.cpu() if hasattr(mask, "cpu") else mask) != 0, dtype=np.uint8)
        if m.shape != (self.height, self.width):
            raise ValueError("mask must be %dx%d" % (self.height, self.width))
        _check(lib().of_set_mask(self._h, m.ctypes.data, self.width))

    def set_graph(self, enable: bool):
        _check(lib().of_set_graph(self._h, 1 if enable else 0))

    def set_persistent(self, enable: bool):
        _check(lib().of_set_persistent(self._h, 1 if enable else 0))

    def set_fused(self, enable: bool):
        _check(lib().of_set_fused(self._h, 1 if enable else 0))

    def set_hoist(self, enable: bool):
        _check(lib().of_set_hoist(self._h, 1 if enable else 0))

    def solve_timeline(self, enable=True, cta=-1):
        """Stamps [ns] of the last profiled solve (NumPy uint64, empty if the hook was off) of CTA
        `cta`, or the maximum over CTAs for cta < 0; then switches the hook on/off."""
        import numpy as np
        buf = np.zeros(4096, dtype=np.uint64)
        n = lib().of_solve_timeline(self._h, 1 if enable else 0, cta, buf.ctypes.data, buf.size)
        if n < 0:
            _check(n)
        return buf[:n]

    def validity(self, stream=None):
        torch = self._torch
        m = torch.empty((self.height, self.width), dtype=torch.uint8, device="cuda")
        _check(lib().of_get_validity(self._h, m.data_ptr(), _stream_ptr(stream)))
        return m

    def level_size(self, level):
        w, h = _i(), _i()
        _check(lib().of_level_size(self._h, level, ctypes.byref(w), ctypes.byref(h)))
        return w.value, h.value

    def last_launch_count(self):
        return int(lib().of_last_launch_count(self._h))

    def debug_plane(self, level, which, stream=None):
        torch = self._torch
        w, h = self.level_size(level)
        out = torch.empty((h, w), dtype=torch.float32, device="cuda")
        _check(lib().of_get_debug_plane(self._h, level, which, out.data_ptr(), _stream_ptr(stream)))
        return out

    def run_step(self, level, which, repeat=1, stream=None):
        _check(lib().of_run_step(self._h, level, which, repeat, _stream_ptr(stream)))

    def run_solve(self, repeat=1, stream=None):
        _check(lib().of_run_solve(self._h, repeat, _stream_ptr(stream)))

    # -- integral quantity, eq. 3 -----------------------------------------------------------
    def field_accumulate(self, total, field, stream=None):
        _check(lib().of_field_accumulate(self._h, total.data_ptr(), field.data_ptr(), _stream_ptr(stream)))

    def field_minmax(self, field, valid=None, stream=None):
        out = self._torch.empty(2, dtype=self._torch.float32, device=field.device)
        _check(lib().of_field_minmax(self._h, field.data_ptr(), valid.data_ptr() if valid is not None else None,
                                     out.data_ptr(), _stream_ptr(stream)))
        return out

    def bubble_count(self, vx, threshold, valid=None, stream=None):
        """Device tensor of two int64: (available vectors with vx <= threshold, available vectors)."""
        out = self._torch.empty(2, dtype=self._torch.int64, device=vx.device)
        _check(lib().of_bubble_count(self._h, vx.data_ptr(), valid.data_ptr() if valid is not None else None,
                                     float(threshold), out.data_ptr(), _stream_ptr(stream)))
        return out

    def bubble_threshold(self, total, n_fields, valid=None, stream=None):
        """Device tensor holding T_v = 0.5 * (min + max) / n_fields of the running sum `total` over the available vectors."""
        out = self._torch.empty(1, dtype=self._torch.float32, device=total.device)
        _check(lib().of_bubble_threshold(self._h, total.data_ptr(), int(n_fields), valid.data_ptr() if valid is not None else None,
                                         out.data_ptr(), _stream_ptr(stream)))
        return out

    def bubble_count_dev(self, vx, threshold_dev, valid=None, stream=None):
        """As bubble_count with the threshold taken from a device tensor (no host round trip)."""
        out = self._torch.empty(2, dtype=self._torch.int64, device=vx.device)
        _check(lib().of_bubble_count_dev(self._h, vx.data_ptr(), valid.data_ptr() if valid is not None else None,
                                         threshold_dev.data_ptr(), out.data_ptr(), _stream_ptr(stream)))
        return out

    # -- frame pipeline -----------------------------------------------------------------------
    def stream_open(self, dtype, mode=OF_STREAM_CONSECUTIVE, result_on_host=True):
        _check(lib().of_stream_open(self._h, dtype, mode, 1 if result_on_host else 0))
        self._s_dtype, self._s_mode, self._s_host = dtype, mode, bool(result_on_host)

    def stream_acquire(self):
        """NumPy view of the pinned slot to fill: (H, W), or (2, H, W) in PAIRS mode."""
        import numpy as np
        p = lib().of_stream_acquire(self._h)
        if not p:
            raise OptflowError("of_stream_acquire failed: %s" % last_error())
        ct = {OF_DTYPE_F32: (ctypes.c_float, np.float32), OF_DTYPE_U8: (ctypes.c_uint8, np.uint8),
              OF_DTYPE_U16: (ctypes.c_uint16, np.uint16)}[self._s_dtype]
        n = self.width * self.height * (2 if self._s_mode == OF_STREAM_PAIRS else 1)
        buf = (ct[0] * n).from_address(p)
        a = np.frombuffer(buf, dtype=ct[1])
        return a.reshape((2, self.height, self.width) if self._s_mode == OF_STREAM_PAIRS else (self.height, self.width))

    def stream_submit(self):
        _check(lib().of_stream_submit(self._h))

    def stream_result(self):
        """Returns (pair_index, u, v).  Host mode: NumPy views of the pinned result buffers (valid
        until the next-but-one call); device mode: raw device pointers (ints)."""
        import numpy as np
        pu, pv, idx = _vp(), _vp(), _i()
        _check(lib().of_stream_result(self._h, ctypes.byref(pu), ctypes.byref(pv), ctypes.byref(idx)))
        if not self._s_host:
            return idx.value, pu.value, pv.value
        n = self.width * self.height
        u = np.frombuffer((ctypes.c_float * n).from_address(pu.value), dtype=np.float32).reshape(self.height, self.width)
        v = np.frombuffer((ctypes.c_float * n).from_address(pv.value), dtype=np.float32).reshape(self.height, self.width)
        return idx.value, u, v

    def stream_result_validity(self):
        """Validity bytes of the field the last stream_result returned (host mode: NumPy view; device mode: raw pointer)."""
        import numpy as np
        pm = _vp()
        _check(lib().of_stream_result_validity(self._h, ctypes.byref(pm)))
        if not self._s_host:
            return pm.value
        n = self.width * self.height
        return np.frombuffer((ctypes.c_uint8 * n).from_address(pm.value), dtype=np.uint8).reshape(self.height, self.width)

    def stream_close(self):
        _check(lib().of_stream_close(self._h))


def device_to_numpy(ptr: int, count: int, dtype):
    """Copy `count` elements from a raw device pointer (as the pipeline hands out in device-result mode) into a NumPy array.
    Synchronous cudaMemcpy through the CUDA runtime that torch has loaded."""
    import numpy as np
    import torch  # noqa: F401  (loads libcudart)
    rt = None
    for name in ("libcudart.so.12", "libcudart.so"):
        try:
            rt = ctypes.CDLL(name)
            break
        except OSError:
            continue
    if rt is None:
        raise OptflowError("libcudart not found")
    out = np.empty(count, dtype=dtype)
    rt.cudaMemcpy.restype = ctypes.c_int
    rt.cudaMemcpy.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int]
    err = rt.cudaMemcpy(out.ctypes.data, ptr, out.nbytes, 2)          # cudaMemcpyDeviceToHost
    if err != 0:
        raise OptflowError("cudaMemcpy failed: error %d" % err)
    return out


def pyramid_down(src, stream=None):
    """Stand-alone pyramid step on a dense float32 CUDA tensor (H, W) -> ((H+1)//2, (W+1)//2)."""
    import torch
    H, W = src.shape
    dst = torch.empty(((H + 1) // 2, (W + 1) // 2), dtype=torch.float32, device=src.device)
    _check(lib().of_pyramid_down(src.data_ptr(), W, H, dst.data_ptr(), _stream_ptr(stream)))
    return dst


def upsample_flow(uc, vc, width, height, stream=None):
    import torch
    hc, wc = uc.shape
    u = torch.empty((height, width), dtype=torch.float32, device=uc.device)
    v = torch.empty((height, width), dtype=torch.float32, device=uc.device)
    _check(lib().of_upsample_flow(uc.data_ptr(), vc.data_ptr(), wc, hc, u.data_ptr(), v.data_ptr(), width, height,
                                  _stream_ptr(stream)))
    return u, v
