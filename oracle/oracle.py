"""ctypes loader for the fp64 CPU oracle (oracle/optflow_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It imports nothing from the CUDA package.  `build()` compiles the C file with gcc (-O2 -fopenmp).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "optflow_oracle.c")
_LIB = os.path.join(_HERE, "liboptflow_oracle.so")

WINDOW_BOX = 0
WINDOW_GAUSSIAN = 1
EPS_REL = 1e-3        # D14
MAX_STEP = 3.0        # D15 (eq. 1)

_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-Wall",
                               "-Wno-misleading-indentation", "-Wno-unknown-pragmas",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_window_weight.restype = ctypes.c_double
        _lib.oracle_window_weight.argtypes = [ctypes.c_int] * 3
        _lib.oracle_solve.restype = ctypes.c_int
        _lib.oracle_solve_masked.restype = ctypes.c_int
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def window_weight(t, R, window_type):
    return float(lib().oracle_window_weight(int(t), int(R), int(window_type)))


def downsample(img):
    src, ps = _d(img)
    H, W = src.shape
    out = np.empty(((H + 1) // 2, (W + 1) // 2))
    lib().oracle_downsample(ps, ctypes.c_int(W), ctypes.c_int(H), out.ctypes.data_as(_dp))
    return out


def upsample_flow(coarse, W, H):
    c, pc = _d(coarse)
    Hc, Wc = c.shape
    out = np.empty((H, W))
    lib().oracle_upsample_flow(pc, ctypes.c_int(Wc), ctypes.c_int(Hc), out.ctypes.data_as(_dp),
                               ctypes.c_int(W), ctypes.c_int(H))
    return out


def equalise(img, r=5):
    """Local equalisation pre-filter, eq. 2."""
    src, ps = _d(img)
    H, W = src.shape
    out = np.empty((H, W))
    lib().oracle_equalise(ps, ctypes.c_int(W), ctypes.c_int(H), ctypes.c_int(r), out.ctypes.data_as(_dp))
    return out


def warp(I2, u, v):
    a, pa = _d(I2)
    uu, pu = _d(u)
    vv, pv = _d(v)
    H, W = a.shape
    out = np.empty((H, W))
    lib().oracle_warp(pa, pu, pv, ctypes.c_int(W), ctypes.c_int(H), out.ctypes.data_as(_dp))
    return out


def gradients(I1):
    a, pa = _d(I1)
    H, W = a.shape
    Ix, Iy = np.empty((H, W)), np.empty((H, W))
    lib().oracle_gradients(pa, ctypes.c_int(W), ctypes.c_int(H), Ix.ctypes.data_as(_dp),
                           Iy.ctypes.data_as(_dp))
    return Ix, Iy


def window_sum(f, R, window_type, direct=False):
    a, pa = _d(f)
    H, W = a.shape
    out = np.empty((H, W))
    fn = lib().oracle_window_sum_direct if direct else lib().oracle_window_sum
    fn(pa, ctypes.c_int(W), ctypes.c_int(H), ctypes.c_int(R), ctypes.c_int(window_type),
       out.ctypes.data_as(_dp))
    return out


def _mask(mask, shape):
    if mask is None:
        return None, None
    m = np.ascontiguousarray(np.asarray(mask) != 0, dtype=np.uint8)
    assert m.shape == shape
    return m, m.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte))


def mask_downsample(mask):
    """One step of the mask pyramid (reading M4): fluid iff any in-image child is fluid."""
    m, pm = _mask(mask, np.asarray(mask).shape)
    H, W = m.shape
    out = np.empty(((H + 1) // 2, (W + 1) // 2), dtype=np.uint8)
    lib().oracle_mask_downsample(pm, ctypes.c_int(W), ctypes.c_int(H),
                                 out.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)))
    return out


def iteration(I1, I2, u, v, R, window_type, eps=EPS_REL, max_step=MAX_STEP, direct=False, mask=None):
    """One iteration; returns (u_new, v_new, sums5[5,H,W], valid[H,W] uint8, det[H,W]).
    mask (optional, f4): non-zero = fluid, readings M1-M3."""
    a, pa = _d(I1)
    b, pb = _d(I2)
    H, W = a.shape
    m, pm = _mask(mask, a.shape)
    un = np.array(u, dtype=np.float64, order="C", copy=True)
    vn = np.array(v, dtype=np.float64, order="C", copy=True)
    sums = np.empty((5, H, W))
    valid = np.empty((H, W), dtype=np.uint8)
    det = np.empty((H, W))
    lib().oracle_iteration_masked(pa, pb, pm, ctypes.c_int(W), ctypes.c_int(H), ctypes.c_int(R),
                           ctypes.c_int(window_type), ctypes.c_double(eps), ctypes.c_double(max_step),
                           un.ctypes.data_as(_dp), vn.ctypes.data_as(_dp), sums.ctypes.data_as(_dp),
                           valid.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)),
                           det.ctypes.data_as(_dp), ctypes.c_int(1 if direct else 0))
    return un, vn, sums, valid, det


def solve(I1, I2, levels, R, iterations, window_type, eps=EPS_REL, max_step=MAX_STEP,
          direct=False, return_levels=False, mask=None):
    """Whole solve.  Returns dict(u, v, valid, det[, level_u, level_v]).
    mask (optional, f4): level-0 bytes, non-zero = fluid, readings M1-M5."""
    a, pa = _d(I1)
    b, pb = _d(I2)
    assert a.shape == b.shape and a.ndim == 2
    H, W = a.shape
    m, pm = _mask(mask, a.shape)
    u, v = np.empty((H, W)), np.empty((H, W))
    valid = np.empty((H, W), dtype=np.uint8)
    det = np.empty((H, W))
    lu = lv = None
    plu = plv = None
    if return_levels:
        lu, lv = [], []
        w, h = W, H
        for _ in range(levels):
            lu.append(np.empty((h, w)))
            lv.append(np.empty((h, w)))
            w, h = (w + 1) // 2, (h + 1) // 2
        plu = (_dp * levels)(*[x.ctypes.data_as(_dp) for x in lu])
        plv = (_dp * levels)(*[x.ctypes.data_as(_dp) for x in lv])
    rc = lib().oracle_solve_masked(pa, pb, pm, ctypes.c_int(W), ctypes.c_int(H), ctypes.c_int(levels),
                            ctypes.c_int(R), ctypes.c_int(iterations), ctypes.c_int(window_type),
                            ctypes.c_double(eps), ctypes.c_double(max_step),
                            u.ctypes.data_as(_dp), v.ctypes.data_as(_dp),
                            valid.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)),
                            det.ctypes.data_as(_dp), plu, plv, ctypes.c_int(1 if direct else 0))
    if rc != 0:
        raise ValueError("oracle_solve: invalid arguments (rc=%d)" % rc)
    out = {"u": u, "v": v, "valid": valid, "det": det}
    if return_levels:
        out["level_u"], out["level_v"] = lu, lv
    return out


# ---------------------------------------------------------------------------------------------
# NEXT item f3: recirculation-bubble surface, eq. 3.  The printed fraction is garbled
# (D20); the text defines it: "the percentage of velocities below a given threshold T_v relative to the
# total number of available velocity vectors", with T_v = 1/2 [min + max] of the longitudinal component
# of the MEAN velocity field.  Plain NumPy, written out as the definition.
# ---------------------------------------------------------------------------------------------
def bubble_threshold(mean_vx, valid=None):
    """T_v = (min + max) / 2 of the mean longitudinal velocity over the available vectors."""
    m = np.asarray(mean_vx, dtype=np.float64)
    if valid is not None:
        m = m[np.asarray(valid).astype(bool)]
    return 0.5 * (float(m.min()) + float(m.max()))


def bubble_counts(vx, threshold, valid=None):
    """(number of available vectors with v_x <= T_v, number of available vectors); S_bubble is their ratio."""
    v = np.asarray(vx)
    ok = np.ones(v.shape, dtype=bool) if valid is None else np.asarray(valid).astype(bool)
    below = 0
    total = 0
    for row_v, row_ok in zip(v, ok):            # explicit count, row by row
        for a, b in zip(row_v.tolist(), row_ok.tolist()):
            if b:
                total += 1
                if a <= threshold:
                    below += 1
    return below, total
