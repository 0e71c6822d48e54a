"""Tolerance rule of the parity tests (BASELINE.json:5; reading D23 in DESIGN.md).

S = {det_oracle > 1e-3 * max det_oracle}, det = a*c - b^2 of level 0 (iteration independent, D9).
On S: max(|du|, |dv|) <= 1e-3 px and RMS <= 1e-4 px; on ALL pixels the validity masks are identical.
"""
import numpy as np

MAX_TOL = 1e-3
RMS_TOL = 1e-4


def compare_flow(gu, gv, gvalid, ref, max_tol=MAX_TOL, rms_tol=RMS_TOL):
    gu = np.asarray(gu, dtype=np.float64)
    gv = np.asarray(gv, dtype=np.float64)
    det = ref["det"]
    S = det > 1e-3 * det.max()
    du = (gu - ref["u"])[S]
    dv = (gv - ref["v"])[S]
    stats = {
        "frac_S": float(S.mean()),
        "max": float(max(np.abs(du).max(), np.abs(dv).max())) if du.size else 0.0,
        "rms": float(np.sqrt(np.mean(du * du + dv * dv))) if du.size else 0.0,
        "mask_mismatch": int(np.count_nonzero(np.asarray(gvalid) != ref["valid"])) if gvalid is not None else 0,
        "max_all": float(max(np.abs(gu - ref["u"]).max(), np.abs(gv - ref["v"]).max())),
    }
    return stats


def assert_parity(gu, gv, gvalid, ref, what=""):
    st = compare_flow(gu, gv, gvalid, ref)
    assert np.isfinite(np.asarray(gu)).all() and np.isfinite(np.asarray(gv)).all(), what
    assert st["frac_S"] > 0.0, (what, st)
    assert st["max"] <= MAX_TOL, (what, st)
    assert st["rms"] <= RMS_TOL, (what, st)
    assert st["mask_mismatch"] == 0, (what, st)
    return st
