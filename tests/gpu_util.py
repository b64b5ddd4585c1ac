"""Helpers for the -m gpu parity tests: tolerance of north_star (2 ulp of (|A||B|)_ij) and handles."""
import json
import os

import numpy as np


def ulp_of(absab, bits=52):
    """2^(floor(log2 x) - bits): one unit in the last place of x (bits = 52 for FP64, 23 for FP32)."""
    absab = np.asarray(absab, dtype=np.float64)
    out = np.zeros_like(absab)
    nz = absab > 0
    out[nz] = np.exp2(np.floor(np.log2(absab[nz])) - bits)
    return out


def assert_within_ulps(got, want, scale, n_ulp=2, bits=52, what=""):
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    tol = n_ulp * ulp_of(scale, bits)
    err = np.abs(got - want)
    bad = err > tol
    if bad.any():
        idx = np.unravel_index(np.argmax(err / np.maximum(tol, 1e-300)), err.shape)
        raise AssertionError(f"{what}: {bad.sum()} / {bad.size} elements beyond {n_ulp} ulp; worst at {idx}: "
                             f"got {got[idx]!r} want {want[idx]!r} err {err[idx]:.3e} tol {tol[idx]:.3e}")
    worst = float((err / np.maximum(ulp_of(scale, bits), 1e-300)).max()) if err.size else 0.0
    log = os.environ.get("EMUGEMM_PARITY_LOG")  # optional record of the measured errors (BASELINE.md section 4's last column)
    if log:
        with open(log, "a") as f:
            f.write(json.dumps({"test": os.environ.get("PYTEST_CURRENT_TEST", "").split(" ")[0], "what": what,
                                "elements": int(err.size), "max_err_ulps": worst, "tolerance_ulps": n_ulp, "bits": bits}) + "\n")
    return worst
