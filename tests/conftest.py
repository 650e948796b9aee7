import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def rel_l2(got, ref, field_ref=None, tol=None, comp_floor=1e-12):
    """Per-component relative L2 error with the zero-component rule (Q10):
    if ||ref_c|| < comp_floor * ||ref field|| (1e-12: an identically-zero component) the error is
    measured against the whole field's norm.  The two fp32 fuzz tests (one-step and series) pass
    comp_floor = 1e-3, a reading stated and derived in DESIGN.md Q10: with one or two observation
    points a component can cancel to 1e-5 of the field, and an fp32 sum of O(field) terms carries
    ~1e-7 of the FIELD whatever the component's size -- 2e-4 of the component needs it >= 1e-3."""
    import numpy as np

    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    fnorm = float(np.linalg.norm(ref if field_ref is None else field_ref))
    out = []
    for c in range(ref.shape[0]):
        rn = float(np.linalg.norm(ref[c]))
        den = rn if rn >= comp_floor * fnorm and rn > 0 else (fnorm if fnorm > 0 else 1.0)
        out.append(float(np.linalg.norm(got[c] - ref[c])) / den)
    return out
