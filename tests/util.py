"""Shared test helpers: the parity metric of BASELINE.json `north_star` (reading A-13)."""
import numpy as np

TOL = 2e-2  # north_star: max|gpu - ref| / rms(ref) <= 2e-2 per tensor


def norm_err(got, ref):
    """max|got - ref| / rms(ref) over the whole tensor, in float64. NaN/Inf -> inf."""
    got = np.asarray(got, np.float64).reshape(-1)
    ref = np.asarray(ref, np.float64).reshape(-1)
    assert got.shape == ref.shape, (got.shape, ref.shape)
    if not np.all(np.isfinite(got)):
        return float("inf")
    rms = float(np.sqrt(np.mean(ref * ref)))
    if rms < 1e-30:
        return 0.0 if not np.any(got) else float("inf")
    return float(np.max(np.abs(got - ref)) / rms)
