"""Shared helpers of the GPU parity tests: tolerance of BASELINE.json north_star (SURVEY A-15) and
oracle-vs-CUDA comparison.  Test infrastructure (may import oracle/)."""
import numpy as np

ABS_TOL, REL_TOL, LSE_TOL = 2e-2, 1e-2, 1e-3


def check_close(x, ref, what):
    """element passes iff |x - ref| <= max(2e-2, 1e-2 |ref|)  (bf16 outputs and gradients)."""
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert x.shape == ref.shape, (what, x.shape, ref.shape)
    assert np.isfinite(x).all(), f"{what}: non-finite values"
    err = np.abs(x - ref)
    tol = np.maximum(ABS_TOL, REL_TOL * np.abs(ref))
    bad = err > tol
    assert not bad.any(), (f"{what}: {int(bad.sum())} of {bad.size} elements out of tolerance; max abs err "
                           f"{err.max():.4e} at {np.unravel_index(err.argmax(), err.shape)}")
    return float(err.max())


def check_lse(x, ref, what):
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    err = np.abs(x - ref)
    assert np.isfinite(x).all() and err.max() <= LSE_TOL, f"{what}: max |dLSE| {err.max():.3e} > {LSE_TOL}"
    return float(err.max())


def to_np(t):
    return t.detach().float().cpu().numpy()
