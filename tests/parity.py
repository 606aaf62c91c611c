"""Shared helpers of the GPU parity tests: tolerance of BASELINE.json north_star (SURVEY A-15) and
oracle-vs-CUDA comparison.  Test infrastructure (may import oracle/)."""
import numpy as np

import os

ABS_TOL, REL_TOL, LSE_TOL = 2e-2, 1e-2, 1e-3
# Norm-relative companion of the element rule.  With N(0,1) inputs |out| ~ sqrt(e / L): on a 128K-token document every
# element is below ABS_TOL, so the element rule alone would pass an all-zero row (and a dropped K/V tile, which moves
# a 1024-tile row by ~3 % of its norm).  Every head vector (last axis: the d values of one token and head) must also
# satisfy
#     ||x - ref||_2 <= VEC_REL * ||ref||_2 + sqrt(d) * (VEC_ABS + VEC_FLOOR * nat)
# Measured on the B200 path against the oracle (10K-token document plus short ones, every vector): the relative L2
# error is <= 0.43 % for out, dK, dV at any length and for dQ from ~33 visible keys on (bf16 rounding of P, dS and of
# the result, R-4, A-12).  Only dQ of rows with a handful of keys goes higher (4 % at 2-4 keys, tails to
# 14 %): dS = P (dP - D) cancels there; its absolute error stays below 8e-3 sqrt(d / n), n = visible keys.  Hence
#     nat = 1 / sqrt(n) for row vectors (out, dQ), 0 for key-column vectors (dK, dV), 1 when the caller does not say.
# At 64K keys the floor is 0.6 % of a typical row norm: a dropped tile still fails.  VEC_ABS serves vectors that are
# zero in exact arithmetic (dQ of the first row of a document: measured 6e-6).
VEC_REL, VEC_FLOOR, VEC_ABS = 1e-2, 8e-3, 1e-4


def row_scale(cu_seqlens, rows):
    """nat of out / dQ vectors of the given rows: 1 / sqrt(visible keys) = 1 / sqrt(t - cu[doc(t)] + 1)"""
    cu = np.asarray(cu_seqlens, dtype=np.int64)
    rows = np.asarray(rows, dtype=np.int64)
    doc = np.searchsorted(cu, rows, side="right") - 1
    return 1.0 / np.sqrt((rows - cu[doc] + 1).astype(np.float64))


def col_scale(cu_seqlens, cols):
    """nat of dK / dV vectors: 0 (they need no floor beyond VEC_ABS)"""
    return np.zeros(len(cols), dtype=np.float64)


def check_close(x, ref, what, nat=None):
    """element passes iff |x - ref| <= max(2e-2, 1e-2 |ref|)  (bf16 outputs and gradients, BASELINE.json north_star),
    and every head vector passes the norm-relative rule above.  x, ref: [tokens, heads, d]; nat: [tokens] or None."""
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert x.shape == ref.shape, (what, x.shape, ref.shape)
    assert np.isfinite(x).all(), f"{what}: non-finite values"
    err = np.abs(x - ref)
    tol = np.maximum(ABS_TOL, REL_TOL * np.abs(ref))
    bad = err > tol
    assert not bad.any(), (f"{what}: {int(bad.sum())} of {bad.size} elements out of tolerance; max abs err "
                           f"{err.max():.4e} at {np.unravel_index(err.argmax(), err.shape)}")
    d = x.shape[-1]
    en = np.sqrt((err ** 2).sum(axis=-1))
    rn = np.sqrt((ref ** 2).sum(axis=-1))
    nat_a = 1.0 if nat is None else np.asarray(nat, dtype=np.float64).reshape((-1,) + (1,) * (en.ndim - 1))
    lim = VEC_REL * rn + np.sqrt(d) * (VEC_ABS + VEC_FLOOR * nat_a)
    ratio = en / lim
    if os.environ.get("SAP_PARITY_STATS"):
        print(f"[parity] {what}: max vector err / limit = {ratio.max():.3f}; median limit / ||ref|| = {np.median(lim / np.maximum(rn, 1e-30)):.3f}")
    worst = np.unravel_index(ratio.argmax(), ratio.shape)
    assert ratio.max() <= 1.0, (f"{what}: head vector {worst} has ||x - ref|| = {en[worst]:.3e} against ||ref|| = {rn[worst]:.3e} "
                                f"(limit {lim[worst]:.3e}); {int((ratio > 1).sum())} of {ratio.size} vectors fail")
    return float(err.max())


def check_lse(x, ref, what):
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    err = np.abs(x - ref)
    assert np.isfinite(x).all() and err.max() <= LSE_TOL, f"{what}: max |dLSE| {err.max():.3e} > {LSE_TOL}"
    return float(err.max())


def to_np(t):
    return t.detach().float().cpu().numpy()
