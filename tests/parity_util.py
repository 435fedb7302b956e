"""Shared helpers of the GPU parity tests: the north_star tolerance and the
oracle-side reference on the same seeded inputs.  No arithmetic of the method
lives here (the oracle is oracle/, the product is the C-ABI library)."""
import numpy as np

REL_TOL = 1e-4      # per bin where oracle >= FLOOR * max(k)      (BASELINE.json north_star)
FLOOR = 1e-8        # absolute tolerance FLOOR * max(k) elsewhere


def check_parity(k_gpu, k_ref, kmax=None, rel=REL_TOL, floor=FLOOR, what=""):
    """Assert the north_star tolerance; returns (max rel err in the relative regime,
    max abs err / kmax in the absolute regime, fraction of bins in the relative regime)."""
    k_gpu = np.asarray(k_gpu, dtype=np.float64)
    k_ref = np.asarray(k_ref, dtype=np.float64)
    assert k_gpu.shape == k_ref.shape
    assert np.all(np.isfinite(k_gpu)), f"{what}: non-finite GPU output"
    if kmax is None:
        kmax = float(k_ref.max()) if k_ref.size else 0.0
    if k_ref.size == 0:
        return 0.0, 0.0, 0.0
    big = k_ref >= floor * kmax
    err = np.abs(k_gpu - k_ref)
    relerr = float((err[big] / k_ref[big]).max()) if big.any() else 0.0
    abserr = float(err[~big].max() / kmax) if (~big).any() and kmax > 0 else 0.0
    assert relerr <= rel, f"{what}: relative error {relerr:.3e} > {rel:g} (bin {np.argmax(np.where(big, err / np.maximum(k_ref, 1e-300), 0))})"
    assert abserr <= floor, f"{what}: absolute error {abserr:.3e} x max(k) > {floor:g}"
    return relerr, abserr, float(big.mean())


def check_parity_plinth(k_gpu, k_ref, k_raw, rel=REL_TOL, floor=FLOOR, what=""):
    """Tolerance with plinth removal (section 2.1.1; R27).  The paper defines the result as
    the line opacity minus its value at the cutting length and stores opacities in single precision (L367): a
    difference of two stored-precision numbers is defined to a fraction of the UNSUBTRACTED value, so the north_star
    pair is applied with the opacity before removal as the reference magnitude: |k - k_ref| <= rel k_raw + floor
    max(k_raw) on every bin.  Where the removed part is negligible this is the plain north_star tolerance."""
    k_gpu = np.asarray(k_gpu, dtype=np.float64)
    assert np.all(np.isfinite(k_gpu)), f"{what}: non-finite GPU output"
    err = np.abs(k_gpu - k_ref)
    kmax = float(k_raw.max()) if k_raw.size else 0.0
    bad = err > rel * k_raw + floor * kmax
    worst = float((err / np.maximum(k_raw, 1e-300))[k_raw >= floor * kmax].max()) if (k_raw >= floor * kmax).any() else 0.0
    assert not bad.any(), f"{what}: {int(bad.sum())} bins beyond {rel:g} x unsubtracted k (worst {worst:.3e})"
    return worst


def check_parity_subtracted(k_gpu, k_ref, k_raw, rel=REL_TOL, floor=FLOOR, rounding=2.0 ** -22, what=""):
    """The accuracy contract of hk_set_plinth for well-conditioned lines (include/hk.h, HK_PLINTH_ROUNDING): the north_star
    pair on the SUBTRACTED opacity, plus the rounding of the two fp32 terms of the difference, 2^-22 of the opacity before
    removal (one to two fp32 ulps of it: what no fp32 evaluation of V - V(cut) can avoid).  Returns the worst relative
    error among the bins of the relative regime."""
    k_gpu = np.asarray(k_gpu, dtype=np.float64)
    assert np.all(np.isfinite(k_gpu)), f"{what}: non-finite GPU output"
    kmax = float(k_ref.max()) if k_ref.size else 0.0
    err = np.abs(k_gpu - k_ref)
    big = k_ref >= floor * kmax
    bad = err > rel * np.where(big, k_ref, 0.0) + floor * kmax * (~big) + rounding * k_raw
    worst = float((err[big] / k_ref[big]).max()) if big.any() else 0.0
    assert not bad.any(), (f"{what}: {int(bad.sum())} bins beyond {rel:g} x subtracted k + 2^-22 x unsubtracted k "
                           f"(worst relative {worst:.3e} at bin {int(np.argmax(np.where(big, err / np.maximum(k_ref, 1e-300), 0)))})")
    return worst


def sample_windows(N, n_windows, width, rng):
    """Stratified windows of `width` contiguous bins incl. the first and last."""
    if N <= n_windows * width:
        return [(0, N)]
    starts = {0, N - width}
    strata = np.linspace(0, N - width, n_windows - 1).astype(np.int64)
    for a, b in zip(strata[:-1], strata[1:]):
        starts.add(int(rng.integers(a, max(a + 1, b))))
    return [(s, s + width) for s in sorted(starts)]
