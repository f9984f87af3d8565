"""Shared helpers of the parity tests (comparison rules of BASELINE.json north_star)."""
import numpy as np

RTOL = 1e-5     # north_star: within 1e-5 relative ...
ATOL = 1e-6     # ... with a 1e-6 absolute floor, for float32 sums, masses and weighted bin contents


def assert_tol(got, want, what=""):
    """|got - want| <= max(RTOL*|want|, ATOL); infinities and NaNs must sit in the same places."""
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    assert got.shape == want.shape, (what, got.shape, want.shape)
    fin = np.isfinite(want)
    np.testing.assert_array_equal(np.isfinite(got), fin, err_msg=f"{what}: finite pattern")
    np.testing.assert_array_equal(got[~fin], want[~fin], err_msg=f"{what}: non-finite values")
    err = np.abs(got[fin] - want[fin])
    bound = np.maximum(RTOL * np.abs(want[fin]), ATOL)
    bad = err > bound
    if bad.any():
        i = np.flatnonzero(bad)[0]
        raise AssertionError(f"{what}: {bad.sum()} of {bad.size} outside tolerance; first: got {got[fin][i]!r} "
                             f"want {want[fin][i]!r} (err {err[i]:.3e}, bound {bound[i]:.3e})")


def assert_exact(got, want, what=""):
    np.testing.assert_array_equal(np.asarray(got), np.asarray(want), err_msg=what)


def to_np(t):
    return t.detach().cpu().numpy()
