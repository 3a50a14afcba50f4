"""Element-wise parity helpers shared by the GPU tests.

Every comparison with the oracle carries TWO bounds:
  * the relative L2 norm of the difference (the tolerance north_star states), and
  * a max-abs bound:  max |a - ref| <= MAXABS_FACTOR * tol * max |ref|.
The second one catches what the first cannot see on large fields: at 256^3 a single boundary cell that is wrong by the
field's RMS moves the relative L2 norm by only 1 / sqrt(N) = 2.4e-4.  MAXABS_FACTOR = 10: rounding errors of a stencil
pass are a few ulps of the LOCAL magnitude, i.e. at most a few times tol * max |ref| at any single point, while a wrong
cell is off by a sizeable fraction of max |ref| -- orders of magnitude above the bound.
"""
import numpy as np

MAXABS_FACTOR = 10.0


def rel_l2(a, ref):
    a = np.asarray(a, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64)
    return float(np.linalg.norm((a - ref).ravel()) / max(np.linalg.norm(ref.ravel()), 1e-300))


def max_abs(a, ref):
    """max |a - ref| relative to max |ref|"""
    a = np.asarray(a, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64)
    return float(np.abs(a - ref).max() / max(np.abs(ref).max(), 1e-300)) if ref.size else 0.0


def close(a, ref, tol, factor=MAXABS_FACTOR):
    """True when both bounds hold; use as `assert close(...)`, failures are explained by `why`."""
    return rel_l2(a, ref) <= tol and max_abs(a, ref) <= factor * tol


def why(a, ref, tol, factor=MAXABS_FACTOR):
    return "rel L2 %.3e (bound %.1e), max-abs/max|ref| %.3e (bound %.1e)" % (rel_l2(a, ref), tol, max_abs(a, ref), factor * tol)


def assert_close(a, ref, tol, what="", factor=MAXABS_FACTOR):
    assert close(a, ref, tol, factor), (what + ": " if what else "") + why(a, ref, tol, factor)
