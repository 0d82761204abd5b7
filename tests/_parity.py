"""Error measures and acceptance checks shared by the GPU parity tests (no arithmetic of the method)."""
import numpy as np

TOL_STATE = 1e-4      # north_star: rel-L2 of psi after the configured steps
TOL_ROUNDTRIP = 1e-5  # north_star: one forward+inverse transform
TOL_NORM = 1e-5       # north_star: relative norm drift


def rel(a, b):
    """||a - b||_2 / ||b||_2, accumulated in float64 (chunked: a 512^3 pair stays within a few GB)."""
    a = np.asarray(a).reshape(-1)
    b = np.asarray(b).reshape(-1)
    num = den = 0.0
    for i in range(0, a.size, 1 << 24):
        x = a[i:i + (1 << 24)].astype(np.complex128 if np.iscomplexobj(a) or np.iscomplexobj(b) else np.float64)
        y = b[i:i + (1 << 24)].astype(x.dtype)
        num += float(np.sum(np.abs(x - y) ** 2))
        den += float(np.sum(np.abs(y) ** 2))
    return float(np.sqrt(num / den))


def maxrel(a, b):
    """max |a - b| / max |b|: an element-wise bound next to the norm (a defect confined to one tile or one row of
    a large grid hides in rel-L2)."""
    a = np.asarray(a).reshape(-1)
    b = np.asarray(b).reshape(-1)
    num = den = 0.0
    for i in range(0, a.size, 1 << 24):
        num = max(num, float(np.max(np.abs(a[i:i + (1 << 24)] - b[i:i + (1 << 24)]))))
        den = max(den, float(np.max(np.abs(b[i:i + (1 << 24)]))))
    return num / den


def assert_state(got, want, tol=TOL_STATE):
    """north_star's acceptance (rel-L2 <= tol) plus the element-wise bound max |dpsi| <= 10 tol max |psi|."""
    e2, em = rel(got, want), maxrel(got, want)
    assert e2 < tol and em < 10 * tol, (e2, em)
    return e2
