"""Test-only helpers: independent brute-force linear algebra (numpy, no oracle, no CUDA)."""
import numpy as np


def gauss_jordan_inverse(A: np.ndarray) -> np.ndarray:
    """Textbook Gauss-Jordan elimination with partial pivoting on [A | I]."""
    n = A.shape[0]
    M = np.concatenate([A.astype(np.float64).copy(), np.eye(n)], axis=1)
    for c in range(n):
        piv = c + int(np.argmax(np.abs(M[c:, c])))
        if piv != c:
            M[[c, piv]] = M[[piv, c]]
        M[c] /= M[c, c]
        for r in range(n):
            if r != c:
                M[r] -= M[r, c] * M[c]
    return M[:, n:]


def se_kernel_numpy(A, B, ell, v, ell_squared=False):
    """Eq. 1 without the noise term, written with numpy broadcasting (independent of oracle)."""
    d = A[:, None, :] - B[None, :, :]
    r2 = np.sum(d * d, axis=2)
    den = 2.0 * ell * ell if ell_squared else 2.0 * ell
    return v * np.exp(-r2 / den)


def relerr(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (nb if nb > 0 else 1.0)
